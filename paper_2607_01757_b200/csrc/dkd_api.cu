// dkd_api.cu — host side of libdkd: the C-ABI of include/dkd.h (argument validation, workspace,
// TMA descriptors, launch plans, the shape-keyed CUDA-graph cache, the host-buffer path).  See DESIGN.md.
#include "dkd.h"

#include <math.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "dkd_kernels.cuh"
#include "dkd_host.h"

using namespace dkd;

namespace {

typedef CUresult (*PFN_tensorMapEncodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                             const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                             CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                             CUtensorMapFloatOOBfill);

thread_local char g_create_error[512] = "";

struct ExtractArgs {                       // one dkd_extract* call
    const float* score;
    int B, H, W;
    const void* desc;
    int desc_dtype, Hd, Wd, D, stride, r;
    float thresh;
    int top_k;
    float T;
    float* out_kpts;
    float* out_scores;
    void* out_desc;
    int32_t* out_count;
    int32_t* out_index;
    float* out_offset;
    // variants (dkd_extract_var)
    const float* score2;                   // reliability map: score = heat x reliability
    const uint8_t* mask;                   // validity mask
    int nms_iters, score_mode;
    int32_t* out_total;
    // derived
    int use_tma;
    int origin_x, origin_y;                // letterbox offset subtracted from the keypoint coordinates
};

// What a cached graph's TOPOLOGY and launch geometry depend on.  Addresses and the scalars thresh / T are
// kernel arguments: a call that differs only in those re-uses the instantiated graph and updates the
// kernel nodes' parameters (cudaGraphExecKernelNodeSetParams) — no capture, no instantiation.
struct ShapeKey {
    int B, H, W, has_desc, desc_dtype, Hd, Wd, D, stride, r, top_k;
    int has_index, has_offset, has_score2, has_mask, has_total, nms_iters, score_mode;
    int use_tma, negt, use_pdl, nms_cpu, split;
    bool operator==(const ShapeKey& o) const {
        return B == o.B && H == o.H && W == o.W && has_desc == o.has_desc && desc_dtype == o.desc_dtype && Hd == o.Hd &&
               Wd == o.Wd && D == o.D && stride == o.stride && r == o.r && top_k == o.top_k && has_index == o.has_index &&
               has_offset == o.has_offset && has_score2 == o.has_score2 && has_mask == o.has_mask &&
               has_total == o.has_total && nms_iters == o.nms_iters && score_mode == o.score_mode && use_tma == o.use_tma &&
               negt == o.negt && use_pdl == o.use_pdl && nms_cpu == o.nms_cpu && split == o.split;
    }
};

bool same_values(const ExtractArgs& x, const ExtractArgs& y) {   // the arguments a graph's kernel nodes embed
    return x.score == y.score && x.desc == y.desc && x.thresh == y.thresh && x.T == y.T && x.out_kpts == y.out_kpts &&
           x.out_scores == y.out_scores && x.out_desc == y.out_desc && x.out_count == y.out_count &&
           x.out_index == y.out_index && x.out_offset == y.out_offset && x.score2 == y.score2 && x.mask == y.mask &&
           x.out_total == y.out_total && x.origin_x == y.origin_x && x.origin_y == y.origin_y;
}

constexpr int MAX_KERNELS = 3;                              // kernels per extract, in launch order:
const char* const KERNEL_NAMES[MAX_KERNELS] = {"nms", "select", "refine_gather"};

struct Plan {                                               // the launches of one extract
    KLaunch k[MAX_KERNELS];
    int n;
};

struct GraphEntry {
    ShapeKey key;
    ExtractArgs last;                                       // the argument values the exec currently embeds
    cudaGraph_t graph;                                      // kept: its kernel nodes address the exec's nodes
    cudaGraphExec_t exec;
    cudaGraphNode_t node[MAX_KERNELS];
    int n_nodes;                                            // 0: node handles unknown, parameters cannot be updated
    unsigned long long last_use;
};

constexpr size_t GRAPH_CACHE_CAP = 64;

}  // namespace

struct dkd_ctx {
    dkd_create_params p;
    int num_sms;
    int nms_ctas_per_sm[MAX_R + 1];
    int nms_ctas_per_sm_prod[MAX_R + 1];
    PFN_tensorMapEncodeTiled encode;
    // workspace (device)
    uint64_t* cand;          // [max_tiles * SEG_CAP] candidate keys, one private segment per NMS unit
    int* tile_cnt;           // [max_tiles] keys in each segment
    int32_t* sel_idx;        // [max_batch * max_top_k]
    size_t max_tiles;
    size_t max_segs;         // ints in tile_cnt: max_tiles, or the tile count of the finest iterated-NMS tiling if larger
    size_t ws_bytes;
    // host-path staging (device), grown on demand
    void* st_score; size_t st_score_bytes;
    void* st_desc;  size_t st_desc_bytes;
    void* st_out;   size_t st_out_bytes;
    void* scratch[2]; size_t scratch_bytes[2];              // dkd_ctx_scratch: match partials, retrieval-scan workspace
    const void* st_desc_src; size_t st_desc_src_bytes;      // the host map st_desc holds as a RESIDENT copy (else NULL)
    // options
    int use_graph, use_tma, use_pdl, profile, nms_cpu, origin_x, origin_y, sel_prefetch;
    cudaEvent_t prof_ev[MAX_KERNELS + 1];                   // measurement mode: event before/after every kernel
    int prof_n;                                             // kernels of the last profiled call (0: none)
    std::vector<GraphEntry> graphs;
    Plan last_plan;                                         // plain-launch path: the most recent plan and what it was built for
    ShapeKey last_plan_key;
    ExtractArgs last_plan_args;
    bool have_last_plan;
    cudaStream_t cap_stream;  // capture-only stream for building the cached graphs
    unsigned long long tick;
    unsigned long long n_instantiated, n_updated, n_replayed, n_stream;   // graph-cache statistics (dkd_graph_stats)
    char err[512];
};

namespace {

int fail(dkd_ctx* ctx, int code, const char* fmt, const char* a = "", const char* b = "") {
    if (ctx) snprintf(ctx->err, sizeof(ctx->err), fmt, a, b);
    return code;
}
int fail_cuda(dkd_ctx* ctx, const char* what, cudaError_t e) {
    return fail(ctx, DKD_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

#define CK(ctx, call)                                                  \
    do {                                                               \
        cudaError_t e_ = (call);                                       \
        if (e_ != cudaSuccess) return fail_cuda((ctx), #call, e_);     \
    } while (0)

bool misaligned(const void* p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }

template <int R>
cudaError_t setup_nms(dkd_ctx* ctx) {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_nms_tma<R, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, NMS_SMEM_BYTES)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_nms_tma<R, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, NMS_SMEM_BYTES)) != cudaSuccess) return e;
    int n = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_nms_tma<R, true, false>, NMS_WARPS * 32, NMS_SMEM_BYTES);
    ctx->nms_ctas_per_sm[R] = n > 0 ? (n < NMS_CTAS ? n : NMS_CTAS) : 1;
    if (e != cudaSuccess) return e;
    ctx->nms_ctas_per_sm_prod[R] = 1;
    if (2 * NMS_SMEM_BYTES > 227 * 1024) return e;          // (tuning builds with a deeper ring: no product variant)
    if ((e = cudaFuncSetAttribute(k_nms_tma<R, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * NMS_SMEM_BYTES)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_nms_tma<R, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * NMS_SMEM_BYTES)) != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_nms_tma<R, true, true>, NMS_WARPS * 32, 2 * NMS_SMEM_BYTES);
    ctx->nms_ctas_per_sm_prod[R] = n > 0 ? n : 1;
    return e;
}

// Strip-tiles per unit: as many as possible (the 2R rows above a unit are fetched once per unit) while
// the units still fill the machine several times over.
NmsPlan nms_plan(const dkd_ctx* ctx, const ExtractArgs& a) {   // (a.use_tma == 0: the plain loader works per strip-tile)
    NmsPlan p;
    p.H = a.H; p.W = a.W;
    p.strips_x = (a.W + STRIP_W - 1) / STRIP_W;
    p.chunks_y = (a.H + TH - 1) / TH;
    // S > thresh  <=>  S >= nextafter(thresh, +inf): the threshold joins the window maximum (dkd_kernels.cuh)
    p.thr_up = nextafterf(a.thresh, INFINITY);
    const long long slots = static_cast<long long>(NMS_CTAS) * ctx->num_sms * NMS_WARPS;  // resident warps
    int best = 1;
    for (int cpu = MAX_CPU; cpu >= 1; --cpu) {
        const int segs = (p.chunks_y + cpu - 1) / cpu;
        if (static_cast<long long>(p.strips_x) * segs * a.B >= 4 * slots) { best = cpu; break; }
    }
    if (ctx->nms_cpu > 0) best = ctx->nms_cpu < MAX_CPU ? ctx->nms_cpu : MAX_CPU;
    if (!a.use_tma) best = 1;
    p.cpu = best;
    p.segs = (p.chunks_y + best - 1) / best;
    p.units = p.strips_x * p.segs * a.B;
    return p;
}

bool encode_map(dkd_ctx* ctx, CUtensorMap* tmap, const float* base, const ExtractArgs& a) {
    const cuuint64_t dims[3] = {(cuuint64_t)a.W, (cuuint64_t)a.H, (cuuint64_t)a.B};
    const cuuint64_t strides[2] = {(cuuint64_t)a.W * 4, (cuuint64_t)a.W * a.H * 4};
    const cuuint32_t box[3] = {(cuuint32_t)BOX_W, (cuuint32_t)TH, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    return ctx->encode(tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(base), dims, strides, box, estr,
                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                       CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int R>
cudaError_t plan_nms(dkd_ctx* ctx, const ExtractArgs& a, const NmsPlan& p, KLaunch& k) {
    const bool prod = a.score2 != nullptr;
    const bool pdl = ctx->use_pdl != 0;                      // (the kernel waits for its predecessor before touching memory)
    if (a.use_tma) {
        CUtensorMap tmap, tmap2;
        if (!encode_map(ctx, &tmap, a.score, a)) return cudaErrorInvalidValue;
        tmap2 = tmap;
        if (prod && !encode_map(ctx, &tmap2, a.score2, a)) return cudaErrorInvalidValue;
        int grid = ctx->num_sms * (prod ? ctx->nms_ctas_per_sm_prod[R] : ctx->nms_ctas_per_sm[R]);
        if (grid > (p.units + NMS_WARPS - 1) / NMS_WARPS) grid = (p.units + NMS_WARPS - 1) / NMS_WARPS;
        const size_t smem = prod ? 2 * NMS_SMEM_BYTES : NMS_SMEM_BYTES;
        const bool negt = !(p.thr_up > 0.0f);                // a -0.0 score may be a candidate: fold it onto +0
#define DKD_PREP_TMA(NEGT, PROD)                                                                                         \
    prep(k, k_nms_tma<R, NEGT, PROD>, dim3(grid), dim3(NMS_WARPS * 32), smem, pdl, tmap, tmap2, p, a.score, a.score2, \
         ctx->cand, ctx->tile_cnt)
        if (prod) { if (negt) DKD_PREP_TMA(true, true); else DKD_PREP_TMA(false, true); }
        else { if (negt) DKD_PREP_TMA(true, false); else DKD_PREP_TMA(false, false); }
#undef DKD_PREP_TMA
    } else {
        const int total = p.strips_x * p.chunks_y * a.B;
        const dim3 grid((total + PLAIN_WARPS - 1) / PLAIN_WARPS);
        if (prod) prep(k, k_nms_plain<R, true>, grid, dim3(PLAIN_WARPS * 32), 0, pdl, a.score, a.score2, p, total, ctx->cand, ctx->tile_cnt);
        else prep(k, k_nms_plain<R, false>, grid, dim3(PLAIN_WARPS * 32), 0, pdl, a.score, a.score2, p, total, ctx->cand, ctx->tile_cnt);
    }
    return cudaSuccess;
}

FastDiv make_fastdiv(uint32_t d) {                          // exact n / d for every 32-bit n (d >= 1)
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;
    FastDiv f;
    f.m = static_cast<uint32_t>(((1ull << 32) * ((1ull << l) - d)) / d + 1);
    f.s1 = l < 1 ? l : 1;
    f.s2 = l > 0 ? l - 1 : 0;
    return f;
}

SampleAxis make_axis(int stride, int n) {
    SampleAxis a;
    a.den = make_fastdiv(2u * static_cast<uint32_t>(stride));
    a.s = stride;
    a.inv_den = 1.0f / (2.0f * static_cast<float>(stride));
    a.inv_s = 1.0f / static_cast<float>(stride);
    a.n = n;
    return a;
}

template <int DT, int G>
void plan_rg_g(const RGParams& p, int B, bool prod, bool pdl, KLaunch& k) {
    const dim3 grid((p.top_k + RG_SLOTS - 1) / RG_SLOTS, B);
    const dim3 block(DT < 0 ? 32 : RG_THREADS);
    if (prod) prep(k, k_refine_gather<DT, G, true>, grid, block, 0, pdl, p);
    else prep(k, k_refine_gather<DT, G, false>, grid, block, 0, pdl, p);
}

template <int DT>
void plan_rg_dt(const RGParams& p, int B, bool prod, bool pdl, KLaunch& k) {
    if (p.nchunk <= 8) plan_rg_g<DT, 8>(p, B, prod, pdl, k);
    else if (p.nchunk <= 16) plan_rg_g<DT, 16>(p, B, prod, pdl, k);
    else plan_rg_g<DT, 32>(p, B, prod, pdl, k);
}

void plan_rg(const ExtractArgs& a, const int32_t* sel, bool pdl, int num_sms, KLaunch& k) {
    RGParams p;
    memset(&p, 0, sizeof(p));
    p.score = a.score; p.score2 = a.score2; p.H = a.H; p.W = a.W;
    p.divW = make_fastdiv(static_cast<uint32_t>(a.W));
    p.sel_idx = sel; p.top_k = a.top_k; p.r = a.r;
    p.kscale = static_cast<float>(1.4426950408889634 / static_cast<double>(a.T));
    p.out_kpts = a.out_kpts; p.out_scores = a.out_scores; p.out_off = a.out_offset;
    p.origin_x = a.origin_x; p.origin_y = a.origin_y;
    p.score_mode = a.score_mode;
    p.vec_window = (a.W % 4 == 0) && !misaligned(a.score, 16) && a.score2 == nullptr;
    p.early_trigger = pdl && static_cast<long long>((a.top_k + RG_SLOTS - 1) / RG_SLOTS) * a.B <= 4LL * num_sms;
    const bool prod = a.score2 != nullptr;
    if (a.desc == nullptr) { plan_rg_g<-1, 8>(p, a.B, prod, pdl, k); return; }
    const size_t esz = a.desc_dtype == DKD_F16 ? 2 : 4;
    p.desc = static_cast<const unsigned char*>(a.desc);
    p.nchunk = static_cast<int>(a.D * esz / 16);
    p.img_bytes = static_cast<size_t>(a.Hd) * a.Wd * a.D * esz;
    p.ax = make_axis(a.stride, a.Wd);
    p.ay = make_axis(a.stride, a.Hd);
    p.out_desc = static_cast<unsigned char*>(a.out_desc);
    if (a.desc_dtype == DKD_F16) plan_rg_dt<DKD_F16>(p, a.B, prod, pdl, k);
    else plan_rg_dt<DKD_F32>(p, a.B, prod, pdl, k);
}

// The launches of one extract (launch geometry + argument values).  Pure host work: nothing touches a stream.
cudaError_t build_plan(dkd_ctx* ctx, const ExtractArgs& a, Plan& pl) {
    const NmsPlan plan = nms_plan(ctx, a);
    int tpi = plan.strips_x * plan.segs;                    // candidate segments (NMS units) per image
    int seg_cap = plan.cpu * SEG_CAP;
    cudaError_t e = cudaSuccess;
    if (a.nms_iters > 0) {                                  // variant V1: tiles of T x T pixels, one segment each
        IterParams ip;
        memset(&ip, 0, sizeof(ip));
        ip.score = a.score; ip.score2 = a.score2; ip.mask = a.mask; ip.H = a.H; ip.W = a.W; ip.r = a.r; ip.iters = a.nms_iters;
        ip.halo = (2 * a.nms_iters + 1) * a.r;
        ip.halo_x = (ip.halo + 3) & ~3;                     // (fits: IT_REG - 2 halo - T >= halo_x - halo, IT_REG % 8 == 0)
        ip.vec = (a.W % 4 == 0) && !misaligned(a.score, 16) && !misaligned(a.score2, 16);
        ip.T = (IT_REG - 2 * ip.halo) & ~7;
        ip.tiles_x = (a.W + ip.T - 1) / ip.T; ip.tiles_y = (a.H + ip.T - 1) / ip.T;
        ip.thresh = a.thresh; ip.cand = ctx->cand; ip.seg_cnt = ctx->tile_cnt;
        const dim3 ig(ip.tiles_x * ip.tiles_y, a.B), ib(IT_THREADS);
        const bool ipdl = ctx->use_pdl != 0;
        switch (a.r) {
            case 1: prep(pl.k[0], k_nms_iter<1>, ig, ib, IT_SMEM_BYTES, ipdl, ip); break;
            case 2: prep(pl.k[0], k_nms_iter<2>, ig, ib, IT_SMEM_BYTES, ipdl, ip); break;
            case 3: prep(pl.k[0], k_nms_iter<3>, ig, ib, IT_SMEM_BYTES, ipdl, ip); break;
            default: prep(pl.k[0], k_nms_iter<4>, ig, ib, IT_SMEM_BYTES, ipdl, ip); break;
        }
        tpi = ip.tiles_x * ip.tiles_y;
        seg_cap = ip.T * ip.T;
    } else {
        switch (a.r) {
            case 1: e = plan_nms<1>(ctx, a, plan, pl.k[0]); break;
            case 2: e = plan_nms<2>(ctx, a, plan, pl.k[0]); break;
            case 3: e = plan_nms<3>(ctx, a, plan, pl.k[0]); break;
            default: e = plan_nms<4>(ctx, a, plan, pl.k[0]); break;
        }
    }
    if (e != cudaSuccess) return e;
    int32_t* sel = a.out_index ? a.out_index : ctx->sel_idx;
    int idx_shift = 0;                                       // (H*W - 1) >> idx_shift < NBT: index buckets of the top ties
    while (((static_cast<long long>(a.H) * a.W - 1) >> idx_shift) >= NBT) ++idx_shift;
    const bool pdl = ctx->use_pdl != 0;
    SelExtra pf;
    memset(&pf, 0, sizeof(pf));
    pf.img_px = static_cast<size_t>(a.H) * a.W;
    // variant V5: the single-pass NMS kernels leave the validity mask to the gather of k_select (one byte per candidate,
    // read where the kernel is latency-bound anyway, instead of a dependent load inside the NMS emit loop)
    if (a.nms_iters == 0) pf.vmask = a.mask;
    if (ctx->sel_prefetch) {
        const FastDiv dw = make_fastdiv(static_cast<uint32_t>(a.W));
        pf.score = a.score; pf.score2 = a.score2; pf.W = a.W; pf.r = a.r;
        pf.div_m = dw.m; pf.div_s1 = dw.s1; pf.div_s2 = dw.s2;
    }
    prep(pl.k[1], k_select, dim3(a.B), dim3(SEL_THREADS), SEL_SMEM_BYTES, pdl, ctx->cand, ctx->tile_cnt, tpi,
         seg_cap, a.top_k, idx_shift, pf, sel, a.out_count, a.out_total);
    plan_rg(a, sel, pdl, ctx->num_sms, pl.k[2]);
    pl.n = 3;
    return cudaSuccess;
}

// Enqueue the kernels of one extract on `st`.  No sync, no allocation: capture-safe.
// prof: measurement mode, an event on `st` before and after every kernel (and no PDL: the events would
// serialise the kernels anyway).
cudaError_t enqueue(dkd_ctx* ctx, const Plan& pl, cudaStream_t st, bool prof = false) {
    cudaError_t e;
    for (int i = 0; i < pl.n; ++i) {
        if (prof && (e = cudaEventRecord(ctx->prof_ev[i], st)) != cudaSuccess) return e;
        if ((e = launch(pl.k[i], st, !prof)) != cudaSuccess) return e;
    }
    if (prof) {
        if ((e = cudaEventRecord(ctx->prof_ev[pl.n], st)) != cudaSuccess) return e;
        ctx->prof_n = pl.n;
    }
    return cudaSuccess;
}

// shape / scalar checks (no pointer is dereferenced, no alignment is looked at): shared by the device and host paths
int validate_shapes(dkd_ctx* ctx, const ExtractArgs& a) {
    if (a.B < 1 || a.H < 1 || a.W < 1 || a.top_k < 1) return fail(ctx, DKD_ERR_INVALID_ARG, "B, H, W, top_k must be >= 1");
    if (a.r < 1) return fail(ctx, DKD_ERR_INVALID_ARG, "r must be >= 1");
    if (!(a.T > 0.0f) || !isfinite(a.T)) return fail(ctx, DKD_ERR_INVALID_ARG, "T must be finite and > 0");
    if (isnan(a.thresh)) return fail(ctx, DKD_ERR_INVALID_ARG, "thresh is NaN");
    if ((a.desc == nullptr) != (a.out_desc == nullptr))
        return fail(ctx, DKD_ERR_INVALID_ARG, "desc and out_desc must both be NULL or both be set");
    if (a.nms_iters < 0) return fail(ctx, DKD_ERR_INVALID_ARG, "nms_iters must be >= 0");
    if (a.score_mode != DKD_SCORE_RAW && a.score_mode != DKD_SCORE_BILINEAR)
        return fail(ctx, DKD_ERR_INVALID_ARG, "score_mode must be DKD_SCORE_RAW or DKD_SCORE_BILINEAR");
    if (a.desc) {
        if (a.Hd < 1 || a.Wd < 1 || a.D < 1 || a.stride < 1)
            return fail(ctx, DKD_ERR_INVALID_ARG, "Hd, Wd, D, stride must be >= 1");
        if (a.desc_dtype != DKD_F32 && a.desc_dtype != DKD_F16)
            return fail(ctx, DKD_ERR_UNSUPPORTED, "desc_dtype must be DKD_F32 or DKD_F16");
    }
    if (a.r > DKD_MAX_RADIUS) return fail(ctx, DKD_ERR_UNSUPPORTED, "r > DKD_MAX_RADIUS");
    if (ctx->p.max_radius > 0 && a.r > ctx->p.max_radius) return fail(ctx, DKD_ERR_CAPACITY, "r above the dkd_create max_radius");
    if (a.nms_iters > 0) {
        const long long halo = (2LL * a.nms_iters + 1) * a.r;
        if (halo > 40) return fail(ctx, DKD_ERR_UNSUPPORTED, "iterated NMS: (2 nms_iters + 1) r must be <= 40");
        const int T = (IT_REG - 2 * static_cast<int>(halo)) & ~7;
        const long long tiles = static_cast<long long>((a.W + T - 1) / T) * ((a.H + T - 1) / T) * a.B;
        if (tiles * T * T > static_cast<long long>(ctx->max_tiles) * SEG_CAP || tiles > static_cast<long long>(ctx->max_segs))
            return fail(ctx, DKD_ERR_CAPACITY, "iterated NMS: candidate workspace too small for these tiles (raise the dkd_create maxima)");
    }
    if (a.B > 65535) return fail(ctx, DKD_ERR_UNSUPPORTED, "B > 65535");
    if (a.desc) {
        const size_t rowb = static_cast<size_t>(a.D) * (a.desc_dtype == DKD_F16 ? 2 : 4);
        if (rowb % 16 != 0 || rowb > DKD_MAX_ROW_BYTES)
            return fail(ctx, DKD_ERR_UNSUPPORTED, "D * elemsize must be a multiple of 16 and <= DKD_MAX_ROW_BYTES");
        if (a.D > ctx->p.max_dim) return fail(ctx, DKD_ERR_CAPACITY, "D > max_dim");
        if (a.stride > (1 << 20)) return fail(ctx, DKD_ERR_UNSUPPORTED, "stride too large");
        if (static_cast<long long>(a.Hd) * a.Wd > 0x7fffffffLL) return fail(ctx, DKD_ERR_UNSUPPORTED, "Hd * Wd >= 2^31");
    }
    if (a.B > ctx->p.max_batch || a.H > ctx->p.max_h || a.W > ctx->p.max_w || a.top_k > ctx->p.max_top_k)
        return fail(ctx, DKD_ERR_CAPACITY, "B, H, W or top_k above the dkd_create maxima");
    return DKD_OK;
}

int validate(dkd_ctx* ctx, const ExtractArgs& a) {
    if (!a.score || !a.out_kpts || !a.out_scores || !a.out_count)
        return fail(ctx, DKD_ERR_INVALID_ARG, "NULL required pointer (score/out_kpts/out_scores/out_count)");
    const int rc = validate_shapes(ctx, a);
    if (rc != DKD_OK) return rc;
    if (misaligned(a.score, 4) || misaligned(a.score2, 4)) return fail(ctx, DKD_ERR_UNSUPPORTED, "score / reliability not 4-byte aligned");
    if (misaligned(a.out_kpts, 8) || misaligned(a.out_offset, 8))
        return fail(ctx, DKD_ERR_UNSUPPORTED, "out_kpts / out_offset not 8-byte aligned");
    if (misaligned(a.out_scores, 4) || misaligned(a.out_count, 4) || misaligned(a.out_index, 4) || misaligned(a.out_total, 4))
        return fail(ctx, DKD_ERR_UNSUPPORTED, "out_scores / out_count / out_index / out_total not 4-byte aligned");
    if (a.desc && (misaligned(a.desc, 16) || misaligned(a.out_desc, 16)))
        return fail(ctx, DKD_ERR_UNSUPPORTED, "desc / out_desc not 16-byte aligned");
    return DKD_OK;
}

ShapeKey shape_key(const dkd_ctx* ctx, const ExtractArgs& a) {
    ShapeKey k;
    memset(&k, 0, sizeof(k));
    k.B = a.B; k.H = a.H; k.W = a.W; k.has_desc = a.desc != nullptr; k.desc_dtype = a.desc_dtype; k.Hd = a.Hd; k.Wd = a.Wd;
    k.D = a.D; k.stride = a.stride; k.r = a.r; k.top_k = a.top_k;
    k.has_index = a.out_index != nullptr; k.has_offset = a.out_offset != nullptr; k.has_score2 = a.score2 != nullptr;
    k.has_mask = a.mask != nullptr; k.has_total = a.out_total != nullptr; k.nms_iters = a.nms_iters; k.score_mode = a.score_mode;
    k.use_tma = a.use_tma; k.negt = !(nextafterf(a.thresh, INFINITY) > 0.0f); k.use_pdl = ctx->use_pdl; k.nms_cpu = ctx->nms_cpu;
    k.split = ctx->sel_prefetch;
    return k;
}

void drop_graphs(dkd_ctx* ctx) {
    for (auto& g : ctx->graphs) {
        cudaGraphExecDestroy(g.exec);
        cudaGraphDestroy(g.graph);
    }
    ctx->graphs.clear();
}

// Capture the launches of `pl` once on the context's capture stream and instantiate them as a graph.  The
// node handle of every kernel is read back right after its launch (the capturing stream's dependency set
// is then exactly that node), so that later calls can re-point the kernels at other buffers.
int build_graph(dkd_ctx* ctx, const Plan& pl, GraphEntry& ge) {
    // (captured on a context-owned stream: the caller's may be the legacy default stream, which
    // cannot be captured; the instantiated graph is then launched on the caller's stream)
    CK(ctx, cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
    cudaError_t e = cudaSuccess;
    ge.n_nodes = pl.n;
    for (int i = 0; i < pl.n; ++i) {
        e = launch(pl.k[i], ctx->cap_stream, i > 0);         // (the first node has no predecessor inside the graph)
        if (e != cudaSuccess) break;
        cudaStreamCaptureStatus cs;
        const cudaGraphNode_t* deps = nullptr;
        const cudaGraphEdgeData* edges = nullptr;
        size_t nd = 0;
        if (cudaStreamGetCaptureInfo_v3(ctx->cap_stream, &cs, nullptr, nullptr, &deps, &edges, &nd) == cudaSuccess &&
            cs == cudaStreamCaptureStatusActive && nd == 1)
            ge.node[i] = deps[0];
        else
            ge.n_nodes = 0;                                  // handles unknown: this entry is replay-only
    }
    cudaGraph_t graph = nullptr;
    const cudaError_t e2 = cudaStreamEndCapture(ctx->cap_stream, &graph);
    if (e != cudaSuccess || e2 != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        (void)cudaGetLastError();
        return fail_cuda(ctx, "graph capture", e != cudaSuccess ? e : e2);
    }
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    if (e != cudaSuccess) {
        cudaGraphDestroy(graph);
        return fail_cuda(ctx, "cudaGraphInstantiate", e);
    }
    ge.graph = graph;
    ge.exec = exec;
    ++ctx->n_instantiated;
    return DKD_OK;
}

// Re-point an instantiated graph at the argument values of `pl` (same launch geometry: same ShapeKey).
cudaError_t update_graph(GraphEntry& ge, const Plan& pl) {
    for (int i = 0; i < pl.n; ++i) {
        void* argp[KLaunch::MAX_ARGS];
        cudaKernelNodeParams np;
        memset(&np, 0, sizeof(np));
        np.func = const_cast<void*>(pl.k[i].func);
        np.gridDim = pl.k[i].grid; np.blockDim = pl.k[i].block;
        np.sharedMemBytes = static_cast<unsigned>(pl.k[i].smem);
        pl.k[i].arg_pointers(argp);
        np.kernelParams = argp;
        const cudaError_t e = cudaGraphExecKernelNodeSetParams(ge.exec, ge.node[i], &np);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

int run(dkd_ctx* ctx, ExtractArgs a, cudaStream_t st) {
    int rc = validate(ctx, a);
    if (rc != DKD_OK) return rc;
    a.origin_x = ctx->origin_x; a.origin_y = ctx->origin_y;
    a.use_tma = ctx->use_tma && ctx->encode && (a.W % 4 == 0) && !misaligned(a.score, 16) && !misaligned(a.score2, 16);

    Plan pl;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    CK(ctx, cudaStreamIsCapturing(st, &cap));
    if (ctx->profile && cap == cudaStreamCaptureStatusNone) {
        ctx->prof_n = 0;
        CK(ctx, build_plan(ctx, a, pl));
        CK(ctx, enqueue(ctx, pl, st, true));
        return DKD_OK;
    }
    if (!ctx->use_graph || cap != cudaStreamCaptureStatusNone) {
        // plain launches: the plan of the previous call is kept (a repeated call with the same arguments skips the
        // tensor-map encoding and the rest of build_plan)
        const ShapeKey key = shape_key(ctx, a);
        if (!(ctx->have_last_plan && ctx->last_plan_key == key && same_values(ctx->last_plan_args, a))) {
            ctx->have_last_plan = false;
            CK(ctx, build_plan(ctx, a, ctx->last_plan));
            ctx->last_plan_key = key;
            ctx->last_plan_args = a;
            ctx->have_last_plan = true;
        }
        CK(ctx, enqueue(ctx, ctx->last_plan, st));
        ++ctx->n_stream;
        return DKD_OK;
    }
    ++ctx->tick;
    const ShapeKey key = shape_key(ctx, a);
    for (size_t gi = 0; gi < ctx->graphs.size(); ++gi) {
        GraphEntry& g = ctx->graphs[gi];
        if (!(g.key == key)) continue;
        g.last_use = ctx->tick;
        if (!same_values(g.last, a)) {                      // other buffers / thresh / T: update the kernel nodes in place
            CK(ctx, build_plan(ctx, a, pl));
            if (g.n_nodes != pl.n || update_graph(g, pl) != cudaSuccess) {
                // Cannot update.  The nodes are updated one by one, so the exec may now mix the new buffers with the old
                // ones: drop the entry (rebuilt by the next call of this shape; an exec still in flight is freed when it
                // completes) and serve this call with plain PDL-linked launches.
                (void)cudaGetLastError();
                cudaGraphExecDestroy(g.exec);
                cudaGraphDestroy(g.graph);
                ctx->graphs[gi] = ctx->graphs.back();
                ctx->graphs.pop_back();
                CK(ctx, enqueue(ctx, pl, st));
                ++ctx->n_stream;
                return DKD_OK;
            }
            g.last = a;
            ++ctx->n_updated;
        } else {
            ++ctx->n_replayed;
        }
        CK(ctx, cudaGraphLaunch(g.exec, st));
        return DKD_OK;
    }
    // first call with this shape: capture the launches once, then replay as one graph launch
    CK(ctx, build_plan(ctx, a, pl));
    GraphEntry ge;
    memset(&ge, 0, sizeof(ge));
    if ((rc = build_graph(ctx, pl, ge)) != DKD_OK) return rc;
    if (ctx->graphs.size() >= GRAPH_CACHE_CAP) {            // evict the least recently used entry
        size_t v = 0;
        for (size_t i = 1; i < ctx->graphs.size(); ++i)
            if (ctx->graphs[i].last_use < ctx->graphs[v].last_use) v = i;
        cudaGraphExecDestroy(ctx->graphs[v].exec);
        cudaGraphDestroy(ctx->graphs[v].graph);
        ctx->graphs[v] = ctx->graphs.back();
        ctx->graphs.pop_back();
    }
    ge.key = key;
    ge.last = a;
    ge.last_use = ctx->tick;
    ctx->graphs.push_back(ge);
    CK(ctx, cudaGraphLaunch(ge.exec, st));
    return DKD_OK;
}

int grow(dkd_ctx* ctx, void** buf, size_t* have, size_t need) {
    if (need <= *have) return DKD_OK;
    if (*buf) CK(ctx, cudaFree(*buf));
    *buf = nullptr;
    *have = 0;
    CK(ctx, cudaMalloc(buf, need));
    *have = need;
    return DKD_OK;
}

template <int CIN, int COUT, int DT>
cudaError_t launch_pre(PreParams& q, cudaStream_t st) {
    const bool vec = q.Wp % 8 == 0;
    const int V = vec ? 8 : 1;
    q.gpr = (q.Wp + V - 1) / V;
    const dim3 grid((q.gpr + 255) / 256, q.Hp, q.B);
    if (vec) k_preprocess<CIN, COUT, DT, 8><<<grid, 256, 0, st>>>(q);
    else k_preprocess<CIN, COUT, DT, 1><<<grid, 256, 0, st>>>(q);
    return cudaGetLastError();
}

size_t align256(size_t x) { return (x + 255) & ~static_cast<size_t>(255); }

// device address of a pinned, mapped host buffer (cudaHostAlloc / cudaHostRegister); NULL for pageable memory
void* mapped_device_pointer(const void* host) {
    if (!host) return nullptr;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, host) != cudaSuccess) {
        (void)cudaGetLastError();
        return nullptr;
    }
    return at.type == cudaMemoryTypeHost ? at.devicePointer : nullptr;
}

ExtractArgs make_args(const float* score, int B, int H, int W, const void* desc, int desc_dtype, int Hd, int Wd, int D,
                      int stride, int r, float thresh, int top_k, float T, float* out_kpts, float* out_scores,
                      void* out_desc, int32_t* out_count, int32_t* out_index, float* out_offset,
                      const dkd_variant_params* v) {
    ExtractArgs a;
    memset(&a, 0, sizeof(a));
    a.score = score; a.B = B; a.H = H; a.W = W;
    a.desc = desc; a.desc_dtype = desc ? desc_dtype : 0; a.Hd = desc ? Hd : 0; a.Wd = desc ? Wd : 0;
    a.D = desc ? D : 0; a.stride = desc ? stride : 1; a.r = r; a.thresh = thresh; a.top_k = top_k; a.T = T;
    a.out_kpts = out_kpts; a.out_scores = out_scores; a.out_desc = out_desc; a.out_count = out_count;
    a.out_index = out_index; a.out_offset = out_offset;
    if (v) {
        a.score2 = v->reliability; a.mask = v->valid_mask; a.nms_iters = v->nms_iters; a.score_mode = v->score_mode;
        a.out_total = v->out_total;
    }
    return a;
}

}  // namespace

// ---- helpers the other translation-unit-less parts of the library use (dkd_host.h) ---------------------------
int dkd_ctx_device(const dkd_ctx* ctx) { return ctx->p.device; }
int dkd_ctx_num_sms(const dkd_ctx* ctx) { return ctx->num_sms; }
int dkd_ctx_fail(dkd_ctx* ctx, int code, const char* msg, const char* detail) {
    return fail(ctx, code, "%s%s", msg, detail ? detail : "");
}

void* dkd_ctx_scratch(dkd_ctx* ctx, int slot, size_t bytes) {
    if (slot < 0 || slot > 1) return nullptr;
    if (bytes < 256) bytes = 256;
    if (grow(ctx, &ctx->scratch[slot], &ctx->scratch_bytes[slot], bytes) != DKD_OK) return nullptr;
    return ctx->scratch[slot];
}
int dkd_internal_select(dkd_ctx* ctx, const uint64_t* cand, const int* seg_cnt, int tpi, int seg_cap, int top_k, int n_items,
                        int32_t* sel_idx, int32_t* out_count, cudaStream_t st) {
    if ((seg_cap & 1) || misaligned(cand, 16)) return fail(ctx, DKD_ERR_INVALID_ARG, "internal: candidate segments must be 16-byte aligned");
    int idx_shift = 0;
    while (((static_cast<long long>(n_items) - 1) >> idx_shift) >= NBT) ++idx_shift;
    SelExtra pf;
    memset(&pf, 0, sizeof(pf));
    KLaunch k;
    prep(k, k_select, dim3(1), dim3(SEL_THREADS), SEL_SMEM_BYTES, false, cand, seg_cnt, tpi, seg_cap, top_k, idx_shift, pf,
         sel_idx, out_count, static_cast<int32_t*>(nullptr));
    const cudaError_t e = launch(k, st, false);
    if (e != cudaSuccess) return fail_cuda(ctx, "k_select launch", e);
    return DKD_OK;
}

extern "C" {

const char* dkd_version(void) {
#ifdef DKD_DEBUG
    return "dkd-b200 0.2 (sm_100a, DKD_DEBUG: device-side bounds checks)";
#else
    return "dkd-b200 0.2 (sm_100a)";
#endif
}

int dkd_create(const dkd_create_params* p, dkd_ctx** out) {
    if (out) *out = nullptr;
    if (!p || !out) { snprintf(g_create_error, sizeof(g_create_error), "NULL argument"); return DKD_ERR_INVALID_ARG; }
    if (p->max_batch < 1 || p->max_h < 1 || p->max_w < 1 || p->max_top_k < 1 || p->max_dim < 0 ||
        static_cast<long long>(p->max_h) * p->max_w > 0x7fffffffLL) {
        snprintf(g_create_error, sizeof(g_create_error), "invalid maxima");
        return DKD_ERR_INVALID_ARG;
    }
    if (p->max_top_k > DKD_MAX_TOP_K) {
        snprintf(g_create_error, sizeof(g_create_error), "max_top_k > DKD_MAX_TOP_K");
        return DKD_ERR_UNSUPPORTED;
    }
    if (p->max_radius < 0 || p->max_match_n < 0 || p->max_match_pairs < 0 || p->max_scan_rows < 0) {
        snprintf(g_create_error, sizeof(g_create_error), "invalid maxima (max_radius / max_match_n / max_match_pairs / max_scan_rows < 0)");
        return DKD_ERR_INVALID_ARG;
    }
    if (p->max_radius > DKD_MAX_RADIUS) {
        snprintf(g_create_error, sizeof(g_create_error), "max_radius > DKD_MAX_RADIUS");
        return DKD_ERR_UNSUPPORTED;
    }
    int prev_dev = -1;
    const bool have_prev = cudaGetDevice(&prev_dev) == cudaSuccess;   // the caller's current device is left unchanged
    (void)cudaGetLastError();
    dkd_ctx* ctx = new dkd_ctx();
    ctx->p = *p;
    ctx->use_graph = 1;
    ctx->use_tma = 1;
    ctx->use_pdl = 1;
    ctx->nms_cpu = 0;
    ctx->sel_prefetch = 0;
    ctx->origin_x = ctx->origin_y = 0;
    ctx->err[0] = 0;
    ctx->tick = 0;
    ctx->have_last_plan = false;
#define CKC(call)                                                                                        \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            snprintf(g_create_error, sizeof(g_create_error), "%s: %s", #call, cudaGetErrorString(e_));   \
            dkd_destroy(ctx);                                                                            \
            if (have_prev) cudaSetDevice(prev_dev);                                                      \
            return DKD_ERR_CUDA;                                                                         \
        }                                                                                                \
    } while (0)
    CKC(cudaSetDevice(p->device));
    CKC(cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, p->device));
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
        ctx->encode = reinterpret_cast<PFN_tensorMapEncodeTiled>(fn);
    (void)cudaGetLastError();
    CKC(setup_nms<1>(ctx));
    CKC(setup_nms<2>(ctx));
    CKC(setup_nms<3>(ctx));
    CKC(setup_nms<4>(ctx));
    CKC(cudaFuncSetAttribute(k_select, cudaFuncAttributeMaxDynamicSharedMemorySize, SEL_SMEM_BYTES));
    CKC(cudaFuncSetAttribute(k_nms_iter<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, IT_SMEM_BYTES));
    CKC(cudaFuncSetAttribute(k_nms_iter<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, IT_SMEM_BYTES));
    CKC(cudaFuncSetAttribute(k_nms_iter<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, IT_SMEM_BYTES));
    CKC(cudaFuncSetAttribute(k_nms_iter<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, IT_SMEM_BYTES));
    CKC(dkd_match_setup_device());
    const size_t tx = (p->max_w + STRIP_W - 1) / STRIP_W, ty = (p->max_h + TH - 1) / TH;
    ctx->max_tiles = tx * (ty + MAX_CPU - 1) * p->max_batch;   // segments of whole units: up to MAX_CPU-1 spare strip-tiles per strip
    const size_t b_cand = align256(ctx->max_tiles * SEG_CAP * sizeof(uint64_t));
    // k_nms_iter writes one count per T x T tile; its smallest tile (halo 40) gives more tiles than there are NMS units
    const size_t it_t_min = (IT_REG - 2 * 40) & ~7;
    const size_t it_tiles = ((p->max_w + it_t_min - 1) / it_t_min) * ((p->max_h + it_t_min - 1) / it_t_min) * p->max_batch;
    ctx->max_segs = ctx->max_tiles > it_tiles ? ctx->max_tiles : it_tiles;
    const size_t b_cnt = align256(ctx->max_segs * sizeof(int));
    const size_t b_sel = align256(static_cast<size_t>(p->max_batch) * p->max_top_k * sizeof(int32_t));
    CKC(cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
    for (int i = 0; i <= MAX_KERNELS; ++i) CKC(cudaEventCreate(&ctx->prof_ev[i]));
    CKC(cudaMalloc(&ctx->cand, b_cand));
    CKC(cudaMalloc(&ctx->tile_cnt, b_cnt));
    CKC(cudaMalloc(&ctx->sel_idx, b_sel));
    ctx->ws_bytes = b_cand + b_cnt + b_sel;
    // Scratch of the descriptor consumers, sized once for the declared maxima (upper bounds of what dkd_match /
    // dkd_retrieval_scan ask dkd_ctx_scratch for), so that those calls never allocate:
    //   match: both directions of P x splits x N partial records of 16 bytes, splits <= min(16, column tiles of 128);
    //   scan:  one key per row plus at most 8 spare per warp of the grid (<= 16 warps per SM), the per-warp counts, and
    //          the similarity of every row when the caller passes out_sim = NULL.
    if (p->max_match_n > 0) {
        const size_t n = p->max_match_n, P = p->max_match_pairs > 0 ? p->max_match_pairs : 2;
        const size_t tiles = (n + 127) / 128, sp = tiles < 16 ? tiles : 16;
        const size_t bytes = align256(2 * P * sp * n * 16);
        CKC(cudaMalloc(&ctx->scratch[0], bytes));
        ctx->scratch_bytes[0] = bytes;
    }
    if (p->max_scan_rows > 0) {
        const size_t n = p->max_scan_rows, nw = 16 * static_cast<size_t>(ctx->num_sms);
        const size_t bytes = align256((n + 8 * nw) * 8) + align256(nw * 4) + align256(n * 4);
        CKC(cudaMalloc(&ctx->scratch[1], bytes));
        ctx->scratch_bytes[1] = bytes;
    }
#undef CKC
    if (have_prev) cudaSetDevice(prev_dev);
    *out = ctx;
    return DKD_OK;
}

int dkd_destroy(dkd_ctx* ctx) {
    if (!ctx) return DKD_OK;
    DeviceGuard dg(ctx->p.device);
    drop_graphs(ctx);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    for (int i = 0; i <= MAX_KERNELS; ++i)
        if (ctx->prof_ev[i]) cudaEventDestroy(ctx->prof_ev[i]);
    if (ctx->cand) cudaFree(ctx->cand);
    if (ctx->tile_cnt) cudaFree(ctx->tile_cnt);
    if (ctx->sel_idx) cudaFree(ctx->sel_idx);
    if (ctx->st_score) cudaFree(ctx->st_score);
    if (ctx->st_desc) cudaFree(ctx->st_desc);
    if (ctx->st_out) cudaFree(ctx->st_out);
    for (int i = 0; i < 2; ++i)
        if (ctx->scratch[i]) cudaFree(ctx->scratch[i]);
    delete ctx;
    return DKD_OK;
}

const char* dkd_last_error(const dkd_ctx* ctx) { return ctx ? ctx->err : g_create_error; }

size_t dkd_workspace_bytes(const dkd_ctx* ctx) {
    return ctx ? ctx->ws_bytes + ctx->st_score_bytes + ctx->st_desc_bytes + ctx->st_out_bytes + ctx->scratch_bytes[0] + ctx->scratch_bytes[1] : 0;
}

int dkd_set_option(dkd_ctx* ctx, int option, int value) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    switch (option) {
        case DKD_OPT_USE_GRAPH: ctx->use_graph = value != 0; return DKD_OK;
        case DKD_OPT_USE_TMA: ctx->use_tma = value != 0; return DKD_OK;
        case DKD_OPT_PROFILE: ctx->profile = value != 0; ctx->prof_n = 0; return DKD_OK;
        case DKD_OPT_USE_PDL: ctx->use_pdl = value != 0; return DKD_OK;          // (part of the graph-cache key)
        case DKD_OPT_NMS_UNIT: ctx->nms_cpu = value > 0 ? value : 0; return DKD_OK;
        case DKD_OPT_SEL_PREFETCH: ctx->sel_prefetch = value != 0; return DKD_OK;   // (kernel argument only)
        case DKD_OPT_ORIGIN_X: ctx->origin_x = value; return DKD_OK;   // (a kernel argument: cached graphs are updated)
        case DKD_OPT_ORIGIN_Y: ctx->origin_y = value; return DKD_OK;
        default: return fail(ctx, DKD_ERR_INVALID_ARG, "unknown option");
    }
}

int dkd_graph_stats(const dkd_ctx* ctx, uint64_t* instantiated, uint64_t* updated, uint64_t* replayed,
                    uint64_t* stream_launched) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (instantiated) *instantiated = ctx->n_instantiated;
    if (updated) *updated = ctx->n_updated;
    if (replayed) *replayed = ctx->n_replayed;
    if (stream_launched) *stream_launched = ctx->n_stream;
    return DKD_OK;
}

int dkd_launches_per_extract(const dkd_ctx* ctx, int with_desc) {
    (void)ctx;
    (void)with_desc;
    return MAX_KERNELS;                                     // k_nms_*, k_select, k_refine_gather
}

const char* dkd_kernel_name(int i) { return (i >= 0 && i < MAX_KERNELS) ? KERNEL_NAMES[i] : ""; }

int dkd_profile_read(dkd_ctx* ctx, float* ms, int n) {
    if (!ctx || !ms || n < 0) return DKD_ERR_INVALID_ARG;
    DeviceGuard dg(ctx->p.device);
    if (ctx->prof_n <= 0) return fail(ctx, DKD_ERR_INVALID_ARG, "no profiled dkd_extract call (set DKD_OPT_PROFILE)");
    CK(ctx, cudaEventSynchronize(ctx->prof_ev[ctx->prof_n]));
    for (int i = 0; i < ctx->prof_n && i < n; ++i) CK(ctx, cudaEventElapsedTime(&ms[i], ctx->prof_ev[i], ctx->prof_ev[i + 1]));
    return ctx->prof_n;
}

int dkd_pre_padded_size(int H, int W, int grid, int* Hp, int* Wp, int* oy, int* ox) {
    if (H < 1 || W < 1 || grid < 1) return DKD_ERR_INVALID_ARG;
    const int hp = (H + grid - 1) / grid * grid, wp = (W + grid - 1) / grid * grid;
    if (Hp) *Hp = hp;
    if (Wp) *Wp = wp;
    if (oy) *oy = (hp - H) / 2;
    if (ox) *ox = (wp - W) / 2;
    return DKD_OK;
}

int dkd_preprocess(dkd_ctx* ctx, const uint8_t* src, int B, int H, int W, const dkd_pre_params* p, void* dst,
                   void* stream) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (!src || !dst || !p || B < 1 || H < 1 || W < 1) return fail(ctx, DKD_ERR_INVALID_ARG, "NULL pointer or size < 1");
    if (p->grid < 1) return fail(ctx, DKD_ERR_INVALID_ARG, "grid must be >= 1");
    if ((p->in_channels != 1 && p->in_channels != 3) || (p->out_channels != 1 && p->out_channels != 3))
        return fail(ctx, DKD_ERR_UNSUPPORTED, "in_channels and out_channels must be 1 or 3");
    if (p->out_dtype != DKD_F32 && p->out_dtype != DKD_F16) return fail(ctx, DKD_ERR_UNSUPPORTED, "out_dtype must be DKD_F32 or DKD_F16");
    if (reinterpret_cast<uintptr_t>(dst) & 15) return fail(ctx, DKD_ERR_UNSUPPORTED, "dst not 16-byte aligned");
    DeviceGuard dg(ctx->p.device);
    PreParams q;
    memset(&q, 0, sizeof(q));
    q.src = src; q.dst = static_cast<unsigned char*>(dst);
    q.B = B; q.H = H; q.W = W;
    dkd_pre_padded_size(H, W, p->grid, &q.Hp, &q.Wp, &q.oy, &q.ox);
    if (B > 65535 || q.Hp > 65535) return fail(ctx, DKD_ERR_UNSUPPORTED, "B and the padded height must be <= 65535");
    q.bgr = p->bgr != 0;
    for (int c = 0; c < 3; ++c) {
        q.a[c] = static_cast<float>(static_cast<double>(p->scale) * static_cast<double>(p->inv_std[c]));
        q.b[c] = static_cast<float>(-static_cast<double>(p->mean[c]) * static_cast<double>(p->inv_std[c]));
    }
    q.pad = p->pad_value;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    const int key = (p->in_channels == 3) * 4 + (p->out_channels == 3) * 2 + (p->out_dtype == DKD_F16);
    switch (key) {
        case 0: e = launch_pre<1, 1, DKD_F32>(q, st); break;
        case 1: e = launch_pre<1, 1, DKD_F16>(q, st); break;
        case 2: e = launch_pre<1, 3, DKD_F32>(q, st); break;
        case 3: e = launch_pre<1, 3, DKD_F16>(q, st); break;
        case 4: e = launch_pre<3, 1, DKD_F32>(q, st); break;
        case 5: e = launch_pre<3, 1, DKD_F16>(q, st); break;
        case 6: e = launch_pre<3, 3, DKD_F32>(q, st); break;
        default: e = launch_pre<3, 3, DKD_F16>(q, st); break;
    }
    if (e != cudaSuccess) return fail_cuda(ctx, "k_preprocess launch", e);
    return DKD_OK;
}

int dkd_extract_var(dkd_ctx* ctx, const float* score, int B, int H, int W, const void* desc, int desc_dtype, int Hd,
                    int Wd, int D, int stride, int r, float thresh, int top_k, float T, float* out_kpts,
                    float* out_scores, void* out_desc, int32_t* out_count, int32_t* out_index, float* out_offset,
                    const dkd_variant_params* v, void* stream) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    DeviceGuard dg(ctx->p.device);
    return run(ctx, make_args(score, B, H, W, desc, desc_dtype, Hd, Wd, D, stride, r, thresh, top_k, T, out_kpts, out_scores,
                              out_desc, out_count, out_index, out_offset, v),
               static_cast<cudaStream_t>(stream));
}

int dkd_extract_ex(dkd_ctx* ctx, const float* score, int B, int H, int W, const void* desc, int desc_dtype, int Hd,
                   int Wd, int D, int stride, int r, float thresh, int top_k, float T, float* out_kpts,
                   float* out_scores, void* out_desc, int32_t* out_count, int32_t* out_index, float* out_offset,
                   void* stream) {
    return dkd_extract_var(ctx, score, B, H, W, desc, desc_dtype, Hd, Wd, D, stride, r, thresh, top_k, T, out_kpts,
                           out_scores, out_desc, out_count, out_index, out_offset, nullptr, stream);
}

int dkd_extract(dkd_ctx* ctx, const float* score, int B, int H, int W, const void* desc, int desc_dtype, int Hd,
                int Wd, int D, int stride, int r, float thresh, int top_k, float T, float* out_kpts, float* out_scores,
                void* out_desc, int32_t* out_count, void* stream) {
    return dkd_extract_var(ctx, score, B, H, W, desc, desc_dtype, Hd, Wd, D, stride, r, thresh, top_k, T, out_kpts,
                           out_scores, out_desc, out_count, nullptr, nullptr, nullptr, stream);
}

int dkd_extract_host(dkd_ctx* ctx, const float* score, int B, int H, int W, const void* desc, int desc_dtype, int Hd,
                     int Wd, int D, int stride, int r, float thresh, int top_k, float T, float* out_kpts,
                     float* out_scores, void* out_desc, int32_t* out_count, int32_t* out_index, float* out_offset,
                     int desc_resident, void* stream) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (!score || !out_kpts || !out_scores || !out_count)
        return fail(ctx, DKD_ERR_INVALID_ARG, "NULL required pointer (score/out_kpts/out_scores/out_count)");
    // every argument check that does not need a device address happens BEFORE anything is allocated or enqueued
    const ExtractArgs chk = make_args(score, B, H, W, desc, desc_dtype, Hd, Wd, D, stride, r, thresh, top_k, T, out_kpts,
                                      out_scores, out_desc, out_count, out_index, out_offset, nullptr);
    int rc = validate_shapes(ctx, chk);
    if (rc != DKD_OK) return rc;
    if (desc_resident < 0 || desc_resident > 2) return fail(ctx, DKD_ERR_INVALID_ARG, "desc_resident must be 0, 1 or 2");
    DeviceGuard dg(ctx->p.device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t esz = desc_dtype == DKD_F16 ? 2 : 4;
    const size_t n_score = static_cast<size_t>(B) * H * W * 4;
    const size_t n_desc = desc ? static_cast<size_t>(B) * Hd * Wd * D * esz : 0;
    const size_t slots = static_cast<size_t>(B) * top_k;
    const size_t o_kpts = 0, o_scores = align256(o_kpts + slots * 8), o_count = align256(o_scores + slots * 4);
    const size_t o_index = align256(o_count + static_cast<size_t>(B) * 4), o_off = align256(o_index + slots * 4);
    const size_t o_desc = align256(o_off + slots * 8), n_out = align256(o_desc + (desc ? slots * D * esz : 0));
    void* d_kpts = mapped_device_pointer(out_kpts);
    void* d_scores = mapped_device_pointer(out_scores);
    void* d_count = mapped_device_pointer(out_count);
    void* d_desc = desc ? mapped_device_pointer(out_desc) : nullptr;
    void* d_index = out_index ? mapped_device_pointer(out_index) : nullptr;
    void* d_off = out_offset ? mapped_device_pointer(out_offset) : nullptr;
    // Pinned (page-locked, mapped) host buffers are addressable from the device.  Two uses:
    //  * descriptor map: only 4 rows per kept keypoint are ever read, so when that is a small part of the map
    //    the gather samples it in place over PCIe instead of uploading all of it;
    //  * outputs: when every output buffer is pinned (and suitably aligned) the kernels store straight into
    //    them (no staging, no device->host copies).
    const bool direct = d_kpts && d_scores && d_count && (!desc || d_desc) && (!out_index || d_index) &&
                        (!out_offset || d_off) && !misaligned(d_desc, 16) && !misaligned(d_kpts, 8) && !misaligned(d_off, 8) &&
                        !misaligned(d_scores, 4) && !misaligned(d_count, 4) && !misaligned(d_index, 4);
    if ((rc = grow(ctx, &ctx->st_score, &ctx->st_score_bytes, n_score)) != DKD_OK) return rc;
    if (!direct && (rc = grow(ctx, &ctx->st_out, &ctx->st_out_bytes, n_out)) != DKD_OK) return rc;
    const void* desc_dev = nullptr;
    bool upload_desc = false;
    if (desc) {
        const void* zc = mapped_device_pointer(desc);
        const size_t touched = slots * 4 * static_cast<size_t>(D) * esz;
        const bool have = desc_resident == 1 && ctx->st_desc && ctx->st_desc_src == desc && ctx->st_desc_src_bytes == n_desc;
        if (have) {
            desc_dev = ctx->st_desc;
        } else if (zc && !desc_resident && touched * 8 <= n_desc && !misaligned(zc, 16)) {
            desc_dev = zc;
        } else {
            if ((rc = grow(ctx, &ctx->st_desc, &ctx->st_desc_bytes, n_desc)) != DKD_OK) return rc;
            upload_desc = true;
            desc_dev = ctx->st_desc;
        }
    }
    // ---- from here on work is enqueued: on any error the stream is drained before returning ----------------
    cudaError_t e = cudaSuccess;
    if (upload_desc) {
        ctx->st_desc_src = nullptr;                         // only an upload made by a resident call may be re-used later
        e = cudaMemcpyAsync(ctx->st_desc, desc, n_desc, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess && desc_resident) { ctx->st_desc_src = desc; ctx->st_desc_src_bytes = n_desc; }
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->st_score, score, n_score, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) {
        cudaStreamSynchronize(st);
        return fail_cuda(ctx, "host -> device copy", e);
    }
    if (direct) {
        rc = dkd_extract_ex(ctx, static_cast<const float*>(ctx->st_score), B, H, W, desc_dev, desc_dtype, Hd, Wd, D, stride,
                            r, thresh, top_k, T, static_cast<float*>(d_kpts), static_cast<float*>(d_scores), d_desc,
                            static_cast<int32_t*>(d_count), static_cast<int32_t*>(d_index), static_cast<float*>(d_off), st);
        e = cudaStreamSynchronize(st);
        if (rc != DKD_OK) return rc;
        if (e != cudaSuccess) return fail_cuda(ctx, "cudaStreamSynchronize", e);
        return DKD_OK;
    }
    char* so = static_cast<char*>(ctx->st_out);
    rc = dkd_extract_ex(ctx, static_cast<const float*>(ctx->st_score), B, H, W, desc_dev,
                        desc_dtype, Hd, Wd, D, stride, r, thresh, top_k, T, reinterpret_cast<float*>(so + o_kpts),
                        reinterpret_cast<float*>(so + o_scores), desc ? so + o_desc : nullptr,
                        reinterpret_cast<int32_t*>(so + o_count),
                        out_index ? reinterpret_cast<int32_t*>(so + o_index) : nullptr,
                        out_offset ? reinterpret_cast<float*>(so + o_off) : nullptr, st);
    if (rc != DKD_OK) {
        cudaStreamSynchronize(st);
        return rc;
    }
    e = cudaMemcpyAsync(out_kpts, so + o_kpts, slots * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out_scores, so + o_scores, slots * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out_count, so + o_count, static_cast<size_t>(B) * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && out_index) e = cudaMemcpyAsync(out_index, so + o_index, slots * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && out_offset) e = cudaMemcpyAsync(out_offset, so + o_off, slots * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && desc) e = cudaMemcpyAsync(out_desc, so + o_desc, slots * D * esz, cudaMemcpyDeviceToHost, st);
    const cudaError_t es = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail_cuda(ctx, "device -> host copy", e);
    if (es != cudaSuccess) return fail_cuda(ctx, "cudaStreamSynchronize", es);
    return DKD_OK;
}

}  // extern "C"
