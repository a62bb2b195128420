// dkd_api.cu — host side of libdkd: the C-ABI of include/dkd.h (argument validation, workspace,
// TMA descriptor, launches, CUDA-graph cache, host-buffer path).  See DESIGN.md.
#include "dkd.h"

#include <math.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "dkd_kernels.cuh"

using namespace dkd;

namespace {

typedef CUresult (*PFN_tensorMapEncodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                             const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                             CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                             CUtensorMapFloatOOBfill);

char g_create_error[512] = "";

struct ExtractArgs {                       // everything that determines the enqueued work
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
    int use_tma;
    int origin_x, origin_y;                // letterbox offset subtracted from the keypoint coordinates
};

struct GraphEntry {
    ExtractArgs key;
    cudaGraphExec_t exec;
    unsigned long long last_use;
};

constexpr size_t GRAPH_CACHE_CAP = 256;
constexpr int MAX_KERNELS = 3;                              // kernels per extract, in launch order:
const char* const KERNEL_NAMES[MAX_KERNELS] = {"nms", "select", "refine_gather"};

}  // namespace

struct dkd_ctx {
    dkd_create_params p;
    int num_sms;
    int nms_ctas_per_sm[MAX_R + 1];
    PFN_tensorMapEncodeTiled encode;
    // workspace (device)
    uint64_t* cand;          // [max_tiles * SEG_CAP] candidate keys, one private segment per NMS unit
    int* tile_cnt;           // [max_tiles] keys in each segment
    int32_t* sel_idx;        // [max_batch * max_top_k]
    size_t max_tiles;
    size_t ws_bytes;
    // host-path staging (device), grown on demand
    void* st_score; size_t st_score_bytes;
    void* st_desc;  size_t st_desc_bytes;
    void* st_out;   size_t st_out_bytes;
    const void* st_desc_src; size_t st_desc_src_bytes;      // what st_desc currently holds
    // options
    int use_graph, use_tma, use_pdl, profile, nms_cpu, origin_x, origin_y;
    cudaEvent_t prof_ev[MAX_KERNELS + 1];                   // measurement mode: event before/after every kernel
    int prof_n;                                             // kernels of the last profiled call (0: none)
    std::vector<GraphEntry> graphs;
    cudaStream_t cap_stream;  // capture-only stream for building the cached graphs
    unsigned long long tick;
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

template <int R>
cudaError_t setup_nms(dkd_ctx* ctx) {
    cudaError_t e = cudaFuncSetAttribute(k_nms_tma<R, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, NMS_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_nms_tma<R, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, NMS_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    int n = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_nms_tma<R, true>, NMS_WARPS * 32, NMS_SMEM_BYTES);
    ctx->nms_ctas_per_sm[R] = n > 0 ? n : 1;
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
    const long long slots = 2LL * ctx->num_sms * NMS_WARPS;  // resident warps
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

template <int R>
cudaError_t launch_nms(dkd_ctx* ctx, const ExtractArgs& a, const NmsPlan& p, cudaStream_t st) {
    if (a.use_tma) {
        CUtensorMap tmap;
        const cuuint64_t dims[3] = {(cuuint64_t)a.W, (cuuint64_t)a.H, (cuuint64_t)a.B};
        const cuuint64_t strides[2] = {(cuuint64_t)a.W * 4, (cuuint64_t)a.W * a.H * 4};
        const cuuint32_t box[3] = {(cuuint32_t)BOX_W, (cuuint32_t)TH, 1};
        const cuuint32_t estr[3] = {1, 1, 1};
        if (ctx->encode(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(a.score), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return cudaErrorInvalidValue;
        int grid = ctx->num_sms * ctx->nms_ctas_per_sm[R];
        if (grid > (p.units + NMS_WARPS - 1) / NMS_WARPS) grid = (p.units + NMS_WARPS - 1) / NMS_WARPS;
        if (p.thr_up > 0.0f)
            k_nms_tma<R, false><<<grid, NMS_WARPS * 32, NMS_SMEM_BYTES, st>>>(tmap, p, a.score, ctx->cand, ctx->tile_cnt);
        else                                                 // a -0.0 score may be a candidate: fold it onto +0
            k_nms_tma<R, true><<<grid, NMS_WARPS * 32, NMS_SMEM_BYTES, st>>>(tmap, p, a.score, ctx->cand, ctx->tile_cnt);
    } else {
        const int total = p.strips_x * p.chunks_y * a.B;
        k_nms_plain<R><<<(total + PLAIN_WARPS - 1) / PLAIN_WARPS, PLAIN_WARPS * 32, 0, st>>>(a.score, p, total, ctx->cand,
                                                                                             ctx->tile_cnt);
    }
    return cudaGetLastError();
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

// Launch with (pdl) or without the programmatic-stream-serialization attribute: with it the kernel may be
// scheduled while its predecessor in the stream still runs (it calls griddepcontrol.wait before it reads
// the predecessor's results), which hides the launch latency between the three kernels of an extract.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                       Args... args) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

template <int DT, int G>
cudaError_t launch_rg_g(const RGParams& p, int B, cudaStream_t st, bool pdl) {
    const dim3 grid((p.top_k + RG_THREADS / G - 1) / (RG_THREADS / G), B);
    return launch_pdl(k_refine_gather<DT, G>, grid, dim3(RG_THREADS), 0, st, pdl, p);
}

template <int DT>
cudaError_t launch_rg_dt(const RGParams& p, int B, cudaStream_t st, bool pdl) {
    if (p.nchunk <= 8) return launch_rg_g<DT, 8>(p, B, st, pdl);
    if (p.nchunk <= 16) return launch_rg_g<DT, 16>(p, B, st, pdl);
    return launch_rg_g<DT, 32>(p, B, st, pdl);
}

cudaError_t launch_rg(const ExtractArgs& a, const int32_t* sel, cudaStream_t st, bool pdl) {
    RGParams p;
    memset(&p, 0, sizeof(p));
    p.score = a.score; p.H = a.H; p.W = a.W;
    p.divW = make_fastdiv(static_cast<uint32_t>(a.W));
    p.sel_idx = sel; p.top_k = a.top_k; p.r = a.r;
    p.kscale = static_cast<float>(1.4426950408889634 / static_cast<double>(a.T));
    p.out_kpts = a.out_kpts; p.out_scores = a.out_scores; p.out_off = a.out_offset;
    p.origin_x = a.origin_x; p.origin_y = a.origin_y;
    if (a.desc == nullptr) return launch_rg_g<-1, 8>(p, a.B, st, pdl);
    const size_t esz = a.desc_dtype == DKD_F16 ? 2 : 4;
    p.desc = static_cast<const unsigned char*>(a.desc);
    p.nchunk = static_cast<int>(a.D * esz / 16);
    p.img_bytes = static_cast<size_t>(a.Hd) * a.Wd * a.D * esz;
    p.ax = make_axis(a.stride, a.Wd);
    p.ay = make_axis(a.stride, a.Hd);
    p.out_desc = static_cast<unsigned char*>(a.out_desc);
    return a.desc_dtype == DKD_F16 ? launch_rg_dt<DKD_F16>(p, a.B, st, pdl) : launch_rg_dt<DKD_F32>(p, a.B, st, pdl);
}

// Enqueue the three kernels of one extract on `st`.  No sync, no allocation: capture-safe.
// prof: measurement mode, an event on `st` before and after every kernel.
cudaError_t enqueue(dkd_ctx* ctx, const ExtractArgs& a, cudaStream_t st, bool prof = false) {
    const NmsPlan plan = nms_plan(ctx, a);
    const int tpi = plan.strips_x * plan.segs;              // candidate segments (NMS units) per image
    cudaError_t e;
    int nk = 0;
    auto mark = [&]() { return prof ? cudaEventRecord(ctx->prof_ev[nk++], st) : cudaSuccess; };
    if ((e = mark()) != cudaSuccess) return e;
    switch (a.r) {
        case 1: e = launch_nms<1>(ctx, a, plan, st); break;
        case 2: e = launch_nms<2>(ctx, a, plan, st); break;
        case 3: e = launch_nms<3>(ctx, a, plan, st); break;
        default: e = launch_nms<4>(ctx, a, plan, st); break;
    }
    if (e != cudaSuccess) return e;
    if ((e = mark()) != cudaSuccess) return e;
    int32_t* sel = a.out_index ? a.out_index : ctx->sel_idx;
    int idx_shift = 0;                                       // (H*W - 1) >> idx_shift < NBT: index buckets of the top ties
    while (((static_cast<long long>(a.H) * a.W - 1) >> idx_shift) >= NBT) ++idx_shift;
    const bool pdl = ctx->use_pdl && !prof;                  // (events between the kernels would serialise them anyway)
    e = launch_pdl(k_select, dim3(a.B), dim3(SEL_THREADS), SEL_SMEM_BYTES, st, pdl, ctx->cand, ctx->tile_cnt, tpi,
                   plan.cpu * SEG_CAP, a.top_k, idx_shift, sel, a.out_count);
    if (e != cudaSuccess) return e;
    if ((e = mark()) != cudaSuccess) return e;
    e = launch_rg(a, sel, st, pdl);
    if (e != cudaSuccess) return e;
    if ((e = mark()) != cudaSuccess) return e;
    if (prof) ctx->prof_n = nk - 1;
    return cudaSuccess;
}

int validate(dkd_ctx* ctx, const ExtractArgs& a) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (!a.score || !a.out_kpts || !a.out_scores || !a.out_count)
        return fail(ctx, DKD_ERR_INVALID_ARG, "NULL required pointer (score/out_kpts/out_scores/out_count)");
    if (a.B < 1 || a.H < 1 || a.W < 1 || a.top_k < 1) return fail(ctx, DKD_ERR_INVALID_ARG, "B, H, W, top_k must be >= 1");
    if (a.r < 1) return fail(ctx, DKD_ERR_INVALID_ARG, "r must be >= 1");
    if (!(a.T > 0.0f) || !isfinite(a.T)) return fail(ctx, DKD_ERR_INVALID_ARG, "T must be finite and > 0");
    if (isnan(a.thresh)) return fail(ctx, DKD_ERR_INVALID_ARG, "thresh is NaN");
    if ((a.desc == nullptr) != (a.out_desc == nullptr))
        return fail(ctx, DKD_ERR_INVALID_ARG, "desc and out_desc must both be NULL or both be set");
    if (a.desc) {
        if (a.Hd < 1 || a.Wd < 1 || a.D < 1 || a.stride < 1)
            return fail(ctx, DKD_ERR_INVALID_ARG, "Hd, Wd, D, stride must be >= 1");
        if (a.desc_dtype != DKD_F32 && a.desc_dtype != DKD_F16)
            return fail(ctx, DKD_ERR_UNSUPPORTED, "desc_dtype must be DKD_F32 or DKD_F16");
    }
    if (a.r > DKD_MAX_RADIUS) return fail(ctx, DKD_ERR_UNSUPPORTED, "r > DKD_MAX_RADIUS");
    if (a.B > 65535) return fail(ctx, DKD_ERR_UNSUPPORTED, "B > 65535");
    if (reinterpret_cast<uintptr_t>(a.score) & 3) return fail(ctx, DKD_ERR_UNSUPPORTED, "score not 4-byte aligned");
    if (a.desc) {
        const size_t rowb = static_cast<size_t>(a.D) * (a.desc_dtype == DKD_F16 ? 2 : 4);
        if (rowb % 16 != 0 || rowb > DKD_MAX_ROW_BYTES)
            return fail(ctx, DKD_ERR_UNSUPPORTED, "D * elemsize must be a multiple of 16 and <= DKD_MAX_ROW_BYTES");
        if ((reinterpret_cast<uintptr_t>(a.desc) & 15) || (reinterpret_cast<uintptr_t>(a.out_desc) & 15))
            return fail(ctx, DKD_ERR_UNSUPPORTED, "desc / out_desc not 16-byte aligned");
        if (a.D > ctx->p.max_dim) return fail(ctx, DKD_ERR_CAPACITY, "D > max_dim");
        if (a.stride > (1 << 20)) return fail(ctx, DKD_ERR_UNSUPPORTED, "stride too large");
    }
    if (a.B > ctx->p.max_batch || a.H > ctx->p.max_h || a.W > ctx->p.max_w || a.top_k > ctx->p.max_top_k)
        return fail(ctx, DKD_ERR_CAPACITY, "B, H, W or top_k above the dkd_create maxima");
    return DKD_OK;
}

bool same_key(const ExtractArgs& x, const ExtractArgs& y) { return memcmp(&x, &y, sizeof(ExtractArgs)) == 0; }

int run(dkd_ctx* ctx, ExtractArgs a, cudaStream_t st) {
    int rc = validate(ctx, a);
    if (rc != DKD_OK) return rc;
    a.origin_x = ctx->origin_x; a.origin_y = ctx->origin_y;
    a.use_tma = ctx->use_tma && ctx->encode && (a.W % 4 == 0) && ((reinterpret_cast<uintptr_t>(a.score) & 15) == 0);

    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    CK(ctx, cudaStreamIsCapturing(st, &cap));
    if (ctx->profile && cap == cudaStreamCaptureStatusNone) {
        ctx->prof_n = 0;
        CK(ctx, enqueue(ctx, a, st, true));
        return DKD_OK;
    }
    if (!ctx->use_graph || cap != cudaStreamCaptureStatusNone) {
        CK(ctx, enqueue(ctx, a, st));
        return DKD_OK;
    }
    ++ctx->tick;
    for (auto& g : ctx->graphs)
        if (same_key(g.key, a)) {
            g.last_use = ctx->tick;
            CK(ctx, cudaGraphLaunch(g.exec, st));
            return DKD_OK;
        }
    // first call with these arguments: capture the launches once, then replay as one graph launch
    cudaGraph_t graph = nullptr;
    // (captured on a context-owned stream: the caller's may be the legacy default stream, which
    // cannot be captured; the instantiated graph is then launched on the caller's stream)
    CK(ctx, cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
    cudaError_t e = enqueue(ctx, a, ctx->cap_stream);
    cudaError_t e2 = cudaStreamEndCapture(ctx->cap_stream, &graph);
    if (e != cudaSuccess || e2 != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        return fail_cuda(ctx, "graph capture", e != cudaSuccess ? e : e2);
    }
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaGraphInstantiate", e);
    if (ctx->graphs.size() >= GRAPH_CACHE_CAP) {            // evict the least recently used entry
        size_t v = 0;
        for (size_t i = 1; i < ctx->graphs.size(); ++i)
            if (ctx->graphs[i].last_use < ctx->graphs[v].last_use) v = i;
        cudaGraphExecDestroy(ctx->graphs[v].exec);
        ctx->graphs[v] = ctx->graphs.back();
        ctx->graphs.pop_back();
    }
    GraphEntry ge;
    ge.key = a;
    ge.exec = exec;
    ge.last_use = ctx->tick;
    ctx->graphs.push_back(ge);
    CK(ctx, cudaGraphLaunch(exec, st));
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

}  // namespace

extern "C" {

const char* dkd_version(void) { return "dkd-b200 0.1 (sm_100a)"; }

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
    dkd_ctx* ctx = new dkd_ctx();
    ctx->p = *p;
    ctx->use_graph = 1;
    ctx->use_tma = 1;
    ctx->use_pdl = 1;
    ctx->nms_cpu = 0;
    ctx->origin_x = ctx->origin_y = 0;
    ctx->err[0] = 0;
    ctx->tick = 0;
#define CKC(call)                                                                                        \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            snprintf(g_create_error, sizeof(g_create_error), "%s: %s", #call, cudaGetErrorString(e_));   \
            dkd_destroy(ctx);                                                                            \
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
    const size_t tx = (p->max_w + STRIP_W - 1) / STRIP_W, ty = (p->max_h + TH - 1) / TH;
    ctx->max_tiles = tx * (ty + MAX_CPU - 1) * p->max_batch;   // segments of whole units: up to MAX_CPU-1 spare strip-tiles per strip
    const size_t b_cand = align256(ctx->max_tiles * SEG_CAP * sizeof(uint64_t));
    const size_t b_cnt = align256(ctx->max_tiles * sizeof(int));
    const size_t b_sel = align256(static_cast<size_t>(p->max_batch) * p->max_top_k * sizeof(int32_t));
    CKC(cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
    for (int i = 0; i <= MAX_KERNELS; ++i) CKC(cudaEventCreate(&ctx->prof_ev[i]));
    CKC(cudaMalloc(&ctx->cand, b_cand));
    CKC(cudaMalloc(&ctx->tile_cnt, b_cnt));
    CKC(cudaMalloc(&ctx->sel_idx, b_sel));
    ctx->ws_bytes = b_cand + b_cnt + b_sel;
#undef CKC
    *out = ctx;
    return DKD_OK;
}

int dkd_destroy(dkd_ctx* ctx) {
    if (!ctx) return DKD_OK;
    for (auto& g : ctx->graphs) cudaGraphExecDestroy(g.exec);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    for (int i = 0; i <= MAX_KERNELS; ++i)
        if (ctx->prof_ev[i]) cudaEventDestroy(ctx->prof_ev[i]);
    if (ctx->cand) cudaFree(ctx->cand);
    if (ctx->tile_cnt) cudaFree(ctx->tile_cnt);
    if (ctx->sel_idx) cudaFree(ctx->sel_idx);
    if (ctx->st_score) cudaFree(ctx->st_score);
    if (ctx->st_desc) cudaFree(ctx->st_desc);
    if (ctx->st_out) cudaFree(ctx->st_out);
    delete ctx;
    return DKD_OK;
}

const char* dkd_last_error(const dkd_ctx* ctx) { return ctx ? ctx->err : g_create_error; }

size_t dkd_workspace_bytes(const dkd_ctx* ctx) {
    return ctx ? ctx->ws_bytes + ctx->st_score_bytes + ctx->st_desc_bytes + ctx->st_out_bytes : 0;
}

int dkd_set_option(dkd_ctx* ctx, int option, int value) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    switch (option) {
        case DKD_OPT_USE_GRAPH: ctx->use_graph = value != 0; return DKD_OK;
        case DKD_OPT_USE_TMA: ctx->use_tma = value != 0; return DKD_OK;
        case DKD_OPT_PROFILE: ctx->profile = value != 0; ctx->prof_n = 0; return DKD_OK;
        case DKD_OPT_USE_PDL:                               // part of what a cached graph contains: drop the cache
        case DKD_OPT_NMS_UNIT:
            for (auto& g : ctx->graphs) cudaGraphExecDestroy(g.exec);
            ctx->graphs.clear();
            if (option == DKD_OPT_USE_PDL) ctx->use_pdl = value != 0;
            else ctx->nms_cpu = value > 0 ? value : 0;
            return DKD_OK;
        case DKD_OPT_ORIGIN_X: ctx->origin_x = value; return DKD_OK;   // (part of the graph-cache key)
        case DKD_OPT_ORIGIN_Y: ctx->origin_y = value; return DKD_OK;
        default: return fail(ctx, DKD_ERR_INVALID_ARG, "unknown option");
    }
}

int dkd_launches_per_extract(const dkd_ctx* ctx, int with_desc) {
    (void)ctx;
    (void)with_desc;
    return MAX_KERNELS;                                     // k_nms_*, k_select, k_refine_gather
}

const char* dkd_kernel_name(int i) { return (i >= 0 && i < MAX_KERNELS) ? KERNEL_NAMES[i] : ""; }

int dkd_profile_read(dkd_ctx* ctx, float* ms, int n) {
    if (!ctx || !ms || n < 0) return DKD_ERR_INVALID_ARG;
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

int dkd_extract_ex(dkd_ctx* ctx, const float* score, int B, int H, int W, const void* desc, int desc_dtype, int Hd,
                   int Wd, int D, int stride, int r, float thresh, int top_k, float T, float* out_kpts,
                   float* out_scores, void* out_desc, int32_t* out_count, int32_t* out_index, float* out_offset,
                   void* stream) {
    ExtractArgs a;
    memset(&a, 0, sizeof(a));                               // key is compared with memcmp: no stray padding
    a.score = score; a.B = B; a.H = H; a.W = W;
    a.desc = desc; a.desc_dtype = desc ? desc_dtype : 0; a.Hd = desc ? Hd : 0; a.Wd = desc ? Wd : 0;
    a.D = desc ? D : 0; a.stride = desc ? stride : 1; a.r = r; a.thresh = thresh; a.top_k = top_k; a.T = T;
    a.out_kpts = out_kpts; a.out_scores = out_scores; a.out_desc = out_desc; a.out_count = out_count;
    a.out_index = out_index; a.out_offset = out_offset;
    return run(ctx, a, static_cast<cudaStream_t>(stream));
}

int dkd_extract(dkd_ctx* ctx, const float* score, int B, int H, int W, const void* desc, int desc_dtype, int Hd,
                int Wd, int D, int stride, int r, float thresh, int top_k, float T, float* out_kpts, float* out_scores,
                void* out_desc, int32_t* out_count, void* stream) {
    return dkd_extract_ex(ctx, score, B, H, W, desc, desc_dtype, Hd, Wd, D, stride, r, thresh, top_k, T, out_kpts,
                          out_scores, out_desc, out_count, nullptr, nullptr, stream);
}

int dkd_extract_host(dkd_ctx* ctx, const float* score, int B, int H, int W, const void* desc, int desc_dtype, int Hd,
                     int Wd, int D, int stride, int r, float thresh, int top_k, float T, float* out_kpts,
                     float* out_scores, void* out_desc, int32_t* out_count, int32_t* out_index, float* out_offset,
                     int desc_resident, void* stream) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (!score || !out_kpts || !out_scores || !out_count || B < 1 || H < 1 || W < 1 || top_k < 1)
        return fail(ctx, DKD_ERR_INVALID_ARG, "NULL required pointer or size < 1");
    if ((desc == nullptr) != (out_desc == nullptr))
        return fail(ctx, DKD_ERR_INVALID_ARG, "desc and out_desc must both be NULL or both be set");
    if (desc && (Hd < 1 || Wd < 1 || D < 1 || (desc_dtype != DKD_F32 && desc_dtype != DKD_F16)))
        return fail(ctx, DKD_ERR_INVALID_ARG, "bad descriptor-map shape or dtype");
    if (B > ctx->p.max_batch || H > ctx->p.max_h || W > ctx->p.max_w || top_k > ctx->p.max_top_k)
        return fail(ctx, DKD_ERR_CAPACITY, "B, H, W or top_k above the dkd_create maxima");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t esz = desc_dtype == DKD_F16 ? 2 : 4;
    const size_t n_score = static_cast<size_t>(B) * H * W * 4;
    const size_t n_desc = desc ? static_cast<size_t>(B) * Hd * Wd * D * esz : 0;
    const size_t slots = static_cast<size_t>(B) * top_k;
    const size_t o_kpts = 0, o_scores = align256(o_kpts + slots * 8), o_count = align256(o_scores + slots * 4);
    const size_t o_index = align256(o_count + static_cast<size_t>(B) * 4), o_off = align256(o_index + slots * 4);
    const size_t o_desc = align256(o_off + slots * 8), n_out = align256(o_desc + (desc ? slots * D * esz : 0));
    int rc;
    if ((rc = grow(ctx, &ctx->st_score, &ctx->st_score_bytes, n_score)) != DKD_OK) return rc;
    // Pinned (page-locked, mapped) host buffers are addressable from the device.  Two uses:
    //  * descriptor map: only 4 rows per kept keypoint are ever read, so when that is a small part of the map
    //    the gather samples it in place over PCIe instead of uploading all of it;
    //  * outputs: when every output buffer is pinned the kernels store straight into them (no staging, no
    //    device->host copies).
    const void* desc_dev = nullptr;
    if (desc) {
        const void* zc = mapped_device_pointer(desc);
        const size_t touched = slots * 4 * static_cast<size_t>(D) * esz;
        const bool have = desc_resident && ctx->st_desc && ctx->st_desc_src == desc && ctx->st_desc_src_bytes == n_desc;
        if (have) {
            desc_dev = ctx->st_desc;
        } else if (zc && !desc_resident && touched * 8 <= n_desc) {
            desc_dev = zc;
        } else {
            if ((rc = grow(ctx, &ctx->st_desc, &ctx->st_desc_bytes, n_desc)) != DKD_OK) return rc;
            CK(ctx, cudaMemcpyAsync(ctx->st_desc, desc, n_desc, cudaMemcpyHostToDevice, st));
            ctx->st_desc_src = desc;
            ctx->st_desc_src_bytes = n_desc;
            desc_dev = ctx->st_desc;
        }
    }
    CK(ctx, cudaMemcpyAsync(ctx->st_score, score, n_score, cudaMemcpyHostToDevice, st));
    void* d_kpts = mapped_device_pointer(out_kpts);
    void* d_scores = mapped_device_pointer(out_scores);
    void* d_count = mapped_device_pointer(out_count);
    void* d_desc = desc ? mapped_device_pointer(out_desc) : nullptr;
    void* d_index = out_index ? mapped_device_pointer(out_index) : nullptr;
    void* d_off = out_offset ? mapped_device_pointer(out_offset) : nullptr;
    const bool direct = d_kpts && d_scores && d_count && (!desc || d_desc) && (!out_index || d_index) &&
                        (!out_offset || d_off) && (!desc || (reinterpret_cast<uintptr_t>(d_desc) & 15) == 0);
    if (direct) {
        rc = dkd_extract_ex(ctx, static_cast<const float*>(ctx->st_score), B, H, W, desc_dev, desc_dtype, Hd, Wd, D, stride,
                            r, thresh, top_k, T, static_cast<float*>(d_kpts), static_cast<float*>(d_scores), d_desc,
                            static_cast<int32_t*>(d_count), static_cast<int32_t*>(d_index), static_cast<float*>(d_off), st);
        if (rc != DKD_OK) return rc;
        CK(ctx, cudaStreamSynchronize(st));
        return DKD_OK;
    }
    if ((rc = grow(ctx, &ctx->st_out, &ctx->st_out_bytes, n_out)) != DKD_OK) return rc;
    char* so = static_cast<char*>(ctx->st_out);
    rc = dkd_extract_ex(ctx, static_cast<const float*>(ctx->st_score), B, H, W, desc_dev,
                        desc_dtype, Hd, Wd, D, stride, r, thresh, top_k, T, reinterpret_cast<float*>(so + o_kpts),
                        reinterpret_cast<float*>(so + o_scores), desc ? so + o_desc : nullptr,
                        reinterpret_cast<int32_t*>(so + o_count),
                        out_index ? reinterpret_cast<int32_t*>(so + o_index) : nullptr,
                        out_offset ? reinterpret_cast<float*>(so + o_off) : nullptr, st);
    if (rc != DKD_OK) return rc;
    CK(ctx, cudaMemcpyAsync(out_kpts, so + o_kpts, slots * 8, cudaMemcpyDeviceToHost, st));
    CK(ctx, cudaMemcpyAsync(out_scores, so + o_scores, slots * 4, cudaMemcpyDeviceToHost, st));
    CK(ctx, cudaMemcpyAsync(out_count, so + o_count, static_cast<size_t>(B) * 4, cudaMemcpyDeviceToHost, st));
    if (out_index) CK(ctx, cudaMemcpyAsync(out_index, so + o_index, slots * 4, cudaMemcpyDeviceToHost, st));
    if (out_offset) CK(ctx, cudaMemcpyAsync(out_offset, so + o_off, slots * 8, cudaMemcpyDeviceToHost, st));
    if (desc) CK(ctx, cudaMemcpyAsync(out_desc, so + o_desc, slots * D * esz, cudaMemcpyDeviceToHost, st));
    CK(ctx, cudaStreamSynchronize(st));
    return DKD_OK;
}

}  // extern "C"
