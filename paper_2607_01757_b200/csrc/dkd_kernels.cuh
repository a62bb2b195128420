// dkd_kernels.cuh — device code of libdkd (sm_100a).  Hand-written CUDA, no tensor cores (nothing on
// this path is a dense contraction), no CPU fallback.
//
// Kernels (reference = /root/reference/PAPER.md):
//   k_nms_tma / k_nms_plain   step a1 + a1'  NMS + border + threshold + warp-ballot compaction
//                             ("NMS" stage; north_star step (1))
//   k_select                  step a2        per-image top-k on the 64-bit key, ordered
//                             ("sorting"; north_star step (2))
//   k_refine_gather           steps a3-a5    soft-argmax refinement, bilinear gather + L2 norm,
//                             zero padding (north_star steps (3),(4))
#pragma once

#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <type_traits>
#include <stdint.h>

#include "dkd.h"

// -DDKD_DEBUG (libdkd_debug.so): device-side bounds checks on every workspace / shared-memory index and on
// the mbarrier ring arithmetic; compiled out of the product library.
#ifdef DKD_DEBUG
#include <assert.h>
#define DKD_ASSERT(c) assert(c)
#else
#define DKD_ASSERT(c) ((void)0)
#endif

namespace dkd {

// ---- geometry -------------------------------------------------------------------------------
// NMS work is cut into STRIP-TILES of STRIP_W x TH output pixels (one candidate segment each).  A
// warp owns a UNIT = up to MAX_CPU vertically consecutive strip-tiles of one strip and walks down it
// keeping the last 2R rows in registers, so the R halo rows above a strip-tile are fetched only once
// per unit.  Shared-memory boxes are BOX_W = 128 floats wide: 4 halo columns each side (>= max
// radius, keeps every lane's float4 16-byte aligned) — one 512-byte row per image row.  Lane l owns
// box columns 4l..4l+3; lanes 0 and 31 hold only halo columns, lanes 1..30 produce the 120 outputs.
constexpr int STRIP_W = 120;             // output columns per strip
constexpr int BOX_W = 128;               // box columns = one 512-byte shared-memory row (32 lanes x float4)
constexpr int HALO_X = 4;
constexpr int TH = 8;                    // output rows per strip-tile = rows of one TMA box
constexpr int SEG_CAP = STRIP_W * TH;    // 960 = worst-case candidates of a strip-tile = segment capacity
constexpr int MAX_R = 4;
constexpr int MAX_CPU = 8;               // strip-tiles (chunks) per unit, chosen per call (nms_plan)
constexpr int SEL_THREADS = 1024;
constexpr int SORT_CAP = 8192;           // keys ordered in shared memory by k_select
constexpr int RG_THREADS = 256;          // k_refine_gather: 8 warps, 8..32 keypoints per CTA

constexpr int BOX_BYTES = BOX_W * TH * 4;                                                // 4 KB
// Every resident warp keeps NMS_STAGES-1 boxes in flight while it works on one: bytes in flight per
// SM >= 2 CTAs x warps x (stages-1) x 4 KB = 128 KB (HBM latency x bandwidth needs ~50 KB per SM).
// (-DDKD_NMS_WARPS / _STAGES / _CTAS: tuning builds only — DESIGN.md 7.5 quotes what 8 and 12 warps per SM cost)
#ifndef DKD_NMS_WARPS
#define DKD_NMS_WARPS 8
#endif
#ifndef DKD_NMS_STAGES
#define DKD_NMS_STAGES 3
#endif
#ifndef DKD_NMS_CTAS
#define DKD_NMS_CTAS 2
#endif
constexpr int NMS_WARPS = DKD_NMS_WARPS;  // per CTA, 2 CTAs/SM: 16 warps x <= 128 registers
constexpr int NMS_STAGES = DKD_NMS_STAGES;
constexpr int NMS_CTAS = DKD_NMS_CTAS;    // CTAs per SM the kernel is compiled and launched for
constexpr int NMS_SMEM_BYTES = NMS_WARPS * NMS_STAGES * BOX_BYTES;                        // 96 KB per CTA

// ---- 64-bit selection key ---------------------------------------------------------------------
// key = (orderable(score bits) << 32) | ~idx : a larger key is a better candidate, i.e. descending
// key order == (score desc, idx asc) — DESIGN.md G6.  -0.0 is folded onto +0.0 so that the order is
// the order of fp32 VALUES; the reported score is re-read from the map (bit-exact, G7).
__device__ __forceinline__ uint64_t make_key(float s, int idx) {
    uint32_t b = __float_as_uint(s + 0.0f);
    b ^= (b & 0x80000000u) ? 0xFFFFFFFFu : 0x80000000u;
    return (static_cast<uint64_t>(b) << 32) | static_cast<uint32_t>(~static_cast<uint32_t>(idx));
}
__device__ __forceinline__ int key_index(uint64_t key) { return static_cast<int>(~static_cast<uint32_t>(key)); }

// ---- mbarrier / TMA (inline PTX) ------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 3-D tiled TMA load (x, y, image) -> shared memory, completion signalled on `bar` (complete_tx).
// Out-of-bounds elements (negative or past-the-end coordinates) are zero-filled by the hardware.
__device__ __forceinline__ void tma_load_tile(void* dst, const CUtensorMap* tmap, uint64_t* bar, int x, int y,
                                              int b, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5}], [%2], %6;"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(b), "l"(policy)
        : "memory");
}
// L2 policy for data that is read once (the score maps): evict first, so the stream does not push the
// candidate lists and the previous call's outputs out of L2
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// The candidate lists are small (a few MB) and are read back by k_select right after the NMS pass has streamed half a
// gigabyte through L2: written with an evict-last policy they are still in L2 when k_select gathers them.
__device__ __forceinline__ uint64_t l2_evict_last_policy() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void st_keep_u64(uint64_t* p, uint64_t v, uint64_t policy) {
    asm volatile("st.global.L2::cache_hint.b64 [%0], %1, %2;" ::"l"(p), "l"(v), "l"(policy) : "memory");
}
__device__ __forceinline__ void st_keep_s32(int* p, int v, uint64_t policy) {
    asm volatile("st.global.L2::cache_hint.b32 [%0], %1, %2;" ::"l"(p), "r"(v), "l"(policy) : "memory");
}
// true in exactly one lane of a converged warp (elect.sync): the compiler then knows the guarded code runs in a single
// thread and emits the uniform-register instructions (UTMALDG) without a per-lane election loop around them
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tmap)) : "memory");
}

// programmatic dependent launch (PDL): a kernel launched with the programmatic-stream-serialization
// attribute may start while its predecessor still runs; pdl_wait() blocks until the predecessor grid
// has completed and its writes are visible, pdl_launch_dependents() lets the successor be scheduled.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }

// 3-input max: one FMNMX3 on sm_100a (alu pipe), halves the op count of the window maxima
__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float d;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}

// ---- step a1: TH new rows of one strip -> candidate bit mask ----------------------------------------
// cat[q] = image row yc-R+q of this lane's 4 columns, q = 0 .. TH+2R-1 (registers): output row yc+o
// needs cat[o] .. cat[o+2R], its centre is cat[o+R].  Pixels outside the image read 0 (never used: a
// kept pixel's window is inside the image, G3).
//
// Separable window maximum, the same ~9 instructions per pixel on any input (no data-dependent
// divergence): vertical max of the 2R+1 rows per column from registers (2 FMNMX3 per column for
// r = 2), the neighbouring lanes' column maxima by shuffle (2R SHFL per row), and the horizontal max
// with the threshold folded in:
//     m_k = max( max over the (2r+1)^2 window of pixel k ,  thr_up ),  thr_up = nextafter(thresh, +inf)
// so that   S > thresh  AND  S >= every window value   <=>   S == m_k   <=>   S - m_k = +0
// (S <= m_k always; the difference of two different finite floats is never 0; S + 0.0f folds -0 onto
// +0; needed only when thr_up <= 0, i.e. NEGT).  neg[k] collects, for pixel column k, the sign bit of
// S - m_k of output rows 0..TH-1 in bits TH-1..0 (one funnel shift per pixel): a 0 bit = candidate.
// The body is branch-free and fully unrolled.
template <int R, bool NEGT>
__device__ __forceinline__ void nms_rows(const float4 (&cat)[TH + 2 * R], float thr_up, unsigned (&neg)[4]) {
    constexpr int N = 2 * R + 1;
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(TH == 8, "8 rows per mask byte");
    neg[0] = neg[1] = neg[2] = neg[3] = 0u;
#pragma unroll
    for (int o = 0; o < TH; ++o) {
        float4 vm = cat[o];                                  // vertical max of the 2R+1 rows, per column
#pragma unroll
        for (int q = 1; q + 1 < N; q += 2) {
            vm.x = fmax3(vm.x, cat[o + q].x, cat[o + q + 1].x);
            vm.y = fmax3(vm.y, cat[o + q].y, cat[o + q + 1].y);
            vm.z = fmax3(vm.z, cat[o + q].z, cat[o + q + 1].z);
            vm.w = fmax3(vm.w, cat[o + q].w, cat[o + q + 1].w);
        }
        // neighbours' column maxima: l[j] = column X-1-j, rt[j] = column X+4+j
        float l[R], rt[R];
        {
            const float lv[4] = {vm.w, vm.z, vm.y, vm.x};    // sender's columns nearest the receiver first
            const float rv[4] = {vm.x, vm.y, vm.z, vm.w};
#pragma unroll
            for (int j = 0; j < R; ++j) {
                l[j] = __shfl_up_sync(FULL, lv[j], 1);
                rt[j] = __shfl_down_sync(FULL, rv[j], 1);
            }
        }
        // horizontal max with the threshold folded in
        float m0, m1, m2, m3;
        if constexpr (R == 1) {
            const float p = fmax3(vm.y, vm.z, thr_up);
            m0 = fmax3(l[0], vm.x, fmaxf(vm.y, thr_up));
            m1 = fmaxf(p, vm.x);
            m2 = fmaxf(p, vm.w);
            m3 = fmax3(vm.z, vm.w, fmaxf(rt[0], thr_up));
        } else if constexpr (R == 2) {
            const float p = fmax3(vm.y, vm.z, thr_up);       // {1,2,thr}
            const float q0 = fmax3(p, vm.x, l[0]);           // {-1..2,thr}
            const float q1 = fmax3(p, vm.w, rt[0]);          // {1..4,thr}
            m0 = fmaxf(q0, l[1]);                            // {-2..2}
            m1 = fmaxf(q0, vm.w);                            // {-1..3}
            m2 = fmaxf(q1, vm.x);                            // {0..4}
            m3 = fmaxf(q1, rt[1]);                           // {1..5}
        } else {
            // R >= 3: every window contains the lane's own 4 columns
            const float core = fmax3(fmax3(vm.x, vm.y, vm.z), vm.w, thr_up);
            float lp[R], rp[R];                              // lp[j] = max(l[0..j]), rp[j] = max(rt[0..j])
            lp[0] = l[0];
            rp[0] = rt[0];
#pragma unroll
            for (int j = 1; j < R; ++j) {
                lp[j] = fmaxf(lp[j - 1], l[j]);
                rp[j] = fmaxf(rp[j - 1], rt[j]);
            }
            // pixel k spans columns k-R .. k+R: left part l[0..R-k-1], right part rt[0..k+R-4]
            m0 = fmaxf(core, lp[R - 1]);
            m1 = fmax3(core, lp[R - 2], rp[R - 3]);
            m2 = fmax3(core, lp[R - 3], rp[R - 2]);
            m3 = fmaxf(core, rp[R - 1]);
            if constexpr (R == 4) m0 = fmaxf(m0, rp[0]), m3 = fmaxf(m3, lp[0]);
        }
        // S - m_k: +0 for a candidate, negative otherwise
        float4 c = cat[o + R];                               // centre row
        if constexpr (NEGT) c = make_float4(c.x + 0.0f, c.y + 0.0f, c.z + 0.0f, c.w + 0.0f);
        neg[0] = __funnelshift_l(__float_as_uint(c.x - m0), neg[0], 1);
        neg[1] = __funnelshift_l(__float_as_uint(c.y - m1), neg[1], 1);
        neg[2] = __funnelshift_l(__float_as_uint(c.z - m2), neg[2], 1);
        neg[3] = __funnelshift_l(__float_as_uint(c.w - m3), neg[3], 1);
    }
}

// ---- step a1': candidate masks of one strip-tile -> keys in its private segment --------------------
// Row validity (R <= y < H-R) and column validity (colmask, one bit per owned column that may emit)
// are applied here.  Candidates are rare (a few per strip-tile): every round, each lane that still
// holds one appends its next candidate at a ballot-ranked slot; the running count is warp-uniform
// (no atomics, no shared counter).  The score of a candidate is re-read from the box `rows` (output
// row o >= R has its centre in box row o - R) or, for the first R rows, from the rows still in
// registers.  Returns the segment's count.
template <int R, bool PROD>
__device__ __forceinline__ int nms_emit(const unsigned (&neg)[4], unsigned colmask, int X, int yc, int H, int W,
                                        const float4 (&cat)[TH + 2 * R], const float* __restrict__ rows,
                                        const float* __restrict__ rows2, uint64_t* __restrict__ seg, int seg_room,
                                        uint64_t keep) {
    constexpr unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    unsigned rowmask = 0xffu;                                // bit TH-1-o = output row o is valid
    if (yc < R || yc + TH > H - R) {                         // warp-uniform: first / last strip-tiles only
        int a = R - yc, b = H - R - yc;                      // valid output rows [a, b) clipped to [0, TH]
        a = a < 0 ? 0 : (a > TH ? TH : a);
        b = b < 0 ? 0 : (b > TH ? TH : b);
        rowmask = b > a ? ((1u << (TH - a)) - 1u) & ~((1u << (TH - b)) - 1u) : 0u;
    }
    unsigned w = 0u;                                         // bit 8k + (TH-1-o): pixel k of output row o is a candidate
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if ((colmask >> k) & 1u) w |= (~neg[k] & rowmask) << (8 * k);
    int cnt = 0;
    unsigned bal = __ballot_sync(FULL, w != 0u);
    while (bal) {                                            // warp-uniform; usually one round
        bool take = false;
        uint64_t key = 0ull;
        if (w != 0u) {
            const int bit = __ffs(w) - 1;
            w &= w - 1u;
            const int k = bit >> 3, o = TH - 1 - (bit & 7);
            const int idx = (yc + o) * W + X + k;
            take = true;                                     // (the validity mask, variant V5, is applied by k_select's gather)
            float v;
            if (o >= R) {
                DKD_ASSERT((o - R) * BOX_W + 4 * lane + k < BOX_W * TH);
                v = rows[(o - R) * BOX_W + 4 * lane + k];
                if constexpr (PROD) v = __fmul_rn(v, rows2[(o - R) * BOX_W + 4 * lane + k]);
            } else {
                float4 tr = cat[R];
#pragma unroll
                for (int j = 1; j < R; ++j)
                    if (o == j) tr = cat[R + j];
                v = k == 0 ? tr.x : (k == 1 ? tr.y : (k == 2 ? tr.z : tr.w));
            }
            key = make_key(v, idx);
        }
        const unsigned tb = __ballot_sync(FULL, take);
        if (take) {
            DKD_ASSERT(cnt + __popc(tb & ((1u << lane) - 1u)) < seg_room);
            st_keep_u64(seg + cnt + __popc(tb & ((1u << lane) - 1u)), key, keep);
        }
        cnt += __popc(tb);
        bal = __ballot_sync(FULL, w != 0u);
    }
    (void)seg_room;
    return cnt;
}

__device__ __forceinline__ unsigned strip_colmask(int X, int W, int R) {
    const int lane = threadIdx.x & 31;
    unsigned colmask = 0;                                    // output columns this lane may emit
    if (lane >= 1 && lane <= 30) {
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (X + k >= R && X + k < W - R) colmask |= 1u << k;
    }
    return colmask;
}

// ---- work decomposition (host: nms_plan) -----------------------------------------------------------
// unit u = (b * segs + sg) * strips_x + sx  covers strip-tiles cy = sg*cpu .. min(sg*cpu + cpu, chunks_y) - 1 of
// strip sx; its candidates go to segment u of `cand` (capacity cpu * SEG_CAP keys), their number to seg_cnt[u].
struct NmsPlan {
    int H, W;
    int strips_x, chunks_y;  // strip-tiles per image row / column
    int cpu, segs;           // strip-tiles per unit, units per strip
    int units;               // strips_x * segs * B
    float thr_up;            // nextafter(thresh, +inf)
};
struct UnitCoords {
    int b, x0, y0, nch;      // image, first output column / row, strip-tiles in the unit
};
__device__ __forceinline__ UnitCoords unit_coords(int u, const NmsPlan& p) {
    const int upi = p.strips_x * p.segs;
    UnitCoords c;
    c.b = u / upi;
    const int rem = u - c.b * upi;
    const int sg = rem / p.strips_x, sx = rem - sg * p.strips_x;
    c.x0 = sx * STRIP_W;
    c.y0 = sg * p.cpu * TH;
    c.nch = p.chunks_y - sg * p.cpu < p.cpu ? p.chunks_y - sg * p.cpu : p.cpu;
    return c;
}

// the 2R rows above a unit (image rows y0-R .. y0+R-1), one float4 per lane and row, straight from
// global memory (once per unit; mostly L2 hits: the unit above has just streamed them); 0 outside the image
__device__ __forceinline__ float4 mul4_rn(const float4 a, const float4 b) {   // heat x reliability, one rounding each
    return make_float4(__fmul_rn(a.x, b.x), __fmul_rn(a.y, b.y), __fmul_rn(a.z, b.z), __fmul_rn(a.w, b.w));
}
template <int R, bool PROD>
__device__ __forceinline__ void load_head(float4 (&cat)[TH + 2 * R], const float* __restrict__ img,
                                          const float* __restrict__ img2, int X, int y0, int H, int W) {
#pragma unroll
    for (int q = 0; q < 2 * R; ++q) {
        const int y = y0 - R + q;
        cat[q] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (y >= 0 && y < H && X >= 0 && X < W) {            // W % 4 == 0 and X % 4 == 0: all four or none
            cat[q] = __ldg(reinterpret_cast<const float4*>(img + static_cast<size_t>(y) * W + X));
            if constexpr (PROD)
                cat[q] = mul4_rn(cat[q], __ldg(reinterpret_cast<const float4*>(img2 + static_cast<size_t>(y) * W + X)));
        }
    }
}

// ---- k_nms_tma: persistent; every warp runs its own TMA/mbarrier pipeline ---------------------------
// grid = min(ceil(units / warps), CTAs that fit); warp g handles units g, g + G, ... (image-major,
// segment-major, strips fastest: neighbouring warps load neighbouring boxes, so the 4 halo columns hit L2).
// Per strip-tile one TMA box of TH rows (image rows yc+R .. yc+R+TH-1, the newest rows its outputs
// need) through a NMS_STAGES-deep ring: while a warp works on one box (8 LDS.128 into registers, the
// arithmetic, the candidate scores picked out of the box), its other NMS_STAGES-1 boxes stay in flight.
// No CTA-wide barrier after set-up: a warp only ever waits for its own boxes.  Dynamic smem:
// NMS_SMEM_BYTES, 128-byte aligned; warp w owns NMS_STAGES boxes.  NEGT: thr_up <= 0 (see nms_rows).
template <int R, bool NEGT, bool PROD>
__global__ void __launch_bounds__(NMS_WARPS * 32, PROD ? 1 : NMS_CTAS) k_nms_tma(const __grid_constant__ CUtensorMap tmap,
                                                                          const __grid_constant__ CUtensorMap tmap2,
                                                                          const __grid_constant__ NmsPlan p,
                                                                          const float* __restrict__ score,
                                                                          const float* __restrict__ score2,
                                                                          uint64_t* __restrict__ cand,
                                                                          int* __restrict__ seg_cnt) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bars[NMS_WARPS * NMS_STAGES];
    constexpr int STAGE_BYTES = PROD ? 2 * BOX_BYTES : BOX_BYTES;      // PROD: heat box | reliability box
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int first = blockIdx.x * NMS_WARPS + warp, step = gridDim.x * NMS_WARPS;
    const int n_my = first < p.units ? (p.units - first + step - 1) / step : 0;
    pdl_launch_dependents();                                 // k_select may fill the SMs this grid leaves
    if (n_my == 0) return;
    unsigned char* my_smem = smem_raw + warp * NMS_STAGES * STAGE_BYTES;
    uint64_t* bar = bars + warp * NMS_STAGES;

    const uint64_t policy = l2_evict_first_policy();
    const uint64_t keep = l2_evict_last_policy();
    // issue side (every lane tracks the cursor, lane 0 issues): next box = chunk ic of unit iteration iit
    int iit = 0, ic = 0, issued = 0;
    UnitCoords iu = unit_coords(first, p);
    auto issue_box = [&]() {
        if (iit >= n_my) return;
        const int s = issued % NMS_STAGES;
        if (elect_one()) {                                   // (the warp is converged here: one elected lane issues)
            mbar_arrive_expect_tx(&bar[s], STAGE_BYTES);
            tma_load_tile(my_smem + s * STAGE_BYTES, &tmap, &bar[s], iu.x0 - HALO_X, iu.y0 + R + TH * ic, iu.b, policy);
            if constexpr (PROD)
                tma_load_tile(my_smem + s * STAGE_BYTES + BOX_BYTES, &tmap2, &bar[s], iu.x0 - HALO_X, iu.y0 + R + TH * ic,
                              iu.b, policy);
        }
        ++issued;
        if (++ic == iu.nch) {
            ic = 0;
            if (++iit < n_my) iu = unit_coords(first + iit * step, p);
        }
    };

    UnitCoords cu = iu;
    if (lane == 0) {
        tma_prefetch_desc(&tmap);
        if constexpr (PROD) tma_prefetch_desc(&tmap2);
#pragma unroll
        for (int s = 0; s < NMS_STAGES; ++s) mbar_init(&bar[s], 1);
        fence_mbar_init();
    }
    __syncwarp();
    // Launched with the programmatic attribute, this grid may have started while the previous kernel of the stream (the
    // previous call's k_refine_gather, or whatever produced the score map) was still running: everything above is
    // set-up; nothing is read from or written to global memory before the predecessor has completed.
    pdl_wait();
#pragma unroll
    for (int s = 0; s < NMS_STAGES; ++s) issue_box();

    int consumed = 0;
    const size_t img_px = static_cast<size_t>(p.H) * p.W;
    for (int it = 0; it < n_my; ++it) {
        const int X = cu.x0 - HALO_X + 4 * lane;             // image column of this lane's first pixel
        float4 cat[TH + 2 * R];                              // rows yc-R .. yc+R+TH-1 of the current strip-tile
        load_head<R, PROD>(cat, score + cu.b * img_px, PROD ? score2 + cu.b * img_px : nullptr, X, cu.y0, p.H, p.W);
        const unsigned colmask = strip_colmask(X, p.W, R);
        const int u = first + it * step;                     // the unit's candidate segment: p.cpu * SEG_CAP keys
        DKD_ASSERT(u >= 0 && u < p.units);
        uint64_t* useg = cand + static_cast<size_t>(u) * (p.cpu * SEG_CAP);
        int ucnt = 0;                                        // warp-uniform running count of the segment
        for (int c = 0; c < cu.nch; ++c) {
            const int s = consumed % NMS_STAGES;
            DKD_ASSERT(consumed < issued && issued - consumed <= NMS_STAGES);
            mbar_wait(&bar[s], (consumed / NMS_STAGES) & 1);
            const float* rows = reinterpret_cast<const float*>(my_smem + s * STAGE_BYTES);
            const float* rows2 = PROD ? rows + BOX_W * TH : nullptr;
            {
                const float4* src = reinterpret_cast<const float4*>(rows) + lane;
#pragma unroll
                for (int o = 0; o < TH; ++o) {
                    cat[2 * R + o] = src[o * 32];
                    if constexpr (PROD) cat[2 * R + o] = mul4_rn(cat[2 * R + o], src[BOX_W * TH / 4 + o * 32]);
                }
            }
            unsigned neg[4];
            nms_rows<R, NEGT>(cat, p.thr_up, neg);
            ucnt += nms_emit<R, PROD>(neg, colmask, X, cu.y0 + TH * c, p.H, p.W, cat, rows, rows2, useg + ucnt,
                                      p.cpu * SEG_CAP - ucnt, keep);
            __syncwarp();                                    // every lane is done with stage s
            issue_box();                                     // (the other NMS_STAGES-1 boxes stay in flight meanwhile)
            ++consumed;
#pragma unroll
            for (int q = 0; q < 2 * R; ++q) cat[q] = cat[TH + q];   // the 2R rows above the next strip-tile
        }
        if (lane == 0) st_keep_s32(seg_cnt + u, ucnt, keep);
        if (it + 1 < n_my) cu = unit_coords(first + (it + 1) * step, p);
    }
}

// ---- k_nms_plain: same strip math, one strip-tile per warp, rows fetched with ordinary loads ---------
// (any W, any alignment: scalar loads, 0 outside the image)
constexpr int PLAIN_WARPS = 4;
template <int R, bool PROD>
__global__ void __launch_bounds__(PLAIN_WARPS * 32) k_nms_plain(const float* __restrict__ score,
                                                                const float* __restrict__ score2,
                                                                const __grid_constant__ NmsPlan p, int total,
                                                                uint64_t* __restrict__ cand,
                                                                int* __restrict__ seg_cnt) {
    __shared__ __align__(16) float boxes[PLAIN_WARPS][BOX_W * TH];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int t = blockIdx.x * PLAIN_WARPS + warp;          // unit == strip-tile (nms_plan: cpu = 1 on this path)
    pdl_launch_dependents();
    if (t >= total) return;
    pdl_wait();                                              // (see k_nms_tma)
    const int tpi = p.strips_x * p.chunks_y;
    const int b = t / tpi, rem = t - b * tpi;
    const int cy = rem / p.strips_x, x0 = (rem - cy * p.strips_x) * STRIP_W, y0 = cy * TH;
    const size_t img_px = static_cast<size_t>(p.H) * p.W;
    const float* img = score + b * img_px;
    const float* img2 = PROD ? score2 + b * img_px : nullptr;
    const int X = x0 - HALO_X + 4 * lane;
    float4 cat[TH + 2 * R];
#pragma unroll
    for (int q = 0; q < TH + 2 * R; ++q) {
        const int gy = y0 - R + q;
        float v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            v[k] = 0.0f;
            if (gy >= 0 && gy < p.H && X + k >= 0 && X + k < p.W) {
                const size_t e = static_cast<size_t>(gy) * p.W + X + k;
                v[k] = __ldg(img + e);
                if constexpr (PROD) v[k] = __fmul_rn(v[k], __ldg(img2 + e));
            }
        }
        cat[q] = make_float4(v[0], v[1], v[2], v[3]);
    }
    float4* box = reinterpret_cast<float4*>(boxes[warp]) + lane;   // (already the product: emit reads it as is)
#pragma unroll
    for (int o = 0; o < TH; ++o) box[o * 32] = cat[2 * R + o];
    __syncwarp();
    unsigned neg[4];
    nms_rows<R, true>(cat, p.thr_up, neg);
    const int cnt = nms_emit<R, false>(neg, strip_colmask(X, p.W, R), X, y0, p.H, p.W, cat, boxes[warp], nullptr,
                                       cand + static_cast<size_t>(t) * SEG_CAP, SEG_CAP, l2_evict_last_policy());
    if (lane == 0) seg_cnt[t] = cnt;
}

// ---- k_nms_iter: the iterated suppress-and-recover NMS variant (V1) -----------------------
//   M = (S == maxpool(S));  repeat n times:  supp = maxpool(M) > 0;  S' = supp ? 0 : S;  M |= (S' == maxpool(S')) & !supp
// with (2r+1)^2 windows clipped at the image edge.  The mask at a pixel depends on S within (2n+1) r pixels, so a CTA
// loads an IT_REG x IT_REG region (out-of-image pixels = -inf) into shared memory, runs every pooling stage on the
// whole region as a separable row / column pass (values near the region's edge are wrong, but no output of the inner
// T x T tile, T = IT_REG - 2 (2n+1) r, depends on them), applies border / threshold / validity mask to the tile and
// appends its candidates to the tile's private segment (block scan, no atomics) for k_select.
// Every pass works on GROUPS of 4 horizontally adjacent pixels: one float4 (scores) or one 32-bit word of four 0/1 bytes
// (masks) per shared-memory access.  A row pass reads the group and its two neighbours (r <= 4: the window never
// reaches further) and slides the window over the 12 values in registers; a column pass reads the 2r+1 groups above /
// below (rows clamped into the region: a repeated row does not change a maximum or an OR).  The radius is a template
// parameter, so all window loops are unrolled.  32 warps per CTA hide the shared-memory latency between the passes.
constexpr int IT_REG = 96;
constexpr int IT_G = IT_REG / 4;                             // pixel groups per region row
constexpr int IT_THREADS = 768;
constexpr int IT_SMEM_BYTES = IT_REG * IT_REG * (2 * 4 + 3); // S, tmp (fp32); M, tb, sup (bytes): 99 KB -> two CTAs per SM,
                                                             // one loads its region while the other runs its passes
static_assert(IT_REG % 8 == 0 && MAX_R <= 4, "pixel groups of 4: a window may reach one group to either side");
static_assert((IT_REG * IT_REG / 4) % IT_THREADS == 0, "every thread owns the same number of pixel groups");
struct IterParams {
    const float* score;
    const float* score2;
    const uint8_t* mask;
    int H, W, r, iters, T, halo, halo_x, tiles_x, tiles_y;   // halo_x = halo rounded up to 4: pixel groups are 4-aligned in the image
    int vec;                                                 // W % 4 == 0 and 16-byte aligned maps: 16-byte global loads
    float thresh;
    uint64_t* cand;
    int* seg_cnt;
};
__device__ __forceinline__ float4 it_max4(const float4& a, const float4& b) {
    return make_float4(fmaxf(a.x, b.x), fmaxf(a.y, b.y), fmaxf(a.z, b.z), fmaxf(a.w, b.w));
}
// the four bytes that start D bytes after the start of word c in the byte sequence (l, c, rr); D in [-4, 4]
template <int D>
__device__ __forceinline__ uint32_t it_shift_bytes(uint32_t l, uint32_t c, uint32_t rr) {
    if constexpr (D == 0) return c;
    else if constexpr (D == -4) return l;
    else if constexpr (D == 4) return rr;
    else if constexpr (D < 0) return __funnelshift_r(l, c, 8 * (4 + D));
    else return __funnelshift_r(c, rr, 8 * D);
}
template <int R, int D = -R>
__device__ __forceinline__ uint32_t it_dilate_row(uint32_t l, uint32_t c, uint32_t rr) {
    if constexpr (D > R) return 0u;
    else return it_shift_bytes<D>(l, c, rr) | it_dilate_row<R, D + 1>(l, c, rr);
}
// S' = supp ? 0 : S of a pixel group (out-of-image pixels stay -inf); sm = the group's four suppression bytes
__device__ __forceinline__ float4 it_suppressed(const float4& v, uint32_t sm) {
    return make_float4(v.x == -INFINITY ? v.x : ((sm & 0xFFu) ? 0.0f : v.x), v.y == -INFINITY ? v.y : ((sm & 0xFF00u) ? 0.0f : v.y),
                       v.z == -INFINITY ? v.z : ((sm & 0xFF0000u) ? 0.0f : v.z), v.w == -INFINITY ? v.w : ((sm & 0xFF000000u) ? 0.0f : v.w));
}
template <int R>
__global__ void __launch_bounds__(IT_THREADS, 2) k_nms_iter(const __grid_constant__ IterParams p) {
    extern __shared__ __align__(16) unsigned char it_smem[];
    constexpr int NPX = IT_REG * IT_REG, NG = NPX / 4;
    float* S = reinterpret_cast<float*>(it_smem);
    float* tmp = S + NPX;
    uint8_t* M = reinterpret_cast<uint8_t*>(tmp + NPX);
    uint8_t* tb = M + NPX;
    uint8_t* sup = tb + NPX;
    float4* S4 = reinterpret_cast<float4*>(S);
    float4* tmp4 = reinterpret_cast<float4*>(tmp);
    uint32_t* M32 = reinterpret_cast<uint32_t*>(M);
    uint32_t* tb32 = reinterpret_cast<uint32_t*>(tb);
    uint32_t* sup32 = reinterpret_cast<uint32_t*>(sup);
    __shared__ int s_scan[IT_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx = blockIdx.x % p.tiles_x, ty = blockIdx.x / p.tiles_x, b = blockIdx.y;
    const int x0 = tx * p.T - p.halo_x, y0 = ty * p.T - p.halo;   // image coordinates of the region's origin (x0 % 4 == 0)
    const size_t img_px = static_cast<size_t>(p.H) * p.W;
    const float* img = p.score + b * img_px;
    const float* img2 = p.score2 ? p.score2 + b * img_px : nullptr;
    DKD_ASSERT(p.r == R && (x0 & 3) == 0);
    pdl_launch_dependents();
    pdl_wait();                                              // (see k_nms_tma)
    const float4 ninf4 = make_float4(-INFINITY, -INFINITY, -INFINITY, -INFINITY);
#pragma unroll
    for (int g = tid; g < NG; g += IT_THREADS) {
        const int ry = g / IT_G, gy = y0 + ry, gx = x0 + 4 * (g - ry * IT_G);
        float4 v = ninf4;
        if (gy >= 0 && gy < p.H && gx + 3 >= 0 && gx < p.W) {
            const size_t e = static_cast<size_t>(gy) * p.W + gx;     // (not formed as a pointer unless in range)
            if (p.vec) {                                     // W % 4 == 0 and gx % 4 == 0: the group is inside the row
                v = __ldg(reinterpret_cast<const float4*>(img + e));
                if (img2) {
                    const float4 q = __ldg(reinterpret_cast<const float4*>(img2 + e));
                    v = make_float4(__fmul_rn(v.x, q.x), __fmul_rn(v.y, q.y), __fmul_rn(v.z, q.z), __fmul_rn(v.w, q.w));
                }
            } else {
                float t[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    t[j] = -INFINITY;
                    if (gx + j >= 0 && gx + j < p.W) {
                        t[j] = __ldg(img + e + j);
                        if (img2) t[j] = __fmul_rn(t[j], __ldg(img2 + e + j));
                    }
                }
                v = make_float4(t[0], t[1], t[2], t[3]);
            }
        }
        S4[g] = v;
    }
    __syncthreads();
    // separable window maximum over the region: the row pass of S (SUPP = false) or of S' = supp ? 0 : S, formed on the
    // fly from S and the suppression bytes (SUPP = true), into tmp; the column pass is folded into its user
    auto row_max = [&](auto supp_tag) {
        constexpr bool SUPP = decltype(supp_tag)::value;
        for (int g = tid; g < NG; g += IT_THREADS) {
            const int gx = g % IT_G;
            float4 c = S4[g];
            float4 l = gx > 0 ? S4[g - 1] : ninf4;
            float4 rr = gx < IT_G - 1 ? S4[g + 1] : ninf4;
            if constexpr (SUPP) {
                c = it_suppressed(c, sup32[g]);
                if (gx > 0) l = it_suppressed(l, sup32[g - 1]);
                if (gx < IT_G - 1) rr = it_suppressed(rr, sup32[g + 1]);
            }
            const float w[12] = {l.x, l.y, l.z, l.w, c.x, c.y, c.z, c.w, rr.x, rr.y, rr.z, rr.w};
            float o[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float m = w[4 + j - R];
#pragma unroll
                for (int d = -R + 1; d <= R; ++d) m = fmaxf(m, w[4 + j + d]);
                o[j] = m;
            }
            tmp4[g] = make_float4(o[0], o[1], o[2], o[3]);
        }
    };
    auto col_max4 = [&](int ry, int gx) {
        float4 m = tmp4[max(ry - R, 0) * IT_G + gx];
#pragma unroll
        for (int d = -R + 1; d <= R; ++d) m = it_max4(m, tmp4[min(max(ry + d, 0), IT_REG - 1) * IT_G + gx]);
        return m;
    };
    // bytes (0 / 1) of the pixels of `v` that are in the image and equal their window maximum `m`
    auto maxima4 = [](const float4& v, const float4& m) {
        return (v.x != -INFINITY && v.x == m.x ? 0x1u : 0u) | (v.y != -INFINITY && v.y == m.y ? 0x100u : 0u) |
               (v.z != -INFINITY && v.z == m.z ? 0x10000u : 0u) | (v.w != -INFINITY && v.w == m.w ? 0x1000000u : 0u);
    };
    row_max(std::false_type{});
    __syncthreads();
    for (int g = tid; g < NG; g += IT_THREADS) {
        const int ry = g / IT_G, gx = g - ry * IT_G;
        M32[g] = maxima4(S4[g], col_max4(ry, gx));               // out-of-image pixels are never maxima
    }
    __syncthreads();
    for (int it = 0; it < p.iters; ++it) {
        for (int g = tid; g < NG; g += IT_THREADS) {             // supp = dilate(M): row pass
            const int gx = g % IT_G;
            tb32[g] = it_dilate_row<R>(gx > 0 ? M32[g - 1] : 0u, M32[g], gx < IT_G - 1 ? M32[g + 1] : 0u);
        }
        __syncthreads();
        for (int g = tid; g < NG; g += IT_THREADS) {             // column pass
            const int ry = g / IT_G, gx = g - ry * IT_G;
            uint32_t m = 0;
#pragma unroll
            for (int d = -R; d <= R; ++d) m |= tb32[min(max(ry + d, 0), IT_REG - 1) * IT_G + gx];
            sup32[g] = m;
        }
        __syncthreads();
        row_max(std::true_type{});
        __syncthreads();
        for (int g = tid; g < NG; g += IT_THREADS) {             // recover: maxima of S' outside the suppression mask
            const int ry = g / IT_G, gx = g - ry * IT_G;
            const uint32_t sm = sup32[g];
            if (sm == 0x01010101u) continue;                     // every pixel of the group is suppressed
            const uint32_t rec = maxima4(it_suppressed(S4[g], sm), col_max4(ry, gx)) & ~sm;
            if (rec) M32[g] |= rec;
        }
        __syncthreads();
    }
    // the inner T x T tile: border exclusion, strict threshold, validity mask -> keys, compacted in pixel order.  The tile
    // starts on a group boundary (halo_x % 4 == 0, T % 8 == 0): it is walked group by group, and a group whose four mask
    // bytes are zero (almost all of them) costs one shared-memory load.
    const int tile_px = p.T * p.T, gpr = p.T >> 2, tile_g = p.T * gpr;
    const uint8_t* vm = p.mask ? p.mask + b * img_px : nullptr;
    // candidates of tile group t (in pixel order): calls emit(v, idx) for each, returns their number
    auto group_cands = [&](int t, auto&& emit) {
        const int ly = t / gpr, lg = t - ly * gpr;
        const int ri = (ly + p.halo) * IT_G + (p.halo_x >> 2) + lg;
        const uint32_t mw = M32[ri];
        if (mw == 0u) return 0;
        const int gy = ty * p.T + ly;
        if (gy < R || gy >= p.H - R) return 0;
        const float4 v4 = S4[ri];
        const float v[4] = {v4.x, v4.y, v4.z, v4.w};
        int n = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int gx = tx * p.T + 4 * lg + j;
            if (!((mw >> (8 * j)) & 0xFFu) || gx < R || gx >= p.W - R || !(v[j] > p.thresh)) continue;
            const int idx = gy * p.W + gx;
            if (vm != nullptr && __ldg(vm + idx) == 0) continue;
            emit(v[j], idx);
            ++n;
        }
        return n;
    };
    // each thread owns a contiguous run of the tile's groups, so the segment is filled in pixel order
    const int per = (tile_g + IT_THREADS - 1) / IT_THREADS;
    const int t_lo = min(tid * per, tile_g), t_hi = min(t_lo + per, tile_g);
    int mine = 0;
    for (int t = t_lo; t < t_hi; ++t) mine += group_cands(t, [](float, int) {});
    int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += up;
    }
    if (lane == 31) s_scan[warp] = incl;
    __syncthreads();
    int base = 0;
    for (int w = 0; w < warp; ++w) base += s_scan[w];
    int pos = base + incl - mine;
    const int seg_id = (b * p.tiles_y + ty) * p.tiles_x + tx;
    uint64_t* seg = p.cand + static_cast<size_t>(seg_id) * tile_px;
    if (mine > 0)
        for (int t = t_lo; t < t_hi; ++t)
            group_cands(t, [&](float v, int idx) { DKD_ASSERT(pos < tile_px); seg[pos++] = make_key(v, idx); });
    if (tid == IT_THREADS - 1) p.seg_cnt[seg_id] = base + incl;
}

// ---- k_select: per-image top-k select + order ---------------------------------------------------
// One CTA per image.  n = sum of the image's strip-tile counts.
//   gather        : every key (n = sum of the image's strip-tile counts) is copied into shared memory.
//   n >  SORT_CAP : (rare) MSB-first radix select (8-bit digits, warp-aggregated shared-memory histogram)
//                   narrows to a lower bound `lo` with  top_k <= #{key >= lo} <= SORT_CAP; gather again,
//                   keys >= lo only.
//   order         : bucket rank (the common case) — one pass of a monotone bucket function over the
//                   score bits (NB buckets spanning [min, max] of the gathered scores; the keys tied at the
//                   maximum score get NBT buckets over their pixel index instead), an exclusive
//                   scan of the bucket counts, a scatter into bucket order, and an exact rank
//                   = keys in better buckets + keys of the own bucket with a larger key.  ~100
//                   lane-instructions per key instead of the ~550 of a 64-bit bitonic network.
//                   Falls back to the in-smem bitonic sort when one bucket holds more than
//                   BUCKET_LIMIT keys (near-constant maps).
// Keys are unique (they embed the pixel index) so the result is the unique (score desc, idx asc) order.
constexpr int NB = 4096;                 // score buckets of the rank pass
constexpr int NBT = 1024;                // index buckets for the keys tied at the maximum score (see k_select)
constexpr int NBK = NBT + NB;
constexpr int BUCKET_LIMIT = 1024;       // largest bucket the rank pass accepts
constexpr int SEL_SMEM_BYTES = 2 * SORT_CAP * 8 + 2 * NBK * 4;    // keys | sorted | base | cur = 168 KB

__device__ __forceinline__ int block_sum_1024(int v, int* s_red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    int r = s_red[lane];                                    // SEL_THREADS / 32 == 32 partials
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    __syncthreads();
    return r;
}

// The refinement that follows reads the (2r+1)^2 window of every kept keypoint: k_select, which knows the kept
// indices first and has bandwidth to spare, asks L2 for those rows (first and last element of each window row:
// one or two sectors), so that k_refine_gather's dependent window loads hit L2 instead of paying a DRAM round trip.
struct SelExtra {
    const uint8_t* vmask;               // validity mask [B,H,W] (variant V5) or NULL: keys on masked pixels are dropped in the gather
    const float* score;                 // NULL: no prefetch
    const float* score2;                // reliability map (product variant) or NULL
    int W, r;
    uint32_t div_m, div_s1, div_s2;     // idx / W (FastDiv)
    size_t img_px;
};
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_window(const SelExtra& pf, int b, int idx) {
    if (pf.score == nullptr) return;
    const uint32_t t = __umulhi(pf.div_m, static_cast<uint32_t>(idx));
    const int y = static_cast<int>((t + ((static_cast<uint32_t>(idx) - t) >> pf.div_s1)) >> pf.div_s2), x = idx - y * pf.W;
    const float* row = pf.score + b * pf.img_px + static_cast<size_t>(y - pf.r) * pf.W + (x - pf.r);
    for (int j = 0; j <= 2 * pf.r; ++j, row += pf.W) {
        prefetch_l2(row);
        prefetch_l2(row + 2 * pf.r);
    }
    if (pf.score2 != nullptr) {
        row = pf.score2 + b * pf.img_px + static_cast<size_t>(y - pf.r) * pf.W + (x - pf.r);
        for (int j = 0; j <= 2 * pf.r; ++j, row += pf.W) {
            prefetch_l2(row);
            prefetch_l2(row + 2 * pf.r);
        }
    }
}

// MSB-first 8-bit radix select over the candidate segments of one image (only when more than SORT_CAP keys were found):
// returns a prefix `lo` with top_k <= #{key >= lo} <= SORT_CAP.  Kept OUT OF LINE: k_select runs once per launch with
// cold instruction caches, so its common path must not jump across kilobytes of code it never executes.
__device__ __noinline__ uint64_t select_radix_prefix(const uint64_t* __restrict__ seg0, const int* __restrict__ cnt, int tpi,
                                                     int seg_cap, const uint8_t* __restrict__ vm, int top_k, int* s_hist,
                                                     int* s_rdx) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = SEL_THREADS / 32;
    constexpr unsigned FULL = 0xffffffffu;
    int& s_digit = s_rdx[0];
    int& s_cum = s_rdx[1];
    int& s_h = s_rdx[2];
    uint64_t prefix = 0;
    int need = top_k;                                   // rank (1-based, from the top) inside the prefix bucket
    int above = 0;                                      // keys strictly above the prefix bucket
    for (int shift = 56; shift >= 0; shift -= 8) {
        for (int i = tid; i < 257; i += SEL_THREADS) s_hist[i] = 0;
        __syncthreads();
        for (int t = warp; t < tpi; t += NW) {
            const int c = cnt[t];
            const uint64_t* seg = seg0 + static_cast<size_t>(t) * seg_cap;
            for (int e0 = 0; e0 < c; e0 += 32) {
                const int e = e0 + lane;
                int digit = 256;                        // dummy bin: past the end / outside the prefix
                if (e < c) {
                    const uint64_t k = seg[e];
                    bool match = (shift == 56) || ((k >> (shift + 8)) == (prefix >> (shift + 8)));
                    if (match && vm != nullptr) match = __ldg(vm + key_index(k)) != 0;
                    if (match) digit = static_cast<int>((k >> shift) & 255u);
                }
                const unsigned peers = __match_any_sync(FULL, digit);
                if (lane == __ffs(peers) - 1) atomicAdd(&s_hist[digit], __popc(peers));
            }
        }
        __syncthreads();
        if (warp == 0) {                                // find the digit holding the need-th largest key
            int grp = 0;                                // lane l owns bins 255-8l .. 248-8l (descending)
#pragma unroll
            for (int q = 0; q < 8; ++q) grp += s_hist[255 - 8 * lane - q];
            int incl = grp;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int up = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += up;
            }
            const unsigned hit = __ballot_sync(FULL, incl >= need);
            const int owner = __ffs(hit) - 1;           // exists: need <= keys in the bucket
            if (lane == owner) {
                int cum = incl - grp;
                int d = 255 - 8 * lane;
                for (int q = 0; q < 8; ++q, --d) {
                    const int h = s_hist[d];
                    if (cum + h >= need) break;
                    cum += h;
                }
                s_digit = d;
                s_cum = cum;
                s_h = s_hist[d];
            }
        }
        __syncthreads();
        prefix |= static_cast<uint64_t>(s_digit) << shift;
        above += s_cum;
        need -= s_cum;
        const bool done = (above + s_h <= SORT_CAP);
        __syncthreads();
        if (done) break;
    }
    return prefix;
}

__global__ void __launch_bounds__(SEL_THREADS, 1) k_select(const uint64_t* __restrict__ cand,
                                                           const int* __restrict__ seg_cnt, int tpi, int seg_cap,
                                                           int top_k, int idx_shift, const SelExtra pf,
                                                           int32_t* __restrict__ sel_idx,
                                                           int32_t* __restrict__ out_count,
                                                           int32_t* __restrict__ out_total) {
    extern __shared__ __align__(16) unsigned char sel_smem[];
    uint64_t* keys = reinterpret_cast<uint64_t*>(sel_smem);            // SORT_CAP entries (gathered, unordered)
    uint64_t* sorted = keys + SORT_CAP;                                // SORT_CAP entries (bucket order)
    int* base = reinterpret_cast<int*>(sorted + SORT_CAP);             // NBK
    int* cur = base + NBK;                                             // NBK
    __shared__ int s_hist[257];
    __shared__ int s_red[32];
    __shared__ int s_n, s_maxb, s_meff, s_rdx[3];
    __shared__ unsigned s_hi, s_lo;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = SEL_THREADS / 32;
    constexpr unsigned FULL = 0xffffffffu;
    const int b = blockIdx.x;
    const int* cnt = seg_cnt + static_cast<size_t>(b) * tpi;             // tpi segments of seg_cap keys per image
    const uint8_t* vm = pf.vmask ? pf.vmask + b * pf.img_px : nullptr;
    const uint64_t* seg0 = cand + static_cast<size_t>(b) * tpi * seg_cap;

    pdl_launch_dependents();
    if (tid == 0) { s_n = 0; s_hi = 0u; s_lo = 0xffffffffu; s_maxb = 0; }
    for (int i = tid; i < NBK; i += SEL_THREADS) cur[i] = 0;

    // Gather layout: LPS = 1, 2, 4 or 8 lanes share one segment (lane sub of a segment copies its items sub, sub + LPS,
    // ...), so a warp iteration covers 32 / LPS segments: an item's position in the concatenation is its segment's
    // exclusive offset (one warp scan of the counts) plus its index — no search.  LPS grows with the unit length (longer
    // units hold more keys per segment) as long as one pass of the CTA still covers about all the segments.
    int lps_log = 0;
    while (lps_log < 3 && (SEG_CAP << lps_log) < seg_cap && (tpi << (lps_log + 1)) <= SEL_THREADS) ++lps_log;
    const int lps = 1 << lps_log, spw = 32 >> lps_log;      // lanes per segment, segments per warp iteration
    const int sub = lane & (lps - 1), sl = lane >> lps_log;
    uint64_t lo = 0;                                        // gather keys >= lo (0: all of them)
    pdl_wait();                                              // the candidates of k_nms_* are complete and visible
    __syncthreads();
    // With a validity mask (V5) the keys are first STAGED in `sorted` by the fast copy and then filtered densely, every
    // thread testing one key (one mask byte each, all in flight); only if more than SORT_CAP keys turn up is the first
    // pass repeated with the per-lane filter, which counts without storing.
    bool stage = vm != nullptr;
    for (int pass = 0; pass < 2; ++pass) {                  // second pass only if the first found n > SORT_CAP
        const bool copy_all = lo == 0 && (vm == nullptr || stage);
        uint64_t* const dst = stage ? sorted : keys;
        unsigned khi = 0u, klo = 0xffffffffu;                   // range of the gathered score words
        int c_next = (warp * spw + sl < tpi) ? cnt[warp * spw + sl] : 0;
        for (int t0 = warp * spw; t0 < tpi; t0 += NW * spw) {
            const int t = t0 + sl;
            const int c = c_next;                               // (the next iteration's counts are already on their way)
            c_next = (t + NW * spw < tpi) ? cnt[t + NW * spw] : 0;
            int incl = sub == 0 ? c : 0;
    #pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int up = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += up;
            }
            const int total = __shfl_sync(FULL, incl, 31);
            if (total == 0) continue;                           // warp-uniform
            const int excl = incl - c;                          // items of the warp's earlier segments
            int gbase = 0;
            if (copy_all) {                                     // all keys are kept: reserve the slots at once
                if (lane == 0) gbase = atomicAdd(&s_n, total);
                gbase = __shfl_sync(FULL, gbase, 0);
                if (gbase + total > SORT_CAP) continue;         // too many candidates (rare): counted, radix select below
            }
            // One SM turns around roughly one scattered load request every 4 cycles, and with a few keys in each of
            // hundreds of segments every request counts: a lane fetches its keys as 16-byte PAIRS (2q, 2q+1) — the
            // segments are 32-byte aligned — and the LPS lanes of a segment read consecutive pairs (one sector per two lanes).
            constexpr int GU = 4;                               // pair loads in flight per lane
            const ulonglong2* seg = reinterpret_cast<const ulonglong2*>(seg0 + static_cast<size_t>(t < tpi ? t : 0) * seg_cap);
            const int cmax = __reduce_max_sync(FULL, c);
            for (int i0 = 0; i0 < cmax; i0 += 2 * lps * GU) {
                uint64_t kk[2 * GU];
#pragma unroll
                for (int u = 0; u < GU; ++u) {
                    const int i = i0 + 2 * (sub + (u << lps_log));  // first key of the pair
                    DKD_ASSERT(i >= c || i + 1 < seg_cap);
                    ulonglong2 q = make_ulonglong2(0ull, 0ull);
                    if (i < c) q = __ldg(seg + (i >> 1));
                    kk[2 * u] = q.x;
                    kk[2 * u + 1] = i + 1 < c ? q.y : 0ull;
                }
                if (vm != nullptr && !copy_all) {               // variant V5: a key on a masked pixel is no candidate
#pragma unroll
                    for (int u = 0; u < 2 * GU; ++u)
                        if (kk[u] != 0ull && __ldg(vm + key_index(kk[u])) == 0) kk[u] = 0ull;
                }
#pragma unroll
                for (int u = 0; u < 2 * GU; ++u) {
                    const int i = i0 + 2 * (sub + ((u >> 1) << lps_log)) + (u & 1);
                    uint64_t k = kk[u];
                    if (copy_all) {
                        if (i < c) { DKD_ASSERT(gbase + excl + i >= 0 && gbase + excl + i < SORT_CAP); dst[gbase + excl + i] = k; }
                        if (stage) k = 0ull;                    // (the range is taken after the filter)
                    } else {
                        const bool take = (i < c) && k != 0ull && (k >= lo);
                        const unsigned bal = __ballot_sync(FULL, take);
                        if (bal) {
                            int pb = 0;
                            if (lane == 0) pb = atomicAdd(&s_n, __popc(bal));
                            pb = __shfl_sync(FULL, pb, 0);
                            // (first pass with a mask: the count may pass SORT_CAP -> counted, not stored, radix select below)
                            if (take && pb + __popc(bal) <= SORT_CAP) keys[pb + __popc(bal & ((1u << lane) - 1u))] = k;
                        }
                        if (!take) k = 0ull;
                    }
                    if (k != 0ull) {
                        const unsigned kb = static_cast<unsigned>(k >> 32);
                        khi = kb > khi ? kb : khi;
                        klo = kb < klo ? kb : klo;
                    }
                }
            }
        }
        khi = __reduce_max_sync(FULL, khi);
        klo = __reduce_min_sync(FULL, klo);
        if (lane == 0 && khi >= klo) { atomicMax(&s_hi, khi); atomicMin(&s_lo, klo); }
        __syncthreads();
        if (stage) {                                        // block-uniform
            stage = false;
            const int n0 = s_n;
            __syncthreads();
            if (tid == 0) s_n = 0;
            __syncthreads();
            if (n0 > SORT_CAP) { --pass; continue; }         // too many to stage: count with the per-lane filter instead
            khi = 0u; klo = 0xffffffffu;
            for (int i0 = 0; i0 < n0; i0 += SEL_THREADS) {   // (warp-uniform trip count: ballots inside)
                const int i = i0 + tid;
                const uint64_t k = i < n0 ? sorted[i] : 0ull;
                const bool take = k != 0ull && __ldg(vm + key_index(k)) != 0;
                const unsigned bal = __ballot_sync(FULL, take);
                if (bal) {
                    int pb = 0;
                    if (lane == 0) pb = atomicAdd(&s_n, __popc(bal));
                    pb = __shfl_sync(FULL, pb, 0);
                    if (take) {
                        DKD_ASSERT(pb + __popc(bal) <= SORT_CAP);
                        keys[pb + __popc(bal & ((1u << lane) - 1u))] = k;
                        const unsigned kb = static_cast<unsigned>(k >> 32);
                        khi = kb > khi ? kb : khi;
                        klo = kb < klo ? kb : klo;
                    }
                }
            }
            khi = __reduce_max_sync(FULL, khi);
            klo = __reduce_min_sync(FULL, klo);
            if (lane == 0 && khi >= klo) { atomicMax(&s_hi, khi); atomicMin(&s_lo, klo); }
            __syncthreads();
        }
        if (pass == 0 && tid == 0 && out_total != nullptr) out_total[b] = s_n;   // C_b: every candidate, before the cap
        if (s_n <= SORT_CAP) break;                         // block-uniform; always true in the second pass
        lo = select_radix_prefix(seg0, cnt, tpi, seg_cap, vm, top_k, s_hist, s_rdx);   // (out of line: rare, and the common
                                                            // path stays one contiguous run of instructions)
        if (tid == 0) { s_n = 0; s_hi = 0u; s_lo = 0xffffffffu; }
        __syncthreads();
    }
    const int m = s_n;
    const int K = m < top_k ? m : top_k;
    int32_t* out = sel_idx + static_cast<size_t>(b) * top_k;
    for (int i = K + tid; i < top_k; i += SEL_THREADS) out[i] = -1;    // step a5: padding slots
    if (tid == 0) out_count[b] = K;
    if (m == 0) return;

    // ---- order, common case: bucket rank ------------------------------------------------------------
    const unsigned hi = s_hi;
    const unsigned range = hi - s_lo;
    const int shift = range >= static_cast<unsigned>(NB) ? (32 - __clz(range)) - 12 : 0;   // (range >> shift) < NB
    // Monotone bucket function (a better key never gets a larger bucket).  Keys TIED at the maximum score
    // (score maps saturate: the clamp at 1.0 ties hundreds of peaks) differ only in their index, so they
    // are spread over NBT buckets by index; every other key goes by its score word.
    auto bucket_of = [&](uint64_t k) -> int {
        const unsigned kb = static_cast<unsigned>(k >> 32);
        return kb == hi ? key_index(k) >> idx_shift : NBT + static_cast<int>((hi - kb) >> shift);
    };
    if (tid == 0) s_meff = m;
    for (int i = tid; i < m; i += SEL_THREADS) {
        DKD_ASSERT(bucket_of(keys[i]) >= 0 && bucket_of(keys[i]) < NBK);
        atomicAdd(&cur[bucket_of(keys[i])], 1);
    }
    __syncthreads();
    {   // exclusive scan of the NBK bucket counts (5 consecutive buckets per thread), largest bucket
        int c4[NBK / SEL_THREADS];
        int sum = 0;
#pragma unroll
        for (int q = 0; q < NBK / SEL_THREADS; ++q) {
            c4[q] = cur[tid * (NBK / SEL_THREADS) + q];
            sum += c4[q];
        }
        int incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int up = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += up;
        }
        if (lane == 31) s_red[warp] = incl;
        __syncthreads();
        int woff = s_red[lane];                             // 32 warp totals -> exclusive offsets
        int wincl = woff;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int up = __shfl_up_sync(FULL, wincl, o);
            if (lane >= o) wincl += up;
        }
        woff = __shfl_sync(FULL, wincl - woff, warp);
        int run = woff + incl - sum;
        // Only the buckets that start before rank K can hold a kept key: the keys of the others are neither scattered
        // nor ranked (m_eff = end of the bucket that contains rank K-1), and only the kept buckets count for the size limit.
        int mx = 0;
#pragma unroll
        for (int q = 0; q < NBK / SEL_THREADS; ++q) {
            base[tid * (NBK / SEL_THREADS) + q] = run;
            cur[tid * (NBK / SEL_THREADS) + q] = 0;
            if (run < K) {
                mx = c4[q] > mx ? c4[q] : mx;
                if (run + c4[q] >= K) s_meff = run + c4[q];  // (exactly one bucket when m >= K)
            }
            run += c4[q];
        }
        mx = __reduce_max_sync(FULL, mx);
        if (lane == 0 && mx > 0) atomicMax(&s_maxb, mx);
        __syncthreads();
    }
    const int m_eff = s_meff;                               // keys in the kept buckets (<= m)
    DKD_ASSERT(m_eff >= K && m_eff <= m);
    if (s_maxb <= BUCKET_LIMIT) {                           // block-uniform
        for (int i = tid; i < m; i += SEL_THREADS) {        // scatter into bucket order
            const uint64_t k = keys[i];
            const int d = bucket_of(k);
            DKD_ASSERT(d >= 0 && d < NBK);
            if (base[d] >= K) continue;                      // every key of this bucket ranks past K
            const int pos = base[d] + atomicAdd(&cur[d], 1);
            DKD_ASSERT(pos >= 0 && pos < m_eff && pos < SORT_CAP);
            sorted[pos] = k;
        }
        __syncthreads();
        for (int i = tid; i < m_eff; i += SEL_THREADS) {    // exact rank inside the own bucket
            const uint64_t k = sorted[i];
            const int d = bucket_of(k);
            const int s0 = base[d], s1 = s0 + cur[d];
            int rank = s0;
            int j = s0;
            for (; j + 8 <= s1; j += 8) {                    // 8 independent loads in flight (tie clusters:
                int r8 = 0;                                  //  the clamp at 1.0 puts hundreds of keys in one bucket)
#pragma unroll
                for (int u = 0; u < 8; ++u) r8 += sorted[j + u] > k ? 1 : 0;
                rank += r8;
            }
            for (; j < s1; ++j) rank += sorted[j] > k ? 1 : 0;
            DKD_ASSERT(rank >= 0 && rank < m);
            if (rank < K) {
                out[rank] = key_index(k);
                prefetch_window(pf, b, key_index(k));
            }
        }
        return;
    }

    // ---- order, fallback: bitonic sort (descending) of the gathered keys in shared memory --------------
    int P = 1;
    while (P < m) P <<= 1;
    for (int i = m + tid; i < P; i += SEL_THREADS) keys[i] = 0ull;     // 0 < every real key
    __syncthreads();
    for (int k2 = 2; k2 <= P; k2 <<= 1) {
        for (int j = k2 >> 1; j > 0; j >>= 1) {
            for (int i = tid; i < P; i += SEL_THREADS) {
                const int q = i ^ j;
                if (q > i) {
                    const uint64_t a = keys[i], c = keys[q];
                    const bool desc = (i & k2) == 0;
                    if (desc ? (a < c) : (a > c)) {
                        keys[i] = c;
                        keys[q] = a;
                    }
                }
            }
            __syncthreads();
        }
    }
    for (int i = tid; i < K; i += SEL_THREADS) {
        out[i] = key_index(keys[i]);
        prefetch_window(pf, b, key_index(keys[i]));
    }
}

// ---- k_refine_gather: steps a3, a4, a5 for RG_SLOTS consecutive output slots of one image per CTA ------
// Phase 1 (warp 0, ONE THREAD PER KEYPOINT): index -> (y, x), the (2r+1)^2 window with every load of a row
//   batch in flight at once, soft-argmax offset, keypoint / score / offset stores (coalesced across the
//   lanes), and the four bilinear corner rows + weights of the keypoint, left in shared memory.  The
//   refinement is scalar work per keypoint: done this way it costs ~8 warp instructions per keypoint
//   instead of the ~110 of a lane-group-per-keypoint layout whose lanes mostly idle.
// Phase 2 (all warps, G lanes per keypoint): G = 8, 16 or 32 = the number of 16-byte chunks of one
//   descriptor row rounded up to a power of two (D=128 f16 / D=64 f32: 16; D=256 f16: 32; D=64 f16: 8),
//   so every lane issues exactly one 16-byte load per corner row; fp32 FMAs, shuffle L2 norm, 16-byte stores.
// grid = (ceil(top_k / RG_SLOTS), B): the image index is blockIdx.y (no division by top_k).
constexpr int RG_SLOTS = 32;             // output slots per CTA = lanes of the refining warp

// exact unsigned division by a runtime constant (Granlund-Montgomery): q = (t + ((n - t) >> s1)) >> s2,
// t = umulhi(m, n); host-computed by make_fastdiv; exact for every 32-bit n.
struct FastDiv {
    uint32_t m, s1, s2;
};
__device__ __forceinline__ uint32_t fast_div(uint32_t n, const FastDiv d) {
    const uint32_t t = __umulhi(d.m, n);
    return (t + ((n - t) >> d.s1)) >> d.s2;
}

struct SampleAxis {          // u = (p + 0.5)/s - 0.5 along one axis, p = xi + d (G12, G13)
    FastDiv den;             // division by 2s
    int s;                   // stride
    float inv_den, inv_s;    // 1/(2s), 1/s (exact for power-of-two strides)
    int n;                   // map extent along this axis
};
// Splits u into an integer cell and a fraction without ever forming the large coordinate in fp32:
// 2u = (2 xi + 1 - s)/s + 2d/s, so u = q + rem/(2s) + d/s with (q, rem) an exact integer division
// (biased by +2s to keep the numerator non-negative).  Clamped to [0, n-1].
__device__ __forceinline__ void sample_axis(int xi, float d, const SampleAxis a, int& i0, int& i1, float& f) {
    float t;
    int q;
    if (a.s == 1) {                                          // warp-uniform
        q = xi;
        t = d;
    } else {
        const uint32_t num = static_cast<uint32_t>(2 * xi + 1 + a.s);    // (2 xi + 1 - s) + 2s  >= 2
        const uint32_t qq = fast_div(num, a.den);
        q = static_cast<int>(qq) - 1;
        t = fmaf(static_cast<float>(num - qq * 2u * static_cast<uint32_t>(a.s)), a.inv_den, d * a.inv_s);
    }
    const float ft = floorf(t);
    i0 = q + static_cast<int>(ft);
    f = t - ft;
    if (i0 < 0) { i0 = 0; f = 0.0f; }
    else if (i0 >= a.n - 1) { i0 = a.n - 1; f = 0.0f; }
    i1 = i0 + 1 < a.n - 1 ? i0 + 1 : a.n - 1;
}

__device__ __forceinline__ uint4 ld_stream16(const void* p, uint64_t policy) {   // read-once data: no L1, L2 evict-first
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p), "l"(policy));
    return r;
}
__device__ __forceinline__ float ex2_approx(float x) {      // 2^x, MUFU.EX2 (max 2 ulp)
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int DT> struct ChunkT;                            // one 16-byte chunk of a descriptor row
template <> struct ChunkT<DKD_F32> { static constexpr int N = 4; };
template <> struct ChunkT<DKD_F16> { static constexpr int N = 8; };

template <int DT>
__device__ __forceinline__ void chunk_to_float(const uint4& q, float* f) {
    if (DT == DKD_F16) {
        const __half2* h = reinterpret_cast<const __half2*>(&q);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 t = __half22float2(h[i]);
            f[2 * i] = t.x;
            f[2 * i + 1] = t.y;
        }
    } else {
        f[0] = __uint_as_float(q.x);
        f[1] = __uint_as_float(q.y);
        f[2] = __uint_as_float(q.z);
        f[3] = __uint_as_float(q.w);
    }
}
template <int DT>
__device__ __forceinline__ uint4 float_to_chunk(const float* f) {
    uint4 q;
    if (DT == DKD_F16) {
        __half2* h = reinterpret_cast<__half2*>(&q);
#pragma unroll
        for (int i = 0; i < 4; ++i) h[i] = __floats2half2_rn(f[2 * i], f[2 * i + 1]);
    } else {
        q.x = __float_as_uint(f[0]);
        q.y = __float_as_uint(f[1]);
        q.z = __float_as_uint(f[2]);
        q.w = __float_as_uint(f[3]);
    }
    return q;
}

struct RGParams {
    const float* score;
    const float* score2;                // reliability map of the heat x reliability variant, else NULL
    int H, W;
    FastDiv divW;                       // idx -> (y, x)
    const int32_t* sel_idx;             // [B, top_k] linear index, -1 in padding
    int top_k, r;
    float kscale;                       // log2(e) / T : w = 2^((S - S_c) * kscale) = exp((S - S_c)/T)
    const unsigned char* desc;
    int nchunk;                         // D * elemsize / 16
    size_t img_bytes;                   // Hd * Wd * D * elemsize
    SampleAxis ax, ay;
    float* out_kpts;
    float* out_scores;
    float* out_off;
    unsigned char* out_desc;
    int origin_x, origin_y;             // letterbox offset subtracted from the stored coordinates
    int score_mode;                     // DKD_SCORE_RAW: S at the integer peak; DKD_SCORE_BILINEAR: S at the refined point
    int vec_window;                     // W % 4 == 0 and a 16-byte aligned map: window rows as aligned 16-byte chunks
    int early_trigger;                  // the grid fits the machine at once: let the stream's next kernel launch early
};

// score value at one pixel: S, or heat x reliability rounded once to fp32 (the product variant)
template <bool PROD>
__device__ __forceinline__ float score_at(const float* __restrict__ S, const float* __restrict__ S2, size_t e) {
    if constexpr (PROD) return __fmul_rn(__ldg(S + e), __ldg(S2 + e));
    else return __ldg(S + e);
}

// ---- step a3 for one keypoint, one thread: soft-argmax over the (2R+1)^2 window ----------------------
// w(i,j) = 2^((S[y+j,x+i] - c) * kscale); column sums Wcol, row sums Wrow in a fixed order, then the
// antisymmetric pairing of the definition (dx = sum_a a (Wcol[+a] - Wcol[-a]) / Z): a window symmetric about
// an axis gives two bitwise-equal sums, i.e. an offset of exactly 0 along it.  RPB rows of loads are in
// flight at once (9 / 25 / 21 / 27 loads for R = 1..4).
template <int R, bool PROD, bool VEC>
__device__ __forceinline__ void refine_window(const float* __restrict__ S, const float* __restrict__ S2, int W,
                                              int y, int x, float c, float kscale, float& dx, float& dy) {
    constexpr int N = 2 * R + 1;
    constexpr int RPB = R <= 2 ? N : 3;
    float col[N], row[N];
#pragma unroll
    for (int i = 0; i < N; ++i) col[i] = 0.0f, row[i] = 0.0f;
#pragma unroll
    for (int j0 = 0; j0 < N; j0 += RPB) {
        float v[RPB][N];
        if constexpr (VEC && !PROD) {
            // Every lane of the refining warp reads its own window: a scalar load per element costs one
            // L1 wavefront per lane and element (26 per keypoint at r = 2).  With W % 4 == 0 and a 16-byte
            // aligned map, a window row is instead the 2 (r <= 2) or 3 aligned 16-byte chunks that contain
            // it, and element i is picked out of them by the lane's chunk offset o = (x - r) & 3.
            constexpr int NCH = R <= 2 ? 2 : 3;
            const int xs = x - R, o = xs & 3;
            float f[RPB][4 * NCH];
#pragma unroll
            for (int jj = 0; jj < RPB; ++jj) {
                if (j0 + jj < N) {
                    const float4* rp = reinterpret_cast<const float4*>(S + static_cast<size_t>(y - R + j0 + jj) * W + (xs - o));
#pragma unroll
                    for (int k = 0; k < NCH; ++k) {
                        float4 q = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                        if (4 * k < o + N) q = __ldg(rp + k);     // (a chunk past the window may lie past the map)
                        f[jj][4 * k] = q.x; f[jj][4 * k + 1] = q.y; f[jj][4 * k + 2] = q.z; f[jj][4 * k + 3] = q.w;
                    }
                }
            }
#pragma unroll
            for (int jj = 0; jj < RPB; ++jj) {
                if (j0 + jj < N) {
#pragma unroll
                    for (int i = 0; i < N; ++i) {
                        const float m0 = (o & 1) ? f[jj][i + 1] : f[jj][i];
                        const float m1 = (o & 1) ? f[jj][i + 3] : f[jj][i + 2];   // i + 3 <= 2R + 3 < 4 NCH
                        v[jj][i] = (o & 2) ? m1 : m0;
                    }
                }
            }
        } else {
#pragma unroll
            for (int jj = 0; jj < RPB; ++jj) {
                if (j0 + jj < N) {
                    const size_t e = static_cast<size_t>(y - R + j0 + jj) * W + (x - R);
#pragma unroll
                    for (int i = 0; i < N; ++i) v[jj][i] = score_at<PROD>(S, S2, e + i);
                }
            }
        }
#pragma unroll
        for (int jj = 0; jj < RPB; ++jj) {
            if (j0 + jj < N) {
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    const float w = ex2_approx((v[jj][i] - c) * kscale);
                    col[i] += w;
                    row[j0 + jj] += w;
                }
            }
        }
    }
    float z = col[0], sx = 0.0f, sy = 0.0f;
#pragma unroll
    for (int i = 1; i < N; ++i) z += col[i];
#pragma unroll
    for (int a = 1; a <= R; ++a) {
        sx = fmaf(static_cast<float>(a), col[R + a] - col[R - a], sx);
        sy = fmaf(static_cast<float>(a), row[R + a] - row[R - a], sy);
    }
    const float inv_z = __frcp_rn(z);                        // z >= 1 (the centre weight is exactly 1)
    dx = sx * inv_z;
    dy = sy * inv_z;
}

template <bool PROD, bool VEC>
__device__ __forceinline__ void refine_dispatch(int r, const float* __restrict__ S, const float* __restrict__ S2, int W,
                                                int y, int x, float c, float kscale, float& dx, float& dy) {
    switch (r) {                                             // (uniform)
        case 1: refine_window<1, PROD, VEC>(S, S2, W, y, x, c, kscale, dx, dy); break;
        case 2: refine_window<2, PROD, VEC>(S, S2, W, y, x, c, kscale, dx, dy); break;
        case 3: refine_window<3, PROD, VEC>(S, S2, W, y, x, c, kscale, dx, dy); break;
        default: refine_window<4, PROD, VEC>(S, S2, W, y, x, c, kscale, dx, dy); break;
    }
}

struct SampleInfo {                     // phase 1 -> phase 2, one per slot (shared memory)
    uint32_t o00, o01, o10, o11;        // descriptor-row index (v * Wd + u) of the four corners; o00 = ~0: padding slot
    float w00, w01, w10, w11;
};

// DT: DKD_F32 / DKD_F16 descriptor maps, or -1 for keypoints only (launched with one warp per CTA).
// G: lanes per keypoint in phase 2.  PROD: score = heat x reliability.
template <int DT, int G, bool PROD>
__global__ void __launch_bounds__(RG_THREADS, 4) k_refine_gather(const __grid_constant__ RGParams p) {
    __shared__ __align__(16) SampleInfo s_info[RG_SLOTS];
    const int b = blockIdx.y;
    const int slot0 = blockIdx.x * RG_SLOTS;                 // first slot (within the image) of this CTA
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // The next call's NMS kernel may be launched while this grid runs (it waits for this grid's completion before it
    // touches memory) — but only when every CTA of this grid is resident at once: waiting CTAs of the successor must
    // not take the place of CTAs of this grid that have not started yet.
    if (p.early_trigger) pdl_launch_dependents();
    pdl_wait();                                              // the selection of k_select is complete and visible

    if (warp == 0) {
        const int i_img = slot0 + lane;
        SampleInfo si;
        si.o00 = 0xffffffffu; si.o01 = si.o10 = si.o11 = 0u;
        si.w00 = si.w01 = si.w10 = si.w11 = 0.0f;
        if (i_img < p.top_k) {
            const size_t slot = static_cast<size_t>(b) * p.top_k + i_img;
            const int idx = __ldg(p.sel_idx + slot);
            float2 kp = make_float2(0.0f, 0.0f), off = make_float2(0.0f, 0.0f);
            float sc = 0.0f;                                 // step a5: zero padding
            if (idx >= 0) {
                const int W = p.W;
                const int y = static_cast<int>(fast_div(static_cast<uint32_t>(idx), p.divW)), x = idx - y * W;
                const float* S = p.score + static_cast<size_t>(b) * p.H * W;
                const float* S2 = PROD ? p.score2 + static_cast<size_t>(b) * p.H * W : nullptr;
                const float c = score_at<PROD>(S, S2, static_cast<size_t>(idx));
                float dx, dy;
                if (p.vec_window) refine_dispatch<PROD, true>(p.r, S, S2, W, y, x, c, p.kscale, dx, dy);
                else refine_dispatch<PROD, false>(p.r, S, S2, W, y, x, c, p.kscale, dx, dy);
                kp = make_float2(static_cast<float>(x - p.origin_x) + dx, static_cast<float>(y - p.origin_y) + dy);
                off = make_float2(dx, dy);
                sc = c;                                      // raw S at the integer peak (G7)
                if (p.score_mode == DKD_SCORE_BILINEAR) {    // variant: S interpolated at the refined point (V2)
                    const float fdx = floorf(dx), fdy = floorf(dy);
                    int x0 = x + static_cast<int>(fdx), y0 = y + static_cast<int>(fdy);
                    float fx = dx - fdx, fy = dy - fdy;
                    if (x0 >= W - 1) { x0 = W - 1; fx = 0.0f; }      // |dx| <= r <= border: x0 >= 0 always
                    if (y0 >= p.H - 1) { y0 = p.H - 1; fy = 0.0f; }
                    const int x1 = x0 + 1 < W - 1 ? x0 + 1 : W - 1, y1 = y0 + 1 < p.H - 1 ? y0 + 1 : p.H - 1;
                    const float s00 = score_at<PROD>(S, S2, static_cast<size_t>(y0) * W + x0);
                    const float s01 = score_at<PROD>(S, S2, static_cast<size_t>(y0) * W + x1);
                    const float s10 = score_at<PROD>(S, S2, static_cast<size_t>(y1) * W + x0);
                    const float s11 = score_at<PROD>(S, S2, static_cast<size_t>(y1) * W + x1);
                    const float top = fmaf(fx, s01 - s00, s00), bot = fmaf(fx, s11 - s10, s10);
                    sc = fmaf(fy, bot - top, top);
                }
                if constexpr (DT >= 0) {
                    int x0, x1, y0, y1;
                    float fx, fy;
                    sample_axis(x, dx, p.ax, x0, x1, fx);
                    sample_axis(y, dy, p.ay, y0, y1, fy);
                    const uint32_t Wd = static_cast<uint32_t>(p.ax.n);
                    si.o00 = static_cast<uint32_t>(y0) * Wd + x0; si.o01 = static_cast<uint32_t>(y0) * Wd + x1;
                    si.o10 = static_cast<uint32_t>(y1) * Wd + x0; si.o11 = static_cast<uint32_t>(y1) * Wd + x1;
                    si.w00 = (1.0f - fy) * (1.0f - fx); si.w01 = (1.0f - fy) * fx;
                    si.w10 = fy * (1.0f - fx); si.w11 = fy * fx;
                }
            }
            reinterpret_cast<float2*>(p.out_kpts)[slot] = kp;
            p.out_scores[slot] = sc;
            if (p.out_off != nullptr) reinterpret_cast<float2*>(p.out_off)[slot] = off;
        }
        if constexpr (DT >= 0) {
            DKD_ASSERT(lane < RG_SLOTS);
            s_info[lane] = si;
        }
    }
    if constexpr (DT < 0) return;                            // keypoints only

    // ---- step a4: bilinear gather of the four corner rows (16-byte loads), fp32 accumulate, L2 norm
    if constexpr (DT >= 0) {
        __syncthreads();
        constexpr int ITERS = (G == 32) ? DKD_MAX_ROW_BYTES / 16 / 32 : 1;   // chunks per lane
        constexpr int KPR = RG_THREADS / G;                  // keypoints per round
        constexpr int N = ChunkT<DT >= 0 ? DT : 0>::N;
        const int gl = threadIdx.x & (G - 1);                // lane within the group
        const unsigned gmask = (G == 32) ? 0xffffffffu : (((1u << G) - 1u) << ((threadIdx.x & 31) & ~(G - 1)));
        const size_t rowb = static_cast<size_t>(p.nchunk) * 16;
        const unsigned char* base = p.desc + static_cast<size_t>(b) * p.img_bytes;
        const uint64_t policy = l2_evict_first_policy();
        if (p.nchunk <= G) {                                 // (uniform) one 16-byte chunk per lane and corner row:
            // the corner loads of TWO of this group's keypoints are issued before any of them is used
            // (8 loads in flight per lane); G = 8: one pass of one keypoint, G = 16: one pass, G = 32: two passes
            constexpr int ROUNDS = RG_SLOTS / KPR;           // keypoints per lane group
            constexpr int U = ROUNDS >= 2 ? 2 : 1;
#pragma unroll 1
            for (int k0 = 0; k0 < ROUNDS; k0 += U) {
                uint4 q[U][4];
                SampleInfo si[U];
                bool live[U];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int k = threadIdx.x / G + (k0 + u) * KPR;
                    si[u] = s_info[k];
                    live[u] = slot0 + k < p.top_k && si[u].o00 != 0xffffffffu && gl < p.nchunk;
                    if (live[u]) {
                        q[u][0] = ld_stream16(reinterpret_cast<const uint4*>(base + si[u].o00 * rowb) + gl, policy);
                        q[u][1] = ld_stream16(reinterpret_cast<const uint4*>(base + si[u].o01 * rowb) + gl, policy);
                        q[u][2] = ld_stream16(reinterpret_cast<const uint4*>(base + si[u].o10 * rowb) + gl, policy);
                        q[u][3] = ld_stream16(reinterpret_cast<const uint4*>(base + si[u].o11 * rowb) + gl, policy);
                    }
                }
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int k = threadIdx.x / G + (k0 + u) * KPR;
                    const int i_img = slot0 + k;
                    if (i_img >= p.top_k) break;             // whole groups leave together
                    uint4* o = reinterpret_cast<uint4*>(p.out_desc + (static_cast<size_t>(b) * p.top_k + i_img) * rowb);
                    if (si[u].o00 == 0xffffffffu) {          // padding slot: zero descriptor
                        if (gl < p.nchunk) o[gl] = make_uint4(0u, 0u, 0u, 0u);
                        continue;
                    }
                    float acc[N];
                    float ss = 0.0f;
                    if (live[u]) {
                        float a[N], bq[N], cq[N], dq[N];
                        chunk_to_float<DT >= 0 ? DT : 0>(q[u][0], a);
                        chunk_to_float<DT >= 0 ? DT : 0>(q[u][1], bq);
                        chunk_to_float<DT >= 0 ? DT : 0>(q[u][2], cq);
                        chunk_to_float<DT >= 0 ? DT : 0>(q[u][3], dq);
#pragma unroll
                        for (int e = 0; e < N; ++e) {
                            const float d = fmaf(si[u].w11, dq[e], fmaf(si[u].w10, cq[e], fmaf(si[u].w01, bq[e], si[u].w00 * a[e])));
                            acc[e] = d;
                            ss = fmaf(d, d, ss);
                        }
                    }
#pragma unroll
                    for (int sft = G / 2; sft > 0; sft >>= 1) ss += __shfl_xor_sync(gmask, ss, sft);
                    const float inv = __frcp_rn(fmaxf(sqrtf(ss), 1e-12f));
                    if (live[u]) {
                        float f[N];
#pragma unroll
                        for (int e = 0; e < N; ++e) f[e] = acc[e] * inv;
                        o[gl] = float_to_chunk<DT >= 0 ? DT : 0>(f);
                    }
                }
            }
        } else {
#pragma unroll 1
            for (int k = threadIdx.x / G; k < RG_SLOTS; k += KPR) {
                const int i_img = slot0 + k;
                if (i_img >= p.top_k) break;                 // whole groups leave together
                const SampleInfo si = s_info[k];
                uint4* o = reinterpret_cast<uint4*>(p.out_desc + (static_cast<size_t>(b) * p.top_k + i_img) * rowb);
                if (si.o00 == 0xffffffffu) {                 // padding slot: zero descriptor
                    for (int ch = gl; ch < p.nchunk; ch += G) o[ch] = make_uint4(0u, 0u, 0u, 0u);
                    continue;
                }
                const uint4* p00 = reinterpret_cast<const uint4*>(base + si.o00 * rowb);
                const uint4* p01 = reinterpret_cast<const uint4*>(base + si.o01 * rowb);
                const uint4* p10 = reinterpret_cast<const uint4*>(base + si.o10 * rowb);
                const uint4* p11 = reinterpret_cast<const uint4*>(base + si.o11 * rowb);
                float acc[ITERS][N];
                float ss = 0.0f;
#pragma unroll
                for (int it = 0; it < ITERS; ++it) {
                    const int ch = gl + G * it;
                    if (ch < p.nchunk) {
                        const uint4 q00 = ld_stream16(p00 + ch, policy), q01 = ld_stream16(p01 + ch, policy);
                        const uint4 q10 = ld_stream16(p10 + ch, policy), q11 = ld_stream16(p11 + ch, policy);
                        float a[N], bq[N], cq[N], dq[N];
                        chunk_to_float<DT >= 0 ? DT : 0>(q00, a);
                        chunk_to_float<DT >= 0 ? DT : 0>(q01, bq);
                        chunk_to_float<DT >= 0 ? DT : 0>(q10, cq);
                        chunk_to_float<DT >= 0 ? DT : 0>(q11, dq);
#pragma unroll
                        for (int e = 0; e < N; ++e) {
                            const float d = fmaf(si.w11, dq[e], fmaf(si.w10, cq[e], fmaf(si.w01, bq[e], si.w00 * a[e])));
                            acc[it][e] = d;
                            ss = fmaf(d, d, ss);
                        }
                    }
                }
#pragma unroll
                for (int sft = G / 2; sft > 0; sft >>= 1) ss += __shfl_xor_sync(gmask, ss, sft);
                const float inv = __frcp_rn(fmaxf(sqrtf(ss), 1e-12f));
#pragma unroll
                for (int it = 0; it < ITERS; ++it) {
                    const int ch = gl + G * it;
                    if (ch < p.nchunk) {
                        float f[N];
#pragma unroll
                        for (int e = 0; e < N; ++e) f[e] = acc[it][e] * inv;
                        o[ch] = float_to_chunk<DT >= 0 ? DT : 0>(f);
                    }
                }
            }
        }
    }
}

// ---- k_preprocess: fused letterbox + colour conversion + normalisation + NCHW packing -------------------
// (P1..P7.)  HBM-bound, write-dominated: one thread produces VEC consecutive
// output columns of one padded row for EVERY output channel, so each source pixel is read once;
// VEC = 8 -> 32-byte (f32) / 16-byte (f16) stores per plane.  Padding pixels get pad_value.
struct PreParams {
    const uint8_t* src;
    unsigned char* dst;
    int B, H, W, Hp, Wp, oy, ox;
    int bgr;
    float a[3], b[3];        // out = value * a[c] + b[c],  a = scale * inv_std, b = -mean * inv_std
    float pad;
    int gpr;                 // groups per padded row = ceil(Wp / VEC)
};

template <int CIN, int COUT, int DT, int VEC>
__global__ void __launch_bounds__(256) k_preprocess(const __grid_constant__ PreParams p) {
    // grid = (ceil(groups per row / 256), Hp, B): no index division
    const int xg = blockIdx.x * 256 + threadIdx.x;
    if (xg >= p.gpr) return;
    const int yp = blockIdx.y, b = blockIdx.z;
    const int xp0 = xg * VEC, y = yp - p.oy;
    float v[COUT][VEC];
    const bool row_in = y >= 0 && y < p.H;
    const int x0 = xp0 - p.ox;                               // source column of the group's first pixel
    // one pixel: 8-bit channel values -> COUT normalised outputs
    auto convert = [&](float c0, float c1, float c2, int i) {
        if constexpr (CIN == 1) {
#pragma unroll
            for (int c = 0; c < COUT; ++c) v[c][i] = fmaf(c0, p.a[c], p.b[c]);
        } else {
            const float R = p.bgr ? c2 : c0, Bl = p.bgr ? c0 : c2;
            if constexpr (COUT == 1) {
                v[0][i] = fmaf(fmaf(0.299f, R, fmaf(0.587f, c1, 0.114f * Bl)), p.a[0], p.b[0]);
            } else {
                v[0][i] = fmaf(R, p.a[0], p.b[0]);
                v[1][i] = fmaf(c1, p.a[1], p.b[1]);
                v[2][i] = fmaf(Bl, p.a[2], p.b[2]);
            }
        }
    };
    if (row_in && x0 >= 0 && x0 + VEC <= p.W) {              // interior group: no per-pixel test, one row pointer
        const uint8_t* q = p.src + ((static_cast<size_t>(b) * p.H + y) * p.W + x0) * CIN;
        constexpr int NB = VEC * CIN;
        uint8_t raw[NB];
        if (NB % 4 == 0 && (reinterpret_cast<uintptr_t>(q) & 3) == 0) {      // (uniform along a row)
#pragma unroll
            for (int w = 0; w < NB / 4; ++w) {
                const uint32_t u = __ldg(reinterpret_cast<const uint32_t*>(q) + w);
                raw[4 * w] = u & 0xff; raw[4 * w + 1] = (u >> 8) & 0xff; raw[4 * w + 2] = (u >> 16) & 0xff; raw[4 * w + 3] = u >> 24;
            }
        } else {
#pragma unroll
            for (int k = 0; k < NB; ++k) raw[k] = __ldg(q + k);
        }
#pragma unroll
        for (int i = 0; i < VEC; ++i)
            convert(static_cast<float>(raw[i * CIN]), CIN == 3 ? static_cast<float>(raw[i * CIN + (CIN == 3 ? 1 : 0)]) : 0.0f,
                    CIN == 3 ? static_cast<float>(raw[i * CIN + (CIN == 3 ? 2 : 0)]) : 0.0f, i);
    } else {                                                 // padding rows / groups straddling the image edge
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
            const int x = x0 + i;
            if (row_in && x >= 0 && x < p.W) {
                const uint8_t* px = p.src + ((static_cast<size_t>(b) * p.H + y) * p.W + x) * CIN;
                convert(static_cast<float>(__ldg(px)), CIN == 3 ? static_cast<float>(__ldg(px + (CIN == 3 ? 1 : 0))) : 0.0f,
                        CIN == 3 ? static_cast<float>(__ldg(px + (CIN == 3 ? 2 : 0))) : 0.0f, i);
            } else {
#pragma unroll
                for (int c = 0; c < COUT; ++c) v[c][i] = p.pad;
            }
        }
    }
    constexpr int ESZ = DT == DKD_F16 ? 2 : 4;
#pragma unroll
    for (int c = 0; c < COUT; ++c) {
        unsigned char* o = p.dst + (((static_cast<size_t>(b) * COUT + c) * p.Hp + yp) * p.Wp + xp0) * ESZ;
        if constexpr (VEC == 8) {                            // Wp % 8 == 0: aligned vector stores
            if constexpr (DT == DKD_F16) {
                uint4 q;
                __half2* h = reinterpret_cast<__half2*>(&q);
#pragma unroll
                for (int i = 0; i < 4; ++i) h[i] = __floats2half2_rn(v[c][2 * i], v[c][2 * i + 1]);
                __stcs(reinterpret_cast<uint4*>(o), q);      // streaming stores: written once, read by the network later
            } else {
                __stcs(reinterpret_cast<float4*>(o), make_float4(v[c][0], v[c][1], v[c][2], v[c][3]));
                __stcs(reinterpret_cast<float4*>(o) + 1, make_float4(v[c][4], v[c][5], v[c][6], v[c][7]));
            }
        } else {
            if constexpr (DT == DKD_F16) *reinterpret_cast<__half*>(o) = __float2half_rn(v[c][0]);
            else *reinterpret_cast<float*>(o) = v[c][0];
        }
    }
}

}  // namespace dkd
