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
#include <stdint.h>

#include "dkd.h"

namespace dkd {

// ---- geometry -------------------------------------------------------------------------------
constexpr int TW = 128;                  // tile width  (pixels)
constexpr int TH = 32;                   // tile height (pixels)
constexpr int HX = 4;                    // x halo kept in smem: >= max radius, multiple of 4 so the
                                         // tile interior stays float4-aligned
constexpr int PITCH = TW + 2 * HX;       // 136 floats = 544 B per smem row (= TMA box width)
constexpr int TILE_PX = TW * TH;         // 4096 = worst-case candidates of a tile = segment capacity
constexpr int MAX_R = 4;
constexpr int NMS_THREADS = 256;
constexpr int NMS_STAGES = 4;            // TMA pipeline depth per CTA
constexpr int SEL_THREADS = 1024;
constexpr int SORT_CAP = 8192;           // keys sorted in shared memory by k_select (64 KB)
constexpr int RG_THREADS = 256;          // k_refine_gather: 8 warps, one warp per output slot

__host__ __device__ constexpr int tile_rows(int R) { return TH + 2 * R; }
__host__ __device__ constexpr int stage_bytes(int R) { return ((PITCH * tile_rows(R) * 4 + 127) / 128) * 128; }
__host__ __device__ constexpr int box_bytes(int R) { return PITCH * tile_rows(R) * 4; }

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
                                              int b) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(b)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tmap)) : "memory");
}

// ---- step a1 + a1': one halo'd tile in shared memory -> candidate keys ------------------------------
// tile: smem, tile_rows(R) x PITCH floats; tile[(row + R) * PITCH + HX + col] is pixel (x0+col, y0+row).
// Pixels outside the image read 0 (never used: a kept pixel's window is inside the image, G3).
// Candidates are appended (unordered) to this tile's private global segment `seg` (capacity TILE_PX);
// the slot comes from a shared-memory counter, one atomic per warp-row (warp-ballot compaction).
template <int R>
__device__ __forceinline__ void process_tile(const float* __restrict__ tile, int x0, int y0, int H, int W,
                                             float thresh, int* s_cnt, uint64_t* __restrict__ seg) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    constexpr int ROWS_PER_WARP = TH / (NMS_THREADS / 32);
    const int gx = x0 + 4 * lane;
#pragma unroll
    for (int rr = 0; rr < ROWS_PER_WARP; ++rr) {
        const int row = warp * ROWS_PER_WARP + rr;
        const int gy = y0 + row;
        const float* ctr = tile + (row + R) * PITCH + HX + 4 * lane;
        const float4 v4 = *reinterpret_cast<const float4*>(ctr);
        const float v[4] = {v4.x, v4.y, v4.z, v4.w};
        unsigned m = 0;
        if (gy >= R && gy < H - R) {                         // warp-uniform
#pragma unroll
            for (int c = 0; c < 4; ++c)
                if (v[c] > thresh && gx + c >= R && gx + c < W - R) m |= 1u << c;
        }
        if (m) {                                             // rare (a few % of pixels pass the threshold)
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                if (m & (1u << c)) {
                    const float* wp = ctr + c - R * PITCH - R;
                    bool ismax = true;
#pragma unroll
                    for (int j = 0; j <= 2 * R; ++j)
#pragma unroll
                        for (int i = 0; i <= 2 * R; ++i) ismax &= !(wp[j * PITCH + i] > v[c]);   // ties keep (G1)
                    if (!ismax) m &= ~(1u << c);
                }
            }
        }
        if (__any_sync(0xffffffffu, m != 0)) {
            unsigned bal[4];
            int tot = 0, mypos[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                bal[c] = __ballot_sync(0xffffffffu, (m >> c) & 1u);
                mypos[c] = tot + __popc(bal[c] & ((1u << lane) - 1u));
                tot += __popc(bal[c]);
            }
            int base = 0;
            if (lane == 0) base = atomicAdd(s_cnt, tot);
            base = __shfl_sync(0xffffffffu, base, 0);
#pragma unroll
            for (int c = 0; c < 4; ++c)
                if ((m >> c) & 1u) seg[base + mypos[c]] = make_key(v[c], gy * W + gx + c);
        }
    }
}

// ---- k_nms_tma: persistent, TMA-staged halo tiles, NMS_STAGES-deep mbarrier pipeline ----------------
// grid = min(total_tiles, CTAs that fit); CTA c handles tiles c, c+grid, ... (image-major order).
// Dynamic smem: NMS_STAGES * stage_bytes(R), 128-byte aligned.
template <int R>
__global__ void __launch_bounds__(NMS_THREADS) k_nms_tma(const __grid_constant__ CUtensorMap tmap, int H, int W,
                                                         int tiles_x, int tiles_y, int total_tiles, float thresh,
                                                         uint64_t* __restrict__ cand, int* __restrict__ tile_cnt) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[NMS_STAGES];
    __shared__ int s_cnt[2];
    constexpr int SB = stage_bytes(R);
    const int tid = threadIdx.x;
    const int tpi = tiles_x * tiles_y;
    const int first = blockIdx.x, step = gridDim.x;
    const int n_my = first < total_tiles ? (total_tiles - first + step - 1) / step : 0;

    auto issue = [&](int it) {
        const int t = first + it * step;
        const int b = t / tpi, rem = t - b * tpi;
        const int ty = rem / tiles_x, tx = rem - ty * tiles_x;
        const int s = it % NMS_STAGES;
        mbar_arrive_expect_tx(&full_bar[s], box_bytes(R));
        tma_load_tile(smem_raw + s * SB, &tmap, &full_bar[s], tx * TW - HX, ty * TH - R, b);
    };

    if (tid == 0) {
        tma_prefetch_desc(&tmap);
#pragma unroll
        for (int s = 0; s < NMS_STAGES; ++s) mbar_init(&full_bar[s], 1);
        s_cnt[0] = 0;
        s_cnt[1] = 0;
        fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0) {
        const int pre = n_my < NMS_STAGES ? n_my : NMS_STAGES;
        for (int it = 0; it < pre; ++it) issue(it);
    }
    for (int it = 0; it < n_my; ++it) {
        const int t = first + it * step;
        const int b = t / tpi, rem = t - b * tpi;
        const int ty = rem / tiles_x, tx = rem - ty * tiles_x;
        const int s = it % NMS_STAGES;
        mbar_wait(&full_bar[s], (it / NMS_STAGES) & 1);
        process_tile<R>(reinterpret_cast<const float*>(smem_raw + s * SB), tx * TW, ty * TH, H, W, thresh,
                        &s_cnt[it & 1], cand + static_cast<size_t>(t) * TILE_PX);
        __syncthreads();                                     // every warp is done with stage s and s_cnt[it&1]
        if (tid == 0) {
            tile_cnt[t] = s_cnt[it & 1];
            s_cnt[it & 1] = 0;
            if (it + NMS_STAGES < n_my) issue(it + NMS_STAGES);
        }
    }
}

// ---- k_nms_plain: same tile math, tile staged with ordinary loads (any W, any alignment) ------------
template <int R>
__global__ void __launch_bounds__(NMS_THREADS) k_nms_plain(const float* __restrict__ score, int H, int W,
                                                           int tiles_x, int tiles_y, float thresh,
                                                           uint64_t* __restrict__ cand, int* __restrict__ tile_cnt) {
    __shared__ __align__(16) float tile[PITCH * tile_rows(R)];
    __shared__ int s_cnt;
    const int t = blockIdx.x;
    const int tpi = tiles_x * tiles_y;
    const int b = t / tpi, rem = t - b * tpi;
    const int ty = rem / tiles_x, tx = rem - ty * tiles_x;
    const int x0 = tx * TW, y0 = ty * TH;
    const float* img = score + static_cast<size_t>(b) * H * W;
    if (threadIdx.x == 0) s_cnt = 0;
    for (int e = threadIdx.x; e < PITCH * tile_rows(R); e += NMS_THREADS) {
        const int ry = e / PITCH, rx = e - ry * PITCH;
        const int gy = y0 - R + ry, gx = x0 - HX + rx;
        tile[e] = (gy >= 0 && gy < H && gx >= 0 && gx < W) ? __ldg(img + static_cast<size_t>(gy) * W + gx) : 0.0f;
    }
    __syncthreads();
    process_tile<R>(tile, x0, y0, H, W, thresh, &s_cnt, cand + static_cast<size_t>(t) * TILE_PX);
    __syncthreads();
    if (threadIdx.x == 0) tile_cnt[t] = s_cnt;
}

// ---- k_select: per-image top-k select + order ---------------------------------------------------
// One CTA per image.  n = sum of the image's tile counts.
//   n <= SORT_CAP : gather every key into shared memory, bitonic sort (descending), emit the first K.
//   n >  SORT_CAP : MSB-first radix select (8-bit digits, warp-aggregated shared-memory histogram)
//                   narrows to a lower bound `lo` with  top_k <= #{key >= lo} <= SORT_CAP, then as above.
// Keys are unique (they embed the pixel index) so the result is the unique (score desc, idx asc) order.
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

__global__ void __launch_bounds__(SEL_THREADS) k_select(const uint64_t* __restrict__ cand,
                                                        const int* __restrict__ tile_cnt, int tpi, int top_k,
                                                        int32_t* __restrict__ sel_idx,
                                                        int32_t* __restrict__ out_count) {
    extern __shared__ __align__(16) unsigned char sel_smem[];
    uint64_t* keys = reinterpret_cast<uint64_t*>(sel_smem);            // SORT_CAP entries
    __shared__ int s_hist[257];
    __shared__ int s_red[32];
    __shared__ int s_n, s_digit, s_cum, s_h;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = SEL_THREADS / 32;
    const int b = blockIdx.x;
    const int* cnt = tile_cnt + static_cast<size_t>(b) * tpi;
    const uint64_t* seg0 = cand + static_cast<size_t>(b) * tpi * TILE_PX;

    int local = 0;
    for (int t = tid; t < tpi; t += SEL_THREADS) local += cnt[t];
    const int n = block_sum_1024(local, s_red);

    uint64_t lo = 0;                                        // gather keys >= lo (0: all of them)
    if (n > SORT_CAP) {
        uint64_t prefix = 0;
        int need = top_k;                                   // rank (1-based, from the top) inside the prefix bucket
        int above = 0;                                      // keys strictly above the prefix bucket
        for (int shift = 56; shift >= 0; shift -= 8) {
            for (int i = tid; i < 257; i += SEL_THREADS) s_hist[i] = 0;
            __syncthreads();
            for (int t = warp; t < tpi; t += NW) {
                const int c = cnt[t];
                const uint64_t* seg = seg0 + static_cast<size_t>(t) * TILE_PX;
                for (int e0 = 0; e0 < c; e0 += 32) {
                    const int e = e0 + lane;
                    int digit = 256;                        // dummy bin: past the end / outside the prefix
                    if (e < c) {
                        const uint64_t k = seg[e];
                        const bool match = (shift == 56) || ((k >> (shift + 8)) == (prefix >> (shift + 8)));
                        if (match) digit = static_cast<int>((k >> shift) & 255u);
                    }
                    const unsigned peers = __match_any_sync(0xffffffffu, digit);
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
                    const int up = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += up;
                }
                const unsigned hit = __ballot_sync(0xffffffffu, incl >= need);
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
        lo = prefix;
    }

    if (tid == 0) s_n = 0;
    __syncthreads();
    for (int t = warp; t < tpi; t += NW) {
        const int c = cnt[t];
        if (c == 0) continue;
        const uint64_t* seg = seg0 + static_cast<size_t>(t) * TILE_PX;
        if (lo == 0) {
            int base = 0;
            if (lane == 0) base = atomicAdd(&s_n, c);
            base = __shfl_sync(0xffffffffu, base, 0);
            for (int e = lane; e < c; e += 32) keys[base + e] = seg[e];
        } else {
            for (int e0 = 0; e0 < c; e0 += 32) {
                const int e = e0 + lane;
                const uint64_t k = e < c ? seg[e] : 0ull;
                const bool take = (e < c) && (k >= lo);
                const unsigned bal = __ballot_sync(0xffffffffu, take);
                if (bal) {
                    int base = 0;
                    if (lane == 0) base = atomicAdd(&s_n, __popc(bal));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (take) keys[base + __popc(bal & ((1u << lane) - 1u))] = k;
                }
            }
        }
    }
    __syncthreads();
    const int m = s_n;
    int P = 1;
    while (P < m) P <<= 1;
    for (int i = m + tid; i < P; i += SEL_THREADS) keys[i] = 0ull;     // 0 < every real key
    __syncthreads();

    for (int k2 = 2; k2 <= P; k2 <<= 1) {
        for (int j = k2 >> 1; j > 0; j >>= 1) {
            for (int i = tid; i < P; i += SEL_THREADS) {
                const int p = i ^ j;
                if (p > i) {
                    const uint64_t a = keys[i], c = keys[p];
                    const bool desc = (i & k2) == 0;
                    if (desc ? (a < c) : (a > c)) {
                        keys[i] = c;
                        keys[p] = a;
                    }
                }
            }
            __syncthreads();
        }
    }

    const int K = m < top_k ? m : top_k;
    int32_t* out = sel_idx + static_cast<size_t>(b) * top_k;
    for (int i = tid; i < top_k; i += SEL_THREADS) out[i] = i < K ? key_index(keys[i]) : -1;
    if (tid == 0) out_count[b] = K;
}

// ---- k_refine_gather: one warp per output slot (b, i) -----------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ uint4 ld_stream16(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
// sample position along one axis: u = (p + 0.5)/s - 0.5 with p = xi + d, split into an integer cell and
// a fraction without ever forming the large coordinate in fp32 (G12); clamped to [0, n-1].
__device__ __forceinline__ void sample_axis(int xi, float d, int s, int n, int& i0, int& i1, float& f) {
    const int num = 2 * xi + 1 - s, den = 2 * s;
    int q = num / den;
    int rem = num - q * den;
    if (rem < 0) { rem += den; --q; }
    const float t = static_cast<float>(rem) / static_cast<float>(den) + d / static_cast<float>(s);
    const float ft = floorf(t);
    i0 = q + static_cast<int>(ft);
    f = t - ft;
    if (i0 < 0) { i0 = 0; f = 0.0f; }
    else if (i0 >= n - 1) { i0 = n - 1; f = 0.0f; }
    i1 = i0 + 1 < n - 1 ? i0 + 1 : n - 1;
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

constexpr int MAX_CHUNK_ITERS = DKD_MAX_ROW_BYTES / 16 / 32;          // 4

// R: window radius; DT: DKD_F32 / DKD_F16 descriptor maps, or -1 for keypoints only.
template <int R, int DT>
__global__ void __launch_bounds__(RG_THREADS) k_refine_gather(
    const float* __restrict__ score, int H, int W, const int32_t* __restrict__ sel_idx, int nslots, int top_k,
    float T, const unsigned char* __restrict__ desc, int Hd, int Wd, int D, int stride,
    float* __restrict__ out_kpts, float* __restrict__ out_scores, float* __restrict__ out_off,
    unsigned char* __restrict__ out_desc) {
    const int lane = threadIdx.x & 31;
    const int slot = blockIdx.x * (RG_THREADS / 32) + (threadIdx.x >> 5);
    if (slot >= nslots) return;
    const int idx = sel_idx[slot];
    constexpr int ESZ = (DT == DKD_F16) ? 2 : 4;
    const int nchunk = (DT >= 0) ? (D * ESZ) >> 4 : 0;

    if (idx < 0) {                                          // step a5: zero padding
        if (lane < 2) out_kpts[2 * static_cast<size_t>(slot) + lane] = 0.0f;
        if (lane == 2) out_scores[slot] = 0.0f;
        if (out_off != nullptr && lane >= 4 && lane < 6) out_off[2 * static_cast<size_t>(slot) + lane - 4] = 0.0f;
        if constexpr (DT >= 0) {
            uint4* o = reinterpret_cast<uint4*>(out_desc + static_cast<size_t>(slot) * D * ESZ);
            for (int ch = lane; ch < nchunk; ch += 32) o[ch] = make_uint4(0u, 0u, 0u, 0u);
        }
        return;
    }

    // ---- step a3: soft-argmax over the (2R+1)^2 window.  Lane q < (R+1)^2 owns the mirror orbit
    // {(+-i, +-j)}, i, j >= 0; differences of mirrored weights are formed first, so a symmetric
    // window refines to exactly (0, 0).
    const int b = slot / top_k;
    const int y = idx / W, x = idx - y * W;
    const float* S = score + static_cast<size_t>(b) * H * W;
    const float c = __ldg(S + idx);
    float sx = 0.0f, sy = 0.0f, z = 0.0f;
    if (lane < (R + 1) * (R + 1)) {
        const int j = lane / (R + 1), i = lane - j * (R + 1);
        const float vpp = __ldg(S + (y + j) * W + (x + i));
        const float vmp = __ldg(S + (y + j) * W + (x - i));
        const float vpm = __ldg(S + (y - j) * W + (x + i));
        const float vmm = __ldg(S + (y - j) * W + (x - i));
        const float wpp = expf(__fdiv_rn(vpp - c, T));
        const float wmp = expf(__fdiv_rn(vmp - c, T));
        const float wpm = expf(__fdiv_rn(vpm - c, T));
        const float wmm = expf(__fdiv_rn(vmm - c, T));
        const float mi = i > 0 ? 1.0f : 0.0f, mj = j > 0 ? 1.0f : 0.0f;
        sx = static_cast<float>(i) * ((wpp - wmp) + mj * (wpm - wmm));
        sy = static_cast<float>(j) * ((wpp - wpm) + mi * (wmp - wmm));
        z = wpp + mi * wmp + mj * (wpm + mi * wmm);
    }
    sx = warp_sum(sx);
    sy = warp_sum(sy);
    z = warp_sum(z);
    const float dx = __fdiv_rn(sx, z), dy = __fdiv_rn(sy, z);
    if (lane == 0) {
        out_kpts[2 * static_cast<size_t>(slot)] = static_cast<float>(x) + dx;
        out_kpts[2 * static_cast<size_t>(slot) + 1] = static_cast<float>(y) + dy;
        out_scores[slot] = c;                               // raw S at the integer peak (G7)
        if (out_off != nullptr) {
            out_off[2 * static_cast<size_t>(slot)] = dx;
            out_off[2 * static_cast<size_t>(slot) + 1] = dy;
        }
    }

    // ---- step a4: bilinear gather of the four corner rows (16-byte loads), fp32 accumulate, L2 norm
    if constexpr (DT >= 0) {
        int x0, x1, y0, y1;
        float fx, fy;
        sample_axis(x, dx, stride, Wd, x0, x1, fx);
        sample_axis(y, dy, stride, Hd, y0, y1, fy);
        const float w00 = (1.0f - fy) * (1.0f - fx), w01 = (1.0f - fy) * fx;
        const float w10 = fy * (1.0f - fx), w11 = fy * fx;
        const size_t rowb = static_cast<size_t>(D) * ESZ;
        const unsigned char* base = desc + static_cast<size_t>(b) * Hd * Wd * rowb;
        const uint4* p00 = reinterpret_cast<const uint4*>(base + (static_cast<size_t>(y0) * Wd + x0) * rowb);
        const uint4* p01 = reinterpret_cast<const uint4*>(base + (static_cast<size_t>(y0) * Wd + x1) * rowb);
        const uint4* p10 = reinterpret_cast<const uint4*>(base + (static_cast<size_t>(y1) * Wd + x0) * rowb);
        const uint4* p11 = reinterpret_cast<const uint4*>(base + (static_cast<size_t>(y1) * Wd + x1) * rowb);
        constexpr int N = ChunkT<DT >= 0 ? DT : 0>::N;
        float acc[MAX_CHUNK_ITERS][N];
        float ss = 0.0f;
#pragma unroll
        for (int it = 0; it < MAX_CHUNK_ITERS; ++it) {
            const int ch = lane + 32 * it;
            if (ch < nchunk) {
                const uint4 q00 = ld_stream16(p00 + ch), q01 = ld_stream16(p01 + ch);
                const uint4 q10 = ld_stream16(p10 + ch), q11 = ld_stream16(p11 + ch);
                float a[N], bq[N], cq[N], dq[N];
                chunk_to_float<DT >= 0 ? DT : 0>(q00, a);
                chunk_to_float<DT >= 0 ? DT : 0>(q01, bq);
                chunk_to_float<DT >= 0 ? DT : 0>(q10, cq);
                chunk_to_float<DT >= 0 ? DT : 0>(q11, dq);
#pragma unroll
                for (int e = 0; e < N; ++e) {
                    const float d = fmaf(w11, dq[e], fmaf(w10, cq[e], fmaf(w01, bq[e], w00 * a[e])));
                    acc[it][e] = d;
                    ss = fmaf(d, d, ss);
                }
            }
        }
        ss = warp_sum(ss);
        const float inv = __fdiv_rn(1.0f, fmaxf(sqrtf(ss), 1e-12f));
        uint4* o = reinterpret_cast<uint4*>(out_desc + static_cast<size_t>(slot) * rowb);
#pragma unroll
        for (int it = 0; it < MAX_CHUNK_ITERS; ++it) {
            const int ch = lane + 32 * it;
            if (ch < nchunk) {
                float f[N];
#pragma unroll
                for (int e = 0; e < N; ++e) f[e] = acc[it][e] * inv;
                o[ch] = float_to_chunk<DT >= 0 ? DT : 0>(f);
            }
        }
    }
}

}  // namespace dkd
