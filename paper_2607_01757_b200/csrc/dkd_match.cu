// dkd_match.cu — the consumers of the descriptor output:
//   k_match_tc        cosine nearest-neighbour matching of two padded, l2-normalised fp16 descriptor sets
//                     (PAPER.md:157): S = A B^T on the 5th-generation tensor cores (tcgen05.mma, fp32
//                     accumulators in TMEM, operands staged by TMA with the 128-byte swizzle), with the
//                     row-wise top-2 fused into the epilogue (tcgen05.ld) — S never reaches memory.
//   k_match_finalize  merge of the column splits, Lowe ratio test, optional mutual check.
//   k_scan            brute-force cosine scan of one global descriptor over the keyframe database
//                     (Eq. 4, 348): an HBM-bound GEMV with the tau gate and the
//                     skip-recent window; the ranked candidate list comes from k_select (dkd_kernels.cuh).
//   k_stereo / k_cov  per-match stereo validation and covariance-weighted square-root
//                     information (Eq. 9-11): elementwise.
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "dkd.h"
#include "dkd_host.h"

#ifdef DKD_DEBUG
#include <assert.h>
#define DKD_ASSERT(c) assert(c)
#else
#define DKD_ASSERT(c) ((void)0)
#endif

namespace dkd {

// ---- PTX wrappers (mbarrier, TMA, tcgen05) ------------------------------------------------------------
__device__ __forceinline__ uint32_t m_smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void m_mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(m_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void m_fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void m_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(m_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void m_mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(m_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void m_mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "MWAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra MDONE;\n"
        "bra MWAIT;\n"
        "MDONE:\n"
        "}" ::"r"(m_smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void m_tma_load_3d(void* dst, const CUtensorMap* tmap, uint64_t* bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(m_smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(m_smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void m_prefetch_tmap(const CUtensorMap* tmap) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(tmap)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// one warp allocates `cols` TMEM columns (power of two >= 32); the base address lands in shared memory
__device__ __forceinline__ void tc_alloc(uint32_t* dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(m_smem_u32(dst_smem)), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tc_dealloc(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc]^T, fp16 inputs, fp32 accumulate; issued by ONE thread
__device__ __forceinline__ void tc_mma_f16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}" ::"r"(tmem_d),
        "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
        : "memory");
}
// the mbarrier receives one arrival when every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(m_smem_u32(bar)) : "memory");
}
// 32 lanes x 32 consecutive fp32 columns: thread t of the warp receives row (lane base + t), columns c .. c+31
__device__ __forceinline__ void tc_ld_32x32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
// true in exactly one lane of a converged warp; the compiler then knows the guarded code runs in a single thread and emits
// the uniform-register instructions (UTCHMMA, UTMALDG) without a per-lane election loop around each of them
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---- k_match_tc -------------------------------------------------------------------------------------------
// One CTA = one block of BM = 128 rows of A (one pair p) against the column tiles [t0, t1) of B, BN = 256 or 128 columns each.
//   warp 0   TMA producer: the A block once (KB boxes of 64 k-elements x 128 rows, 128-byte swizzle), then the B stream in
//            ring UNITS of one k-box (BN rows x 128 bytes: BN / 128 boxes one below the other = one N = BN operand);
//   warp 1   allocates TMEM and, one elect.sync lane of the converged warp, issues the MMAs: per unit 4 tcgen05.mma of
//            128 x BN x 16 into one of two accumulator buffers (128 lanes x BN fp32 columns each); tcgen05.commit frees the
//            unit's shared memory, and after the tile's last unit publishes the accumulator;
//   warps 2..9  epilogue: warp w reads TMEM lanes 32 (w % 4) .. +31 (the hardware's lane quadrant of the warp), the
//            column half h = (w - 2) / 4 of the tile: every thread owns ONE ROW of S and keeps its running
//            (best, arg best, second best) in registers — no cross-thread reduction; columns are visited in
//            increasing order and the comparison is strict, so ties keep the smallest column (M2).
// Rows >= count_a and columns >= count_b (the zero padding of PAPER.md:139) are masked out.
constexpr int MT_BM = 128, MT_KBOX = 64;                         // KBOX fp16 = 128 bytes = the swizzle span
// (the tile width BN = 256 or 128 columns of S is a template parameter: 256-wide MMAs when the problem fills the machine
// with them — they use the tensor pipe better —, 128 for small sets, where more and smaller CTAs finish sooner)
constexpr int MT_BOX_ROWS = 128;                                 // rows of one TMA box (A block: one box per k-box; B unit: two)
constexpr int MT_THREADS = 320;                                  // 10 warps
constexpr int MT_MAX_STAGES = 8;                                 // ring units of the B stream
constexpr int MT_MAX_KB = 4;                                     // D <= 256

struct MatchRec {                      // partial result of one row over one column split
    float best, second;
    int arg;
    int pad;
};

struct MatchParams {
    const int32_t* count_a;            // [P] valid rows of A, device (NULL: Na)
    const int32_t* count_b;            // [P]
    int Na, Nb, KB;                    // KB = D / 64
    int splits, stages;
    MatchRec* part;                    // [P, splits, Na]
};

__device__ __forceinline__ uint64_t mt_desc(uint32_t smem_addr) {
    // K-major operand, 128-byte swizzle: rows of 128 bytes, 8-row groups 1024 bytes apart (SBO), LBO unused (1),
    // descriptor version 1 (sm_100), layout type 2 = SWIZZLE_128B
    return static_cast<uint64_t>((smem_addr >> 4) & 0x3FFFu) | (1ull << 16) | (static_cast<uint64_t>(1024 >> 4) << 32) |
           (1ull << 46) | (2ull << 61);
}

template <int MT_BN>
__global__ void __launch_bounds__(MT_THREADS, 1) k_match_tc(const __grid_constant__ CUtensorMap tmap_a,
                                                            const __grid_constant__ CUtensorMap tmap_b,
                                                            const __grid_constant__ MatchParams p) {
    extern __shared__ __align__(1024) unsigned char mt_smem[];
    __shared__ __align__(8) uint64_t bar_a, bar_full[MT_MAX_STAGES], bar_empty[MT_MAX_STAGES], bar_tfull[2], bar_tempty[2];
    __shared__ uint32_t s_tmem;
    __shared__ MatchRec s_half[MT_BM];                           // the upper column half's result of every row

    constexpr int MT_TMEM_COLS = 2 * MT_BN;                      // two accumulator buffers (BN = 256: all of TMEM)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rb = blockIdx.x, sp = blockIdx.y, pr = blockIdx.z;
    // programmatic dependent launch: the next kernel of the call (the reverse direction, k_match_finalize) may be
    // scheduled while this grid runs; k_match_finalize waits for its predecessor before it reads the partials
    asm volatile("griddepcontrol.launch_dependents;");
    const int na = p.count_a ? min(max(p.count_a[pr], 0), p.Na) : p.Na;
    const int nb = p.count_b ? min(max(p.count_b[pr], 0), p.Nb) : p.Nb;
    const int tiles = (nb + MT_BN - 1) / MT_BN;
    const int t0 = static_cast<int>(static_cast<long long>(tiles) * sp / p.splits);
    const int t1 = static_cast<int>(static_cast<long long>(tiles) * (sp + 1) / p.splits);
    const int row0 = rb * MT_BM;
    const bool active = row0 < na && t1 > t0;                    // (block-uniform)

    const uint32_t a_bytes = static_cast<uint32_t>(p.KB) * MT_BM * 128u;          // A block: KB x 16 KB
    // The B stream moves UNITS of one k-box: 256 rows x 128 bytes = 32 KB (two TMA boxes of 128 rows, one below the other,
    // so that the 8-row groups of the whole unit are 1024 bytes apart: one N = 256 operand).  A tile of 256 columns of S is
    // KB units; a unit's shared memory is released as soon as its four MMAs have read it.
    const uint32_t b_bytes = static_cast<uint32_t>(MT_BN) * 128u;                 // one unit
    unsigned char* smem_a = mt_smem + ((1024u - (m_smem_u32(mt_smem) & 1023u)) & 1023u);   // the swizzle atom is 1024 bytes
    unsigned char* smem_b = smem_a + a_bytes;

    if (threadIdx.x == 0) {
        m_mbar_init(&bar_a, 1);
        for (int s = 0; s < MT_MAX_STAGES; ++s) { m_mbar_init(&bar_full[s], 1); m_mbar_init(&bar_empty[s], 1); }
        for (int a = 0; a < 2; ++a) { m_mbar_init(&bar_tfull[a], 1); m_mbar_init(&bar_tempty[a], 256); }
        m_fence_mbar_init();
    }
    if (warp == 1) tc_alloc(&s_tmem, MT_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;

    if (active) {
        if (warp == 0) {
            if (lane == 0) {                                     // ===== TMA producer =====
                m_prefetch_tmap(&tmap_a);
                m_prefetch_tmap(&tmap_b);
                m_mbar_expect_tx(&bar_a, a_bytes);
                for (int kb = 0; kb < p.KB; ++kb) m_tma_load_3d(smem_a + kb * (MT_BM * 128), &tmap_a, &bar_a, kb * MT_KBOX, row0, pr);
                for (int t = t0, iu = 0; t < t1; ++t) {
                    for (int kb = 0; kb < p.KB; ++kb, ++iu) {
                        const int s = iu % p.stages;
                        if (iu >= p.stages) m_mbar_wait(&bar_empty[s], ((iu / p.stages) - 1) & 1);
                        m_mbar_expect_tx(&bar_full[s], b_bytes);
                        m_tma_load_3d(smem_b + s * b_bytes, &tmap_b, &bar_full[s], kb * MT_KBOX, t * MT_BN, pr);
                        if (MT_BN > MT_BOX_ROWS)
                            m_tma_load_3d(smem_b + s * b_bytes + MT_BOX_ROWS * 128, &tmap_b, &bar_full[s], kb * MT_KBOX, t * MT_BN + MT_BOX_ROWS, pr);
                    }
                }
            }
        } else if (warp == 1) {
            {                                                    // ===== MMA issuer: the warp stays converged, one elected lane issues =====
                // instruction descriptor: D = F32 (bits 4-5 = 1), A = B = F16 (0), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
                const uint32_t idesc = (1u << 4) | (static_cast<uint32_t>(MT_BN >> 3) << 17) | (static_cast<uint32_t>(MT_BM >> 4) << 24);
                m_mbar_wait(&bar_a, 0);
                const uint64_t a_base = mt_desc(m_smem_u32(smem_a));
                for (int t = t0, it = 0, iu = 0; t < t1; ++t, ++it) {
                    const int acc = it & 1;
                    if (it >= 2) m_mbar_wait(&bar_tempty[acc], ((it >> 1) - 1) & 1);   // the epilogue has drained this buffer
                    const uint32_t d_tmem = tmem + acc * MT_BN;
                    for (int kb = 0; kb < p.KB; ++kb, ++iu) {
                        const int s = iu % p.stages;
                        m_mbar_wait(&bar_full[s], (iu / p.stages) & 1);
                        tc_fence_after();
                        // One thread issues every tcgen05.mma, and the tensor pipe is busy for only ~128 cycles per 128 x 256 x
                        // 16 MMA: the descriptors must not cost a dependent chain each.  The 14-bit address field holds
                        // (address >> 4) of a buffer below 256 KB, so the descriptor of a later K step is the base descriptor
                        // plus a constant — one independent add per MMA.
                        const uint64_t b_base = mt_desc(m_smem_u32(smem_b + s * b_bytes));
                        const uint64_t a_kb = a_base + static_cast<uint64_t>((kb * (MT_BM * 128)) >> 4);
                        if (elect_one()) {
#pragma unroll
                            for (int k = 0; k < MT_KBOX / 16; ++k)   // UMMA_K = 16 fp16 = 32 bytes inside the swizzle atom
                                tc_mma_f16(d_tmem, a_kb + static_cast<uint64_t>((k * 32) >> 4), b_base + static_cast<uint64_t>((k * 32) >> 4),
                                           idesc, (kb | k) != 0);
                            tc_commit(&bar_empty[s]);            // the unit's shared memory is free once these MMAs have read it
                            if (kb + 1 == p.KB) tc_commit(&bar_tfull[acc]);   // accumulator complete
                        }
                        __syncwarp();
                    }
                }
            }
        } else {                                                 // ===== epilogue: one thread per row and column half =====
            const int q = warp & 3, h = (warp - 2) >> 2;
            const int row = row0 + 32 * q + lane;
            float best = -INFINITY, second = -INFINITY;
            int arg = -1;
            for (int t = t0, it = 0; t < t1; ++t, ++it) {
                const int acc = it & 1;
                m_mbar_wait(&bar_tfull[acc], (it >> 1) & 1);
                tc_fence_after();
#pragma unroll
                for (int c = 0; c < MT_BN / 2; c += 32) {
                    uint32_t v[32];
                    tc_ld_32x32(tmem + (static_cast<uint32_t>(32 * q) << 16) + acc * MT_BN + (MT_BN / 2) * h + c, v);
                    tc_wait_ld();
                    const int col0 = t * MT_BN + (MT_BN / 2) * h + c;
                    if (col0 + 32 <= nb) {
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const float x = __uint_as_float(v[j]);
                            const bool gt = x > best;
                            second = gt ? best : fmaxf(second, x);
                            arg = gt ? col0 + j : arg;
                            best = gt ? x : best;
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const float x = col0 + j < nb ? __uint_as_float(v[j]) : -INFINITY;
                            const bool gt = x > best;
                            second = gt ? best : fmaxf(second, x);
                            arg = gt ? col0 + j : arg;
                            best = gt ? x : best;
                        }
                    }
                }
                tc_fence_before();
                m_mbar_arrive(&bar_tempty[acc]);
            }
            // combine the two column halves of a row (lower columns first: ties keep the smaller column)
            if (h == 1) {
                MatchRec r;
                r.best = best; r.second = second; r.arg = arg; r.pad = 0;
                s_half[32 * q + lane] = r;
            }
            asm volatile("bar.sync 1, 256;" ::: "memory");      // the 8 epilogue warps only
            if (h == 0 && row < p.Na) {
                // per tile the halves interleave (cols 0-63 | 64-127 | 128-191 ...): merge by value, ties by column
                const MatchRec o = s_half[32 * q + lane];
                MatchRec r;
                if (o.best > best || (o.best == best && o.arg >= 0 && (arg < 0 || o.arg < arg))) {
                    r.best = o.best; r.arg = o.arg; r.second = fmaxf(best, o.second);
                } else {
                    r.best = best; r.arg = arg; r.second = fmaxf(second, o.best);
                }
                r.pad = 0;
                p.part[(static_cast<size_t>(pr) * p.splits + sp) * p.Na + row] = r;
            }
        }
    } else if (warp >= 2 && (warp - 2) < 4) {                    // no work for this CTA: neutral partials
        const int row = row0 + 32 * (warp & 3) + lane;
        if (row < p.Na) {
            MatchRec r;
            r.best = -INFINITY; r.second = -INFINITY; r.arg = -1; r.pad = 0;
            p.part[(static_cast<size_t>(pr) * p.splits + sp) * p.Na + row] = r;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tc_dealloc(tmem, MT_TMEM_COLS);
    }
    // Launched with the programmatic attribute (the reverse direction of a mutual match) this grid read nothing its
    // predecessor wrote; it only must not COMPLETE before it, so that k_match_finalize's wait covers both directions.
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// merge of the column splits (in column order), ratio test (M3), mutual check (M4)
struct FinalizeParams {
    const MatchRec* part;              // [P, splits, Na]
    const MatchRec* rpart;             // [P, rsplits, Nb]: the reverse direction (mutual check) or NULL
    const int32_t* count_a;
    int Na, Nb, splits, rsplits, P;
    float ratio2;                      // rho^2, or < 0: ratio test disabled
    int32_t* out_match;                // [P, Na]
    float* out_sim;                    // [P, Na, 2] or NULL
};
__device__ __forceinline__ MatchRec merge_splits(const MatchRec* part, int splits, size_t stride) {
    MatchRec r = part[0];
    for (int s = 1; s < splits; ++s) {
        const MatchRec o = part[s * stride];
        if (o.best > r.best) { r.second = fmaxf(r.best, o.second); r.best = o.best; r.arg = o.arg; }
        else r.second = fmaxf(r.second, o.best);
    }
    return r;
}
__global__ void __launch_bounds__(256) k_match_finalize(const __grid_constant__ FinalizeParams p) {
    const int i = blockIdx.x * 256 + threadIdx.x, pr = blockIdx.y;
    asm volatile("griddepcontrol.wait;" ::: "memory");      // the partials of k_match_tc are complete and visible
    if (i >= p.Na) return;
    const int na = p.count_a ? min(max(p.count_a[pr], 0), p.Na) : p.Na;
    int m = -1;
    float s1 = 0.0f, s2 = 0.0f;
    if (i < na) {
        const MatchRec r = merge_splits(p.part + static_cast<size_t>(pr) * p.splits * p.Na + i, p.splits, p.Na);
        if (r.arg >= 0) {
            s1 = r.best;
            s2 = r.second == -INFINITY ? -1.0f : r.second;       // a single column: the smallest cosine (M2)
            bool keep = true;
            if (p.ratio2 >= 0.0f) {
                const float d1 = fmaxf(2.0f - 2.0f * s1, 0.0f), d2 = fmaxf(2.0f - 2.0f * s2, 0.0f);
                keep = d1 < p.ratio2 * d2;
            }
            if (keep && p.rpart != nullptr) {
                const MatchRec rr = merge_splits(p.rpart + static_cast<size_t>(pr) * p.rsplits * p.Nb + r.arg, p.rsplits, p.Nb);
                keep = rr.arg == i;
            }
            if (keep) m = r.arg;
        }
    }
    p.out_match[static_cast<size_t>(pr) * p.Na + i] = m;
    if (p.out_sim) {
        p.out_sim[(static_cast<size_t>(pr) * p.Na + i) * 2] = s1;
        p.out_sim[(static_cast<size_t>(pr) * p.Na + i) * 2 + 1] = s2;
    }
}

// ---- k_scan: sim_k = q . db_k over the keyframe database ------------------------------------------------------
// One WARP per database row, SC_R rows at a time: lane l owns the 16-byte chunks l, l + 32, ... of a row, SC_R x SC_U of
// them in flight per lane (streaming loads, no L1 allocation), multiplied with the query held in shared memory as
// fp32.  No block-wide barrier after the query is staged, no cross-warp reduction: a row's sum is its lanes' sequential
// partial sums combined by a shuffle tree — a fixed order that does not depend on the grid.  Rows that pass the gate
// (k < n - n_exclude, sim > tau) are appended by lane 0 to the warp's private key segment in row order (no atomics) for
// k_select to rank.  Every row is read exactly once: HBM-bound.
constexpr int SC_THREADS = 256;
constexpr int SC_U = 4;                                            // chunks per lane and row in flight
constexpr int SC_R = 4;                                            // rows per warp step (the query chunk is unpacked once for all of them)
__device__ __forceinline__ uint4 ld_stream16_plain(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
template <int DT> struct ScanChunk;
template <> struct ScanChunk<DKD_F16> { static constexpr int N = 8; };
template <> struct ScanChunk<DKD_F32> { static constexpr int N = 4; };
template <int DT>
__device__ __forceinline__ void scan_unpack(const uint4& q, float* f) {
    if constexpr (DT == DKD_F16) {
        const __half2* h = reinterpret_cast<const __half2*>(&q);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 t = __half22float2(h[i]);
            f[2 * i] = t.x;
            f[2 * i + 1] = t.y;
        }
    } else {
        f[0] = __uint_as_float(q.x); f[1] = __uint_as_float(q.y); f[2] = __uint_as_float(q.z); f[3] = __uint_as_float(q.w);
    }
}
__device__ __forceinline__ uint64_t scan_key(float s, int k) {     // same key as the DKD selection: (score desc, index asc)
    uint32_t b = __float_as_uint(s + 0.0f);
    b ^= (b & 0x80000000u) ? 0xFFFFFFFFu : 0x80000000u;
    return (static_cast<uint64_t>(b) << 32) | static_cast<uint32_t>(~static_cast<uint32_t>(k));
}

struct ScanParams {
    const unsigned char* db;
    const unsigned char* q;
    int n, chunks;                     // rows; 16-byte chunks per row
    int n_eligible;                    // rows k < n_eligible may be candidates (n - n_exclude)
    float tau;
    float* out_sim;                    // [n]
    uint64_t* seg;                     // [warps of the grid, seg_cap] candidate keys
    int* seg_cnt;                      // [warps of the grid]
    int seg_cap;
};

template <int DT>
__global__ void __launch_bounds__(SC_THREADS, 2) k_scan(const __grid_constant__ ScanParams p) {
    constexpr int N = ScanChunk<DT>::N;
    extern __shared__ __align__(16) float s_q[];                  // the query as fp32: chunks * N floats
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int ch = tid; ch < p.chunks; ch += SC_THREADS) {
        float f[N];
        scan_unpack<DT>(__ldg(reinterpret_cast<const uint4*>(p.q) + ch), f);
#pragma unroll
        for (int e = 0; e < N; ++e) s_q[ch * N + e] = f[e];
    }
    __syncthreads();
    const int gw = blockIdx.x * (SC_THREADS / 32) + warp, nw = gridDim.x * (SC_THREADS / 32);
    const size_t rowb = static_cast<size_t>(p.chunks) * 16;
    uint64_t* my_seg = p.seg + static_cast<size_t>(gw) * p.seg_cap;
    int cnt = 0;
    for (int k0 = SC_R * gw; k0 < p.n; k0 += SC_R * nw) {
        const uint4* rp[SC_R];
#pragma unroll
        for (int r = 0; r < SC_R; ++r)                            // rows past the end alias the last row (discarded below)
            rp[r] = reinterpret_cast<const uint4*>(p.db + static_cast<size_t>(k0 + r < p.n ? k0 + r : p.n - 1) * rowb);
        float acc[SC_R];
#pragma unroll
        for (int r = 0; r < SC_R; ++r) acc[r] = 0.0f;
        for (int c0 = lane; c0 < p.chunks; c0 += 32 * SC_U) {
            uint4 raw[SC_U][SC_R];
#pragma unroll
            for (int u = 0; u < SC_U; ++u) {
                const int ch = c0 + 32 * u;
#pragma unroll
                for (int r = 0; r < SC_R; ++r) {
                    raw[u][r] = make_uint4(0u, 0u, 0u, 0u);
                    if (ch < p.chunks) raw[u][r] = ld_stream16_plain(rp[r] + ch);
                }
            }
#pragma unroll
            for (int u = 0; u < SC_U; ++u) {
                const int ch = c0 + 32 * u;
                if (ch < p.chunks) {
                    float fq[N];
                    const float4* qp = reinterpret_cast<const float4*>(s_q + ch * N);
#pragma unroll
                    for (int v = 0; v < N / 4; ++v) {
                        const float4 t = qp[v];
                        fq[4 * v] = t.x; fq[4 * v + 1] = t.y; fq[4 * v + 2] = t.z; fq[4 * v + 3] = t.w;
                    }
#pragma unroll
                    for (int r = 0; r < SC_R; ++r) {
                        float f[N];
                        scan_unpack<DT>(raw[u][r], f);
#pragma unroll
                        for (int e = 0; e < N; ++e) acc[r] = fmaf(f[e], fq[e], acc[r]);
                    }
                }
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int r = 0; r < SC_R; ++r) acc[r] += __shfl_xor_sync(0xffffffffu, acc[r], o);
        }
        if (lane == 0) {
#pragma unroll
            for (int r = 0; r < SC_R; ++r) {
                const int k = k0 + r;
                if (k < p.n) {
                    p.out_sim[k] = acc[r];
                    if (k < p.n_eligible && acc[r] > p.tau) { DKD_ASSERT(cnt < p.seg_cap); my_seg[cnt++] = scan_key(acc[r], k); }
                }
            }
        }
    }
    if (lane == 0) p.seg_cnt[gw] = cnt;
}

__global__ void k_cand_sims(const int32_t* __restrict__ cand, const float* __restrict__ sim, int max_cand, float* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < max_cand) out[i] = cand[i] >= 0 ? sim[cand[i]] : 0.0f;
}

// ---- f4: per-match stereo validation (S1..S4) and covariance-weighted sqrt information (C1..C4) -------------------
struct StereoKParams {
    const float* kl; const float* kr; const int32_t* match;
    int n;
    float fx, fy, cx, cy, baseline, d_min, z_min, z_max, max_reproj;
    float* xyz; float* disp; float* err; uint8_t* valid;
};
__global__ void __launch_bounds__(256) k_stereo(const __grid_constant__ StereoKParams p) {
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= p.n) return;
    const int j = p.match ? p.match[i] : i;
    float X = 0.0f, Y = 0.0f, z = 0.0f, d = 0.0f, e = 0.0f;
    uint8_t ok = 0;
    if (j >= 0) {
        const float2 l = reinterpret_cast<const float2*>(p.kl)[i], r = reinterpret_cast<const float2*>(p.kr)[j];
        d = l.x - r.x;                                               // S1
        if (d > p.d_min) {
            z = __fdiv_rn(p.fx * p.baseline, d);                     // S2
            const float vm = 0.5f * (l.y + r.y);
            X = __fdiv_rn((l.x - p.cx) * z, p.fx);
            Y = __fdiv_rn((vm - p.cy) * z, p.fy);
            // S4: in this rectified model both views are off by |vL - vR| / 2 (the u residual is zero by construction)
            e = 0.5f * fabsf(l.y - r.y);
            ok = (z > p.z_min && z < p.z_max && e <= p.max_reproj) ? 1 : 0;
        }
    }
    p.xyz[3 * i] = X; p.xyz[3 * i + 1] = Y; p.xyz[3 * i + 2] = z;
    if (p.disp) p.disp[i] = d;
    if (p.err) p.err[i] = e;
    p.valid[i] = ok;
}

struct CovKParams {
    const float* L;
    int n;
    float s2, floor_px, inv_fx2, inv_fy2, inv_fxfy, lam, inv_sigma0;
    float* omega; uint8_t* ok;
};
__global__ void __launch_bounds__(256) k_cov(const __grid_constant__ CovKParams p) {
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= p.n) return;
    const float l11 = p.L[3 * i], l21 = p.L[3 * i + 1], l22 = p.L[3 * i + 2];
    const float a = p.s2 * (l11 * l11) + p.floor_px, b = p.s2 * (l11 * l21), c = p.s2 * (l21 * l21 + l22 * l22) + p.floor_px;
    const float na = a * p.inv_fx2, nb = b * p.inv_fxfy, nc = c * p.inv_fy2;              // Eq. 9
    // det(Sigma_px) as a sum of non-negative terms (C4): its sign cannot be flipped by rounding
    const float det_px = p.s2 * p.s2 * (l11 * l11) * (l22 * l22) + p.floor_px * p.s2 * (l11 * l11 + l21 * l21 + l22 * l22) +
                         p.floor_px * p.floor_px;
    const float det = det_px * p.inv_fx2 * p.inv_fy2;
    bool ok = isfinite(na) && isfinite(nb) && isfinite(nc) && na > 0.0f && det > 0.0f && isfinite(det);
    float o00 = p.inv_sigma0, o01 = 0.0f, o11 = p.inv_sigma0;
    if (ok) {
        // Omega^T Omega = lam Sigma_n^-1 = (lam / det) [[nc, -nb], [-nb, na]]; its Cholesky factor in closed form:
        // c11 = sqrt(lam nc / det), c21 = -lam nb / (det c11), c22^2 = lam na / det - c21^2 = lam / nc  (no cancellation)
        const float ia = p.lam * nc / det;
        const float c11 = sqrtf(ia);
        const float c21 = -p.lam * nb / (det * c11);
        const float c22 = sqrtf(p.lam / nc);
        if (ia > 0.0f && nc > 0.0f && isfinite(c11) && isfinite(c21) && isfinite(c22) && c22 > 0.0f) { o00 = c11; o01 = c21; o11 = c22; }
        else ok = false;
    }
    p.omega[4 * i] = o00; p.omega[4 * i + 1] = o01; p.omega[4 * i + 2] = 0.0f; p.omega[4 * i + 3] = o11;
    if (p.ok) p.ok[i] = ok ? 1 : 0;
}

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
PFN_encodeTiled get_encode() {
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<PFN_encodeTiled>(f);
        (void)cudaGetLastError();
    }
    return fn;
}
// [P, N, D] fp16 row-major -> 3-D map (k, row, pair), box (64, 128, 1), 128-byte swizzle, zero fill past the end
bool encode_desc_map(CUtensorMap* m, const void* base, int N, int D, int P) {
    PFN_encodeTiled enc = get_encode();
    if (!enc) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)N, (cuuint64_t)P};
    const cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)D * 2 * N};
    const cuuint32_t box[3] = {(cuuint32_t)MT_KBOX, (cuuint32_t)MT_BOX_ROWS, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// tile width: 256 columns when row blocks x pairs x 256-wide tiles fill the machine, else 128
int match_bn(int num_sms, int Na, int Nb, int P) {
    const long long work = static_cast<long long>((Na + MT_BM - 1) / MT_BM) * P * ((Nb + 255) / 256);
    return work >= num_sms ? 256 : 128;
}
int match_splits(int num_sms, int Na, int Nb, int P) {
    const int bn = match_bn(num_sms, Na, Nb, P);
    const int rbs = (Na + MT_BM - 1) / MT_BM, tiles = (Nb + bn - 1) / bn;
    int s = num_sms / (rbs * P > 0 ? rbs * P : 1);               // fill the machine once
    if (s < 1) s = 1;
    if (s > tiles) s = tiles;
    if (s > 16) s = 16;
    return s;
}

// One direction of the match.  The first direction of a call must be launched with pdl = false: k_match_tc reads the
// counts and issues its TMA loads BEFORE its griddepcontrol.wait (which sits at the kernel's end), so only a launch that
// read nothing its predecessor wrote — the reverse direction — may carry the programmatic attribute.
cudaError_t launch_match_dir(int num_sms, const void* A, const int32_t* ca, int Na, const void* B, const int32_t* cb, int Nb, int D,
                             int P, int splits, MatchRec* part, cudaStream_t st, bool pdl) {
    CUtensorMap ta, tb;
    if (!encode_desc_map(&ta, A, Na, D, P) || !encode_desc_map(&tb, B, Nb, D, P)) return cudaErrorInvalidValue;
    MatchParams mp;
    memset(&mp, 0, sizeof(mp));
    mp.count_a = ca; mp.count_b = cb; mp.Na = Na; mp.Nb = Nb; mp.KB = D / MT_KBOX; mp.splits = splits; mp.part = part;
    const int bn = match_bn(num_sms, Na, Nb, P);
    const size_t a_bytes = static_cast<size_t>(mp.KB) * MT_BM * 128, b_bytes = static_cast<size_t>(bn) * 128;   // A block, one B unit
    int stages = static_cast<int>((200 * 1024 - a_bytes) / b_bytes);
    if (stages > MT_MAX_STAGES) stages = MT_MAX_STAGES;
    mp.stages = stages;
    const size_t smem = a_bytes + stages * b_bytes + 1024;
    const dim3 grid((Na + MT_BM - 1) / MT_BM, splits, P);
    KLaunch k;
    if (bn == 256) prep(k, k_match_tc<256>, grid, dim3(MT_THREADS), smem, pdl, ta, tb, mp);
    else prep(k, k_match_tc<128>, grid, dim3(MT_THREADS), smem, pdl, ta, tb, mp);
    return launch(k, st, true);
}

// ---- dkd_match_static: the matcher with its partials in memory that is part of the loaded library ---------------------
// The column-split partials of k_match_tc normally live in a context-owned buffer that dkd_create / dkd_match obtain
// with cudaMalloc.  This array is the same buffer as a file-scope device variable: it comes into existence when the
// library's module is loaded on a GPU and stays until the process exits (1 MiB on every GPU that loads the library).
constexpr size_t MT_STATIC_RECS = DKD_MATCH_STATIC_MAX_RECS;
static __device__ __align__(256) MatchRec g_match_static[MT_STATIC_RECS];

// `g_match_static` named in HOST code is only the host-side handle of the variable, not an address the GPU can use;
// the device address is asked for once per device (with that device current) and kept here with the SM count.
constexpr int MT_STATIC_MAX_DEVICES = 64;
struct MatchStaticDev {
    MatchRec* part;                    // device address of g_match_static on this device
    int num_sms;
    bool ready;
};
static MatchStaticDev g_ms_dev[MT_STATIC_MAX_DEVICES];
static std::mutex g_ms_mutex;

// set-up of the current device `dev` (first call on it): symbol address, SM count, shared-memory limits of k_match_tc
cudaError_t match_static_setup(int dev, MatchStaticDev* out) {
    std::lock_guard<std::mutex> lk(g_ms_mutex);
    MatchStaticDev& d = g_ms_dev[dev];
    if (!d.ready) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_match_static);
        if (e != cudaSuccess) return e;
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        e = dkd_match_setup_device();
        if (e != cudaSuccess) return e;
        d.part = static_cast<MatchRec*>(ptr);
        d.num_sms = sms;
        d.ready = true;
    }
    *out = d;
    return cudaSuccess;
}

int match_static_fail(char* err, int err_len, int code, const char* msg, const char* detail) {
    if (err && err_len > 0) snprintf(err, static_cast<size_t>(err_len), "%s%s", msg, detail ? detail : "");
    return code;
}

}  // namespace dkd

using namespace dkd;

// Dynamic shared-memory limits of the kernels of this file.  cudaFuncSetAttribute acts on the CURRENT device only, so
// this runs once per context from dkd_create (with the context's device current), not once per process.
cudaError_t dkd_match_setup_device() {
    cudaError_t e = cudaFuncSetAttribute(k_match_tc<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, 204 * 1024);   // (static smem takes ~3 KB of the 227)
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_match_tc<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, 204 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scan<DKD_F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_scan<DKD_F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    // The remaining kernels of this file are loaded now as well (the runtime loads device functions lazily, on first use):
    // a first dkd_match / dkd_retrieval_scan made inside a stream capture must not trigger a module load there.
    cudaFuncAttributes fa;
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, k_match_finalize);
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, k_cand_sims);
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, k_stereo);
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, k_cov);
    if (e == cudaSuccess && get_encode() == nullptr) e = cudaErrorNotSupported;   // (also resolves cuTensorMapEncodeTiled once)
    return e;
}

extern "C" {

int dkd_match(dkd_ctx* ctx, const void* desc_a, const int32_t* count_a, int Na, const void* desc_b, const int32_t* count_b,
              int Nb, int D, int dtype, int P, float ratio, int mutual, int32_t* out_match, float* out_sim, void* stream) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (!desc_a || !desc_b || !out_match || Na < 1 || Nb < 1 || D < 1 || P < 1 || !(ratio > 0.0f))
        return dkd_ctx_fail(ctx, DKD_ERR_INVALID_ARG, "dkd_match: NULL pointer, size < 1 or ratio <= 0", nullptr);
    if (dtype != DKD_F16) return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_match: descriptors must be DKD_F16 (tcgen05 kind::f16)", nullptr);
    if (D % MT_KBOX != 0 || D > MT_KBOX * MT_MAX_KB)
        return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_match: D must be 64, 128, 192 or 256", nullptr);
    if (P > 65535) return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_match: P > 65535", nullptr);
    if ((reinterpret_cast<uintptr_t>(desc_a) & 15) || (reinterpret_cast<uintptr_t>(desc_b) & 15))
        return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_match: descriptor sets not 16-byte aligned", nullptr);
    DeviceGuard dg(dkd_ctx_device(ctx));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int sms = dkd_ctx_num_sms(ctx);
    const int s_ab = match_splits(sms, Na, Nb, P), s_ba = mutual ? match_splits(sms, Nb, Na, P) : 0;
    const size_t n_ab = static_cast<size_t>(P) * s_ab * Na, n_ba = static_cast<size_t>(P) * s_ba * Nb;
    MatchRec* part = static_cast<MatchRec*>(dkd_ctx_scratch(ctx, 0, (n_ab + n_ba) * sizeof(MatchRec)));
    if (!part) return DKD_ERR_CUDA;
    // the first kernel waits for whatever precedes it on the stream (it produced the descriptors); the reverse direction and
    // the finalize kernel are programmatic dependents
    cudaError_t e = launch_match_dir(sms, desc_a, count_a, Na, desc_b, count_b, Nb, D, P, s_ab, part, st, false);
    if (e == cudaSuccess && mutual) e = launch_match_dir(sms, desc_b, count_b, Nb, desc_a, count_a, Na, D, P, s_ba, part + n_ab, st, true);
    if (e != cudaSuccess) return dkd_ctx_fail(ctx, DKD_ERR_CUDA, "dkd_match launch: ", cudaGetErrorString(e));
    FinalizeParams fp;
    memset(&fp, 0, sizeof(fp));
    fp.part = part; fp.rpart = mutual ? part + n_ab : nullptr; fp.count_a = count_a; fp.Na = Na; fp.Nb = Nb; fp.splits = s_ab;
    fp.rsplits = s_ba; fp.P = P; fp.ratio2 = ratio >= 1e9f ? -1.0f : ratio * ratio; fp.out_match = out_match; fp.out_sim = out_sim;
    {
        KLaunch k;
        prep(k, k_match_finalize, dim3((Na + 255) / 256, P), dim3(256), 0, true, fp);
        e = launch(k, st, true);
    }
    if (e != cudaSuccess) return dkd_ctx_fail(ctx, DKD_ERR_CUDA, "k_match_finalize launch: ", cudaGetErrorString(e));
    return DKD_OK;
}

int dkd_match_static(const void* desc_a, const int32_t* count_a, int Na, const void* desc_b, const int32_t* count_b, int Nb,
                     int D, int dtype, int P, float ratio, int mutual, int32_t* out_match, float* out_sim, void* stream,
                     char* err, int err_len) {
    if (err && err_len > 0) err[0] = '\0';
    if (!desc_a || !desc_b || !out_match || Na < 1 || Nb < 1 || D < 1 || P < 1 || !(ratio > 0.0f))
        return match_static_fail(err, err_len, DKD_ERR_INVALID_ARG, "dkd_match_static: NULL pointer, size < 1 or ratio <= 0", nullptr);
    if (dtype != DKD_F16)
        return match_static_fail(err, err_len, DKD_ERR_UNSUPPORTED, "dkd_match_static: descriptors must be DKD_F16", nullptr);
    if (D % MT_KBOX != 0 || D > MT_KBOX * MT_MAX_KB)
        return match_static_fail(err, err_len, DKD_ERR_UNSUPPORTED, "dkd_match_static: D must be 64, 128, 192 or 256", nullptr);
    if (P > 65535) return match_static_fail(err, err_len, DKD_ERR_UNSUPPORTED, "dkd_match_static: P > 65535", nullptr);
    if ((reinterpret_cast<uintptr_t>(desc_a) & 15) || (reinterpret_cast<uintptr_t>(desc_b) & 15))
        return match_static_fail(err, err_len, DKD_ERR_UNSUPPORTED, "dkd_match_static: descriptor sets not 16-byte aligned", nullptr);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return match_static_fail(err, err_len, DKD_ERR_CUDA, "dkd_match_static: cudaGetDevice: ", cudaGetErrorString(e));
    if (dev < 0 || dev >= MT_STATIC_MAX_DEVICES)
        return match_static_fail(err, err_len, DKD_ERR_UNSUPPORTED, "dkd_match_static: device ordinal above 63", nullptr);
    MatchStaticDev d;
    e = match_static_setup(dev, &d);
    if (e != cudaSuccess) return match_static_fail(err, err_len, DKD_ERR_CUDA, "dkd_match_static: device set-up: ", cudaGetErrorString(e));
    const int s_ab = match_splits(d.num_sms, Na, Nb, P), s_ba = mutual ? match_splits(d.num_sms, Nb, Na, P) : 0;
    const size_t n_ab = static_cast<size_t>(P) * s_ab * Na, n_ba = static_cast<size_t>(P) * s_ba * Nb;
    if (n_ab + n_ba > MT_STATIC_RECS) {
        char buf[160];
        snprintf(buf, sizeof(buf), "needs %zu partial records (P x column splits x rows, both directions if mutual), the built-in buffer holds %zu",
                 n_ab + n_ba, MT_STATIC_RECS);
        return match_static_fail(err, err_len, DKD_ERR_CAPACITY, "dkd_match_static: problem too large: ", buf);
    }
    // Nothing in the buffer has to be cleared: every record k_match_finalize reads (rows < Na of every split and pair,
    // rows < Nb of the reverse direction) is written by k_match_tc earlier in this same call.
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    MatchRec* part = d.part;
    e = launch_match_dir(d.num_sms, desc_a, count_a, Na, desc_b, count_b, Nb, D, P, s_ab, part, st, false);
    if (e == cudaSuccess && mutual)
        e = launch_match_dir(d.num_sms, desc_b, count_b, Nb, desc_a, count_a, Na, D, P, s_ba, part + n_ab, st, true);
    if (e != cudaSuccess) return match_static_fail(err, err_len, DKD_ERR_CUDA, "dkd_match_static: k_match_tc launch: ", cudaGetErrorString(e));
    FinalizeParams fp;
    memset(&fp, 0, sizeof(fp));
    fp.part = part; fp.rpart = mutual ? part + n_ab : nullptr; fp.count_a = count_a; fp.Na = Na; fp.Nb = Nb; fp.splits = s_ab;
    fp.rsplits = s_ba; fp.P = P; fp.ratio2 = ratio >= 1e9f ? -1.0f : ratio * ratio; fp.out_match = out_match; fp.out_sim = out_sim;
    KLaunch k;
    prep(k, k_match_finalize, dim3((Na + 255) / 256, P), dim3(256), 0, true, fp);
    e = launch(k, st, true);
    if (e != cudaSuccess) return match_static_fail(err, err_len, DKD_ERR_CUDA, "dkd_match_static: k_match_finalize launch: ", cudaGetErrorString(e));
    return DKD_OK;
}

int dkd_retrieval_scan(dkd_ctx* ctx, const void* db, int dtype, int n, int D, const void* query, int n_exclude, float tau,
                       int max_cand, float* out_sim, int32_t* out_cand, float* out_cand_sim, int32_t* out_count, void* stream) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (!query || !out_cand || !out_count || n < 0 || (n > 0 && !db) || D < 1 || n_exclude < 0 || max_cand < 1 || isnan(tau))
        return dkd_ctx_fail(ctx, DKD_ERR_INVALID_ARG, "dkd_retrieval_scan: NULL pointer or bad size", nullptr);
    if (dtype != DKD_F16 && dtype != DKD_F32) return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_retrieval_scan: dtype must be DKD_F16 or DKD_F32", nullptr);
    const size_t rowb = static_cast<size_t>(D) * (dtype == DKD_F16 ? 2 : 4);
    if (rowb % 16 != 0 || D > 16384)
        return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_retrieval_scan: D * elemsize must be a multiple of 16 and D <= 16384", nullptr);
    if ((reinterpret_cast<uintptr_t>(db) & 15) || (reinterpret_cast<uintptr_t>(query) & 15))
        return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_retrieval_scan: db / query not 16-byte aligned", nullptr);
    if (max_cand > DKD_MAX_TOP_K) return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_retrieval_scan: max_cand > DKD_MAX_TOP_K", nullptr);
    DeviceGuard dg(dkd_ctx_device(ctx));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    constexpr int WPB = SC_THREADS / 32;
    int grid = 2 * dkd_ctx_num_sms(ctx);
    if (grid > (n + SC_R * WPB - 1) / (SC_R * WPB)) grid = (n + SC_R * WPB - 1) / (SC_R * WPB);
    if (grid < 1) grid = 1;
    const int nwarps = grid * WPB;
    const int seg_cap = SC_R * ((n + SC_R * nwarps - 1) / (SC_R * nwarps)) + SC_R;      // rows one warp can see
    const size_t b_seg = (static_cast<size_t>(nwarps) * seg_cap * 8 + 255) & ~static_cast<size_t>(255);
    const size_t b_cnt = (static_cast<size_t>(nwarps) * 4 + 255) & ~static_cast<size_t>(255);
    const size_t b_sim = out_sim ? 0 : ((static_cast<size_t>(n > 0 ? n : 1) * 4 + 255) & ~static_cast<size_t>(255));
    unsigned char* ws = static_cast<unsigned char*>(dkd_ctx_scratch(ctx, 1, b_seg + b_cnt + b_sim));
    if (!ws) return DKD_ERR_CUDA;
    ScanParams sp;
    memset(&sp, 0, sizeof(sp));
    sp.db = static_cast<const unsigned char*>(db); sp.q = static_cast<const unsigned char*>(query);
    sp.n = n; sp.chunks = static_cast<int>(rowb / 16); sp.n_eligible = n - n_exclude; sp.tau = tau;
    sp.out_sim = out_sim ? out_sim : reinterpret_cast<float*>(ws + b_seg + b_cnt);
    sp.seg = reinterpret_cast<uint64_t*>(ws); sp.seg_cnt = reinterpret_cast<int*>(ws + b_seg); sp.seg_cap = seg_cap;
    const size_t smem_q = static_cast<size_t>(D) * 4;
    if (dtype == DKD_F16) k_scan<DKD_F16><<<grid, SC_THREADS, smem_q, st>>>(sp);
    else k_scan<DKD_F32><<<grid, SC_THREADS, smem_q, st>>>(sp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return dkd_ctx_fail(ctx, DKD_ERR_CUDA, "k_scan launch: ", cudaGetErrorString(e));
    const int rc = dkd_internal_select(ctx, sp.seg, sp.seg_cnt, nwarps, seg_cap, max_cand, n > 0 ? n : 1, out_cand, out_count, st);
    if (rc != DKD_OK) return rc;
    if (out_cand_sim) {
        k_cand_sims<<<(max_cand + 255) / 256, 256, 0, st>>>(out_cand, sp.out_sim, max_cand, out_cand_sim);
        e = cudaGetLastError();
        if (e != cudaSuccess) return dkd_ctx_fail(ctx, DKD_ERR_CUDA, "k_cand_sims launch: ", cudaGetErrorString(e));
    }
    return DKD_OK;
}

int dkd_stereo_validate(dkd_ctx* ctx, const float* kpts_l, const float* kpts_r, const int32_t* match, int n,
                        const dkd_stereo_params* sp, float* out_xyz, float* out_disp, float* out_err, uint8_t* out_valid,
                        void* stream) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (!kpts_l || !kpts_r || !sp || !out_xyz || !out_valid || n < 0)
        return dkd_ctx_fail(ctx, DKD_ERR_INVALID_ARG, "dkd_stereo_validate: NULL pointer or n < 0", nullptr);
    if (!(sp->fx > 0.0f) || !(sp->fy > 0.0f) || !(sp->baseline > 0.0f))
        return dkd_ctx_fail(ctx, DKD_ERR_INVALID_ARG, "dkd_stereo_validate: fx, fy, baseline must be > 0", nullptr);
    if ((reinterpret_cast<uintptr_t>(kpts_l) & 7) || (reinterpret_cast<uintptr_t>(kpts_r) & 7))
        return dkd_ctx_fail(ctx, DKD_ERR_UNSUPPORTED, "dkd_stereo_validate: keypoints not 8-byte aligned", nullptr);
    if (n == 0) return DKD_OK;
    DeviceGuard dg(dkd_ctx_device(ctx));
    StereoKParams k;
    memset(&k, 0, sizeof(k));
    k.kl = kpts_l; k.kr = kpts_r; k.match = match; k.n = n;
    k.fx = sp->fx; k.fy = sp->fy; k.cx = sp->cx; k.cy = sp->cy; k.baseline = sp->baseline; k.d_min = sp->d_min;
    k.z_min = sp->z_min; k.z_max = sp->z_max; k.max_reproj = sp->max_reproj;
    k.xyz = out_xyz; k.disp = out_disp; k.err = out_err; k.valid = out_valid;
    k_stereo<<<(n + 255) / 256, 256, 0, static_cast<cudaStream_t>(stream)>>>(k);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return dkd_ctx_fail(ctx, DKD_ERR_CUDA, "k_stereo launch: ", cudaGetErrorString(e));
    return DKD_OK;
}

int dkd_cov_sqrt_info(dkd_ctx* ctx, const float* L, int n, const dkd_cov_params* cp, float* out_omega, uint8_t* out_ok,
                      void* stream) {
    if (!ctx) return DKD_ERR_INVALID_ARG;
    if (!L || !cp || !out_omega || n < 0) return dkd_ctx_fail(ctx, DKD_ERR_INVALID_ARG, "dkd_cov_sqrt_info: NULL pointer or n < 0", nullptr);
    if (!(cp->fx > 0.0f) || !(cp->fy > 0.0f) || !(cp->sigma0 > 0.0f) || !(cp->floor_px >= 0.0f) || !(cp->lambda_min >= 0.0f) ||
        !(fmaxf(cp->lambda, cp->lambda_min) > 0.0f))
        return dkd_ctx_fail(ctx, DKD_ERR_INVALID_ARG, "dkd_cov_sqrt_info: fx, fy, sigma0, max(lambda, lambda_min) must be > 0; floor >= 0", nullptr);
    if (n == 0) return DKD_OK;
    DeviceGuard dg(dkd_ctx_device(ctx));
    CovKParams k;
    memset(&k, 0, sizeof(k));
    k.L = L; k.n = n;
    k.s2 = cp->scale * cp->scale; k.floor_px = cp->floor_px;
    k.inv_fx2 = static_cast<float>(1.0 / (static_cast<double>(cp->fx) * cp->fx));
    k.inv_fy2 = static_cast<float>(1.0 / (static_cast<double>(cp->fy) * cp->fy));
    k.inv_fxfy = static_cast<float>(1.0 / (static_cast<double>(cp->fx) * cp->fy));
    k.lam = fmaxf(cp->lambda, cp->lambda_min);
    k.inv_sigma0 = 1.0f / cp->sigma0;
    k.omega = out_omega; k.ok = out_ok;
    k_cov<<<(n + 255) / 256, 256, 0, static_cast<cudaStream_t>(stream)>>>(k);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return dkd_ctx_fail(ctx, DKD_ERR_CUDA, "k_cov launch: ", cudaGetErrorString(e));
    return DKD_OK;
}

}  // extern "C"
