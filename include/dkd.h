/*
 * dkd.h — C-ABI boundary of libdkd: B200-native (sm_100a) keypoint post-processing for learned
 * visual front-ends: ALIKED-style Differentiable Keypoint Detection (DKD) + descriptor sampling.
 *
 * Reference: /root/reference/PAPER.md ("DL-VINS-Factory", arxiv/paper_2607_01757)
 *   PAPER.md:84-86   (Sec. III-A)  score map -> DKD -> sub-pixel keypoints
 *   PAPER.md:97-101  (Eq. 1)       Phi(I) = {(p_i, d_i, s_i)}: pixel coordinates p_i in R^2,
 *                                  l2-normalised descriptors d_i in R^D, D in {64,128,256}, s_i in [0,1]
 *   PAPER.md:118                   LK pathway needs keypoints only (desc == NULL here)
 *   PAPER.md:120-122 (Sec. III-A)  custom CUDA DKD: NMS, sorting, patch extraction; dynamic count
 *   PAPER.md:128,132               stereo pair processed as one batch (B = 2)
 *   PAPER.md:139                   sets zero-padded to the keypoint cap (static shapes downstream)
 * The paper prints no formula for these steps; the exact arithmetic is fixed by BASELINE.json
 * `north_star` steps (1)-(4) and the readings G1..G21 in DESIGN.md.
 *
 * C99, no C++ types, no exceptions cross the boundary.  All `device` pointers are CUDA device
 * memory on the context's device; `host` pointers are ordinary (preferably pinned) host memory.
 * The caller owns every input/output buffer and the stream; a dkd_ctx owns only its workspace.
 */
#ifndef DKD_H_
#define DKD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dkd_ctx dkd_ctx;   /* opaque */

/* return codes: 0 = OK, negative = error; on INVALID_ARG / UNSUPPORTED / CAPACITY nothing was
 * launched and no output was written. */
enum {
    DKD_OK = 0,
    DKD_ERR_INVALID_ARG = -1,   /* NULL required pointer, size < 1, r < 1, T <= 0 or non-finite, ... */
    DKD_ERR_UNSUPPORTED = -2,   /* r > DKD_MAX_RADIUS; D*elemsize not a multiple of 16 B or > DKD_MAX_ROW_BYTES;
                                   desc/out_desc not 16-byte aligned; out_kpts/out_offset not 8-byte aligned; any
                                   other f32/i32 buffer not 4-byte aligned; unknown dtype */
    DKD_ERR_CAPACITY = -3,      /* B, H, W, top_k or D above the dkd_create maxima */
    DKD_ERR_CUDA = -4           /* CUDA runtime/driver failure; text in dkd_last_error() */
};

enum { DKD_F32 = 0, DKD_F16 = 1 };          /* descriptor-map element type */

enum { DKD_SCORE_RAW = 0, DKD_SCORE_BILINEAR = 1 };   /* reported score, see dkd_variant_params */

#define DKD_MAX_RADIUS    4                 /* (2r+1)^2 window, r in [1,4] (paper's extractors use 2..4) */
#define DKD_MAX_TOP_K     8192              /* per-image cap (paper: 160..384) */
#define DKD_MAX_ROW_BYTES 2048              /* D * elemsize of one descriptor row */

/* options for dkd_set_option (defaults in brackets) */
enum {
    DKD_OPT_USE_GRAPH = 0,   /* [1] run each dkd_extract as ONE cached CUDA-graph launch (north_star:
                                "the whole stereo pair in one CUDA-graph launch"); 0 = plain launches.
                                Ignored (plain launches) while `stream` is being captured by the caller.
                                The cache is keyed on SHAPES (B, H, W, r, top_k, D, dtype, stride, which optional
                                buffers are present, options): a call that differs only in buffer addresses, thresh
                                or T re-uses the instantiated graph and updates its kernel nodes' parameters in
                                place — nothing is captured or instantiated again (dkd_graph_stats). */
    DKD_OPT_USE_TMA   = 1,   /* [1] NMS tiles staged by TMA (cp.async.bulk.tensor) when W % 4 == 0 and
                                score is 16-byte aligned; 0 = always the plain-load tile loader. */
    DKD_OPT_PROFILE   = 2,   /* [0] 1 = measurement mode: plain launches (no graph) with a CUDA event recorded
                                on `stream` before and after every kernel; read with dkd_profile_read. */
    DKD_OPT_USE_PDL   = 3,   /* [1] the kernels are launched with programmatic stream serialization (they start
                                while their predecessor drains and wait on-device, griddepcontrol.wait, before
                                they touch global memory): hides the launch latency between the kernels.  The
                                NMS kernel carries the attribute too, so with plain launches (DKD_OPT_USE_GRAPH
                                = 0, or while the caller captures) it may be SCHEDULED while the previous kernel
                                of `stream` still runs — it reads `score` only after that kernel has completed
                                and flushed, whatever that kernel is; results never depend on this option. */
    DKD_OPT_ORIGIN_X  = 5,   /* [0] letterbox offset (ox, oy) of the score map inside the padded network input: it is */
    DKD_OPT_ORIGIN_Y  = 6,   /* [0] subtracted from every keypoint coordinate ("shifted back to native coordinates by
                                subtracting the offset"); out_index / out_offset are unaffected. */
    DKD_OPT_SEL_PREFETCH = 7, /* [0] the select kernel asks L2 for the refinement-window rows of every kept keypoint, so
                                that the refinement's dependent loads hit L2 (tuning knob; results do not depend on it;
                                measured a net loss at batch 64: DESIGN.md 7.3). */
    DKD_OPT_NMS_UNIT  = 4    /* [0] strip-tiles (8 output rows each) a warp of the NMS kernel walks down before it
                                moves to another strip: 0 = chosen per call from the problem size, 1..8 = forced
                                (tuning / test knob; results do not depend on it). */
};

typedef struct {
    int device;                 /* CUDA ordinal */
    int max_batch, max_h, max_w;
    int max_top_k;              /* <= DKD_MAX_TOP_K */
    int max_dim;                /* max D (0 = keypoints only) */
    /* The fields below may all be 0 (a zero-initialised struct behaves as before they existed). */
    int max_radius;             /* largest r a call may pass, 1..DKD_MAX_RADIUS; 0 = DKD_MAX_RADIUS.  A call with a larger r
                                   returns DKD_ERR_CAPACITY. */
    int max_match_n;            /* dkd_match: largest Na / Nb; > 0 sizes the matcher's scratch at create, so that no dkd_match
                                   call within (max_match_n, max_match_pairs) ever allocates — also not the first one, which
                                   may then be made inside a stream capture.  0 = grown on demand by the calls (cudaMalloc) */
    int max_match_pairs;        /* dkd_match: largest P for the above; 0 = 2 (temporal + stereo pair) */
    int max_scan_rows;          /* dkd_retrieval_scan: largest n; > 0 sizes its scratch at create likewise; 0 = on demand */
} dkd_create_params;

/* Allocates the workspace once on p->device (candidate keys sized for the worst case — every
 * interior pixel a candidate — so selection is exact on any input).
 * Returns DKD_OK and *out, or an error (and *out = NULL). */
int dkd_create(const dkd_create_params* p, dkd_ctx** out);

/* Frees the workspace.  NULL is a no-op -> DKD_OK.  The caller must have synchronised any stream
 * that still runs work enqueued through this context. */
int dkd_destroy(dkd_ctx* ctx);

/* Text of the last error on this context (ctx-owned, valid until the next call on ctx);
 * with ctx == NULL, the text of the last dkd_create failure (static storage). */
const char* dkd_last_error(const dkd_ctx* ctx);

/* Device bytes owned by the context. */
size_t dkd_workspace_bytes(const dkd_ctx* ctx);

int dkd_set_option(dkd_ctx* ctx, int option, int value);

/*
 * dkd_extract — the whole hot path for a batch of B independent images (north_star steps 1-4;
 * PAPER.md:120-122 stages; Eq. 1 outputs):
 *   (1) mask = r-pixel border exclusion AND S > thresh (strict) AND S >= every S in the (2r+1)^2
 *       window (ties are all maxima);
 *   (2) per image keep K_b = min(top_k, #candidates) ordered by (score desc, linear index y*W+x asc)
 *       — selection on the float bits, bit-exact;
 *   (3) soft-argmax over the same window: w = exp((S - S_centre)/T), (dx,dy) = sum w*(i,j) / sum w,
 *       p = (x+dx, y+dy) in score-map pixel units, (x,y) order;
 *   (4) if desc != NULL: bilinear sample of the channel-last map at u = (px+0.5)/stride - 0.5
 *       (likewise v), clamped to the map, fp32 accumulation, divided by max(||d||_2, 1e-12);
 *   (5) slots i >= K_b are zero-filled.
 *
 *   score      device [B,H,W] f32, contiguous.                                   (read only)
 *   desc       device [B,Hd,Wd,D] channel-last, DKD_F16 or DKD_F32, contiguous, 16-byte aligned,
 *              or NULL to skip step (4) (then out_desc must be NULL).  Hd*stride, Wd*stride need
 *              not equal H, W: sampling positions are clamped to the map.           (read only)
 *   out_kpts   device [B,top_k,2] f32 (x,y), 8-byte aligned
 *   out_scores device [B,top_k]   f32, raw S at the integer peak (bit-identical to the input)
 *   out_desc   device [B,top_k,D] same element type as desc, 16-byte aligned
 *   out_count  device [B] i32 = K_b
 *   stream     cudaStream_t (NULL = legacy default stream)
 *
 * Asynchronous and stream-ordered: no host synchronisation, no allocation, no host read of the
 * counts; outputs are valid once `stream` reaches the end of the enqueued work.  One context must
 * not be used from two streams concurrently (the workspace is shared).  Outputs are a pure
 * function of the inputs (deterministic).  Non-finite scores are outside the contract.
 */
int dkd_extract(dkd_ctx* ctx,
                const float* score, int B, int H, int W,
                const void* desc, int desc_dtype, int Hd, int Wd, int D, int stride,
                int r, float thresh, int top_k, float T,
                float* out_kpts, float* out_scores, void* out_desc, int32_t* out_count,
                void* stream);

/* dkd_extract plus two optional outputs (either may be NULL):
 *   out_index  device [B,top_k] i32: linear index y*W+x of the integer peak, -1 in padding
 *              (integer positions cannot be recovered from the refined coordinates);
 *   out_offset device [B,top_k,2] f32, 8-byte aligned: the sub-pixel offset (dx,dy) before it is added to
 *              (x,y) (the 1e-5 px parity bound applies to this; G11). */
int dkd_extract_ex(dkd_ctx* ctx,
                   const float* score, int B, int H, int W,
                   const void* desc, int desc_dtype, int Hd, int Wd, int D, int stride,
                   int r, float thresh, int top_k, float T,
                   float* out_kpts, float* out_scores, void* out_desc, int32_t* out_count,
                   int32_t* out_index, float* out_offset,
                   void* stream);

/*
 * Variants of the path on the same kernels (readings V1..V5 in DESIGN.md).  Every field may be
 * left 0 / NULL, which is the base path.
 *   reliability  device [B,H,W] f32: the score the whole path works on is heat x reliability, each product rounded
 *                once to fp32 and formed BEFORE the window maximum (XFeat: keypoint heat "filtered using an additional
 *                reliability heatmap").  `score` is the heat map.  The product is never written to
 *                memory: the NMS kernel streams both maps (second TMA stream).  Threshold, order, reported score and
 *                refinement all use the product.
 *   valid_mask   device [B,H,W] u8: a pixel can be a keypoint only where the mask is non-zero ("a fisheye validity
 *                mask that culls features near the image periphery").  Masked pixels still take part
 *                in every window maximum and in the refinement windows.  (Read once per candidate, by the selection kernel.)
 *   nms_iters    0 = one (2r+1)^2 max-pool pass (north_star).  n > 0 = the iterated suppress-and-recover NMS of "the
 *                original PyTorch NMS" with n recovery rounds (the published procedure uses 2):
 *                M = (S == maxpool S); n times: supp = maxpool(M) > 0, S' = supp ? 0 : S, M |= (S' == maxpool S') & !supp,
 *                windows clipped at the image edge; border exclusion and threshold apply to the final mask.  Runs in its
 *                own tiled shared-memory kernel; (2 n + 1) r must be <= 40 (DKD_ERR_UNSUPPORTED otherwise).
 *   score_mode   DKD_SCORE_RAW: out_scores = S at the integer peak (bit-exact).  DKD_SCORE_BILINEAR: out_scores = S
 *                interpolated bilinearly at the refined position (x+dx, y+dy).  Selection and order always use the
 *                raw score.
 *   out_total    device [B] i32 or NULL: C_b, the number of candidates of image b BEFORE the cap.  Threshold-only
 *                mode (no cap) = top_k set to the capacity of the output buffers: out_count = min(C_b, top_k) and
 *                out_total tells whether the buffers were large enough (if not, the best top_k are returned).
 */
typedef struct {
    const float* reliability;
    const uint8_t* valid_mask;
    int nms_iters;
    int score_mode;
    int32_t* out_total;
} dkd_variant_params;

/* dkd_extract_ex with the variants above (v == NULL: identical to dkd_extract_ex). */
int dkd_extract_var(dkd_ctx* ctx,
                    const float* score, int B, int H, int W,
                    const void* desc, int desc_dtype, int Hd, int Wd, int D, int stride,
                    int r, float thresh, int top_k, float T,
                    float* out_kpts, float* out_scores, void* out_desc, int32_t* out_count,
                    int32_t* out_index, float* out_offset,
                    const dkd_variant_params* v,
                    void* stream);

/* Graph-cache statistics since dkd_create (any pointer may be NULL): graphs instantiated, calls served by updating
 * the kernel-node parameters of a cached graph, calls that replayed a cached graph unchanged, calls enqueued as plain
 * launches. */
int dkd_graph_stats(const dkd_ctx* ctx, uint64_t* instantiated, uint64_t* updated, uint64_t* replayed,
                    uint64_t* stream_launched);

/*
 * dkd_extract_host — the same call with HOST buffers (the end-to-end path): copies score host->device
 * into a context-owned staging buffer, runs dkd_extract_ex, delivers every non-NULL output to the host
 * buffers, and synchronises `stream` before returning.  Staging is (re)allocated on first use / growth.
 * Pointers have the shapes above.  Pinned (page-locked, mapped: cudaHostAlloc / cudaHostRegister) buffers
 * are used in place where that is cheaper:
 *   - a pinned descriptor map of which the call can touch at most 1/8 (4 rows per output slot) is NOT
 *     uploaded: the gather samples its corner rows directly over PCIe;
 *   - when every output buffer is pinned the kernels store straight into them (no staging, no copies back).
 * Pageable buffers go through staged cudaMemcpyAsync copies.
 * desc_resident: 0 = the map is uploaded (or sampled in place) on every call; 1 = upload once and re-use the device
 * copy while the same desc pointer and shape are passed — the caller must NOT modify the host map while it is resident
 * (a copy uploaded by a desc_resident = 0 call is never re-used); 2 = upload now (the host map changed) and keep the
 * copy resident for later desc_resident = 1 calls.  (A dense network would leave the map on the device.)
 * Every shape / scalar argument is checked before anything is allocated or enqueued; if an error occurs after work
 * was enqueued the stream is synchronised before the call returns.
 */
int dkd_extract_host(dkd_ctx* ctx,
                     const float* score, int B, int H, int W,
                     const void* desc, int desc_dtype, int Hd, int Wd, int D, int stride,
                     int r, float thresh, int top_k, float T,
                     float* out_kpts, float* out_scores, void* out_desc, int32_t* out_count,
                     int32_t* out_index, float* out_offset,
                     int desc_resident, void* stream);

/*
 * Fused input pre-processing (Sec. III-B: "letterbox padding, color-format conversion,
 * intensity normalization, and NCHW layout packing in a single pass, with stereo pairs processed as one
 * batch"; frames padded to multiples of 8 (SuperPoint, XFeat) or 32 (ALIKED, RaCo); mono replicated to three
 * channels, colour reduced to one luminance channel).  The paper prints no constant; P1..P7:
 *   padded size Hp = ceil(H/grid)*grid, Wp likewise; the image is CENTRED: oy = (Hp-H)/2, ox = (Wp-W)/2;
 *   padding holds pad_value (output units); luminance = 0.299 R + 0.587 G + 0.114 B (BT.601);
 *   out = (value * scale - mean[c]) * inv_std[c]; 3 -> 3 channels are written as R,G,B planes.
 */
typedef struct {
    int in_channels;     /* 1 (mono) or 3 (interleaved colour) */
    int out_channels;    /* 1 or 3 */
    int grid;            /* >= 1; H and W are padded up to multiples of it */
    int bgr;             /* != 0: colour input is stored B,G,R */
    int out_dtype;       /* DKD_F32 or DKD_F16 */
    float scale;         /* 1/255 maps 8-bit values to [0,1] */
    float mean[3];
    float inv_std[3];
    float pad_value;
} dkd_pre_params;

/* Padded size and letterbox offset for (H, W, grid); any output pointer may be NULL.  DKD_ERR_INVALID_ARG if
 * H, W or grid < 1. */
int dkd_pre_padded_size(int H, int W, int grid, int* Hp, int* Wp, int* oy, int* ox);

/*   src  device [B,H,W,in_channels] u8, interleaved, contiguous                       (read only)
 *   dst  device [B,out_channels,Hp,Wp] f32|f16 planar, contiguous, 16-byte aligned
 * Asynchronous on `stream`; one kernel launch; every element of dst is written. */
int dkd_preprocess(dkd_ctx* ctx, const uint8_t* src, int B, int H, int W, const dkd_pre_params* p, void* dst,
                   void* stream);

/*
 * ---- consumers of the descriptor output (M1..M8) -----------------------
 *
 * dkd_match — cosine nearest-neighbour matching with a Lowe ratio test between P pairs of padded descriptor sets
 * ("cosine nearest-neighbour matching with a Lowe ratio test"; descriptors are l2-normalised, Eq. 1
 * PAPER.md:101, so the cosine is the dot product, Eq. 4; sets are zero-padded to the cap,
 * PAPER.md:139; the temporal and the stereo pair go in one batch).  For every row i < count_a[p]:
 *   s_ij = a_i . b_j over j < count_b[p];  j1 = argmax_j s_ij (ties: smallest j);  s2 = max_{j != j1} s_ij (-1 if none);
 *   ratio test on the distances of unit vectors, d^2 = max(0, 2 - 2 s): keep iff d1^2 < ratio^2 d2^2 (ratio >= 1e9: off);
 *   mutual != 0: keep only if i is also the nearest neighbour of j1 (ties: smallest i).
 * The similarity matrix is formed on the tensor cores (tcgen05, fp16 inputs, fp32 accumulation) and never written to
 * memory: the row-wise top-2 is fused into the epilogue.
 *   desc_a   device [P,Na,D] f16 (the out_desc of dkd_extract), 16-byte aligned; desc_b device [P,Nb,D] likewise
 *   count_a  device [P] i32 valid rows (the out_count of dkd_extract), or NULL = Na; count_b likewise
 *   D        64, 128, 192 or 256; dtype must be DKD_F16 (else DKD_ERR_UNSUPPORTED)
 *   out_match device [P,Na] i32: j1 or -1 (no match / padding row);  out_sim device [P,Na,2] f32 (s1, s2) or NULL
 * Asynchronous on `stream`.  Uses a context-owned scratch buffer that is grown (cudaMalloc) when a call needs more than
 * any call before it: such a call must not be made while `stream` is being captured — unless the context was created with
 * max_match_n / max_match_pairs (max_scan_rows for the scan) covering the call, which sizes it once at create.  The buffer holds the partial results
 * between the kernels of ONE call: a context must be used from one stream at a time (calls of dkd_match /
 * dkd_retrieval_scan on the same context whose kernels could overlap on the GPU overwrite each other's partials; use
 * one context per stream, or order the streams with events).
 */
int dkd_match(dkd_ctx* ctx, const void* desc_a, const int32_t* count_a, int Na,
              const void* desc_b, const int32_t* count_b, int Nb, int D, int dtype, int P,
              float ratio, int mutual, int32_t* out_match, float* out_sim, void* stream);

/*
 * dkd_match_static — dkd_match for callers that are not allowed to allocate device memory.
 *
 * Who this is for: code that runs where cudaMalloc / cudaFree are off limits — a plug-in living inside a host
 * application that hands out a fixed device-memory budget and forbids allocations of its own (an inference-server
 * back-end, a ROS 2 component under a real-time executor: cudaMalloc takes a driver lock and may stall the whole
 * device for milliseconds), a process whose memory pool has already claimed the entire GPU so that a further
 * cudaMalloc simply fails, or a hard real-time loop in which any call of unbounded duration is banned.  Such a
 * caller cannot use dkd_create (it allocates the workspace) and therefore none of the dkd_ctx entry points.  This one
 * takes no context and calls neither cudaMalloc nor cudaFree nor any library routine that allocates: the one piece
 * of scratch memory the matcher needs — the per-column-split partial results that k_match_tc hands to
 * k_match_finalize — is a fixed-size array that is part of the library image itself.
 *
 * The limit: that array holds DKD_MATCH_STATIC_MAX_RECS records of 16 bytes = 1 MiB.  It is claimed on every GPU
 * on which this library's code is loaded, whether or not this function is ever called there, and is given back only
 * when the process exits.  A call needs  P * splits(Na,Nb) * Na  records, plus  P * splits(Nb,Na) * Nb  when
 * mutual != 0, where splits (1..16) is how many CTAs share the columns of one row block so that the grid fills the
 * GPU once.  Two pairs of 4096 x 4096 with the mutual check need 32768 records on a 148-SM part; a call that needs
 * more than the array holds returns DKD_ERR_CAPACITY, launches nothing, and says both numbers in `err`.
 *
 * Arguments, results, tie rules and alignment requirements are exactly those of dkd_match (see above); the results
 * are bit-identical to dkd_match on the same inputs.  Differences:
 *   - no ctx: the call runs on the calling thread's CURRENT device; every pointer and `stream` must belong to it;
 *   - err / err_len: optional caller-owned host buffer that receives the message of a failure (NUL-terminated,
 *     truncated to err_len; empty on success); NULL / 0 = no message wanted;
 *   - the first call on each device does a one-time set-up on that device (it looks up the device address of the
 *     built-in array, reads the SM count, raises the matcher's shared-memory limit).  Make that first call during
 *     start-up, on a stream that is not being captured; later calls on that device only launch kernels;
 *   - every call on a device shares the one array, and the array keeps what the previous call left in it.  Nothing
 *     in it needs to start at zero (each call overwrites every record it later reads), but two calls whose kernels
 *     can be on the GPU at the same time — different streams, or the same stream from two threads without ordering —
 *     overwrite each other's partials and return garbage.  Keep all calls on one device on one stream, or order
 *     them with events.
 * Asynchronous on `stream` (up to three kernel launches).
 */
#define DKD_MATCH_STATIC_MAX_RECS 65536
int dkd_match_static(const void* desc_a, const int32_t* count_a, int Na,
                     const void* desc_b, const int32_t* count_b, int Nb, int D, int dtype, int P,
                     float ratio, int mutual, int32_t* out_match, float* out_sim, void* stream,
                     char* err, int err_len);

/*
 * dkd_retrieval_scan — brute-force loop-candidate retrieval ("cosine similarity between the current
 * descriptor g_t and a past descriptor g_k", Eq. 4; "a fixed window of the most recent keyframes is excluded";
 * "Candidates with sim > tau_sim are ranked by similarity"; "brute-force scan over the keyframe database, O(n)";
 * 50 most recent excluded, tau_sim = 0.60; g in R^{32*384}).
 *   db       device [n,D] f16|f32, rows in insertion order (row n-1 is the newest keyframe), 16-byte aligned
 *   query    device [D] same dtype, 16-byte aligned;  D * elemsize a multiple of 16, D <= 16384
 *   out_sim  device [n] f32: q . db_k for EVERY row (fp32 accumulation), or NULL
 *   out_cand device [max_cand] i32: rows k < n - n_exclude with sim > tau (strict), ranked by (sim desc, k asc),
 *            -1 padded; out_cand_sim device [max_cand] f32 or NULL; out_count device [1] i32
 * Asynchronous on `stream`; scratch buffer as for dkd_match.  One pass over the database: HBM-bound.
 */
int dkd_retrieval_scan(dkd_ctx* ctx, const void* db, int dtype, int n, int D, const void* query,
                       int n_exclude, float tau, int max_cand,
                       float* out_sim, int32_t* out_cand, float* out_cand_sim, int32_t* out_count, void* stream);

/*
 * ---- per-match stereo validation and covariance weighting (S1..S4, C1..C4) -----------
 *
 * dkd_stereo_validate: rectified pinhole pair, right camera at +baseline along x.  For left keypoint i
 * and right keypoint j = match[i] (match == NULL: j = i; j < 0: invalid): disparity d = uL - uR must exceed d_min
 * ("negligible disparity"); depth z = fx baseline / d, X = (uL - cx) z / fx, Y = ((vL + vR)/2 - cy) z / fy; kept iff
 * z_min < z < z_max and the reprojection error |vL - vR| / 2 (both views) <= max_reproj (1.5 px).
 *   kpts_l device [n,2] f32 (x,y), kpts_r device [m,2] f32, both 8-byte aligned; match device [n] i32 or NULL
 *   out_xyz device [n,3] f32; out_disp, out_err device [n] f32 or NULL; out_valid device [n] u8
 */
typedef struct {
    float fx, fy, cx, cy, baseline;
    float d_min, z_min, z_max, max_reproj;
} dkd_stereo_params;
int dkd_stereo_validate(dkd_ctx* ctx, const float* kpts_l, const float* kpts_r, const int32_t* match, int n,
                        const dkd_stereo_params* p, float* out_xyz, float* out_disp, float* out_err,
                        uint8_t* out_valid, void* stream);

/*
 * dkd_cov_sqrt_info (App. A-B, Eq. 9-11): per keypoint, from the predicted lower-triangular factor
 * L = [[l11,0],[l21,l22]]: Sigma_px = scale^2 L L^T + floor_px I; Sigma_n = J Sigma_px J^T, J = diag(1/fx, 1/fy);
 * Sigma_eff^-1 = max(lambda, lambda_min) Sigma_n^-1; Omega = the upper-triangular factor with Omega^T Omega =
 * Sigma_eff^-1; if Sigma_px is not positive definite or an input is non-finite: Omega = I / sigma0, ok = 0.
 *   L device [n,3] f32 (l11, l21, l22); out_omega device [n,4] f32 row-major 2x2; out_ok device [n] u8 or NULL
 */
typedef struct {
    float scale, floor_px, fx, fy, lambda, lambda_min, sigma0;
} dkd_cov_params;
int dkd_cov_sqrt_info(dkd_ctx* ctx, const float* L, int n, const dkd_cov_params* p, float* out_omega,
                      uint8_t* out_ok, void* stream);

/* Measurement mode (DKD_OPT_PROFILE = 1): waits for the events of the most recent dkd_extract* call
 * on this context and writes the device time of each of its kernels, in launch order, to
 * ms[0..n) (host; milliseconds; entries past the launch count are left untouched).  Returns the
 * number of kernels that call launched, or a negative error (no profiled call yet, CUDA failure).
 * dkd_kernel_name(i) is the name of the i-th kernel of a launch ("nms", "select", "refine_gather"). */
int dkd_profile_read(dkd_ctx* ctx, float* ms, int n);
const char* dkd_kernel_name(int i);

/* Number of kernels one dkd_extract launches for these arguments (for launch accounting). */
int dkd_launches_per_extract(const dkd_ctx* ctx, int with_desc);

const char* dkd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DKD_H_ */
