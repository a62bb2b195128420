/*
 * dkd_oracle.c — CPU ORACLE for the DKD + descriptor-sampling hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA library (libdkd).
 *
 * What it is: the plain definition of each step, written as naive loops in
 * double precision (input floats are widened exactly), in the order and notation of
 * SURVEY.md §8(c) O1..O5 / DESIGN.md "Readings".  No blocking, fusion or reordering.
 *
 * Passages followed (reference = /root/reference/PAPER.md):
 *   PAPER.md:84-86   (Sec. III-A)  score map -> DKD -> sub-pixel keypoints
 *   PAPER.md:97-101  (Eq. 1)       output contract {(p_i, d_i, s_i)}: pixel coords, l2-normalised
 *                                  descriptors, D in {64,128,256}, scores in [0,1]
 *   PAPER.md:120-122 (Sec. III-A)  three stages: NMS, sorting, patch extraction; cost ~ N
 *   PAPER.md:139     (Sec. III-C)  sets zero-padded to the keypoint cap
 *   PAPER.md:210                   thresholding, NMS, top-N retention
 *   BASELINE.json north_star steps (1)-(4) fix the arithmetic the paper leaves open;
 *   every such reading is listed in DESIGN.md (G1..G21).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"):
 *   O1: brute-force python window loops; torch max_pool2d equality mask; planted cases.
 *   O2: python sorted() on (-score, idx); O(C^2) rank counting; invariants.
 *   O3: closed form 1/(1+e^{D/T}) two-pixel window; exact 0 on symmetric peaks; mirror
 *       antisymmetry; |offset| <= r; T->inf centroid; independent numpy softmax expectation.
 *   O4: affine maps (bilinear exact); constant maps; torch grid_sample(border,
 *       align_corners=False); unit norm; zero-map guard.
 *   O5: direct equality.
 *   pre-processing (dkd_oracle_preprocess, tests/test_preprocess_pins.py): hand-worked 2x3 fixture;
 *       exact copy / pad-value / centred-offset invariants; BT.601 closed forms; an independent torch
 *       pad + permute + matmul routine in float64; keypoint un-shift round trip.
 * Unpinned: agreement with the paper's own kernel / ALIKED's DKD (no worked example, no code,
 *   no printed number for this path exists in PAPER.md) — "parity unpinned" w.r.t. the paper's
 *   kernel; parity is against this definition only.
 *
 * Build: gcc -O2 -std=c99 -fopenmp -shared -fPIC dkd_oracle.c -o libdkd_oracle.so -lm
 *        (no -ffast-math).  OpenMP only splits independent rows / keypoints.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_F32 0
#define ORACLE_F16 1

int dkd_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* exact IEEE binary16 -> double (descriptor maps may be stored as f16; PAPER.md:171 FP16 engines) */
static double half_to_double(uint16_t h) {
    int sign = (h >> 15) & 1;
    int e = (h >> 10) & 0x1f;
    int m = h & 0x3ff;
    double v;
    if (e == 0)
        v = ldexp((double)m, -24);            /* subnormal: m * 2^-24 */
    else if (e == 31)
        v = m ? NAN : INFINITY;
    else
        v = ldexp((double)(m + 1024), e - 25); /* (1 + m/1024) * 2^(e-15) */
    return sign ? -v : v;
}

/* ---------------------------------------------------------------------------------------------
 * O1  NMS + border + threshold (north_star step (1); "NMS", 210 "thresholding").
 *   mask[y*W+x] = 1 iff  r <= x < W-r  and  r <= y < H-r          (G3: r-pixel border exclusion)
 *                    and S[y,x] > thresh                          (G4: strict, fp32 compare)
 *                    and no S in the (2r+1)^2 window is > S[y,x]  (G1: ties do NOT suppress)
 * Returns the number of candidates.  One image.
 * ------------------------------------------------------------------------------------------- */
long dkd_oracle_nms(const float* S, int H, int W, int r, float thresh, uint8_t* mask) {
    long n = 0;
    memset(mask, 0, (size_t)H * (size_t)W);
    #pragma omp parallel for schedule(static) reduction(+ : n)
    for (int y = r; y < H - r; ++y) {
        for (int x = r; x < W - r; ++x) {
            float c = S[(size_t)y * W + x];
            if (!(c > thresh)) continue;
            int ismax = 1;
            for (int j = -r; j <= r; ++j)
                for (int i = -r; i <= r; ++i)
                    if (S[(size_t)(y + j) * W + (x + i)] > c) ismax = 0;
            if (ismax) { mask[(size_t)y * W + x] = 1; ++n; }
        }
    }
    return n;
}

/* ---------------------------------------------------------------------------------------------
 * O2  top-k select + order (north_star step (2); "sorting", 210 "top-N retention").
 *   Sort all candidates by (score descending, linear index ascending) — a total order (G6) —
 *   keep the first K = min(top_k, C) (G5).  Scores are compared as fp32 VALUES.
 *   idx_out[top_k], score_out[top_k]; slots >= K get idx -1, score 0 (O5).
 * Returns K.
 * ------------------------------------------------------------------------------------------- */
typedef struct { float s; int32_t idx; } cand_t;

static int cand_cmp(const void* a, const void* b) {
    const cand_t* p = (const cand_t*)a;
    const cand_t* q = (const cand_t*)b;
    if (p->s > q->s) return -1;
    if (p->s < q->s) return 1;
    if (p->idx < q->idx) return -1;
    if (p->idx > q->idx) return 1;
    return 0;
}

int dkd_oracle_topk(const float* S, const uint8_t* mask, int H, int W, int top_k,
                    int32_t* idx_out, float* score_out) {
    size_t npx = (size_t)H * (size_t)W;
    size_t C = 0;
    for (size_t p = 0; p < npx; ++p) C += mask[p] ? 1 : 0;
    cand_t* cand = (cand_t*)malloc((C ? C : 1) * sizeof(cand_t));
    size_t n = 0;
    for (size_t p = 0; p < npx; ++p)
        if (mask[p]) { cand[n].s = S[p]; cand[n].idx = (int32_t)p; ++n; }
    qsort(cand, C, sizeof(cand_t), cand_cmp);
    int K = (C < (size_t)top_k) ? (int)C : top_k;
    for (int i = 0; i < top_k; ++i) {
        if (i < K) { idx_out[i] = cand[i].idx; score_out[i] = cand[i].s; }
        else       { idx_out[i] = -1;          score_out[i] = 0.0f; }
    }
    free(cand);
    return K;
}

/* ---------------------------------------------------------------------------------------------
 * O3  soft-argmax sub-pixel refinement (north_star step (3); "subpixel keypoints",
 *     120-122 "patch extraction ... refinement cost scales with the keypoint count N").
 *   For a kept pixel (x,y) with centre value c = S[y,x] (== the window max, by O1):
 *     w(i,j) = exp( (S[y+j,x+i] - c) / T ),  i,j in [-r, r]        (G8: raw scores, max = centre)
 *     Wcol_i = sum_j w(i,j),  Wrow_j = sum_i w(i,j),  Z = sum_i Wcol_i   (Z >= 1)
 *     dx = ( sum_{i=1..r} i * (Wcol_{+i} - Wcol_{-i}) ) / Z        (antisymmetric pairing:
 *     dy = ( sum_{j=1..r} j * (Wrow_{+j} - Wrow_{-j}) ) / Z         exact 0 on symmetric input)
 *     p  = (x + dx, y + dy)                                         (G10: (x,y), pixel units)
 *   T is the fp32 value widened to double (G9).  off[n][2] = (dx,dy), kpt[n][2] = (px,py).
 *   idx[t] < 0 (padding) -> zeros.
 * ------------------------------------------------------------------------------------------- */
void dkd_oracle_refine(const float* S, int H, int W, int r, float T, int n,
                       const int32_t* idx, double* off, double* kpt) {
    (void)H;
    const double Td = (double)T;
    const int nw = 2 * r + 1;
    #pragma omp parallel for schedule(static)
    for (int t = 0; t < n; ++t) {
        if (idx[t] < 0) { off[2*t] = off[2*t+1] = 0.0; kpt[2*t] = kpt[2*t+1] = 0.0; continue; }
        int y = idx[t] / W, x = idx[t] % W;
        double c = (double)S[(size_t)y * W + x];
        double Wcol[64], Wrow[64];   /* nw <= 63 */
        for (int a = 0; a < nw; ++a) { Wcol[a] = 0.0; Wrow[a] = 0.0; }
        for (int j = -r; j <= r; ++j)
            for (int i = -r; i <= r; ++i) {
                double w = exp(((double)S[(size_t)(y + j) * W + (x + i)] - c) / Td);
                Wcol[i + r] += w;
                Wrow[j + r] += w;
            }
        double Z = 0.0;
        for (int a = 0; a < nw; ++a) Z += Wcol[a];
        double sx = 0.0, sy = 0.0;
        for (int a = 1; a <= r; ++a) {
            sx += (double)a * (Wcol[r + a] - Wcol[r - a]);
            sy += (double)a * (Wrow[r + a] - Wrow[r - a]);
        }
        double dx = sx / Z, dy = sy / Z;
        off[2*t] = dx;  off[2*t+1] = dy;
        kpt[2*t] = (double)x + dx;  kpt[2*t+1] = (double)y + dy;
    }
}

/* ---------------------------------------------------------------------------------------------
 * O4  bilinear descriptor gather + L2 normalisation (north_star step (4)
 *     "l2-normalized descriptors d_i in R^D"; 88-89 descriptors sampled from the model's map).
 *   F [Hd, Wd, D] channel-last, one image.  For keypoint p = (px,py) in score-map pixels:
 *     u = (px + 0.5)/s - 0.5,  v = (py + 0.5)/s - 0.5             (G13: pixel-centre alignment)
 *     u = clamp(u, 0, Wd-1),   v = clamp(v, 0, Hd-1)
 *     x0 = floor(u), y0 = floor(v), x1 = min(x0+1, Wd-1), y1 = min(y0+1, Hd-1), fx = u-x0, fy = v-y0
 *     d[c] = (1-fy)*((1-fx)*F[y0,x0,c] + fx*F[y0,x1,c]) + fy*((1-fx)*F[y1,x0,c] + fx*F[y1,x1,c])
 *     out[c] = d[c] / max(||d||_2, 1e-12)                          (G14)
 *   valid[t] == 0 (padding) -> zeros.  out [n, D] double.
 * ------------------------------------------------------------------------------------------- */
static double fetch(const void* F, int dtype, size_t e) {
    if (dtype == ORACLE_F16) return half_to_double(((const uint16_t*)F)[e]);
    return (double)((const float*)F)[e];
}

void dkd_oracle_gather(const void* F, int dtype, int Hd, int Wd, int D, int stride, int n,
                       const double* kpt, const int32_t* valid, double* out) {
    const double s = (double)stride;
    #pragma omp parallel for schedule(static)
    for (int t = 0; t < n; ++t) {
        double* o = out + (size_t)t * D;
        if (valid && valid[t] < 0) { for (int c = 0; c < D; ++c) o[c] = 0.0; continue; }
        double u = (kpt[2*t]   + 0.5) / s - 0.5;
        double v = (kpt[2*t+1] + 0.5) / s - 0.5;
        if (u < 0.0) u = 0.0;
        if (u > (double)(Wd - 1)) u = (double)(Wd - 1);
        if (v < 0.0) v = 0.0;
        if (v > (double)(Hd - 1)) v = (double)(Hd - 1);
        int x0 = (int)floor(u), y0 = (int)floor(v);
        int x1 = x0 + 1 < Wd - 1 ? x0 + 1 : Wd - 1;
        int y1 = y0 + 1 < Hd - 1 ? y0 + 1 : Hd - 1;
        double fx = u - (double)x0, fy = v - (double)y0;
        double ss = 0.0;
        for (int c = 0; c < D; ++c) {
            double f00 = fetch(F, dtype, ((size_t)y0 * Wd + x0) * D + c);
            double f01 = fetch(F, dtype, ((size_t)y0 * Wd + x1) * D + c);
            double f10 = fetch(F, dtype, ((size_t)y1 * Wd + x0) * D + c);
            double f11 = fetch(F, dtype, ((size_t)y1 * Wd + x1) * D + c);
            double d = (1.0 - fy) * ((1.0 - fx) * f00 + fx * f01)
                     +        fy  * ((1.0 - fx) * f10 + fx * f11);
            o[c] = d;
            ss += d * d;
        }
        double nrm = sqrt(ss);
        if (nrm < 1e-12) nrm = 1e-12;
        for (int c = 0; c < D; ++c) o[c] /= nrm;
    }
}

/* ---------------------------------------------------------------------------------------------
 * Whole path O1..O5 over a batch (images independent, G19; stereo = B 2).
 *   score  [B,H,W] f32;  desc [B,Hd,Wd,D] f16|f32 channel-last or NULL (LK pathway,
 *   keypoints only).
 *   out_kpts [B,k,2] f64 (x,y) ; out_off [B,k,2] f64 (dx,dy) ; out_scores [B,k] f32 ;
 *   out_desc [B,k,D] f64 (NULL iff desc NULL) ; out_count [B] ; out_index [B,k] (-1 padding).
 * Returns 0, or -1 on a bad argument.
 * ------------------------------------------------------------------------------------------- */
int dkd_oracle_extract(const float* score, int B, int H, int W,
                       const void* desc, int desc_dtype, int Hd, int Wd, int D, int stride,
                       int r, float thresh, int top_k, float T,
                       double* out_kpts, double* out_off, float* out_scores, double* out_desc,
                       int32_t* out_count, int32_t* out_index) {
    if (!score || B < 1 || H < 1 || W < 1 || r < 1 || r > 31 || top_k < 1 || !(T > 0.0f)) return -1;
    if (desc && (Hd < 1 || Wd < 1 || D < 1 || stride < 1 || !out_desc)) return -1;
    uint8_t* mask = (uint8_t*)malloc((size_t)H * W);
    size_t esz = desc_dtype == ORACLE_F16 ? 2 : 4;
    for (int b = 0; b < B; ++b) {
        const float* S = score + (size_t)b * H * W;
        int32_t* idx = out_index + (size_t)b * top_k;
        dkd_oracle_nms(S, H, W, r, thresh, mask);                                    /* O1 */
        out_count[b] = dkd_oracle_topk(S, mask, H, W, top_k, idx,
                                       out_scores + (size_t)b * top_k);              /* O2, O5 */
        dkd_oracle_refine(S, H, W, r, T, top_k, idx, out_off + (size_t)b * top_k * 2,
                          out_kpts + (size_t)b * top_k * 2);                         /* O3, O5 */
        if (desc) {
            const char* F = (const char*)desc + (size_t)b * Hd * Wd * D * esz;
            dkd_oracle_gather(F, desc_dtype, Hd, Wd, D, stride, top_k,
                              out_kpts + (size_t)b * top_k * 2, idx,
                              out_desc + (size_t)b * top_k * D);                     /* O4, O5 */
        }
    }
    free(mask);
    return 0;
}

/* =============================================================================================
 * Fused input pre-processing (Sec. III-B): letterbox padding to
 * the resolution grid (multiples of 8 / 32), colour-format conversion (mono -> 3 channels by
 * replication, colour -> one luminance channel), intensity normalisation, NCHW packing, stereo pair =
 * batch.  The paper prints no constant; the readings (P1..P7):
 *   P1 padded size Hp = ceil(H/g)*g, Wp = ceil(W/g)*g;
 *   P2 letterbox is CENTRED: oy = (Hp-H)/2, ox = (Wp-W)/2 (integer division), source pixel (y,x) lands
 *      at (y+oy, x+ox); keypoints are shifted back by subtracting (ox,oy);
 *   P3 padding holds pad_value (a value in OUTPUT units, i.e. after normalisation);
 *   P4 luminance = 0.299 R + 0.587 G + 0.114 B (ITU-R BT.601) on the 8-bit values; `bgr` says the
 *      interleaved input is B,G,R; 3 -> 3 channels re-orders to R,G,B planes;
 *   P5 normalisation: out = (value * scale - mean[c]) * inv_std[c]  (scale = 1/255 for [0,1]);
 *   P6 mono -> 3 channels: the same 8-bit value in every plane, each with its own mean / inv_std;
 *   P7 output planar [B,Cout,Hp,Wp].
 * src [B,H,W,Cin] u8 interleaved; out [B,Cout,Hp,Wp] double.  Returns 0, -1 on a bad argument.
 * ============================================================================================= */
int dkd_oracle_preprocess(const uint8_t* src, int B, int H, int W, int Cin, int Cout, int grid, int bgr,
                          double scale, const double* mean, const double* inv_std, double pad_value,
                          double* out) {
    if (!src || !out || B < 1 || H < 1 || W < 1 || grid < 1) return -1;
    if (!((Cin == 1 || Cin == 3) && (Cout == 1 || Cout == 3))) return -1;
    int Hp = (H + grid - 1) / grid * grid, Wp = (W + grid - 1) / grid * grid;
    int oy = (Hp - H) / 2, ox = (Wp - W) / 2;
    for (int b = 0; b < B; ++b)
        for (int c = 0; c < Cout; ++c)
            for (int yp = 0; yp < Hp; ++yp)
                for (int xp = 0; xp < Wp; ++xp) {
                    double* o = out + (((size_t)b * Cout + c) * Hp + yp) * Wp + xp;
                    int y = yp - oy, x = xp - ox;
                    if (y < 0 || y >= H || x < 0 || x >= W) { *o = pad_value; continue; }
                    const uint8_t* px = src + (((size_t)b * H + y) * W + x) * Cin;
                    double v;
                    if (Cin == 1) {
                        v = (double)px[0];                                   /* P6 (or 1 -> 1) */
                    } else {
                        double R = (double)px[bgr ? 2 : 0], G = (double)px[1], Bl = (double)px[bgr ? 0 : 2];
                        if (Cout == 1) v = 0.299 * R + 0.587 * G + 0.114 * Bl;          /* P4 */
                        else v = c == 0 ? R : (c == 1 ? G : Bl);
                    }
                    *o = (v * scale - mean[c]) * inv_std[c];                 /* P5 */
                }
    return 0;
}

