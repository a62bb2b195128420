/*
 * dkd_variants.c — CPU ORACLE for the DKD VARIANTS on top of dkd_oracle.c.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as dkd_oracle.c: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build or call it; it
 * shares no code with the CUDA library).  Plain C99, fp64, naive loops, no blocking or fusion.
 *
 * Passages followed (reference = /root/reference/PAPER.md) and the readings taken where the paper is silent
 * (V1..V5):
 *   V1  iterated suppress-and-recover NMS — "the original PyTorch NMS" that the paper's kernel fuses
 *        is, for ALIKED / SuperPoint-family detectors, the published iterative max-pool NMS:
 *           M   = (S == maxpool(S))
 *           repeat n times:  supp = maxpool(M) > 0 ;  S' = supp ? 0 : S ;
 *                            M   = M  or  ((S' == maxpool(S')) and not supp)
 *       with a (2r+1)^2 window clipped at the image edge (max-pool padding never wins).  The paper prints
 *       neither the procedure nor n; n is a parameter (the published procedure uses 2), n = 0 is the single
 *       pass of north_star step (1).  Border exclusion and threshold are applied to the final mask.
 *   V2  reported score = S interpolated bilinearly at the refined position ("detection scores
 *       s_i"; the paper does not say where the score is read).  Selection and order keep using the raw score.
 *   V3  threshold-only mode: no cap.  The outputs have a capacity (top_k); count = min(C_b, capacity) and the
 *       total C_b is reported beside it ("dynamically shaped output").
 *   V4  score = keypoint heat x reliability (XFeat: "filtered using an additional reliability heatmap",
 *       PAPER.md:89-95).  The product is formed in the precision of the maps (fp32, one rounding) BEFORE
 *       the window maximum; threshold, order, reported score and refinement all use the product.
 *   V5  validity mask ("a fisheye validity mask that culls features near the image periphery",
 *       PAPER.md:326): a pixel can be a keypoint only where mask != 0.  Masked pixels still take part in the
 *       window maxima and in the refinement windows (they are real score values).
 *
 * Pins (tests/test_variant_pins.py, -m "not gpu"):
 *   V1: an independent torch restatement with F.max_pool2d; planted A > B > C chain where C is recovered;
 *       n = 0 equals dkd_oracle_nms.   V2: torch grid_sample(align_corners=True) at the refined points;
 *       symmetric peak -> raw score.   V3: total == mask sum, count == min(total, capacity).
 *   V4: base oracle on the numpy float32 product map; reliability 1 -> base; reliability 0 at a peak -> gone.
 *   V5: python filter of the base candidate list; all-ones -> base; a masked neighbour still suppresses.
 * Unpinned: agreement with the paper's own kernels (nothing printed).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* from dkd_oracle.c (linked into the same shared object) */
long dkd_oracle_nms(const float* S, int H, int W, int r, float thresh, uint8_t* mask);
int dkd_oracle_topk(const float* S, const uint8_t* mask, int H, int W, int top_k, int32_t* idx_out, float* score_out);
void dkd_oracle_refine(const float* S, int H, int W, int r, float T, int n, const int32_t* idx, double* off, double* kpt);
void dkd_oracle_gather(const void* F, int dtype, int Hd, int Wd, int D, int stride, int n, const double* kpt,
                       const int32_t* valid, double* out);

/* (2r+1)^2 max-pool with the window clipped at the image edge (V1) */
static void maxpool_clipped(const float* in, int H, int W, int r, float* out) {
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            float m = -INFINITY;
            for (int j = -r; j <= r; ++j)
                for (int i = -r; i <= r; ++i) {
                    int yy = y + j, xx = x + i;
                    if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
                    float v = in[(size_t)yy * W + xx];
                    if (v > m) m = v;
                }
            out[(size_t)y * W + x] = m;
        }
}

/* V1: iterated suppress-and-recover NMS + border + threshold.  iters = 0 is the single pass.  Returns the
 * number of candidates; mask[y*W+x] = 1 for candidates. */
long dkd_oracle_nms_iter(const float* S, int H, int W, int r, float thresh, int iters, uint8_t* mask) {
    size_t n = (size_t)H * W;
    float* mp = (float*)malloc(n * sizeof(float));
    float* M = (float*)malloc(n * sizeof(float));       /* the max mask as 0 / 1 floats (it is max-pooled) */
    float* Sp = (float*)malloc(n * sizeof(float));
    float* t = (float*)malloc(n * sizeof(float));
    maxpool_clipped(S, H, W, r, mp);
    for (size_t p = 0; p < n; ++p) M[p] = (S[p] == mp[p]) ? 1.0f : 0.0f;
    for (int it = 0; it < iters; ++it) {
        maxpool_clipped(M, H, W, r, t);                  /* supp = maxpool(M) > 0 */
        for (size_t p = 0; p < n; ++p) Sp[p] = (t[p] > 0.0f) ? 0.0f : S[p];
        maxpool_clipped(Sp, H, W, r, mp);
        for (size_t p = 0; p < n; ++p)
            if (Sp[p] == mp[p] && !(t[p] > 0.0f)) M[p] = 1.0f;
    }
    long cnt = 0;
    memset(mask, 0, n);
    for (int y = r; y < H - r; ++y)
        for (int x = r; x < W - r; ++x) {
            size_t p = (size_t)y * W + x;
            if (M[p] != 0.0f && S[p] > thresh) { mask[p] = 1; ++cnt; }
        }
    free(mp); free(M); free(Sp); free(t);
    return cnt;
}

/* V2: S interpolated bilinearly at (px, py); corners clamped to the image like O4's */
double dkd_oracle_bilinear_score(const float* S, int H, int W, double px, double py) {
    if (px < 0.0) px = 0.0;
    if (px > (double)(W - 1)) px = (double)(W - 1);
    if (py < 0.0) py = 0.0;
    if (py > (double)(H - 1)) py = (double)(H - 1);
    int x0 = (int)floor(px), y0 = (int)floor(py);
    int x1 = x0 + 1 < W - 1 ? x0 + 1 : W - 1, y1 = y0 + 1 < H - 1 ? y0 + 1 : H - 1;
    double fx = px - (double)x0, fy = py - (double)y0;
    double s00 = S[(size_t)y0 * W + x0], s01 = S[(size_t)y0 * W + x1];
    double s10 = S[(size_t)y1 * W + x0], s11 = S[(size_t)y1 * W + x1];
    return (1.0 - fy) * ((1.0 - fx) * s00 + fx * s01) + fy * ((1.0 - fx) * s10 + fx * s11);
}

/*
 * Whole path with the variants.  score = heat [B,H,W]; rel = reliability [B,H,W] or NULL (V4); vmask [B,H,W]
 * u8 or NULL (V5); nms_iters (V1); score_mode 0 raw / 1 bilinear (V2); out_total [B] or NULL (V3).
 * Outputs as dkd_oracle_extract, except out_scores is double (V2 yields non-fp32 values; in raw mode it holds
 * the fp32 score widened exactly).  Returns 0, -1 on a bad argument.
 */
int dkd_oracle_extract_var(const float* score, const float* rel, const uint8_t* vmask, int B, int H, int W,
                           const void* desc, int desc_dtype, int Hd, int Wd, int D, int stride,
                           int r, float thresh, int top_k, float T, int nms_iters, int score_mode,
                           double* out_kpts, double* out_off, double* out_scores, double* out_desc,
                           int32_t* out_count, int32_t* out_index, int32_t* out_total) {
    if (!score || B < 1 || H < 1 || W < 1 || r < 1 || r > 31 || top_k < 1 || !(T > 0.0f) || nms_iters < 0) return -1;
    if (desc && (Hd < 1 || Wd < 1 || D < 1 || stride < 1 || !out_desc)) return -1;
    size_t n = (size_t)H * W;
    uint8_t* mask = (uint8_t*)malloc(n);
    float* Sb = (float*)malloc(n * sizeof(float));
    float* sc32 = (float*)malloc((size_t)top_k * sizeof(float));
    size_t esz = desc_dtype == 1 ? 2 : 4;
    for (int b = 0; b < B; ++b) {
        const float* heat = score + (size_t)b * n;
        for (size_t p = 0; p < n; ++p) {                                    /* V4: fp32 product, one rounding */
            if (rel) { volatile float prod = heat[p] * rel[(size_t)b * n + p]; Sb[p] = prod; }
            else Sb[p] = heat[p];
        }
        long C;
        if (nms_iters > 0) C = dkd_oracle_nms_iter(Sb, H, W, r, thresh, nms_iters, mask);   /* V1 */
        else C = dkd_oracle_nms(Sb, H, W, r, thresh, mask);
        if (vmask)                                                          /* V5: candidates only where valid */
            for (size_t p = 0; p < n; ++p)
                if (mask[p] && vmask[(size_t)b * n + p] == 0) { mask[p] = 0; --C; }
        if (out_total) out_total[b] = (int32_t)C;                           /* V3 */
        int32_t* idx = out_index + (size_t)b * top_k;
        out_count[b] = dkd_oracle_topk(Sb, mask, H, W, top_k, idx, sc32);
        double* kp = out_kpts + (size_t)b * top_k * 2;
        dkd_oracle_refine(Sb, H, W, r, T, top_k, idx, out_off + (size_t)b * top_k * 2, kp);
        for (int i = 0; i < top_k; ++i) {
            double s = (double)sc32[i];
            if (idx[i] >= 0 && score_mode == 1) s = dkd_oracle_bilinear_score(Sb, H, W, kp[2 * i], kp[2 * i + 1]);   /* V2 */
            out_scores[(size_t)b * top_k + i] = s;
        }
        if (desc) {
            const char* F = (const char*)desc + (size_t)b * Hd * Wd * D * esz;
            dkd_oracle_gather(F, desc_dtype, Hd, Wd, D, stride, top_k, kp, idx, out_desc + (size_t)b * top_k * D);
        }
    }
    free(mask); free(Sb); free(sc32);
    return 0;
}
