/*
 * match_oracle.c — CPU ORACLE for the consumers of the descriptor output:
 *   (1) cosine nearest-neighbour matching of two padded descriptor sets with a Lowe ratio test,
 *   (2) the brute-force cosine retrieval scan of a global descriptor over the keyframe database,
 *   (3) per-match stereo validation, and (4) covariance-weighted square-root information.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as dkd_oracle.c).  Plain C99, fp64, naive loops
 * in the order of the definitions; shares no code with the CUDA library.
 *
 * Passages followed (reference = /root/reference/PAPER.md) and readings (M1..M8,
 * "Stereo validation", S1..S4, "Covariance", C1..C4):
 *
 * (1) PAPER.md:157 (Sec. III-D): "Geometric verification reuses the active local descriptors of the selected
 *     front-end through cosine nearest-neighbour matching with a Lowe ratio test".  Descriptors are
 *     l2-normalised (Eq. 1), so cosine similarity is the dot product (Eq. 4).
 *     M1  s_ij = sum_c a_ic b_jc over the first na rows of A and nb rows of B (sets are zero-padded to the
 *         cap; padding rows never match and are never matched).
 *     M2  nearest neighbour of i: j1 = argmax_j s_ij, ties -> the smallest j; second best s2 = max_{j != j1}
 *         s_ij (s2 = -1, the smallest cosine, when nb == 1).
 *     M3  ratio test in its usual form on Euclidean distances between unit vectors, d^2 = 2 - 2 s (clamped at
 *         0): keep iff d1 < rho * d2, i.e. d1^2 < rho^2 d2^2.  rho is not printed; it is a parameter
 *         (0.8, Lowe's published value, in the tests and the bench).  rho >= 1e9 disables the test.
 *     M4  optional mutual check: keep (i, j1) only if i = argmax_i' s_i'j1 (ties -> smallest i').
 *     M5  output per row: match index j1 or -1; s1; s2 (rows >= na: -1, 0, 0).
 * (2) PAPER.md:147-157: "Loop candidates are retrieved using cosine similarity between the current
 *     descriptor g_t and a past descriptor g_k" (Eq. 4); "a fixed window of the most recent keyframes is
 *     excluded"; "Candidates with sim > tau_sim are ranked by similarity"; "brute-force scan over the keyframe
 *     database, O(n)"; "the 50 most recent keyframes are excluded", "tau_sim = 0.60";
 *     g in R^{32*384}.
 *     M6  database rows are in insertion order; rows k >= n - n_exclude are the excluded recent window.
 *     M7  sim_k = g . db_k in fp64 (both unit-norm: Eq. 4's final equality); gate strict: sim_k > tau.
 *     M8  candidates ranked by (sim desc, k asc), truncated to max_cand.
 * (3) PAPER.md:145: "Matches with negligible disparity are discarded.  The remaining pairs are triangulated
 *     using the known ... stereo baseline and are retained exclusively if they yield a positive depth within a
 *     valid range and exhibit a reprojection error of no more than 1.5-pixel across both views."
 *     S1  rectified pinhole pair (fx, fy, cx, cy shared; right camera at +baseline along x):
 *         disparity d = uL - uR; "negligible" = d <= d_min (parameter).
 *     S2  triangulation = the least-squares point of the rectified pair: depth z = fx * baseline / d,
 *         X = (uL - cx) z / fx, Y = (vm - cy) z / fy with vm = (vL + vR) / 2 (the two rays meet exactly in u
 *         and are split evenly in v).
 *     S3  valid range: z_min < z < z_max (parameters).
 *     S4  reprojection error of a view = Euclidean pixel distance between the observation and the projection of
 *         (X, Y, z): here |vL - vm| = |vR - vm| = |vL - vR| / 2 in both views; keep iff max of the two <= max_reproj
 *         (1.5 px).  Output: valid flag, (X, Y, z), disparity, reprojection error.
 * (4) PAPER.md:586-603 (App. A-B, Eq. 9-11): Sigma_px = L L^T from the predicted lower-triangular factor
 *     L = [[l11, 0], [l21, l22]], rescaled to native pixels "by the squared letterbox factor"; Sigma_n = J Sigma_px
 *     J^T with J = diag(1/fx, 1/fy) (pinhole, Eq. 9); Sigma_eff^-1 = lambda Sigma_n^-1 (Eq. 11) with "a lower clamp
 *     on the gain and, optionally, a small additive floor on Sigma_px"; Omega = chol(Sigma_eff^-1) (Eq. 10) with
 *     "the isotropic sigma_0^-1 I retained as a fallback whenever the Cholesky factorization fails".
 *     C1  Sigma_px = s^2 L L^T + floor I (s = letterbox scale factor; floor >= 0).
 *     C2  lambda_eff = max(lambda, lambda_min).
 *     C3  Omega is the UPPER-triangular factor with Omega^T Omega = Sigma_eff^-1 (so that ||Omega r||^2 =
 *         r^T Sigma_eff^-1 r, the property Eq. 10 states): Omega = Lc^T, Lc = lower Cholesky factor of Sigma_eff^-1.
 *     C4  failure -> Omega = I / sigma0, flag 0.  The factorisation fails iff an input is non-finite or Sigma_px is
 *         not positive definite; the latter is decided on det(Sigma_px) expanded into its non-negative terms,
 *         s^4 l11^2 l22^2 + floor s^2 (l11^2 + l21^2 + l22^2) + floor^2 > 0, whose sign no rounding can flip (the
 *         textbook a c - b^2 cancels to a rounding residue for a singular prediction); a non-positive second pivot
 *         of the Cholesky recursion is a failure as well.
 *
 * Pins (tests/test_match_pins.py — matching, retrieval, stereo and covariance alike —, -m "not gpu"): brute-force python loops on tiny
 * sets; torch.topk on a float64 matmul; planted duplicates / orthogonal sets / exact ties; the Lowe test on hand
 * distances; closed-form triangulation of planted 3-D points; a 2x2 Cholesky worked by hand
 * (tests/golden/chol2x2.txt); Omega^T Omega Sigma_eff = I; the isotropic fallback.
 * Unpinned: agreement with the paper's implementation (nothing printed; rho, d_min, z range are unprinted).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define MO_F32 0
#define MO_F16 1

static double mo_half(uint16_t h) {           /* exact IEEE binary16 -> double */
    int sign = (h >> 15) & 1, e = (h >> 10) & 0x1f, m = h & 0x3ff;
    double v;
    if (e == 0) v = ldexp((double)m, -24);
    else if (e == 31) v = m ? NAN : INFINITY;
    else v = ldexp((double)(m + 1024), e - 25);
    return sign ? -v : v;
}
static double mo_get(const void* p, int dtype, size_t e) {
    return dtype == MO_F16 ? mo_half(((const uint16_t*)p)[e]) : (double)((const float*)p)[e];
}

/* (1) M1..M5.  A [Na, D], B [Nb, D] row-major, f16 or f32; na <= Na, nb <= Nb valid rows.
 * out_idx [Na] i32, out_s1 [Na], out_s2 [Na] double.  S (optional, may be NULL): the full na x nb similarity
 * matrix, row-major with leading dimension nb.  Returns the number of accepted matches, -1 on a bad argument. */
int match_oracle_nn(const void* A, const void* Bm, int dtype, int Na, int Nb, int D, int na, int nb,
                    double ratio, int mutual, int32_t* out_idx, double* out_s1, double* out_s2, double* S) {
    if (!A || !Bm || Na < 1 || Nb < 1 || D < 1 || na < 0 || nb < 0 || na > Na || nb > Nb) return -1;
    double* sim = S ? S : (double*)malloc(((size_t)na * nb + 1) * sizeof(double));
    for (int i = 0; i < na; ++i)                                               /* M1 */
        for (int j = 0; j < nb; ++j) {
            double s = 0.0;
            for (int c = 0; c < D; ++c) s += mo_get(A, dtype, (size_t)i * D + c) * mo_get(Bm, dtype, (size_t)j * D + c);
            sim[(size_t)i * nb + j] = s;
        }
    int accepted = 0;
    for (int i = 0; i < Na; ++i) {
        out_idx[i] = -1; out_s1[i] = 0.0; out_s2[i] = 0.0;
        if (i >= na || nb < 1) continue;
        int j1 = 0;                                                            /* M2: ties -> smallest j */
        for (int j = 1; j < nb; ++j)
            if (sim[(size_t)i * nb + j] > sim[(size_t)i * nb + j1]) j1 = j;
        double s1 = sim[(size_t)i * nb + j1], s2 = -1.0;
        int have2 = 0;
        for (int j = 0; j < nb; ++j) {
            if (j == j1) continue;
            if (!have2 || sim[(size_t)i * nb + j] > s2) { s2 = sim[(size_t)i * nb + j]; have2 = 1; }
        }
        out_s1[i] = s1; out_s2[i] = s2;
        int keep = 1;
        if (ratio < 1e9) {                                                     /* M3 */
            double d1 = 2.0 - 2.0 * s1, d2 = 2.0 - 2.0 * s2;
            if (d1 < 0.0) d1 = 0.0;
            if (d2 < 0.0) d2 = 0.0;
            keep = d1 < ratio * ratio * d2;
        }
        if (keep && mutual) {                                                  /* M4: ties -> smallest i' */
            int i1 = 0;
            for (int ii = 1; ii < na; ++ii)
                if (sim[(size_t)ii * nb + j1] > sim[(size_t)i1 * nb + j1]) i1 = ii;
            keep = i1 == i;
        }
        if (keep) { out_idx[i] = j1; ++accepted; }
    }
    if (!S) free(sim);
    return accepted;
}

/* (2) M6..M8.  db [n, D] f16|f32, q [D] same dtype.  out_sim [n] double (every row, also the excluded window);
 * out_cand [max_cand] i32 (-1 padded), returns the number of candidates written, -1 on a bad argument. */
typedef struct { double s; int32_t k; } mo_cand;
static int mo_cand_cmp(const void* a, const void* b) {
    const mo_cand* p = (const mo_cand*)a; const mo_cand* q = (const mo_cand*)b;
    if (p->s > q->s) return -1;
    if (p->s < q->s) return 1;
    return p->k < q->k ? -1 : (p->k > q->k ? 1 : 0);
}
int retrieval_oracle_scan(const void* db, const void* q, int dtype, int n, int D, int n_exclude, double tau,
                          int max_cand, double* out_sim, int32_t* out_cand) {
    if (!db || !q || n < 0 || D < 1 || n_exclude < 0 || max_cand < 0) return -1;
    mo_cand* c = (mo_cand*)malloc(((size_t)n + 1) * sizeof(mo_cand));
    int m = 0;
    for (int k = 0; k < n; ++k) {
        double s = 0.0;
        for (int e = 0; e < D; ++e) s += mo_get(q, dtype, (size_t)e) * mo_get(db, dtype, (size_t)k * D + e);   /* M7 */
        out_sim[k] = s;
        if (k < n - n_exclude && s > tau) { c[m].s = s; c[m].k = k; ++m; }     /* M6, M7 (strict) */
    }
    qsort(c, (size_t)m, sizeof(mo_cand), mo_cand_cmp);                         /* M8 */
    int K = m < max_cand ? m : max_cand;
    for (int i = 0; i < max_cand; ++i) out_cand[i] = i < K ? c[i].k : -1;
    free(c);
    return K;
}

/* (3) S1..S4.  pl, pr [n,2] double (u,v) pixel observations of matched keypoints in the left / right view.
 * out_xyz [n,3], out_disp [n], out_err [n] double; out_valid [n] u8.  Returns the number of valid matches. */
int stereo_oracle_validate(const double* pl, const double* pr, int n, double fx, double fy, double cx, double cy,
                           double baseline, double d_min, double z_min, double z_max, double max_reproj,
                           double* out_xyz, double* out_disp, double* out_err, uint8_t* out_valid) {
    int nv = 0;
    for (int i = 0; i < n; ++i) {
        double uL = pl[2 * i], vL = pl[2 * i + 1], uR = pr[2 * i], vR = pr[2 * i + 1];
        double d = uL - uR;                                                    /* S1 */
        out_disp[i] = d;
        out_valid[i] = 0; out_xyz[3 * i] = out_xyz[3 * i + 1] = out_xyz[3 * i + 2] = 0.0; out_err[i] = 0.0;
        if (!(d > d_min)) continue;
        double z = fx * baseline / d;                                          /* S2 */
        double vm = 0.5 * (vL + vR);
        double X = (uL - cx) * z / fx, Y = (vm - cy) * z / fy;
        /* reprojection into both views (S4), written out in full */
        double uLp = fx * X / z + cx, vLp = fy * Y / z + cy;
        double uRp = fx * (X - baseline) / z + cx, vRp = vLp;
        double eL = sqrt((uLp - uL) * (uLp - uL) + (vLp - vL) * (vLp - vL));
        double eR = sqrt((uRp - uR) * (uRp - uR) + (vRp - vR) * (vRp - vR));
        double e = eL > eR ? eL : eR;
        out_xyz[3 * i] = X; out_xyz[3 * i + 1] = Y; out_xyz[3 * i + 2] = z; out_err[i] = e;
        if (!(z > z_min && z < z_max)) continue;                               /* S3 */
        if (!(e <= max_reproj)) continue;
        out_valid[i] = 1; ++nv;
    }
    return nv;
}

/* (4) C1..C4.  Lf [n,3] double = (l11, l21, l22).  out_omega [n,4] row-major 2x2, out_ok [n] u8.
 * Returns the number of keypoints whose factorisation succeeded. */
int cov_oracle_sqrt_info(const double* Lf, int n, double scale, double floor_px, double fx, double fy, double lambda,
                         double lambda_min, double sigma0, double* out_omega, uint8_t* out_ok) {
    int ok_n = 0;
    for (int i = 0; i < n; ++i) {
        double l11 = Lf[3 * i], l21 = Lf[3 * i + 1], l22 = Lf[3 * i + 2];
        double s2 = scale * scale;
        double a = s2 * (l11 * l11) + floor_px;                                /* C1: Sigma_px = s^2 L L^T + floor I */
        double b = s2 * (l11 * l21);
        double c = s2 * (l21 * l21 + l22 * l22) + floor_px;
        double na = a / (fx * fx), nb = b / (fx * fy), nc = c / (fy * fy);     /* Eq. 9: Sigma_n = J Sigma_px J^T */
        double det_px = s2 * s2 * (l11 * l11) * (l22 * l22)                    /* C4: det(Sigma_px), non-negative terms */
                      + floor_px * s2 * (l11 * l11 + l21 * l21 + l22 * l22) + floor_px * floor_px;
        double det = det_px / (fx * fx * fy * fy);                             /* det(Sigma_n) */
        double lam = lambda > lambda_min ? lambda : lambda_min;                /* C2 */
        int ok = isfinite(na) && isfinite(nb) && isfinite(nc) && na > 0.0 && det > 0.0 && isfinite(det);
        double o00 = 1.0 / sigma0, o01 = 0.0, o10 = 0.0, o11 = 1.0 / sigma0;   /* C4 fallback */
        if (ok) {
            double ia = lam * nc / det, ib = -lam * nb / det, ic = lam * na / det;   /* Eq. 11: lambda Sigma_n^-1 */
            double c11 = sqrt(ia);                                             /* lower Cholesky of [[ia, ib], [ib, ic]] */
            double c21 = ib / c11;
            double piv = ic - c21 * c21;
            if (ia > 0.0 && piv > 0.0 && isfinite(c11) && isfinite(piv)) {
                double c22 = sqrt(piv);
                o00 = c11; o01 = c21; o10 = 0.0; o11 = c22;                    /* C3: Omega = Lc^T (upper) */
            } else ok = 0;
        }
        out_omega[4 * i] = o00; out_omega[4 * i + 1] = o01; out_omega[4 * i + 2] = o10; out_omega[4 * i + 3] = o11;
        out_ok[i] = (uint8_t)ok;
        ok_n += ok;
    }
    return ok_n;
}
