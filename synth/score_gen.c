/*
 * score_gen.c — seeded synthetic SCORE-MAP generator (inputs only; none of the method's
 * arithmetic lives here).  Serves both the CPU oracle and the CUDA path: the same bytes go to
 * both.  Recipe: DESIGN.md "Input recipe" (from BASELINE.json configs 1-5 / SURVEY.md §8(d)):
 *
 *   value(b,y,x) = clamp( base * U24(b, y*W+x)  +  sum_{k < nblobs} A_k exp(-d^2 / (2 sigma_k^2)), 0, 1 )
 *
 *   U24        : 24-bit uniform in [0,1) from a counter-based mixer (splitmix64 finaliser)
 *   blob k     : centre (cx,cy) ~ U[0,W) x U[0,H) (real-valued), A ~ U(0.3,1), sigma ~ U(0.8,2.0) px,
 *                added (in blob-index order, in double) to pixels with
 *                |x - floor(cx)| <= ceil(5 sigma) and |y - floor(cy)| <= ceil(5 sigma)
 *   the sum is formed in double and rounded ONCE to fp32 after the clamp.  The clamp is what
 *   produces exact-1.0 ties (G1).
 *
 * Build: gcc -O2 -std=c99 -fopenmp -shared -fPIC score_gen.c -o libscore_gen.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static uint64_t splitmix64(uint64_t x) {
    uint64_t z = x + 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

/* tags: 1 = noise, 2 = blob parameters, 3 = descriptors (torch side, synth/__init__.py) */
static uint64_t draw(uint64_t seed, uint64_t tag, uint64_t b, uint64_t counter) {
    return splitmix64(seed ^ (tag << 56) ^ (b << 40) ^ counter);
}

static double u53(uint64_t h) { return (double)(h >> 11) * (1.0 / 9007199254740992.0); }

/* out [B,H,W] fp32.  Returns 0, -1 on allocation failure. */
int synth_score_maps(float* out, int B, int H, int W, uint64_t seed, double base, int nblobs) {
    int fail = 0;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < B; ++b) {
        size_t npx = (size_t)H * (size_t)W;
        double* acc = (double*)malloc(npx * sizeof(double));
        if (!acc) { fail = 1; continue; }
        for (size_t p = 0; p < npx; ++p)
            acc[p] = base * ((double)(draw(seed, 1, (uint64_t)b, (uint64_t)p) >> 40) * (1.0 / 16777216.0));
        for (int k = 0; k < nblobs; ++k) {
            double cx = u53(draw(seed, 2, (uint64_t)b, 4ULL * k + 0)) * (double)W;
            double cy = u53(draw(seed, 2, (uint64_t)b, 4ULL * k + 1)) * (double)H;
            double A  = 0.3 + 0.7 * u53(draw(seed, 2, (uint64_t)b, 4ULL * k + 2));
            double sg = 0.8 + 1.2 * u53(draw(seed, 2, (uint64_t)b, 4ULL * k + 3));
            int R = (int)ceil(5.0 * sg);
            int ix = (int)floor(cx), iy = (int)floor(cy);
            double inv = 1.0 / (2.0 * sg * sg);
            for (int y = iy - R; y <= iy + R; ++y) {
                if (y < 0 || y >= H) continue;
                for (int x = ix - R; x <= ix + R; ++x) {
                    if (x < 0 || x >= W) continue;
                    double ddx = (double)x - cx, ddy = (double)y - cy;
                    acc[(size_t)y * W + x] += A * exp(-(ddx * ddx + ddy * ddy) * inv);
                }
            }
        }
        float* o = out + (size_t)b * npx;
        for (size_t p = 0; p < npx; ++p) {
            double v = acc[p];
            if (v < 0.0) v = 0.0;
            if (v > 1.0) v = 1.0;
            o[p] = (float)v;
        }
        free(acc);
    }
    return fail ? -1 : 0;
}
