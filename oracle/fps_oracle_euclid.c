/*
 * oracle/fps_oracle_euclid.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Classical O(N*M) farthest point sampling with the EUCLIDEAN distance, i.e. the
 * paper's literal formulation (Alg. 1; dist = ||p - s||_2, Eq. 1
 * PAPER.md:122 and Eq. 29), as opposed to the squared distance that
 * BASELINE.json fixes for the main path (oracle/fps_oracle.c).  It is the
 * reference for the FPS_FLAG_EUCLIDEAN mode of the CUDA library (SURVEY.md 8(f)
 * NEXT-4) and shares no code with it.
 *
 * Distance: d = sqrtf(((dx*dx + dy*dy) + dz*dz)), every operation fp32,
 * round-to-nearest-even, no FMA; sqrtf is the correctly rounded IEEE square
 * root (x86-64 sqrtss).  Everything else as in fps_oracle.c: strict "<" update
 * (Eq. 2), argmax ties -> smallest original index,
 * first sample = start, out_mindist[0] = +inf.
 *
 * In fp32 this is a different FUNCTION from the squared-distance FPS: sqrt maps
 * about half of all pairs of adjacent fp32 values to the same result, so maxima
 * that are distinct in the squared domain can tie here and go to the lower index.
 *
 * Pins (tests/test_oracle_pins.py): brute force from Eq. 3 with sqrt on N<=64,
 * closed forms (integer line), agreement with sqrt(squared oracle) where no such
 * collapse occurs, and a constructed collapse where the two oracles must differ.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_fps_euclid(const float *P, int32_t N, int32_t M, int32_t start,
                      int32_t *out_idx, float *out_mindist)
{
    if (!P || !out_idx || !out_mindist) return -1;
    if (N < 1 || M < 1 || M > N || start < 0 || start >= N) return -1;
    float *D = (float *)malloc((size_t)N * sizeof(float));
    if (!D) return -2;
    for (int32_t i = 0; i < N; ++i) D[i] = INFINITY;
    int32_t cur = start;
    out_idx[0] = start;
    out_mindist[0] = INFINITY;
    for (int32_t j = 1; j < M; ++j) {
        const float xs = P[3 * (size_t)cur + 0];
        const float ys = P[3 * (size_t)cur + 1];
        const float zs = P[3 * (size_t)cur + 2];
        float best = -1.0f;
        int32_t besti = 0;
        for (int32_t i = 0; i < N; ++i) {
            const float dx = P[3 * (size_t)i + 0] - xs;
            const float dy = P[3 * (size_t)i + 1] - ys;
            const float dz = P[3 * (size_t)i + 2] - zs;
            const float d = sqrtf(((dx * dx + dy * dy) + dz * dz));   /* Eq. 1 / Eq. 29 */
            if (d < D[i]) D[i] = d;                                    /* Eq. 2, strict < */
            if (D[i] > best) { best = D[i]; besti = i; }               /* lowest index wins ties */
        }
        cur = besti;
        out_idx[j] = besti;
        out_mindist[j] = best;
    }
    free(D);
    return 0;
}

int oracle_fps_euclid_batch(const float *P, int32_t B, int32_t N, int32_t M, int32_t start,
                            int32_t *out_idx, float *out_mindist, int32_t threads)
{
    if (B < 1) return -1;
    int used = 1;
    int err = 0;
#ifdef _OPENMP
    int t = threads > 0 ? threads : omp_get_max_threads();
    if (t > B) t = B;
    used = t;
#pragma omp parallel for num_threads(t) schedule(dynamic, 1)
#endif
    for (int32_t b = 0; b < B; ++b) {
        int r = oracle_fps_euclid(P + (size_t)b * N * 3, N, M, start,
                                  out_idx + (size_t)b * M, out_mindist + (size_t)b * M);
        if (r != 0) {
#ifdef _OPENMP
#pragma omp critical
#endif
            err = r;
        }
    }
    (void)threads;
    return err ? err : used;
}
