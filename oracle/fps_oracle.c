/*
 * oracle/fps_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, classical O(N*M) farthest point sampling on the CPU.  It is the
 * definition the CUDA path (paper_2606_06255_b200/csrc) is checked against and
 * it shares no code, header, table or helper with that path.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call it.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md, arxiv/paper_2606_06255):
 *   - Alg. 1 "Standard FPS Algorithm": D = +inf, seed the set
 *     with p_start, then repeat { D[i] = min(D[i], dist(p_i, s_last)) for all
 *     i; p_next = argmax_i D[i] }.
 *   - Eq. 3-4: s_j = argmax_p min_{s in S_{j-1}} dist(p, s),
 *     D[i] caches the inner min.
 *   - Exactness contract: same seed, same floating-point
 *     precision, argmax ties -> smallest original input index.
 *   - Effective update is a strict "<", Eq. 2 PAPER.md:124.
 * Readings fixed by BASELINE.json north_star / DESIGN.md (paper is silent or
 * differs):
 *   - R1 the distance is the SQUARED Euclidean distance evaluated in fp32 as
 *        ((dx*dx + dy*dy) + dz*dz), dx = x_i - x_s etc., every operation
 *        rounded to nearest-even, no FMA contraction (the paper writes the
 *        Euclidean norm with a square root, Eq. 1/29 PAPER.md:122,340).
 *   - R2 the first sample is the caller's start index (random in the paper,
 *        Eq. 12).
 *   - R3 out_mindist[0] = +inf (the value of max_i D[i] when s_0 is taken,
 *        Alg. 1 l.2 PAPER.md:56); D[start] becomes +0 through the ordinary
 *        update of iteration 1.
 *   - R4 the update after the last selection is not needed and is skipped.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math (x86-64: SSE scalar fp32,
 * never x87).  -ffp-contract=off is what forbids FMA; the volatile-free code
 * below has no other way to change rounding.
 *
 * Pins (tests/test_oracle_pins.py): brute force straight from Eq. 3 on N<=64,
 * closed forms (integer line, cube corners, identical points), M=2 = one
 * NumPy argmax, O(M^2) recomputation of out_mindist from the outputs alone,
 * invariants, metamorphic scaling, and the arithmetic-sensitivity lattice.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* One cloud.  P: [N][3] fp32 row-major.  Returns 0, or -1 on bad arguments.
 * out_idx[M] int32 original indices in selection order; out_mindist[M] fp32. */
int oracle_fps(const float *P, int32_t N, int32_t M, int32_t start,
               int32_t *out_idx, float *out_mindist)
{
    if (!P || !out_idx || !out_mindist) return -1;
    if (N < 1 || M < 1 || M > N || start < 0 || start >= N) return -1;

    float *D = (float *)malloc((size_t)N * sizeof(float));
    if (!D) return -2;
    for (int32_t i = 0; i < N; ++i) D[i] = INFINITY;          /* Alg. 1 l.2 */

    int32_t cur = start;                                       /* R2 */
    out_idx[0] = start;
    out_mindist[0] = INFINITY;                                 /* R3 */

    for (int32_t j = 1; j < M; ++j) {                          /* Alg. 1 l.6 */
        const float xs = P[3 * (size_t)cur + 0];
        const float ys = P[3 * (size_t)cur + 1];
        const float zs = P[3 * (size_t)cur + 2];
        float best = -1.0f;
        int32_t besti = 0;
        for (int32_t i = 0; i < N; ++i) {                      /* Alg. 1 l.8 */
            const float dx = P[3 * (size_t)i + 0] - xs;
            const float dy = P[3 * (size_t)i + 1] - ys;
            const float dz = P[3 * (size_t)i + 2] - zs;
            const float d = ((dx * dx + dy * dy) + dz * dz);   /* R1 */
            if (d < D[i]) D[i] = d;                            /* Eq. 2, strict < */
            if (D[i] > best) { best = D[i]; besti = i; }       /* strict >: lowest index wins ties */
        }
        cur = besti;                                           /* Alg. 1 l.12 */
        out_idx[j] = besti;
        out_mindist[j] = best;
    }
    free(D);
    return 0;
}

/* B independent clouds of equal size, same start index (BASELINE.json configs);
 * one OpenMP thread per cloud, at most `threads` (<=0: library default).
 * P: [B][N][3]; out_idx, out_mindist: [B][M].  Returns the number of threads
 * actually used (>=1), or a negative error code. */
int oracle_fps_batch(const float *P, int32_t B, int32_t N, int32_t M, int32_t start,
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
        int r = oracle_fps(P + (size_t)b * N * 3, N, M, start,
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
