/*
 * oracle/fps_pruned_cpu.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * The paper's CPU RadiusFPS (section 3 of arxiv/paper_2606_06255) written out
 * step by step, as an independent cross-check of oracle/fps_oracle.c (it must
 * return bit-identical indices and min-distances) and as the second timed CPU
 * baseline.  It shares no code with fps_oracle.c nor with the CUDA path; only
 * tests/, __graft_entry__.smoke() and bench.py's CPU legs may use it.
 *
 * Steps and the passages they follow (PAPER.md = /root/reference/PAPER.md):
 *   preprocessing   Eq. 6-8  PAPER.md:187-200  bbox, alpha = 1+eps, L, floor+clamp voxel coords
 *                   Eq. 31   PAPER.md:372      V_id = vz n^2 + vy n + vx
 *                   Eq. 9-10 PAPER.md:202-210  active voxels only; centre c_k and radius r_k
 *                   Eq. 11   PAPER.md:212-216  Dist_p = +inf, Dist_v
 *   selection       Eq. 15-18 PAPER.md:244-259 two-level argmax == global argmax
 *   radius prune    Eq. 23-26 PAPER.md:295-313 skip voxel if LB(v_k,s_j) >= Dist_v[k]
 *   point skip      Eq. 27-28 PAPER.md:327-336 skip p_i if an axis difference alone is >= Dist_p[i]
 *   update + sync   Eq. 29-30 PAPER.md:338-350 Dist_p[i] = min(...), Dist_v[k] = max over voxel
 *
 * Readings (SURVEY.md 8(c) A-numbers):
 *   A1  squared fp32 distance ((dx*dx + dy*dy) + dz*dz), no FMA; all tests re-derived in the
 *       squared domain.
 *   A4  voxel-level tie-break: each voxel stores (max Dist_p, LOWEST ORIGINAL INDEX attaining
 *       it); the voxel-level argmax compares that pair, so it equals the global argmax.
 *   A8  point skip in the squared domain with the SAME rounded products that feed the sum:
 *       skip if dx*dx >= D or dy*dy >= D or dz*dz >= D.  Exact with no margin because fp32
 *       addition of non-negative terms is monotone.
 *   A9  Eq. 25 is proved over the reals; here it is applied with fp32 safety margins:
 *         build:  r_k = sqrtf(max_p d2(p,c_k)) * (1+2^-20)
 *         test:   dc = sqrtf(d2(s,c_k)) * (1-2^-20);  t = (dc - r_k) * (1-2^-20)
 *                 prune iff Dist_v[k] == 0, or
 *                           t > 0 and (t*t)*(1-2^-20) >= Dist_v[k] and Dist_v[k] >= 1e-30f
 *       (Dist_v[k] == 0: no squared distance is < 0, so the strict-< update of Eq. 2 cannot fire;
 *       the 1e-30f clause keeps the relative-error argument clear of underflow).
 *   A10 c_k = midpoint of the axis-aligned bounding box of the voxel's own points, r_k tight
 *       (any enclosing sphere is valid; Eq. 10's sqrt(3)/2 L is one).
 *   A11 Dist_v starts at +inf instead of 0, so iteration 1 prunes nothing and the "initial
 *       update" (Eq. 13-14) is the general step.
 *   A12 eps = 1e-3.
 *
 * Build: gcc -O2 -ffp-contract=off (no fast-math).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int64_t voxel_tests;      /* Eq. 25 evaluations                                  */
    int64_t voxels_visited;   /* voxels that survived the prune                      */
    int64_t points_visited;   /* points of visited voxels                            */
    int64_t points_computed;  /* points that passed the skip test (Eq. 28 not taken) */
    int64_t effective;        /* strict decreases of Dist_p (Eq. 2)                  */
    int32_t K;                /* active voxels                                       */
    int32_t n_vox;
} pruned_stats;

static inline float sq_dist(float x, float y, float z, float xs, float ys, float zs)
{
    const float dx = x - xs, dy = y - ys, dz = z - zs;
    return ((dx * dx + dy * dy) + dz * dz);
}

/* One cloud.  flags bit0: disable radius prune; bit1: disable point skip;
 * bit2: NEGATIVE CONTROL, centroid-only prune r_k := 0 with no margins (Fig. 5/6 PAPER.md:265-276,
 * expected to break exactness).  stats may be NULL. */
int pruned_fps_cpu(const float *P, int32_t N, int32_t M, int32_t start, int32_t n_vox,
                   int32_t flags, int32_t *out_idx, float *out_mindist, pruned_stats *stats)
{
    if (!P || !out_idx || !out_mindist) return -1;
    if (N < 1 || M < 1 || M > N || start < 0 || start >= N || n_vox < 1 || n_vox > 256) return -1;
    const int no_prune = flags & 1, no_skip = flags & 2, centroid_only = flags & 4;
    const float UP = 1.0f + 0x1p-20f, DN = 1.0f - 0x1p-20f;

    /* ---- Eq. 6-7: bounding box and voxel side ---- */
    float lo[3] = {P[0], P[1], P[2]}, hi[3] = {P[0], P[1], P[2]};
    for (int32_t i = 1; i < N; ++i)
        for (int a = 0; a < 3; ++a) {
            const float v = P[3 * (size_t)i + a];
            if (v < lo[a]) lo[a] = v;
            if (v > hi[a]) hi[a] = v;
        }
    float Emax = hi[0] - lo[0];
    if (hi[1] - lo[1] > Emax) Emax = hi[1] - lo[1];
    if (hi[2] - lo[2] > Emax) Emax = hi[2] - lo[2];
    float L = (1.0f + 1e-3f) * Emax / (float)n_vox;            /* A12 */
    if (!(L > 0.0f)) L = 1.0f;                                 /* all points identical */

    /* ---- Eq. 8 + Eq. 31: voxel id per point ---- */
    const size_t nbins = (size_t)n_vox * n_vox * n_vox;
    int32_t *vid = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int32_t *binstart = (int32_t *)calloc(nbins + 1, sizeof(int32_t));
    int32_t *order = (int32_t *)malloc((size_t)N * sizeof(int32_t));   /* sorted pos -> original index */
    float *D = (float *)malloc((size_t)N * sizeof(float));
    if (!vid || !binstart || !order || !D) return -2;
    for (int32_t i = 0; i < N; ++i) {
        int32_t v[3];
        for (int a = 0; a < 3; ++a) {
            int32_t c = (int32_t)floorf((P[3 * (size_t)i + a] - lo[a]) / L);
            if (c < 0) c = 0;
            if (c > n_vox - 1) c = n_vox - 1;
            v[a] = c;
        }
        vid[i] = (v[2] * n_vox + v[1]) * n_vox + v[0];
        binstart[vid[i] + 1]++;
    }
    /* stable counting sort by V_id (the paper's radix sort, Alg. 2 l.11 PAPER.md:399):
     * original indices stay ascending inside each voxel. */
    for (size_t b = 0; b < nbins; ++b) binstart[b + 1] += binstart[b];
    {
        int32_t *cursor = (int32_t *)malloc(nbins * sizeof(int32_t));
        if (!cursor) return -2;
        memcpy(cursor, binstart, nbins * sizeof(int32_t));
        for (int32_t i = 0; i < N; ++i) order[cursor[vid[i]]++] = i;
        free(cursor);
    }

    /* ---- Eq. 9-10: active voxels, centre, radius ---- */
    int32_t K = 0;
    for (size_t b = 0; b < nbins; ++b) K += binstart[b + 1] > binstart[b];
    int32_t *voff = (int32_t *)malloc(((size_t)K + 1) * sizeof(int32_t));
    float *vc = (float *)malloc((size_t)K * 3 * sizeof(float));
    float *vr = (float *)malloc((size_t)K * sizeof(float));
    float *Dv = (float *)malloc((size_t)K * sizeof(float));
    int32_t *Dv_idx = (int32_t *)malloc((size_t)K * sizeof(int32_t));
    if (!voff || !vc || !vr || !Dv || !Dv_idx) return -2;
    {
        int32_t k = 0;
        for (size_t b = 0; b < nbins; ++b) {
            const int32_t s = binstart[b], e = binstart[b + 1];
            if (e == s) continue;
            voff[k] = s;
            float mn[3], mx[3];
            for (int a = 0; a < 3; ++a) mn[a] = mx[a] = P[3 * (size_t)order[s] + a];
            for (int32_t q = s + 1; q < e; ++q)
                for (int a = 0; a < 3; ++a) {
                    const float v = P[3 * (size_t)order[q] + a];
                    if (v < mn[a]) mn[a] = v;
                    if (v > mx[a]) mx[a] = v;
                }
            for (int a = 0; a < 3; ++a) vc[3 * (size_t)k + a] = 0.5f * mn[a] + 0.5f * mx[a];   /* A10 */
            float r2 = 0.0f;
            for (int32_t q = s; q < e; ++q) {
                const float *p = P + 3 * (size_t)order[q];
                const float d = sq_dist(p[0], p[1], p[2], vc[3 * (size_t)k], vc[3 * (size_t)k + 1],
                                        vc[3 * (size_t)k + 2]);
                if (d > r2) r2 = d;
            }
            vr[k] = centroid_only ? 0.0f : sqrtf(r2) * UP;                                  /* A9 build */
            Dv[k] = INFINITY;                                                               /* A11 */
            Dv_idx[k] = order[s];                                                           /* lowest original index in voxel */
            ++k;
        }
        voff[K] = N;
    }
    for (int32_t i = 0; i < N; ++i) D[i] = INFINITY;

    pruned_stats st;
    memset(&st, 0, sizeof st);
    st.K = K;
    st.n_vox = n_vox;

    int32_t cur = start;
    out_idx[0] = start;
    out_mindist[0] = INFINITY;
    for (int32_t j = 1; j < M; ++j) {
        const float xs = P[3 * (size_t)cur], ys = P[3 * (size_t)cur + 1], zs = P[3 * (size_t)cur + 2];
        float gbest = -1.0f;
        int32_t gidx = 0;
        for (int32_t k = 0; k < K; ++k) {
            /* ---- Eq. 25 with the A9 margins ---- */
            int prune = 0;
            if (!no_prune) {
                st.voxel_tests++;
                const float d2c = sq_dist(vc[3 * (size_t)k], vc[3 * (size_t)k + 1], vc[3 * (size_t)k + 2], xs, ys, zs);
                if (centroid_only) {
                    prune = d2c >= Dv[k];
                } else {
                    const float dc = sqrtf(d2c) * DN;
                    const float t = (dc - vr[k]) * DN;
                    prune = (Dv[k] == 0.0f) ||
                            ((t > 0.0f) && ((t * t) * DN >= Dv[k]) && (Dv[k] >= 1e-30f));
                }
            }
            if (!prune) {
                st.voxels_visited++;
                float best = -1.0f;
                int32_t besti = 0;
                for (int32_t q = voff[k]; q < voff[k + 1]; ++q) {
                    const int32_t i = order[q];
                    st.points_visited++;
                    const float dx = P[3 * (size_t)i] - xs, dy = P[3 * (size_t)i + 1] - ys, dz = P[3 * (size_t)i + 2] - zs;
                    const float dx2 = dx * dx, dy2 = dy * dy, dz2 = dz * dz;
                    const float dold = D[i];
                    if (no_skip || !(dx2 >= dold || dy2 >= dold || dz2 >= dold)) {   /* Eq. 28, A8 */
                        st.points_computed++;
                        const float d = ((dx2 + dy2) + dz2);                          /* Eq. 29, A1 */
                        if (d < dold) { D[i] = d; st.effective++; }
                    }
                    /* Eq. 30; original indices ascend with q, so strict > keeps the lowest (A4) */
                    if (D[i] > best) { best = D[i]; besti = i; }
                }
                Dv[k] = best;
                Dv_idx[k] = besti;
            }
            /* Eq. 15-18 with the A4 pair compare */
            if (Dv[k] > gbest || (Dv[k] == gbest && Dv_idx[k] < gidx)) { gbest = Dv[k]; gidx = Dv_idx[k]; }
        }
        cur = gidx;
        out_idx[j] = gidx;
        out_mindist[j] = gbest;
    }
    if (stats) *stats = st;
    free(vid); free(binstart); free(order); free(D);
    free(voff); free(vc); free(vr); free(Dv); free(Dv_idx);
    return 0;
}

/* B equal-size clouds, one OpenMP thread per cloud (<= threads).  Returns threads used or <0.
 * stats (may be NULL): array of B. */
int pruned_fps_cpu_batch(const float *P, int32_t B, int32_t N, int32_t M, int32_t start, int32_t n_vox,
                         int32_t flags, int32_t *out_idx, float *out_mindist, pruned_stats *stats,
                         int32_t threads)
{
    if (B < 1) return -1;
    int used = 1, err = 0;
#ifdef _OPENMP
    int t = threads > 0 ? threads : omp_get_max_threads();
    if (t > B) t = B;
    used = t;
#pragma omp parallel for num_threads(t) schedule(dynamic, 1)
#endif
    for (int32_t b = 0; b < B; ++b) {
        int r = pruned_fps_cpu(P + (size_t)b * N * 3, N, M, start, n_vox, flags,
                               out_idx + (size_t)b * M, out_mindist + (size_t)b * M,
                               stats ? stats + b : NULL);
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
