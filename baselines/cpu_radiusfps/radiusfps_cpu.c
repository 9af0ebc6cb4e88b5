/*
 * radiusfps_cpu.c -- a TUNED, multi-threaded CPU RadiusFPS: the paper's section-3 program
 * (arxiv/paper_2606_06255) as a BASELINE PROGRAM for bench.py's cpu_baseline leg
 * (third part; the paper's CPU claims PAPER.md:697-705, Fig. 15b).
 *
 * It is NOT the oracle (oracle/ holds that: plain and slow on purpose) and NOT product code: nothing
 * under paper_2606_06255_b200/ links, imports or calls it, and it shares no code with either.  It must
 * return, bit for bit, what classical FPS returns (tests/test_cpu_radiusfps.py checks it
 * against oracle.fps):
 *
 *     s_0 = P[start];  s_j = argmax_i min_{j'<j} d2(P[i], s_j'),  ties -> lowest original index,
 *     d2(p,s) = ((dx*dx + dy*dy) + dz*dz) in fp32, round to nearest, no FMA (compiled -ffp-contract=off).
 *
 * What "tuned" means here, next to oracle/fps_pruned_cpu.c (the plain cross-check):
 *   - structure-of-arrays points sorted by voxel (Alg. 2 Phase 2), voxel ids on a
 *     Morton curve so that 16 consecutive active voxels form a spatially compact GROUP;
 *   - two-level radius prune (Eq. 25): group spheres first, then the voxels of surviving
 *     groups; both tests are sqrt-free (squared-domain thresholds cached per voxel / group and refreshed
 *     only when the voxel is visited) and run as vectorisable loops over contiguous float arrays;
 *   - tight per-voxel spheres (midpoint of the voxel's own bounding box, radius rounded up) instead of
 *     the cell centre and sqrt(3)/2 L (Eq. 10): any enclosing sphere is valid;
 *   - the visit of a voxel (Eq. 27-30) is a branch-free vector loop: Dist_p = min(Dist_p, d2), running max;
 *     the coordinate-wise point skip of Eq. 28 is available as an option (flag 1) -- with 8-wide SIMD
 *     the test costs more than the three operations it avoids, so it is off by default;
 *   - the argmax (Eq. 15-18) is a scan over the GROUP keys only (K/16 entries);
 *   - clouds of a batch run on OpenMP threads (one cloud per thread; the M picks of one cloud are
 *     sequentially dependent, and one pick is ~1 us of work, so a single cloud stays on
 *     one thread).
 *
 * fp32 safety of the prune (restated): u = 2^-24;  R_k = sqrtf(max_p d2(p,c_k)) (1+2^-20);
 * a voxel with Dist_v = Dv is skipped for pick s iff d2(s,c_k) >= thr_k,
 *     thr_k = ((sqrtf(Dv) (1+2^-20) + 2^-40) + R_k)^2 (1+2^-18)     (thr = 0 when Dv == 0, +inf when Dv == +inf);
 * then ||s-c|| >= sqrt(Dv)(1+3u) + R_k, so every point of the voxel has fl_d2(p,s) >= Dv >= Dist_p[p] and the
 * strict '<' update cannot fire.  The same with the group sphere and Dv := max over the group.
 */
#include <math.h>
#include <omp.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define GROUP 16

typedef struct {
    int64_t group_tests, voxel_tests, voxels_visited, points_visited;
    int32_t K, n_vox;
} rcpu_stats;

static inline float d2f(float x, float y, float z, float sx, float sy, float sz)
{
    const float dx = x - sx, dy = y - sy, dz = z - sz;
    return ((dx * dx + dy * dy) + dz * dz);
}

static inline float prune_thr(float Dv, float R)
{
    if (Dv == 0.0f) return 0.0f;
    if (!(Dv < INFINITY)) return INFINITY;
    const float q = sqrtf(Dv) * (1.0f + 0x1p-20f) + 0x1p-40f;
    const float a = q + R;
    return (a * a) * (1.0f + 0x1p-18f);
}

static inline uint32_t spread3(uint32_t v)
{
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

static int auto_n_vox(int N)
{   /* some tens of points per active voxel on surface-like clouds */
    double c = cbrt((double)N / 8.0);
    int n = (int)(c + 0.5);
    if (n < 2) n = 2;
    if (n > 512) n = 512;
    return n;
}

typedef struct {
    int N, K, G;
    float *x, *y, *z, *D;        /* [N] sorted by voxel                                   */
    int32_t *orig;               /* [N] sorted position -> original index                 */
    int32_t *off;                /* [K+1] segment starts                                  */
    float *vcx, *vcy, *vcz, *vR, *vthr, *vD;   /* [Kp] voxel sphere, threshold, Dist_v     */
    int32_t *vO;                 /* [Kp] lowest original index attaining Dist_v           */
    float *gcx, *gcy, *gcz, *gR, *gthr, *gD;   /* [Gp] group sphere, threshold, max Dist_v */
    int32_t *gO;                 /* [Gp] lowest original index attaining gD               */
    int32_t *surv;               /* scratch: surviving groups / voxels                    */
} cloud_t;

static void *xalloc(size_t n) { void *p = NULL; if (posix_memalign(&p, 64, n ? n : 64)) return NULL; return p; }

static void cloud_free(cloud_t *c)
{
    free(c->x); free(c->y); free(c->z); free(c->D); free(c->orig); free(c->off);
    free(c->vcx); free(c->vcy); free(c->vcz); free(c->vR); free(c->vthr); free(c->vD); free(c->vO);
    free(c->gcx); free(c->gcy); free(c->gcz); free(c->gR); free(c->gthr); free(c->gD); free(c->gO); free(c->surv);
}

/* Eq. 6-10 + Alg. 2: bbox, voxel ids, stable sort, SoA, segments, spheres */
static int cloud_build(cloud_t *c, const float *P, int N, int n_vox)
{
    memset(c, 0, sizeof *c);
    c->N = N;
    float mn[3] = {P[0], P[1], P[2]}, mx[3] = {P[0], P[1], P[2]};
    for (int i = 1; i < N; ++i)
        for (int a = 0; a < 3; ++a) {
            const float v = P[3 * (size_t)i + a];
            if (v < mn[a]) mn[a] = v;
            if (v > mx[a]) mx[a] = v;
        }
    float E = fmaxf(fmaxf(mx[0] - mn[0], mx[1] - mn[1]), mx[2] - mn[2]);
    float L = (1.0f + 1e-3f) * E / (float)n_vox;             /* Eq. 7, alpha = 1 + 1e-3 */
    if (!(L > 0.0f)) L = 1.0f;
    uint32_t *key = xalloc(sizeof(uint32_t) * (size_t)N), *key2 = xalloc(sizeof(uint32_t) * (size_t)N);
    int32_t *val = xalloc(sizeof(int32_t) * (size_t)N), *val2 = xalloc(sizeof(int32_t) * (size_t)N);
    if (!key || !key2 || !val || !val2) return -1;
    for (int i = 0; i < N; ++i) {
        uint32_t v[3];
        for (int a = 0; a < 3; ++a) {
            int q = (int)floorf((P[3 * (size_t)i + a] - mn[a]) / L);    /* Eq. 8: floor, then clamp */
            if (q < 0) q = 0;
            if (q > n_vox - 1) q = n_vox - 1;
            v[a] = (uint32_t)q;
        }
        key[i] = spread3(v[0]) | (spread3(v[1]) << 1) | (spread3(v[2]) << 2);
        val[i] = i;
    }
    /* stable LSD radix sort, 3 passes of 10 bits: original indices stay ascending inside a voxel */
    for (int pass = 0; pass < 3; ++pass) {
        int cnt[1025];
        memset(cnt, 0, sizeof cnt);
        const int sh = 10 * pass;
        for (int i = 0; i < N; ++i) cnt[((key[i] >> sh) & 1023u) + 1]++;
        for (int d = 0; d < 1024; ++d) cnt[d + 1] += cnt[d];
        for (int i = 0; i < N; ++i) {
            const int dst = cnt[(key[i] >> sh) & 1023u]++;
            key2[dst] = key[i];
            val2[dst] = val[i];
        }
        uint32_t *tk = key; key = key2; key2 = tk;
        int32_t *tv = val; val = val2; val2 = tv;
    }
    int K = 0;
    for (int p = 0; p < N; ++p) K += (p == 0 || key[p] != key[p - 1]);
    const int G = (K + GROUP - 1) / GROUP, Kp = G * GROUP + 16, Gp = G + 16;
    c->K = K; c->G = G;
    c->x = xalloc(4 * (size_t)N + 64); c->y = xalloc(4 * (size_t)N + 64); c->z = xalloc(4 * (size_t)N + 64);
    c->D = xalloc(4 * (size_t)N + 64); c->orig = xalloc(4 * (size_t)N + 64); c->off = xalloc(4 * ((size_t)Kp + 1));
    c->vcx = xalloc(4 * (size_t)Kp); c->vcy = xalloc(4 * (size_t)Kp); c->vcz = xalloc(4 * (size_t)Kp); c->vR = xalloc(4 * (size_t)Kp);
    c->vthr = xalloc(4 * (size_t)Kp); c->vD = xalloc(4 * (size_t)Kp); c->vO = xalloc(4 * (size_t)Kp);
    c->gcx = xalloc(4 * (size_t)Gp); c->gcy = xalloc(4 * (size_t)Gp); c->gcz = xalloc(4 * (size_t)Gp); c->gR = xalloc(4 * (size_t)Gp);
    c->gthr = xalloc(4 * (size_t)Gp); c->gD = xalloc(4 * (size_t)Gp); c->gO = xalloc(4 * (size_t)Gp);
    c->surv = xalloc(4 * ((size_t)Kp + Gp));
    if (!c->x || !c->y || !c->z || !c->D || !c->orig || !c->off || !c->vcx || !c->vcy || !c->vcz || !c->vR || !c->vthr || !c->vD ||
        !c->vO || !c->gcx || !c->gcy || !c->gcz || !c->gR || !c->gthr || !c->gD || !c->gO || !c->surv) return -1;
    int k = -1;
    for (int p = 0; p < N; ++p) {
        const int i = val[p];
        c->x[p] = P[3 * (size_t)i]; c->y[p] = P[3 * (size_t)i + 1]; c->z[p] = P[3 * (size_t)i + 2];
        c->orig[p] = i;
        c->D[p] = INFINITY;
        if (p == 0 || key[p] != key[p - 1]) c->off[++k] = p;
    }
    for (int q = K; q <= Kp; ++q) c->off[q] = N;
    free(key); free(key2); free(val); free(val2);
    /* tight spheres (readings A9 / A10): centre = midpoint of the voxel's own bounding box */
    for (k = 0; k < Kp; ++k) {
        if (k >= K) {       /* padding voxel: threshold 0 prunes it for ever, key below every real key */
            c->vcx[k] = c->vcy[k] = c->vcz[k] = c->vR[k] = 0.0f; c->vthr[k] = 0.0f; c->vD[k] = -1.0f; c->vO[k] = 0x7fffffff;
            continue;
        }
        float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
        for (int p = c->off[k]; p < c->off[k + 1]; ++p) {
            lo[0] = fminf(lo[0], c->x[p]); hi[0] = fmaxf(hi[0], c->x[p]);
            lo[1] = fminf(lo[1], c->y[p]); hi[1] = fmaxf(hi[1], c->y[p]);
            lo[2] = fminf(lo[2], c->z[p]); hi[2] = fmaxf(hi[2], c->z[p]);
        }
        const float cx = 0.5f * lo[0] + 0.5f * hi[0], cy = 0.5f * lo[1] + 0.5f * hi[1], cz = 0.5f * lo[2] + 0.5f * hi[2];
        float r2 = 0.0f;
        for (int p = c->off[k]; p < c->off[k + 1]; ++p) r2 = fmaxf(r2, d2f(c->x[p], c->y[p], c->z[p], cx, cy, cz));
        c->vcx[k] = cx; c->vcy[k] = cy; c->vcz[k] = cz;
        c->vR[k] = sqrtf(r2) * (1.0f + 0x1p-20f);
        c->vthr[k] = INFINITY;                 /* Dist_v = +inf: the first pick visits every voxel (Eq. 13-14) */
        c->vD[k] = INFINITY;
        c->vO[k] = c->orig[c->off[k]];         /* lowest original index of the voxel (stable sort) */
    }
    for (int g = 0; g < Gp; ++g) {
        if (g >= G) { c->gcx[g] = c->gcy[g] = c->gcz[g] = c->gR[g] = 0.0f; c->gthr[g] = 0.0f; c->gD[g] = -1.0f; c->gO[g] = 0x7fffffff; continue; }
        float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
        int o = 0x7fffffff;
        for (k = g * GROUP; k < (g + 1) * GROUP && k < K; ++k) {
            lo[0] = fminf(lo[0], c->vcx[k] - c->vR[k]); hi[0] = fmaxf(hi[0], c->vcx[k] + c->vR[k]);
            lo[1] = fminf(lo[1], c->vcy[k] - c->vR[k]); hi[1] = fmaxf(hi[1], c->vcy[k] + c->vR[k]);
            lo[2] = fminf(lo[2], c->vcz[k] - c->vR[k]); hi[2] = fmaxf(hi[2], c->vcz[k] + c->vR[k]);
            if (c->vO[k] < o) o = c->vO[k];
        }
        const float cx = 0.5f * lo[0] + 0.5f * hi[0], cy = 0.5f * lo[1] + 0.5f * hi[1], cz = 0.5f * lo[2] + 0.5f * hi[2];
        float r = 0.0f;
        for (k = g * GROUP; k < (g + 1) * GROUP && k < K; ++k)
            r = fmaxf(r, (sqrtf(d2f(c->vcx[k], c->vcy[k], c->vcz[k], cx, cy, cz)) * (1.0f + 0x1p-20f) + c->vR[k]) * (1.0f + 0x1p-20f));
        c->gcx[g] = cx; c->gcy[g] = cy; c->gcz[g] = cz; c->gR[g] = r;
        c->gthr[g] = INFINITY; c->gD[g] = INFINITY; c->gO[g] = o;
    }
    return 0;
}

/* Eq. 27-30 on one voxel: update, per-voxel max with the lowest original index (first position attaining it) */
static inline void visit_voxel(cloud_t *c, int k, float sx, float sy, float sz, int point_skip)
{
    const int p0 = c->off[k], p1 = c->off[k + 1];
    float *restrict x = c->x, *restrict y = c->y, *restrict z = c->z, *restrict D = c->D;
    float best = -1.0f;
    if (point_skip) {
        for (int p = p0; p < p1; ++p) {
            const float dx = x[p] - sx, dy = y[p] - sy, dz = z[p] - sz;
            const float dx2 = dx * dx, dy2 = dy * dy, dz2 = dz * dz, Dp = D[p];
            if (!(dx2 >= Dp || dy2 >= Dp || dz2 >= Dp)) {         /* Eq. 28 in the squared domain (A8) */
                const float d = (dx2 + dy2) + dz2;
                if (d < Dp) D[p] = d;                               /* Eq. 29, strict '<' */
            }
            best = fmaxf(best, D[p]);
        }
    } else {
#pragma omp simd reduction(max : best)
        for (int p = p0; p < p1; ++p) {
            const float dx = x[p] - sx, dy = y[p] - sy, dz = z[p] - sz;
            const float d = (dx * dx + dy * dy) + dz * dz;
            const float nd = d < D[p] ? d : D[p];
            D[p] = nd;
            best = nd > best ? nd : best;
        }
    }
    int pb = p0;
    while (D[pb] != best) ++pb;                    /* first = lowest original index inside the voxel */
    c->vD[k] = best;
    c->vO[k] = c->orig[pb];
    c->vthr[k] = prune_thr(best, c->vR[k]);
}

static void refresh_group(cloud_t *c, int g)
{
    float bd = -1.0f;
    int bo = 0x7fffffff;
    for (int k = g * GROUP; k < (g + 1) * GROUP; ++k) {
        const float d = c->vD[k];
        if (d > bd || (d == bd && c->vO[k] < bo)) { bd = d; bo = c->vO[k]; }
    }
    c->gD[g] = bd;
    c->gO[g] = bo;
    c->gthr[g] = prune_thr(bd, c->gR[g]);
}

static int fps_one(const float *P, int N, int M, int start, int n_vox, int flags, int32_t *idx, float *mind, rcpu_stats *st)
{
    cloud_t c;
    if (cloud_build(&c, P, N, n_vox > 0 ? n_vox : auto_n_vox(N)) != 0) { cloud_free(&c); return -1; }
    const int point_skip = flags & 1;
    const int G = c.G;
    int32_t *sg = c.surv, *sv = c.surv + G + 16;
    float sx = P[3 * (size_t)start], sy = P[3 * (size_t)start + 1], sz = P[3 * (size_t)start + 2];
    int64_t gt = 0, vt = 0, vv = 0, pv = 0;
    idx[0] = start;
    mind[0] = INFINITY;
    for (int j = 1; j < M; ++j) {
        /* Eq. 25 on the groups: flags first (vectorisable), then compaction */
        int ns = 0;
        {
            const float *restrict gx = c.gcx, *restrict gy = c.gcy, *restrict gz = c.gcz, *restrict gth = c.gthr;
            for (int g = 0; g < G; ++g) {
                const float dx = gx[g] - sx, dy = gy[g] - sy, dz = gz[g] - sz;
                const float t = (dx * dx + dy * dy) + dz * dz;
                sg[ns] = g;
                ns += !(t >= gth[g]);
            }
        }
        gt += G;
        for (int a = 0; a < ns; ++a) {
            const int g = sg[a];
            int nv = 0;
            for (int k = g * GROUP; k < (g + 1) * GROUP; ++k) {
                const float dx = c.vcx[k] - sx, dy = c.vcy[k] - sy, dz = c.vcz[k] - sz;
                const float t = (dx * dx + dy * dy) + dz * dz;
                sv[nv] = k;
                nv += !(t >= c.vthr[k]);
            }
            vt += GROUP;
            if (!nv) continue;
            for (int b = 0; b < nv; ++b) {
                visit_voxel(&c, sv[b], sx, sy, sz, point_skip);
                pv += c.off[sv[b] + 1] - c.off[sv[b]];
            }
            vv += nv;
            refresh_group(&c, g);
        }
        /* Eq. 15-18: argmax over the group keys, ties to the lowest original index */
        float bd = -1.0f;
        int bo = 0x7fffffff;
        for (int g = 0; g < G; ++g) {
            const float d = c.gD[g];
            if (d > bd || (d == bd && c.gO[g] < bo)) { bd = d; bo = c.gO[g]; }
        }
        idx[j] = bo;
        mind[j] = bd;
        sx = P[3 * (size_t)bo]; sy = P[3 * (size_t)bo + 1]; sz = P[3 * (size_t)bo + 2];
    }
    if (st) { st->group_tests = gt; st->voxel_tests = vt; st->voxels_visited = vv; st->points_visited = pv; st->K = c.K; st->n_vox = n_vox > 0 ? n_vox : auto_n_vox(N); }
    cloud_free(&c);
    return 0;
}

/* points [B][N][3] fp32; idx / mind [B][M]; n_vox 0 = choose; flags: 1 = coordinate-wise point skip (Eq. 28);
 * threads 0 = all.  Returns the number of threads used, or a negative value on bad arguments / allocation failure. */
int radiusfps_cpu_batch(const float *points, int32_t B, int32_t N, int32_t M, int32_t start, int32_t n_vox, int32_t flags,
                        int32_t *idx, float *mind, rcpu_stats *stats, int32_t threads)
{
    if (!points || !idx || !mind || B < 1 || N < 1 || M < 1 || M > N || start < 0 || start >= N || n_vox < 0 || n_vox > 1024) return -1;
    int nt = threads > 0 ? threads : omp_get_max_threads();
    if (nt > B) nt = B;
    int bad = 0;
#pragma omp parallel for num_threads(nt) schedule(dynamic, 1)
    for (int b = 0; b < B; ++b) {
        if (fps_one(points + 3 * (size_t)N * b, N, M, start, n_vox, flags, idx + (size_t)M * b, mind + (size_t)M * b,
                    stats ? stats + b : NULL) != 0) {
#pragma omp atomic write
            bad = 1;
        }
    }
    return bad ? -2 : nt;
}
