// sample_whole.cu -- steps a7-a13 for SMALL clouds (every cloud of the index holds <= 8 192 points): the whole
// cloud lives in the registers of ONE CTA (k_fps_whole; one CTA per cloud, no cluster, no worker CTAs, no
// global rounds).  It is the first sampling layer of a point-cloud network (B x 1 024 .. 4 096 points) and
// BASELINE.json's config 1.
//
// The rules are the paper's: fp32 min-distance update with strict '<' (Eq. 29 / Eq. 2),
// argmax with lowest-index ties (Eq. 15-18), radius prune (Eq. 23-26) -- rescheduled as in sample_batched.cuh:
//   * the picks are resolved in parallel STEPS (local_fps_par of sample_batched.cuh: the top <= 64 points by
//     distance are the MEMBERS of a step; all pairs of members are compared with ballots and one warp derives
//     the exact pick sequence with bit operations).  DESIGN.md section 6 has the exactness argument;
//   * the radius prune works on BLOBS instead of the index's voxels: thread t holds the points 2t, 2t+1 (+1 024,
//     ...) of the voxel-sorted arrays (Hilbert order, Alg. 2 Phase 2), so the 64 points a warp
//     holds at one register position are one contiguous run of the space-filling curve -- a compact blob with its
//     own axis-aligned box and its own Dist_v = max Dist_p (Eq. 30).  A pick s is applied to a blob only if
//     LB(s, box) < Dist_v, where LB evaluates the library's d2 expression on the per-axis gaps
//     max(0, lo - s, s - hi).  That bound is exact in fp32 without any margin: for every point p of the blob
//     |fl(p.x - s.x)| >= fl(gap.x) because rounding is monotone, squares and sums of non-negative terms are
//     monotone as well, hence d2_rn(p, s) >= LB >= Dist_v >= Dist_p[p] and the strict-'<' update cannot fire
//     (Eq. 26 with equality included).  The same Dist_v lets a warp skip the selection histogram for blobs that
//     lie below the step's lower bin edge.
// Results are bit-identical to the oracle (tests/test_gpu_parity.py; the small clouds of every parity test run
// here by default).
#include <cfloat>
#include <cstring>

#include "sample_batched.cuh"

namespace rfps {

// picks taken one at a time (block-wide argmax: ~1 500 cycles each, a parallel step ~9 500) at the start of a cloud,
// after a parallel step that yielded fewer than STEP_MIN_YIELD picks, and when the first bin overflows (then in
// runs that double while the steps keep failing).  Measured on C1, 32 x {1 024, 2 048, 4 096} and the tie-heavy lattice:
// (24, 4, 5) is within 2 % of the best of six settings on every one of them
constexpr int SINGLES_FIRST = 24, SINGLES_AFTER = 4, STEP_MIN_YIELD = 5;
constexpr int SINGLES_UNTESTED = 16;   // the first picks of a cloud reach nearly every blob: no box tests for them

constexpr int WHOLE_HR16 = 2;       // 16 points per thread: coordinate pairs kept in registers (the other 6 live in shared memory)

struct __align__(16) WholeSmem {
    float4 sC[KS];                 // members {x, y, z, D}
    unsigned long long aff[KS];    // members ranked before i whose pick would lower D_i
    unsigned long long bef[KS];    // members ranked before i
    unsigned sO[KS];               // ~orig of the members
    int hist[2][16][32];           // per-warp histograms, double-buffered by step parity
    uint4 wb[16];
    unsigned wmax[16];
    unsigned stop[2];              // bit i: a member of aff_i may leave D_i >= the smallest member distance
    int npk;                       // picks accepted by the step
    unsigned hi;                   // upper bound of every distance after the step (bits)
    float4 pick[KS];               // the step's picks {x, y, z, -}
    float4 bmin[128], bmax[128];   // box of blob q = warp + 16 h
    float4 sp[2][16];              // single picks: every warp's best point {x, y, z, ~orig}, double-buffered by pick parity
    unsigned spd[2][16];           //               and its distance (bits)
};

__device__ __forceinline__ float warp_min_f(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(FULL, v, o));
    return v;
}
__device__ __forceinline__ float warp_max_f(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(FULL, v, o));
    return v;
}
// lower bound of d2_rn(p, s) over every p with lo <= p <= hi (component-wise): the d2 expression on the gaps
__device__ __forceinline__ float box_lb(const float4 lo, const float4 hi, const float4 s)
{
    const float gx = fmaxf(fmaxf(__fsub_rn(lo.x, s.x), __fsub_rn(s.x, hi.x)), 0.0f);
    const float gy = fmaxf(fmaxf(__fsub_rn(lo.y, s.y), __fsub_rn(s.y, hi.y)), 0.0f);
    const float gz = fmaxf(fmaxf(__fsub_rn(lo.z, s.z), __fsub_rn(s.z, hi.z)), 0.0f);
    return __fadd_rn(__fadd_rn(__fmul_rn(gx, gx), __fmul_rn(gy, gy)), __fmul_rn(gz, gz));
}

template <int CPT1, bool STATS, bool EUC>
__global__ void __launch_bounds__(BT, 1) k_fps_whole(const BatchParams P, const int flags)
{
    static_assert(CPT1 % 2 == 0 && CPT1 <= 16 && BT == 512 && KS == 64, "shape");
    // H1 pairs of points per thread: the coordinates of the first HR pairs live in registers, those of the other HS
    // (clouds of 4 097 .. 8 192 points) in shared memory; every distance lives in a register
    constexpr int H1 = CPT1 / 2, TC = CPT1 * BT, HR = H1 <= 4 ? H1 : WHOLE_HR16, HS = H1 - HR;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned *cO = reinterpret_cast<unsigned *>(smem_raw);                    // [TC] ~orig of sorted position i
    f32x2 *sXYZ = reinterpret_cast<f32x2 *>(smem_raw + sizeof(unsigned) * TC);   // [3][HS][BT] packed coordinate pairs
    WholeSmem *ws = reinterpret_cast<WholeSmem *>(smem_raw + sizeof(unsigned) * TC + sizeof(f32x2) * 3 * HS * BT);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const bool no_prune = flags & FPS_FLAG_NO_PRUNE;
    const int b = blockIdx.x;
    const size_t po = (size_t)P.poff[b];
    const int Nb = P.poff[b + 1] - P.poff[b];
    const int M = P.rag ? P.rag[b] : P.M;
    const int startb = P.rag ? P.rag[(P.B + 1) + b] : P.start_idx;
    const size_t obase = P.rag ? (size_t)P.rag[2 * (P.B + 1) + b] : (size_t)b * P.M;
    const float *__restrict__ px = P.px + po;
    const float *__restrict__ py = P.py + po;
    const float *__restrict__ pz = P.pz + po;
    const int *__restrict__ porig = P.porig + po;
    int *out_idx = P.out_idx + obase;
    float *out_mind = P.out_mind + obase;

    // ---- a7 + the initial update (Eq. 13-14): Dist_p = d(p, s_0), straight into registers ----
    const int p0 = P.pinv[po + startb];
    const float s0x = px[p0], s0y = py[p0], s0z = pz[p0];
    f32x2 X[HR] = {}, Y[HR] = {}, Z[HR] = {};
    float D[CPT1];
    // coordinate pair h of this thread (h is a compile-time constant wherever this is called)
    auto cx = [&](const int h) -> f32x2 { return h < HR ? X[h < HR ? h : 0] : sXYZ[(0 * HS + (h - HR)) * BT + tid]; };
    auto cy = [&](const int h) -> f32x2 { return h < HR ? Y[h < HR ? h : 0] : sXYZ[(1 * HS + (h - HR)) * BT + tid]; };
    auto cz = [&](const int h) -> f32x2 { return h < HR ? Z[h < HR ? h : 0] : sXYZ[(2 * HS + (h - HR)) * BT + tid]; };
    unsigned Dm[H1];                     // Dist_v of the warp's blobs (bits; warp-uniform)
    unsigned long long c_eff = 0;        // STATS: effective updates (Eq. 2), the initial one included
    const float inf = __uint_as_float(F32_INF_BITS);
#pragma unroll
    for (int h = 0; h < H1; ++h) {
        const int i0 = h * 2 * BT + 2 * tid, i1 = i0 + 1;
        const bool ok0 = i0 < Nb, ok1 = i1 < Nb;
        const float x0 = ok0 ? px[i0] : 0.0f, y0 = ok0 ? py[i0] : 0.0f, z0 = ok0 ? pz[i0] : 0.0f;
        const float x1 = ok1 ? px[i1] : 0.0f, y1 = ok1 ? py[i1] : 0.0f, z1 = ok1 ? pz[i1] : 0.0f;
        if (h < HR) {
            X[h < HR ? h : 0] = pack2(x0, x1);
            Y[h < HR ? h : 0] = pack2(y0, y1);
            Z[h < HR ? h : 0] = pack2(z0, z1);
        } else {
            sXYZ[(0 * HS + (h - HR)) * BT + tid] = pack2(x0, x1);
            sXYZ[(1 * HS + (h - HR)) * BT + tid] = pack2(y0, y1);
            sXYZ[(2 * HS + (h - HR)) * BT + tid] = pack2(z0, z1);
        }
        D[2 * h] = ok0 ? distf<EUC>(d2_rn(x0, y0, z0, s0x, s0y, s0z)) : 0.0f;      // padding: D = 0 is never picked
        D[2 * h + 1] = ok1 ? distf<EUC>(d2_rn(x1, y1, z1, s0x, s0y, s0z)) : 0.0f;
        if (STATS) c_eff += (ok0 ? 1 : 0) + (ok1 ? 1 : 0);
        cO[i0] = ok0 ? ~(unsigned)porig[i0] : 0u;
        cO[i1] = ok1 ? ~(unsigned)porig[i1] : 0u;
        // the blob's box over its real points (an empty blob gets lo = +inf, hi = -inf: every bound is +inf)
        const float lx = warp_min_f(fminf(ok0 ? x0 : inf, ok1 ? x1 : inf)), hx = warp_max_f(fmaxf(ok0 ? x0 : -inf, ok1 ? x1 : -inf));
        const float ly = warp_min_f(fminf(ok0 ? y0 : inf, ok1 ? y1 : inf)), hy = warp_max_f(fmaxf(ok0 ? y0 : -inf, ok1 ? y1 : -inf));
        const float lz = warp_min_f(fminf(ok0 ? z0 : inf, ok1 ? z1 : inf)), hz = warp_max_f(fmaxf(ok0 ? z0 : -inf, ok1 ? z1 : -inf));
        if (lane == 0) {
            ws->bmin[warp + 16 * h] = make_float4(lx, ly, lz, 0.0f);
            ws->bmax[warp + 16 * h] = make_float4(hx, hy, hz, 0.0f);
        }
        Dm[h] = __reduce_max_sync(FULL, __float_as_uint(fmaxf(D[2 * h], D[2 * h + 1])));
    }
    ws->hist[0][warp][lane] = 0;
    ws->hist[1][warp][lane] = 0;
    if (tid == 0) {
        ws->stop[0] = ws->stop[1] = 0u;
        out_idx[0] = startb;
        out_mind[0] = inf;
    }
    int jl = 1;
    unsigned long long c_steps = 0, c_fallback = 0, c_vtest = 0, c_vvisit = 0, c_pvisit = 0;
    long long t_sel = 0, t_pairs = 0, t_pick = 0, t_upd = 0, t_single = 0, tt0 = 0, tt1 = 0;

    auto block_max = [&]() -> unsigned {
        unsigned m = Dm[0];
#pragma unroll
        for (int h = 1; h < H1; ++h) m = max(m, Dm[h]);
        if (lane == 0) ws->wmax[warp] = m;
        __syncthreads();
        return __reduce_max_sync(FULL, lane < BT / 32 ? ws->wmax[lane] : 0u);
    };
    // ---- a9-a12: the picks ws->pick[0, npk) -> every blob they can reach ----
    auto apply_picks = [&](const int npk) {
        const float4 sa = lane < npk ? ws->pick[lane] : make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 sb = lane + 32 < npk ? ws->pick[lane + 32] : make_float4(0.f, 0.f, 0.f, 0.f);
        // the box tests of all blobs first, without a branch between them (their dependent chains overlap)
        unsigned M0[H1], M1[H1];
#pragma unroll
        for (int h = 0; h < H1; ++h) {
            const float dm = __uint_as_float(Dm[h]);
            if (no_prune) {
                M0[h] = Dm[h] == 0u ? 0u : (npk >= 32 ? FULL : ((1u << npk) - 1u));
                M1[h] = Dm[h] == 0u || npk <= 32 ? 0u : (npk >= 64 ? FULL : ((1u << (npk - 32)) - 1u));
            } else {
                const float4 lo = ws->bmin[warp + 16 * h], hi = ws->bmax[warp + 16 * h];
                // Eq. 25 on the blob: the pick is skipped iff its lower bound to the box is >= Dist_v (Dist_v = +0:
                // nothing left to lower, or an empty blob -- every bound is >= 0)
                M0[h] = __ballot_sync(FULL, lane < npk && !(distf<EUC>(box_lb(lo, hi, sa)) >= dm));
                M1[h] = __ballot_sync(FULL, lane + 32 < npk && !(distf<EUC>(box_lb(lo, hi, sb)) >= dm));
            }
        }
#pragma unroll
        for (int h = 0; h < H1; ++h) {
            unsigned m0 = M0[h], m1 = M1[h];
            if (STATS && Dm[h] != 0u) { c_vtest += (unsigned)npk; c_vvisit += __popc(m0) + __popc(m1); c_pvisit += 64ull * (__popc(m0) + __popc(m1)); }
            if (!(m0 | m1)) continue;
            // Euclidean mode: min and the monotone sqrt_rn commute, so the picks are applied in the squared domain
            // and folded into the distances once
            float a0 = EUC ? inf : D[2 * h], a1 = EUC ? inf : D[2 * h + 1];
            const f32x2 xh = cx(h), yh = cy(h), zh = cz(h);
            auto one = [&](const float4 s) {
                const f32x2 dx = sub2(xh, pack2(s.x, s.x)), dy = sub2(yh, pack2(s.y, s.y)), dz = sub2(zh, pack2(s.z, s.z));
                float x0, x1, y0, y1, z0, z1;
                unpack2(mul2(dx, dx), x0, x1);
                unpack2(mul2(dy, dy), y0, y1);
                unpack2(mul2(dz, dz), z0, z1);
                const float e0 = __fadd_rn(__fadd_rn(x0, y0), z0), e1 = __fadd_rn(__fadd_rn(x1, y1), z1);
                if (STATS && !EUC) c_eff += (e0 < a0 ? 1 : 0) + (e1 < a1 ? 1 : 0);
                a0 = fminf(a0, e0);
                a1 = fminf(a1, e1);
            };
            while (m0) {
                const int i = __ffs(m0) - 1;
                m0 &= m0 - 1u;
                one(ws->pick[i]);
            }
            while (m1) {
                const int i = __ffs(m1) - 1;
                m1 &= m1 - 1u;
                one(ws->pick[32 + i]);
            }
            if (EUC) {
                D[2 * h] = fminf(D[2 * h], __fsqrt_rn(a0));
                D[2 * h + 1] = fminf(D[2 * h + 1], __fsqrt_rn(a1));
            } else {
                D[2 * h] = a0;
                D[2 * h + 1] = a1;
            }
            Dm[h] = __reduce_max_sync(FULL, __float_as_uint(fmaxf(D[2 * h], D[2 * h + 1])));       // a12 (Eq. 30)
        }
    };

    // ---- one pick by the block-wide argmax of Eq. 15-18, literally: every warp offers its best point (largest
    // distance, ties to the lowest original index), one barrier, every warp reduces the 16 offers.  Cheaper than a
    // parallel step while a step yields few picks (the first picks of a cloud each reach most of it; many equal
    // distances).  Returns the maximum before the pick (bits; 0 = nothing left, no pick was made). ----
    int spar = 0;
    auto single_pick = [&](const bool test_boxes) -> unsigned {
        // the warp's maximum is the largest blob maximum (warp-uniform, kept current by every update); only the blobs
        // that attain it -- normally one -- are searched for the point, ties to the lowest original index
        unsigned wm = Dm[0];
#pragma unroll
        for (int h = 1; h < H1; ++h) wm = max(wm, Dm[h]);
        const float wmf = __uint_as_float(wm);
        unsigned o = 0u;
        bool have = false;
        float bx = 0.0f, by = 0.0f, bz = 0.0f;
#pragma unroll
        for (int h = 0; h < H1; ++h) {
            if (Dm[h] != wm) continue;                       // warp-uniform
            const bool e0 = D[2 * h] == wmf, e1 = D[2 * h + 1] == wmf;
            if (e0 || e1) {
                const unsigned o0 = e0 ? cO[h * 2 * BT + 2 * tid] : 0u, o1 = e1 ? cO[h * 2 * BT + 2 * tid + 1] : 0u;
                const bool second = e1 && (!e0 || o1 > o0);
                const unsigned oc = second ? o1 : o0;
                if (!have || oc > o) {
                    float x0, x1, y0, y1, z0, z1;
                    unpack2(cx(h), x0, x1);
                    unpack2(cy(h), y0, y1);
                    unpack2(cz(h), z0, z1);
                    o = oc; have = true;
                    bx = second ? x1 : x0; by = second ? y1 : y0; bz = second ? z1 : z0;
                }
            }
        }
        const unsigned wo = __reduce_max_sync(FULL, have ? o : 0u);
        const int wl = __ffs(__ballot_sync(FULL, have && o == wo)) - 1;
        if (lane == wl) {
            ws->sp[spar][warp] = make_float4(bx, by, bz, __uint_as_float(wo));
            ws->spd[spar][warp] = wm;
        }
        __syncthreads();
        // every warp reduces the 16 offers (loaded together; the winner's coordinates travel by shuffle)
        const unsigned d = lane < BT / 32 ? ws->spd[spar][lane] : 0u;
        const float4 off = lane < BT / 32 ? ws->sp[spar][lane] : make_float4(0.f, 0.f, 0.f, 0.f);
        const unsigned gm = __reduce_max_sync(FULL, d);
        if (gm == 0u) return 0u;
        const unsigned oo = (lane < BT / 32 && d == gm) ? __float_as_uint(off.w) : 0u;
        const unsigned go = __reduce_max_sync(FULL, oo);
        const int wl2 = __ffs(__ballot_sync(FULL, lane < BT / 32 && d == gm && oo == go)) - 1;
        const float4 s = make_float4(__shfl_sync(FULL, off.x, wl2), __shfl_sync(FULL, off.y, wl2), __shfl_sync(FULL, off.z, wl2), 0.0f);
        if (tid == 0) {
            out_idx[jl] = (int)(~go);
            out_mind[jl] = __uint_as_float(gm);
        }
        spar ^= 1;
        // a9-a12 without a branch between the blobs, so that their box tests, updates and reductions overlap
        bool reach[H1];
#pragma unroll
        for (int h = 0; h < H1; ++h) {
            reach[h] = Dm[h] != 0u;
            if (test_boxes) reach[h] = reach[h] && !(distf<EUC>(box_lb(ws->bmin[warp + 16 * h], ws->bmax[warp + 16 * h], s)) >= __uint_as_float(Dm[h]));
        }
        const f32x2 SX = pack2(s.x, s.x), SY = pack2(s.y, s.y), SZ = pack2(s.z, s.z);
#pragma unroll
        for (int h = 0; h < H1; ++h) {
            if (STATS) { if (Dm[h] != 0u) c_vtest++; if (reach[h]) { c_vvisit++; c_pvisit += 64ull; } }
            if (h >= HR && !reach[h]) continue;              // (coordinates in shared memory: not loaded for nothing)
            const f32x2 dx = sub2(cx(h), SX), dy = sub2(cy(h), SY), dz = sub2(cz(h), SZ);
            float x0, x1, y0, y1, z0, z1;
            unpack2(mul2(dx, dx), x0, x1);
            unpack2(mul2(dy, dy), y0, y1);
            unpack2(mul2(dz, dz), z0, z1);
            const float e0 = distf<EUC>(__fadd_rn(__fadd_rn(x0, y0), z0)), e1 = distf<EUC>(__fadd_rn(__fadd_rn(x1, y1), z1));
            if (STATS && reach[h]) c_eff += (e0 < D[2 * h] ? 1 : 0) + (e1 < D[2 * h + 1] ? 1 : 0);
            D[2 * h] = reach[h] ? fminf(D[2 * h], e0) : D[2 * h];
            D[2 * h + 1] = reach[h] ? fminf(D[2 * h + 1], e1) : D[2 * h + 1];
        }
#pragma unroll
        for (int h = 0; h < H1; ++h) Dm[h] = __reduce_max_sync(FULL, __float_as_uint(fmaxf(D[2 * h], D[2 * h + 1])));
        return gm;
    };

    unsigned hibits = block_max();       // (its barrier also publishes the initialisation above)
    bool hi_exact = true, keep_blo = false;
    float g = 0.125f;                    // the bins span (hi (1 - g), hi]; g follows the counts
    float blo = 0.0f;
    int refine = 0, hp = 0;
    int singles = SINGLES_FIRST;         // picks to take one at a time before the next parallel step
    int single_len = SINGLES_AFTER;
    while (jl < M && hibits != 0u) {     // hi == +0: every distance is +0 (reading A7, after the loop)
        if (STATS) tt0 = clock64();
        if (singles > 0) {
            // (the first picks of a cloud reach nearly every blob: the box tests are left out there)
            hibits = single_pick(!no_prune && jl > SINGLES_UNTESTED);      // the maximum before the pick bounds everything after it
            hi_exact = false;
            if (hibits == 0u) break;
            ++jl;
            --singles;
            c_fallback++;
            if (STATS) t_single += clock64() - tt0;
            continue;
        }
        const float hi = __uint_as_float(hibits);
        const bool finite = hibits < F32_INF_BITS;           // d2 overflowed to +inf somewhere: single picks until it is gone
        if (!keep_blo) {
            blo = g >= 1.0f ? 0.0f : __fmul_rn(hi, __fsub_rn(1.0f, g));
            if (!(blo < hi)) blo = 0.0f;
        }
        keep_blo = false;
        hp ^= 1;
        const float scale = fminf(__fdiv_rn(32.0f, __fsub_rn(hi, blo)), FLT_MAX);
        // bin(d): 0 for d = hi, growing as d falls; monotone because fp32 subtraction and multiplication by a
        // positive constant are monotone
#define RFPS_BIN(d) ((int)fminf(fmaxf(__fmul_rn(__fsub_rn(hi, (d)), scale), 0.0f), 31.0f))
        int bstar = 0, total = 0, nmem = 0, mbase = 0;
        const unsigned blobits = __float_as_uint(blo);
        if (finite) {
            // ---- (1) per-warp histogram of the points above blo; blobs whose Dist_v is not above it are skipped whole ----
#pragma unroll
            for (int h = 0; h < H1; ++h) {
                if (Dm[h] > blobits) {                       // warp-uniform
#pragma unroll
                    for (int c = 2 * h; c < 2 * h + 2; ++c)
                        if (D[c] > blo) atomicAdd(&ws->hist[hp][warp][RFPS_BIN(D[c])], 1);
                }
            }
            __syncthreads();
            ws->hist[hp ^ 1][warp][lane] = 0;                // the other buffer: every warp is done with it
            __syncwarp();
            int tot = 0, before = 0;                         // bin `lane`: all warps / the warps before this one
#pragma unroll
            for (int w = 0; w < BT / 32; ++w) {
                const int v = ws->hist[hp][w][lane];
                tot += v;
                before += w < warp ? v : 0;
            }
            int incl = tot;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += t;
            }
            total = __shfl_sync(FULL, incl, 31);
            bstar = __popc(__ballot_sync(FULL, incl <= KS));
            // members = the points of the bins < bstar: their number, and how many of them the warps before this one hold
            nmem = bstar > 0 ? __shfl_sync(FULL, incl, bstar - 1) : 0;
            mbase = __reduce_add_sync(FULL, lane < bstar ? before : 0);
            if (total == 0) {
                // nothing above blo: blo is a bound of everything (it replaces hi), or -- blo == 0 -- nothing is left
                if (blo == 0.0f) { hibits = 0u; break; }
                hibits = __float_as_uint(blo);
                hi_exact = false;
                refine = 0;
                g = fminf(1.0f, g * 2.0f);
                continue;
            }
            if (refine == 0) {           // aim the next step's bin range at ~3 x KS points
                if (total > 6 * KS) g = fmaxf(0x1p-16f, g * 0.5f);
                else if (total < 2 * KS) g = fminf(1.0f, g * 2.0f);
            }
        }
        if (bstar == 0) {
            // the first bin alone holds more than KS points (or a distance is +inf)
            if (!hi_exact) {                                 // the bins hang on a bound: redo them from the true maximum
                hibits = block_max();
                hi_exact = true;
                continue;
            }
            const float nlo = finite ? __fsub_rn(hi, __fmul_rn(__fsub_rn(hi, blo), 0x1p-5f)) : hi;
            if (finite && refine < 2 && nlo > blo && nlo < hi) {     // narrow the bin range to (about) the first bin
                blo = nlo;
                keep_blo = true;
                ++refine;
                continue;
            }
            // many (nearly) equal distances, or an infinite one: picks one at a time
            singles = single_len;
            single_len = min(256, 2 * single_len);           // ... and longer runs of them while the steps keep failing
            refine = 0;
            continue;
        }
        // ---- (2) members (bin < bstar) -> shared memory, in the order (warp, blob, point) the histogram rows give ----
        {
            int base = mbase;
#pragma unroll
            for (int h = 0; h < H1; ++h) {
                if (!(Dm[h] > blobits)) continue;                // warp-uniform: no point of this blob was counted
                const bool m0 = D[2 * h] > blo && RFPS_BIN(D[2 * h]) < bstar, m1 = D[2 * h + 1] > blo && RFPS_BIN(D[2 * h + 1]) < bstar;
                const unsigned b0 = __ballot_sync(FULL, m0), b1 = __ballot_sync(FULL, m1);
                if (b0 | b1) {
                    float x0, x1, y0, y1, z0, z1;
                    unpack2(cx(h), x0, x1);
                    unpack2(cy(h), y0, y1);
                    unpack2(cz(h), z0, z1);
                    if (m0) {
                        const int sl = base + __popc(b0 & lt);
                        ws->sC[sl] = make_float4(x0, y0, z0, D[2 * h]);
                        ws->sO[sl] = cO[h * 2 * BT + 2 * tid];
                    }
                    if (m1) {
                        const int sl = base + __popc(b0) + __popc(b1 & lt);
                        ws->sC[sl] = make_float4(x1, y1, z1, D[2 * h + 1]);
                        ws->sO[sl] = cO[h * 2 * BT + 2 * tid + 1];
                    }
                    base += __popc(b0) + __popc(b1);
                }
            }
        }
        __syncthreads();
        const int n = nmem;
        if (STATS) { tt1 = clock64(); t_sel += tt1 - tt0; tt0 = tt1; }
        // ---- (3) all pairs: warp w takes the members i = 4w .. 4w+3 in turn, its lanes the partners j = lane and
        // lane + 32 (loaded once, consecutive addresses); a mask word is then ONE ballot ----
        unsigned thmbits;
        {
            const int j0 = lane, j1 = lane + 32;
            const bool v0 = j0 < n, v1 = j1 < n;
            const float4 c0 = v0 ? ws->sC[j0] : make_float4(0.f, 0.f, 0.f, 0.f), c1 = v1 ? ws->sC[j1] : make_float4(0.f, 0.f, 0.f, 0.f);
            // rank key (distance bits, ~orig): unsigned order = "larger distance first, ties to the lowest index"; the keys
            // of two different points differ, and an absent partner (key 0) ranks before nobody
            const unsigned long long k0 = v0 ? ((unsigned long long)__float_as_uint(c0.w) << 32) | ws->sO[j0] : 0ull;
            const unsigned long long k1 = v1 ? ((unsigned long long)__float_as_uint(c1.w) << 32) | ws->sO[j1] : 0ull;
            // smallest member distance (members are > 0, so the bits order like the values)
            thmbits = __reduce_min_sync(FULL, min(v0 ? __float_as_uint(c0.w) : 0xffffffffu, v1 ? __float_as_uint(c1.w) : 0xffffffffu));
            const float thm = __uint_as_float(thmbits);
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                // (no early exit: without a branch between the four members their dependent chains overlap; a member
                // slot beyond n is computed on slot 0 and not stored)
                const bool live = 4 * warp + ii < n;
                const int i = live ? 4 * warp + ii : 0;
                const float4 ci = ws->sC[i];
                const unsigned long long ki = ((unsigned long long)__float_as_uint(ci.w) << 32) | ws->sO[i];
                const float d0 = distf<EUC>(d2_rn(ci.x, ci.y, ci.z, c0.x, c0.y, c0.z));
                const float d1 = distf<EUC>(d2_rn(ci.x, ci.y, ci.z, c1.x, c1.y, c1.z));
                const bool b0 = k0 > ki, b1 = k1 > ki;
                const bool l0 = b0 && d0 < ci.w, l1 = b1 && d1 < ci.w;
                const unsigned bw0 = __ballot_sync(FULL, b0), bw1 = __ballot_sync(FULL, b1);
                const unsigned aw0 = __ballot_sync(FULL, l0), aw1 = __ballot_sync(FULL, l1);
                const bool sany = __any_sync(FULL, (l0 && !(d0 < thm)) || (l1 && !(d1 < thm)));
                if (lane == 0 && live) {
                    ws->aff[i] = ((unsigned long long)aw1 << 32) | aw0;
                    ws->bef[i] = ((unsigned long long)bw1 << 32) | bw0;
                    if (sany) atomicOr(&ws->stop[i >> 5], 1u << (i & 31));
                }
            }
        }
        __syncthreads();
        if (STATS) { tt1 = clock64(); t_pairs += tt1 - tt0; tt0 = tt1; }
        // ---- (4) one warp resolves the pick sequence (sample_batched.cuh, local_fps_par step 4) ----
        if (warp == 0) {
            const int ia = lane, ib = lane + 32;
            const bool va = ia < n, vb = ib < n;
            const unsigned long long affa = va ? ws->aff[ia] : 0ull, affb = vb ? ws->aff[ib] : 0ull;
            const unsigned long long befa = va ? ws->bef[ia] : 0ull, befb = vb ? ws->bef[ib] : 0ull;
            const float4 ca = va ? ws->sC[ia] : make_float4(0.f, 0.f, 0.f, 0.f), cb = vb ? ws->sC[ib] : make_float4(0.f, 0.f, 0.f, 0.f);
            const bool sta = (ws->stop[0] >> lane) & 1u, stb = (ws->stop[1] >> lane) & 1u;
            __syncwarp();
            if (lane == 0) ws->stop[0] = ws->stop[1] = 0u;   // for the next step
            bool acca = false, accb = false, reja = !va, rejb = !vb;
            unsigned long long A = 0ull, R = ballot64(reja, rejb);
            for (;;) {
                const bool nra = !acca && !reja && (affa & A) != 0ull, nrb = !accb && !rejb && (affb & A) != 0ull;
                reja |= nra; rejb |= nrb;
                const unsigned long long dR = ballot64(nra, nrb);
                R |= dR;
                const bool naa = !acca && !reja && (affa & ~R) == 0ull, nab = !accb && !rejb && (affb & ~R) == 0ull;
                acca |= naa; accb |= nab;
                const unsigned long long dA = ballot64(naa, nab);
                A |= dA;
                if (!(dR | dA)) break;
            }
            // cut at the first (in rank order) rejected member that may stay in contention
            const int ranka = __popcll(befa), rankb = __popcll(befb);
            const unsigned rmin = __reduce_min_sync(FULL, min(reja && va && sta ? (unsigned)ranka : 255u, rejb && vb && stb ? (unsigned)rankb : 255u));
            acca &= (unsigned)ranka < rmin; accb &= (unsigned)rankb < rmin;
            A = ballot64(acca, accb);
            const int lim = M - jl;                          // >= 1 here
            const int posa = __popcll(A & befa), posb = __popcll(A & befb);
            acca &= posa < lim; accb &= posb < lim;
            A = ballot64(acca, accb);
            if (acca) {
                out_idx[jl + posa] = (int)(~ws->sO[ia]);
                out_mind[jl + posa] = ca.w;
                ws->pick[posa] = make_float4(ca.x, ca.y, ca.z, 0.0f);
            }
            if (accb) {
                out_idx[jl + posb] = (int)(~ws->sO[ib]);
                out_mind[jl + posb] = cb.w;
                ws->pick[posb] = make_float4(cb.x, cb.y, cb.z, 0.0f);
            }
            // bound of what is left: members neither picked nor surely below every member, else the smallest
            // member distance (everything outside the members is below it)
            const bool la = va && !acca && !(reja && !sta && (unsigned)ranka < rmin), lb = vb && !accb && !(rejb && !stb && (unsigned)rankb < rmin);
            const unsigned hin = __reduce_max_sync(FULL, max(la ? __float_as_uint(ca.w) : 0u, lb ? __float_as_uint(cb.w) : 0u));
            if (lane == 0) { ws->npk = __popcll(A); ws->hi = max(hin, thmbits); }
        }
        __syncthreads();
        const int npk = ws->npk;
        hibits = ws->hi;
        hi_exact = false;
        refine = 0;
        c_steps++;
        if (STATS) { tt1 = clock64(); t_pick += tt1 - tt0; tt0 = tt1; }
        // ---- (5) the step's picks -> the blobs they can reach ----
        apply_picks(npk);
        jl += npk;
        // a step costs about as much as STEP_MIN_YIELD single picks
        if (npk < STEP_MIN_YIELD) { singles = single_len; single_len = min(256, 2 * single_len); }
        else single_len = SINGLES_AFTER;
        if (STATS) t_upd += clock64() - tt0;
#undef RFPS_BIN
    }
    // ---- every distance is +0 (duplicates exhausted, reading A7): the argmax is the lowest index, again and again ----
    __syncthreads();
    if (jl < M) {
        unsigned o = 0u;
        for (int i = tid; i < Nb; i += BT) o = max(o, cO[i]);
        o = __reduce_max_sync(FULL, o);
        if (lane == 0) ws->wmax[warp] = o;
        __syncthreads();
        const unsigned go = __reduce_max_sync(FULL, lane < BT / 32 ? ws->wmax[lane] : 0u);
        for (int q = jl + tid; q < M; q += BT) {
            out_idx[q] = (int)(~go);
            out_mind[q] = 0.0f;
        }
    }
    if (STATS) {
        if (lane == 0) {             // (blob, pick) tests and visits are counted once per warp; a visit touches 64 points
            atomicAdd(P.counters + CNT_VTEST, c_vtest);
            atomicAdd(P.counters + CNT_VVISIT, c_vvisit);
            atomicAdd(P.counters + CNT_PVISIT, c_pvisit);
            atomicAdd(P.counters + CNT_PCOMP, c_pvisit);
        }
        atomicAdd(P.counters + CNT_EFF, c_eff);
        if (tid == 0) {
            atomicAdd(P.counters + CNT_ROUNDS, 1ull);
            atomicAdd(P.counters + CNT_CANDS, (unsigned long long)Nb);
            atomicAdd(P.counters + CNT_SUBROUNDS, c_steps);
            atomicAdd(P.counters + CNT_FALLBACK, c_fallback);
            atomicAdd(P.counters + CNT_LSEL, (unsigned long long)t_sel);
            atomicAdd(P.counters + CNT_LPAIRS, (unsigned long long)t_pairs);
            atomicAdd(P.counters + CNT_LPICK, (unsigned long long)(t_pairs + t_pick));
            atomicAdd(P.counters + CNT_LUPD, (unsigned long long)t_upd);
            atomicAdd(P.counters + CNT_CYC_MAX, (unsigned long long)t_single);
            atomicAdd(P.counters + CNT_SINGLES, c_fallback);
            atomicAdd(P.counters + CNT_CYC_LOCAL, (unsigned long long)(t_sel + t_pairs + t_pick + t_upd + t_single));
        }
    }
}

size_t whole_smem_bytes(int cpt)
{
    const int h1 = cpt / 2, hs = h1 > 4 ? h1 - WHOLE_HR16 : 0;
    return sizeof(unsigned) * (size_t)cpt * BT + sizeof(f32x2) * 3 * (size_t)hs * BT + sizeof(WholeSmem);
}

template <int CPT1, bool STATS, bool EUC>
static int launch_whole_one(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st)
{
    auto kern = k_fps_whole<CPT1, STATS, EUC>;
    const size_t smem = whole_smem_bytes(CPT1);
    RFPS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<dim3((unsigned)ix.B), dim3(BT), smem, st>>>(bp, ix.flags);
    RFPS_CUDA(cudaGetLastError());
    return FPS_OK;
}

template <int CPT1>
static int launch_whole_c(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st)
{
    const bool stats = ix.flags & FPS_FLAG_STATS;
    if (ix.flags & FPS_FLAG_EUCLIDEAN) return stats ? launch_whole_one<CPT1, true, true>(bp, ix, st) : launch_whole_one<CPT1, false, true>(bp, ix, st);
    return stats ? launch_whole_one<CPT1, true, false>(bp, ix, st) : launch_whole_one<CPT1, false, false>(bp, ix, st);
}

int launch_sample_whole(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st)
{
    switch (ix.cand_per_thread) {
        case 2: return launch_whole_c<2>(bp, ix, st);
        case 4: return launch_whole_c<4>(bp, ix, st);
        case 8: return launch_whole_c<8>(bp, ix, st);
        case 16: return launch_whole_c<16>(bp, ix, st);
    }
    set_error("whole-cloud kernel: cand_per_thread=%d must be 2, 4, 8 or 16", ix.cand_per_thread);
    return FPS_ERR_INVALID;
}

}  // namespace rfps
