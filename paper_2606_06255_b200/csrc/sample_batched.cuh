// sample_batched.cuh -- steps a7-a13 with EXACT BATCHED PICKING: the same rules as the paper's
// iteration (radius prune Eq. 25, point skip Eq. 28, fp32 min-distance update Eq. 29, per-voxel max
// Eq. 30, lowest-index argmax Eq. 15-18), rescheduled so that the M-1
// sequentially dependent picks no longer pay one cluster-wide exchange each.
//
// Why it is exact.  Let Dist_p be exact with respect to all picks so far and
// tau < max Dist_p.  Put C = {p : Dist_p[p] > tau}.  Dist_p never increases, so every point outside
// C stays <= tau for ever; hence, while the maximum over C is > tau, the argmax over C (same key:
// distance, then lowest original index) IS the global argmax of Eq. 3 -- ties included, because all
// points tied at the maximum are in C.  Plain FPS restricted to C therefore emits exactly the
// oracle's picks until its maximum drops to <= tau.  The picks of such a batch are then applied to
// the whole cloud at once: min is order-independent, so Dist_p ends bit-identical to applying them
// one by one, and a voxel may be tested against a pick with a stale (larger) Dist_v because that
// only makes the prune test of Eq. 25 more conservative.
//
// One thread-block cluster per cloud.  With more than one CTA, CTA 0 is the PICKER (LOCAL) and CTAs
// 1..C-1 are the WORKERS (own the voxels: APPLY, MAX, EXTRACT); the workers apply a batch while the
// picker is still producing it (release/acquire flag + DSMEM copies).  One round:
//   APPLY    the nb picks of the previous batch, 128 at a time.  Prune (a9, squared-domain Eq. 25 with
//            fp32 margins) on two levels: a work unit = (group of 32 voxels, 32 picks) tests the picks
//            against the group sphere, then the group's voxels against the survivors; voxels with
//            survivors are queued with their pick mask.  Warps pop queued voxels and walk their points
//            once for all surviving picks (a10 skip, a11 update) and refresh the voxel key (a12).
//   MAX      CTA argmax of the voxel keys, then cluster argmax over DSMEM (a8).
//   EXTRACT  tau = Dmax * (1 - g): points with Dist_p > tau are appended to the candidate buffer in
//            CTA 0's shared memory over DSMEM (atom.shared::cluster + st.shared::cluster).  If more
//            than TC candidates turn up, tau is raised and the step repeated; if that fails the
//            batch is the single global argmax (the paper's own per-pick iteration).
//   LOCAL    (CTA 0) FPS restricted to the <= TC candidates, hierarchical by default: all warps hold
//            the candidates in registers, one warp picks from the top <= 128 of them with no barrier
//            per pick (local_fps_hier); stops when the maximum is <= tau, after PB picks, or at M.
//            Picks go to out_idx / out_mindist and to the next round's batch.
//
// Arithmetic: d2 only via __fsub_rn/__fmul_rn/__fadd_rn (never FMA); the local phase uses
// fminf(D, d2), which is value-identical to the strict '<' update for non-NaN operands.
#include <cfloat>
#include <algorithm>
#include <cstring>

#pragma once
#include "device_utils.cuh"
#include "internal.h"
#include "sample_batched_shapes.h"

namespace rfps {

enum { CNT_VTEST = 0, CNT_VVISIT, CNT_PVISIT, CNT_PCOMP, CNT_EFF, CNT_ROUNDS, CNT_RETRIES, CNT_SINGLES, CNT_CANDS,
       CNT_XVOX, CNT_XPTS, CNT_CYC_APPLY, CNT_CYC_MAX, CNT_CYC_EXTRACT, CNT_CYC_LOCAL, CNT_GTEST, CNT_CYC_A_SUM, CNT_CYC_B_SUM, CNT_CYC_A_MAX, CNT_CYC_B_MAX, CNT_SUBS, CNT_LSEL, CNT_LPICK, CNT_LUPD, CNT_SUBROUNDS, CNT_FALLBACK, CNT_LPAIRS, CNT_LPUB, CNT_W_TAIL, CNT_W_XSCAN, CNT_W_IDLE, CNT_W_PIECES, CNT_N };

// ---------------------------------------------------------------------------------------------
// packed fp32x2 arithmetic (sm_100: FADD2 / FMUL2).  Each half is an ordinary IEEE round-to-nearest
// fp32 operation, so the results are bit-identical to the scalar __f*_rn intrinsics.
// ---------------------------------------------------------------------------------------------
// The distance the algorithm works with: the squared fp32 expression d2 (the main path, BASELINE.json), or
// EUC: its correctly rounded square root, the paper's literal ||p - s|| (Eq. 1 / Eq. 29).
// Everything else -- min, strict '<', argmax with lowest-index ties, the exact-batching argument -- only
// needs a distance that is a fixed monotone function of d2, so both modes share all of the code below.
template <bool EUC>
__device__ __forceinline__ float distf(const float d2) { return EUC ? __fsqrt_rn(d2) : d2; }
// prune threshold for the Euclidean mode: Dist_v already is a (rounded) distance, so no square root; the
// voxel is pruned iff d2(s, c) >= thr.  Then ||p - s|| >= Dv (1 + 3u) for every point p of the voxel, hence
// fl_d2(p, s) >= Dv^2 and sqrt_rn(fl_d2) >= Dv >= Dist_p[p] (sqrt_rn is monotone, Dv representable).
__device__ __forceinline__ float prune_threshold_euc(unsigned dv_bits, float R)
{
    if (dv_bits == 0u) return 0.0f;
    const float q = __fadd_rn(__fmul_rn(__uint_as_float(dv_bits), 1.0f + 0x1p-20f), 0x1p-40f);
    const float a = __fadd_rn(q, R);
    const float t = __fmul_rn(__fmul_rn(a, a), 1.0f + 0x1p-18f);
    return (t < __uint_as_float(F32_INF_BITS)) ? t : __uint_as_float(F32_NAN_BITS);
}

typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float a, float b)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
// NOTE: there is deliberately no add2(): ptxas (12.9) contracts mul.rn.f32x2 + add.rn.f32x2 into FFMA2
// even under --fmad=false, which changes the rounding.  The two additions of d2 are therefore done
// with scalar __fadd_rn on the unpacked halves (scalar .rn adds are never contracted), and
// tests/test_abi_cpu.py checks that the built library holds no FFMA2 at all.

// How the picker tells its workers how far the running batch has got: a release store of
// (batch id << PUB_SHIFT | count) to the exchange block's `pub` word -- in its own shared memory (cluster) or in
// global memory (grid; the picks themselves are then mirrored to `gpick`).  Inactive for a single-CTA cloud.
struct Publisher {
    unsigned local_addr = 0u;              // cluster: shared::cta address of ctl->pub
    unsigned long long *gptr = nullptr;    // grid: the packed word cmd << 32 | pub (GX_PC)
    unsigned cmd_hi = 0u;                  // grid: the command word that stays in its upper half while the batch runs
    float4 *gpick = nullptr;               // grid: global mirror of the batch buffer
    unsigned base = 0u;                    // batch id << PUB_SHIFT
    __device__ __forceinline__ bool on() const { return local_addr != 0u || gptr != nullptr; }
    __device__ __forceinline__ void operator()(const unsigned count_and_flags) const
    {
        if (gptr) st_release_gpu_u64(gptr, ((unsigned long long)cmd_hi << 32) | (base | count_and_flags));
        else if (local_addr) st_release_cluster_u32(local_addr, base | count_and_flags);
    }
};

// ---------------------------------------------------------------------------------------------
// LOCAL: register-resident FPS over the candidate set (CTA 0, warps 0..LW-1).  Thread t keeps the
// candidates i = c*(LW*32) + t, c < CPT: coordinates (packed in pairs) and D in registers; the
// original indices stay in shared memory and are only read to break exact ties and to emit.
// One pick = CPT d2 evaluations per thread (FADD2/FMUL2 for the differences and squares), one redux + one vote per warp, one
// 8-byte slot {D bits, candidate index} per warp, one named barrier.  Slots are double-buffered by
// pick parity, so a single barrier per pick is enough.  Exact ties of the maximum (inside a lane,
// between lanes, between warps) take a slow path that compares ~orig, i.e. lowest index wins.
// ---------------------------------------------------------------------------------------------
template <int CPT, int LW>
__device__ __forceinline__ void local_fps(const float *cX, const float *cY, const float *cZ, const float *cD,
                                          const unsigned *cO, const int cnt, const unsigned taubits, int &j, int &nb,
                                          const int M, uint2 *lslot, float4 *bpick, int *out_idx, float *out_mind,
                                          const int ltid)
{
    static_assert(CPT % 2 == 0, "candidates are processed in pairs");
    constexpr int H = CPT / 2, LT = LW * 32;
    const int lane = ltid & 31, w = ltid >> 5;
    f32x2 X[H], Y[H], Z[H];
    float D[CPT];
#pragma unroll
    for (int h = 0; h < H; ++h) {
        const int i0 = (2 * h) * LT + ltid, i1 = (2 * h + 1) * LT + ltid;
        const bool ok0 = i0 < cnt, ok1 = i1 < cnt;
        X[h] = pack2(ok0 ? cX[i0] : 0.0f, ok1 ? cX[i1] : 0.0f);
        Y[h] = pack2(ok0 ? cY[i0] : 0.0f, ok1 ? cY[i1] : 0.0f);
        Z[h] = pack2(ok0 ? cZ[i0] : 0.0f, ok1 ? cZ[i1] : 0.0f);
        D[2 * h] = ok0 ? cD[i0] : 0.0f;          // padding: D = 0 never exceeds tau
        D[2 * h + 1] = ok1 ? cD[i1] : 0.0f;
    }
    int par = 0;
    nb = 0;
    for (;;) {
        // ---- warp level: max D, its owner lane and candidate slot ----
        float m = D[0];
#pragma unroll
        for (int c = 1; c < CPT; ++c) m = fmaxf(m, D[c]);
        const unsigned hi = __float_as_uint(m);
        const unsigned mhi = __reduce_max_sync(FULL, hi);
        const bool top = hi == mhi;
        unsigned eq = 0u;                        // bit c set iff D[c] == m (only meaningful on top lanes)
#pragma unroll
        for (int c = 0; c < CPT; ++c) eq |= (D[c] == m ? 1u : 0u) << c;
        const unsigned tops = __ballot_sync(FULL, top);
        const bool multi = __any_sync(FULL, top && (eq & (eq - 1u)));
        int cstar = __ffs(eq) - 1;
        int wlane = __ffs(tops) - 1;
        if (multi || (tops & (tops - 1u))) {     // exact tie inside the warp: lowest original index wins
            unsigned lo = 0u;
            if (top) {
#pragma unroll
                for (int c = 0; c < CPT; ++c)
                    if (eq & (1u << c)) {
                        const unsigned o = cO[c * LT + ltid];
                        if (o >= lo) { lo = o; cstar = c; }
                    }
            }
            const unsigned mlo = __reduce_max_sync(FULL, lo);
            wlane = __ffs(__ballot_sync(FULL, top && lo == mlo)) - 1;
        }
        if (lane == wlane) lslot[par * LW + w] = make_uint2(mhi, (unsigned)(cstar * LT + ltid));
        if (LW > 1) named_bar_sync(1, LT);
        else __syncwarp();
        // ---- CTA level: every thread reads the LW slots ----
        unsigned ghi = 0u, gidx = 0u;
        int nties = 0;
#pragma unroll
        for (int s = 0; s < LW; ++s) {
            const uint2 v = lslot[par * LW + s];
            if (v.x > ghi) { ghi = v.x; gidx = v.y; nties = 1; }
            else if (v.x == ghi) ++nties;
        }
        if (!(ghi > taubits)) break;            // restricted max <= tau: the candidate set no longer decides
        if (nties > 1) {                         // exact tie between warps: lowest original index wins
            unsigned bo = 0u;
#pragma unroll
            for (int s = 0; s < LW; ++s) {
                const uint2 v = lslot[par * LW + s];
                if (v.x == ghi) {
                    const unsigned o = cO[v.y];
                    if (o >= bo) { bo = o; gidx = v.y; }
                }
            }
        }
        const float sx = cX[gidx], sy = cY[gidx], sz = cZ[gidx];
        if (ltid == 0) {
            out_idx[j] = (int)(~cO[gidx]);
            out_mind[j] = __uint_as_float(ghi);
            bpick[nb] = make_float4(sx, sy, sz, 0.0f);
        }
        ++j;
        ++nb;
        if (j >= M || nb >= PB) break;
        // ---- update: D = min(D, d2(candidate, pick)), two candidates per instruction ----
        const f32x2 SX = pack2(sx, sx), SY = pack2(sy, sy), SZ = pack2(sz, sz);
#pragma unroll
        for (int h = 0; h < H; ++h) {
            const f32x2 dx = sub2(X[h], SX), dy = sub2(Y[h], SY), dz = sub2(Z[h], SZ);
            float x0, x1, y0, y1, z0, z1;
            unpack2(mul2(dx, dx), x0, x1);
            unpack2(mul2(dy, dy), y0, y1);
            unpack2(mul2(dz, dz), z0, z1);
            D[2 * h] = fminf(D[2 * h], __fadd_rn(__fadd_rn(x0, y0), z0));
            D[2 * h + 1] = fminf(D[2 * h + 1], __fadd_rn(__fadd_rn(x1, y1), z1));
        }
        par ^= 1;
    }
}

// ---------------------------------------------------------------------------------------------
// LOCAL, hierarchical form (the default): the same exact-batching argument applied once more inside
// the CTA.  All 16 warps keep the candidate set C1 in registers (CPT1 per thread).  A sub-round
//   (a) finds the block maximum m1,
//   (b) histograms the live candidates (D > tau) over 64 bins of [tau, m1] with a bin function that
//       is monotone in D,
//   (c) takes the longest prefix of bins holding <= T2 = 32*CPT2 candidates (B* bins),
//   (d) moves those candidates (C2) to shared memory,
//   (e) lets ONE warp run FPS on C2 in registers -- no barrier, vote or shuffle per pick: two redux
//       levels and three broadcast loads -- while the maximum stays in the first B* bins, i.e. above
//       tau2 = the largest live distance left outside C2.  Exact for the same
//       reason as the outer level: every candidate outside C2 sits in a bin >= B* and can only move
//       to later bins, so while the restricted maximum is in a bin < B* it is the maximum over C1,
//       hence (outer argument) over the whole cloud; equal distances share a bin, so ties are
//       complete inside C2 and go to the lowest original index,
//   (f) applies the sub-round's picks to all of C1 (all warps, FADD2/FMUL2).
// If the first bin alone overflows T2 (many equal or nearly equal distances) the sub-round is a
// single block-wide argmax with the full tie-break.
// ---------------------------------------------------------------------------------------------
struct __align__(16) HierSmem {
    uint4 wb[16];
    float sD[128], sX[128], sY[128], sZ[128];
    unsigned sO[128];
    int hist[64];
    unsigned wmax[16], wmax2[16];
    uint2 plist[PB];               // picks of the running sub-round: {slot id in s*, D bits}
    int cnt2;
    int npub;                      // picks of the running sub-round visible in plist (| NP_FINAL: no more will come)
};
constexpr int NP_FINAL = 1 << 30;

template <int CPT1, int CPT2, bool STATS, bool EUC>
__device__ __forceinline__ void local_fps_hier(const float *cX, const float *cY, const float *cZ, const float *cD,
                                               const unsigned *cO, const int cnt, const unsigned taubits, int &j, int &nb,
                                               const int M, HierSmem *hs, float4 *bpick, int *out_idx, float *out_mind,
                                               const int tid, unsigned long long &c_subrounds, unsigned long long &c_fallback,
                                               long long &t_sel, long long &t_loop, long long &t_app, const Publisher &pubr)
{
    static_assert(CPT1 % 2 == 0 && CPT2 >= 1 && CPT2 <= 4, "shape");
    constexpr int H1 = CPT1 / 2, T2 = 32 * CPT2;
    // the pick warp is the LAST warp: its own candidate slots are padding unless the buffer is full, so it
    // rarely has anything to catch up on after its loop, while the other warps follow the picks as they appear
    constexpr int PW = BT / 32 - 1;
    const int lane = tid & 31, warp = tid >> 5;
    static_assert(BT == 512, "the slot permutation below is written for 16 warps");
    // candidate slots are dealt to the warps so that the four warps of the pick warp's scheduler (warp % 4 == 3)
    // come last: with a buffer that is not nearly full they hold padding only and leave that scheduler alone
    const int wr = (warp & 3) == 3 ? 12 + (warp >> 2) : 3 * (warp >> 2) + (warp & 3);
    const int st = 32 * wr + lane;
    const float tau = __uint_as_float(taubits);
    f32x2 X[H1], Y[H1], Z[H1];
    float D[CPT1];
#pragma unroll
    for (int h = 0; h < H1; ++h) {
        // candidate slots 2t, 2t+1 (then 2*BT + 2t, ...): a buffer that is not full leaves whole warps with
        // padding only, and those warps drop out of the update loop (f)
        const int i0 = h * 2 * BT + 2 * st, i1 = i0 + 1;
        const bool ok0 = i0 < cnt, ok1 = i1 < cnt;
        X[h] = pack2(ok0 ? cX[i0] : 0.0f, ok1 ? cX[i1] : 0.0f);
        Y[h] = pack2(ok0 ? cY[i0] : 0.0f, ok1 ? cY[i1] : 0.0f);
        Z[h] = pack2(ok0 ? cZ[i0] : 0.0f, ok1 ? cZ[i1] : 0.0f);
        D[2 * h] = ok0 ? cD[i0] : 0.0f;          // padding: D = 0 is never above tau
        D[2 * h + 1] = ok1 ? cD[i1] : 0.0f;
    }
    int jl = j, nbl = 0, applied = 0;
    long long tt0 = 0, tt1 = 0;
    unsigned bound_bits = 0u;            // an upper bound of every candidate's distance left by the last sub-round
    bool have_bound = false;
    for (;;) {
        if (STATS) tt0 = clock64();
        // ---- (a) block maximum.  After a sub-round that ended on tau2 every candidate is <= tau2, which
        // serves as the origin of the bins just as well: the reduction and its barrier are skipped ----
        float m = D[0];
#pragma unroll
        for (int c = 1; c < CPT1; ++c) m = fmaxf(m, D[c]);
        unsigned m1 = bound_bits;
        if (!have_bound) {
            const unsigned wm = __reduce_max_sync(FULL, __float_as_uint(m));
            if (lane == 0) hs->wmax[warp] = wm;
            if (tid < 64) hs->hist[tid] = 0;
            if (tid == 0) hs->cnt2 = 0;
            __syncthreads();
            m1 = __reduce_max_sync(FULL, lane < BT / 32 ? hs->wmax[lane] : 0u);
        }
        if (!(m1 > taubits)) break;
        const float fm1 = __uint_as_float(m1);
        const float scale = fminf(__fdiv_rn(64.0f, __fsub_rn(fm1, tau)), FLT_MAX);
        // bin(d): 0 for d = m1, growing as d falls; monotone because fp32 subtraction and multiplication
        // by a positive constant are monotone
#define RFPS_BIN(d) ((int)fminf(__fmul_rn(__fsub_rn(fm1, (d)), scale), 63.0f))
        // ---- (b) histogram of the live candidates ----
#pragma unroll
        for (int c = 0; c < CPT1; ++c)
            if (D[c] > tau) atomicAdd(&hs->hist[RFPS_BIN(D[c])], 1);
        __syncthreads();
        // ---- (c) B* = number of leading bins that together hold <= T2 candidates ----
        int bstar;
        {
            const int h0 = hs->hist[2 * lane], h1 = hs->hist[2 * lane + 1];
            int incl = h0 + h1;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += t;
            }
            const int excl = incl - (h0 + h1);
            bstar = __popc(__ballot_sync(FULL, excl + h0 <= T2)) + __popc(__ballot_sync(FULL, incl <= T2));
            if (__shfl_sync(FULL, incl, 31) == 0) break;      // no live candidate (only possible with a bound as m1)
        }
        if (bstar == 0 && have_bound) {
            // the first bin overflows and m1 is only a bound: redo the sub-round from the true maximum, which
            // the fallback below needs (all warps have read the histogram before it is cleared again)
            have_bound = false;
            __syncthreads();
            continue;
        }
        if (bstar == 0) {
            // ---- fallback: one pick by a block-wide argmax with the full tie-break ----
            unsigned o = 0u, oi = 0u;
            if (__float_as_uint(m) == m1) {
#pragma unroll
                for (int c = 0; c < CPT1; ++c)
                    if (D[c] == m) {
                        const unsigned i = (unsigned)((c >> 1) * 2 * BT + 2 * st + (c & 1));
                        const unsigned oc = cO[i];
                        if (oc >= o) { o = oc; oi = i; }
                    }
            }
            const unsigned wo = __reduce_max_sync(FULL, o);
            const int wl = __ffs(__ballot_sync(FULL, o == wo)) - 1;
            const unsigned widx = __shfl_sync(FULL, oi, wl);
            if (lane == 0) hs->wb[warp] = make_uint4(wo, widx, 0u, 0u);
            __syncthreads();
            uint4 v = lane < BT / 32 ? hs->wb[lane] : make_uint4(0u, 0u, 0u, 0u);
            const unsigned go = __reduce_max_sync(FULL, v.x);
            const unsigned gidx = __shfl_sync(FULL, v.y, __ffs(__ballot_sync(FULL, v.x == go)) - 1);
            if (tid == 0) {
                out_idx[jl] = (int)(~go);
                out_mind[jl] = fm1;
                bpick[nbl] = make_float4(cX[gidx], cY[gidx], cZ[gidx], 0.0f);
                c_fallback++;
            }
            ++jl;
            ++nbl;
            have_bound = false;          // no tau2 from this path: the next sub-round reduces the maximum again
            __syncthreads();
        } else {
            // ---- (d) C2 -> shared memory; tau2 = the largest live distance left outside C2 (>= tau), so
            // that C2 = {D > tau2} exactly and the pick loop needs one integer compare to know when to stop ----
            float exmax = tau;
#pragma unroll
            for (int c = 0; c < CPT1; ++c)
                if (D[c] > tau) {
                    if (RFPS_BIN(D[c]) < bstar) {
                        const int sl = atomicAdd(&hs->cnt2, 1);
                        const int i = (c >> 1) * 2 * BT + 2 * st + (c & 1);
                        hs->sD[sl] = D[c];
                        hs->sX[sl] = cX[i];
                        hs->sY[sl] = cY[i];
                        hs->sZ[sl] = cZ[i];
                        hs->sO[sl] = cO[i];
                    } else {
                        exmax = fmaxf(exmax, D[c]);
                    }
                }
            {
                const unsigned we = __reduce_max_sync(FULL, __float_as_uint(exmax));
                if (lane == 0) hs->wmax2[warp] = we;
            }
            if (tid == 0) hs->npub = 0;
            __syncthreads();
            // every warp is past (c): clean for the next sub-round.  Done by the pick warp, so that it is ordered
            // before the end-of-loop flag the other warps wait for (no barrier ends the sub-round any more)
            if (warp == PW) { hs->hist[lane] = 0; hs->hist[32 + lane] = 0; }
            // tau2 = the largest live distance outside C2: where the pick loop stops, and the bound the next
            // sub-round hangs its bins on
            const unsigned tau2bits = __reduce_max_sync(FULL, lane < BT / 32 ? hs->wmax2[lane] : 0u);
            if (STATS) { tt1 = clock64(); t_sel += tt1 - tt0; tt0 = tt1; }
            // ---- (e) one warp: FPS over C2 in registers.  No barrier and no vote/shuffle per pick: the
            // chain is update -> lane max -> redux(max D) -> redux(slot id) -> 3 broadcast loads. ----
            if (warp == PW) {
                const int n2 = hs->cnt2;
                __syncwarp();
                if (lane == 0) hs->cnt2 = 0;
                float x2[CPT2], y2[CPT2], z2[CPT2], d2v[CPT2];
#pragma unroll
                for (int c = 0; c < CPT2; ++c) {
                    const int i = c * 32 + lane;
                    const bool ok = i < n2;
                    x2[c] = ok ? hs->sX[i] : 0.0f;
                    y2[c] = ok ? hs->sY[i] : 0.0f;
                    z2[c] = ok ? hs->sZ[i] : 0.0f;
                    d2v[c] = ok ? hs->sD[i] : 0.0f;         // padding never exceeds tau2
                }
                // The picks of the sub-round are logged as {slot id, D bits} in shared memory and emitted after
                // the loop.  Fast path: KCH picks at a time, speculatively and without a branch in the dependent
                // chain -- termination (max <= tau2) and exact ties are only recorded; afterwards the prefix of
                // picks before the first such event is accepted.  Picks computed beyond it are discarded with
                // the register state (the sub-round ends there, or the chunk is redone pick by pick).
                const int nb0 = nbl, j0 = jl;
                // one pick, fully checked: returns false when the sub-round is over
                auto careful_pick = [&]() -> bool {
                    float bm = d2v[0];
#pragma unroll
                    for (int c = 1; c < CPT2; ++c) bm = fmaxf(bm, d2v[c]);
                    // slot ids (+1) of this lane's candidates at its maximum: largest and smallest
                    unsigned idmx = 0u, idmn = 0x7fffffffu;
#pragma unroll
                    for (int c = 0; c < CPT2; ++c)
                        if (d2v[c] == bm) { idmx = max(idmx, (unsigned)(c * 32 + lane + 1)); idmn = min(idmn, (unsigned)(c * 32 + lane + 1)); }
                    const unsigned hi = __float_as_uint(bm);
                    const unsigned ghi = __reduce_max_sync(FULL, hi);
                    if (!(ghi > tau2bits)) return false;     // restricted max no longer above everything outside C2
                    const bool top = hi == ghi;
                    const unsigned gmx = __reduce_max_sync(FULL, top ? idmx : 0u);
                    const unsigned gmn = __reduce_min_sync(FULL, top ? idmn : 0x7fffffffu);
                    unsigned wid = gmx - 1u;
                    if (gmx != gmn) {                        // exact tie: lowest original index wins
                        unsigned lo = 0u;
                        if (top) {
#pragma unroll
                            for (int c = 0; c < CPT2; ++c)
                                if (d2v[c] == bm) lo = max(lo, hs->sO[c * 32 + lane]);
                        }
                        const unsigned glo = __reduce_max_sync(FULL, lo);
                        unsigned mine = 0u;
                        if (top) {
#pragma unroll
                            for (int c = 0; c < CPT2; ++c)
                                if (d2v[c] == bm && hs->sO[c * 32 + lane] == glo) mine = (unsigned)(c * 32 + lane + 1);
                        }
                        wid = __reduce_max_sync(FULL, mine) - 1u;
                    }
                    const float sx = hs->sX[wid], sy = hs->sY[wid], sz = hs->sZ[wid];
                    if (lane == 0) {
                        hs->plist[nbl - nb0] = make_uint2(wid, ghi);
                        bpick[nbl] = make_float4(sx, sy, sz, 0.0f);
                    }
                    ++jl;
                    ++nbl;
                    if (jl >= M || nbl >= PB) return false;
#pragma unroll
                    for (int c = 0; c < CPT2; ++c) d2v[c] = fminf(d2v[c], distf<EUC>(d2_rn(x2[c], y2[c], z2[c], sx, sy, sz)));
                    return true;
                };
                for (bool go = true; go;) {
                    if (min(M - jl, PB - nbl) <= KCH) {      // near the end of the output or of the batch buffer
                        go = careful_pick();
                        continue;
                    }
                    float dsave[CPT2];
#pragma unroll
                    for (int c = 0; c < CPT2; ++c) dsave[c] = d2v[c];
                    bool over = false, tie = false;          // "max <= tau2 seen" / "exact tie seen before that"
                    int acc = 0;                             // picks before the first "max <= tau2"
#pragma unroll
                    for (int p = 0; p < KCH; ++p) {
                        // one uniform exit test every four picks bounds the speculation past the end of the
                        // sub-round without putting a branch behind every redux
                        if ((p & 3) == 0 && p > 0 && over) break;
                        // half-way publish: the picks before the first "over" or tie stand whatever follows (a tie
                        // redoes the chunk with the same arithmetic), and what the other warps have not applied when
                        // the loop ends is on the critical path of the sub-round
                        if (p == KCH / 2 && !tie && lane == 0) {
                            __threadfence_block();
                            *(volatile int *)&hs->npub = nbl - nb0 + p;
                        }
                        float bm = d2v[0];
#pragma unroll
                        for (int c = 1; c < CPT2; ++c) bm = fmaxf(bm, d2v[c]);
                        unsigned idmx = 0u, idmn = 0x7fffffffu;
#pragma unroll
                        for (int c = 0; c < CPT2; ++c)
                            if (d2v[c] == bm) { idmx = max(idmx, (unsigned)(c * 32 + lane + 1)); idmn = min(idmn, (unsigned)(c * 32 + lane + 1)); }
                        const unsigned hi = __float_as_uint(bm);
                        const unsigned ghi = __reduce_max_sync(FULL, hi);
                        const bool top = hi == ghi;
                        const unsigned gmx = __reduce_max_sync(FULL, top ? idmx : 0u);
                        const unsigned gmn = __reduce_min_sync(FULL, top ? idmn : 0x7fffffffu);
                        const unsigned wid = gmx - 1u;       // always a valid slot: some lane is top
                        over |= !(ghi > tau2bits);
                        tie |= (gmx != gmn) && !over;
                        acc += over ? 0 : 1;
                        const float sx = hs->sX[wid], sy = hs->sY[wid], sz = hs->sZ[wid];
                        if (lane == 0) {                     // logged speculatively, off the dependent chain
                            hs->plist[nbl - nb0 + p] = make_uint2(wid, ghi);
                            bpick[nbl + p] = make_float4(sx, sy, sz, 0.0f);
                        }
#pragma unroll
                        for (int c = 0; c < CPT2; ++c) d2v[c] = fminf(d2v[c], distf<EUC>(d2_rn(x2[c], y2[c], z2[c], sx, sy, sz)));
                    }
                    if (tie) {                               // rare: redo this chunk pick by pick
#pragma unroll
                        for (int c = 0; c < CPT2; ++c) d2v[c] = dsave[c];
                        for (int p = 0; p < KCH && go; ++p) go = careful_pick();
                        continue;
                    }
                    jl += acc;
                    nbl += acc;
                    go = acc == KCH;
                    if (lane == 0) {                         // the other warps may apply these picks now
                        __threadfence_block();
                        *(volatile int *)&hs->npub = nbl - nb0;
                    }
                }
                if (lane == 0) {
                    __threadfence_block();
                    *(volatile int *)&hs->npub = (nbl - nb0) | NP_FINAL;
                }
                __syncwarp();
                asm volatile("bar.arrive 1, %0;" ::"n"(BT) : "memory");      // wakes the warps that only wait (below)
                {
                    const int n = nbl - nb0;                 // emit the sub-round's picks
                    __syncwarp();
                    for (int i = lane; i < n; i += 32) {
                        const uint2 pk = hs->plist[i];
                        out_idx[j0 + i] = (int)(~hs->sO[pk.x]);
                        out_mind[j0 + i] = __uint_as_float(pk.y);
                    }
                }
            } else {
                // ---- (f), streamed: the other warps apply the sub-round's picks to their candidates while the
                // pick warp is still producing them; after the loop only the last few picks are left ----
                bool live = false;
#pragma unroll
                for (int c = 0; c < CPT1; ++c) live |= D[c] > tau;
                // a warp whose candidates are all dead only needs the final count: it sleeps on a named barrier
                // that the pick warp and the working warps arrive at without waiting (polling would take issue
                // slots from the pick warp)
                const bool wlive = __any_sync(FULL, live);
                {
                    int done = 0;
                    if (!wlive) asm volatile("bar.sync 1, %0;" ::"n"(BT) : "memory");
                    for (;;) {
                        const int v = *(volatile int *)&hs->npub;
                        const int n = v & 0xffff;
                        if (n > done) {
                            __threadfence_block();
                            for (int i = done; wlive && i < n; ++i) {
                                const float4 sp = bpick[nbl + i];
                                const f32x2 SX = pack2(sp.x, sp.x), SY = pack2(sp.y, sp.y), SZ = pack2(sp.z, sp.z);
#pragma unroll
                                for (int h = 0; h < H1; ++h) {
                                    const f32x2 dx = sub2(X[h], SX), dy = sub2(Y[h], SY), dz = sub2(Z[h], SZ);
                                    float x0, x1, y0, y1, z0, z1;
                                    unpack2(mul2(dx, dx), x0, x1);
                                    unpack2(mul2(dy, dy), y0, y1);
                                    unpack2(mul2(dz, dz), z0, z1);
                                    D[2 * h] = fminf(D[2 * h], distf<EUC>(__fadd_rn(__fadd_rn(x0, y0), z0)));
                                    D[2 * h + 1] = fminf(D[2 * h + 1], distf<EUC>(__fadd_rn(__fadd_rn(x1, y1), z1)));
                                }
                            }
                            done = n;
                        } else if (v & NP_FINAL) {
                            break;
                        } else {
                            __nanosleep(POLL_NS);
                        }
                    }
                    if (wlive) asm volatile("bar.arrive 1, %0;" ::"n"(BT) : "memory");
                    nbl += done;                             // the final count is the sub-round's result: no barrier
                    jl += done;
                    applied = nbl;
                }
            }
            bound_bits = tau2bits;       // the pick loop stopped at or below tau2, and so did everything outside C2
            have_bound = true;
        }
#undef RFPS_BIN
        c_subrounds++;
        // the workers may start applying these picks now.  The release is issued by the thread that wrote bpick
        // (lane 0 of the pick warp; after a barrier on the fallback path); its fence overlaps the other warps'
        // selection of the next sub-round
        if (pubr.on() && tid == BT - 32) pubr((unsigned)nbl);
        if (STATS) { tt1 = clock64(); t_loop += tt1 - tt0; tt0 = tt1; }
        // ---- (f) the sub-round's picks -> all of C1.  Candidates at or below tau are out of the round for
        // good; neighbours in the buffer come from the same voxel and tend to die together, so whole
        // warps drop out of this loop as the round proceeds ----
        bool live = false;
#pragma unroll
        for (int c = 0; c < CPT1; ++c) live |= D[c] > tau;
        if (__any_sync(FULL, live))
        for (int i = applied; i < nbl; ++i) {
            const float4 s = bpick[i];
            const f32x2 SX = pack2(s.x, s.x), SY = pack2(s.y, s.y), SZ = pack2(s.z, s.z);
#pragma unroll
            for (int h = 0; h < H1; ++h) {
                const f32x2 dx = sub2(X[h], SX), dy = sub2(Y[h], SY), dz = sub2(Z[h], SZ);
                float x0, x1, y0, y1, z0, z1;
                unpack2(mul2(dx, dx), x0, x1);
                unpack2(mul2(dy, dy), y0, y1);
                unpack2(mul2(dz, dz), z0, z1);
                D[2 * h] = fminf(D[2 * h], distf<EUC>(__fadd_rn(__fadd_rn(x0, y0), z0)));
                D[2 * h + 1] = fminf(D[2 * h + 1], distf<EUC>(__fadd_rn(__fadd_rn(x1, y1), z1)));
            }
        }
        applied = nbl;
        if (STATS) t_app += clock64() - tt0;
        if (jl >= M || nbl >= PB) break;
    }
    j = jl;
    nb = nbl;
}

// ---------------------------------------------------------------------------------------------
// LOCAL, parallel resolution (the default, local_warps = LW_PAR): the sequential pick chain is broken up.
// All 16 warps keep the candidate set C1 in registers (CPT1 per thread), exact with respect to every pick so
// far.  One STEP:
//   (1) histogram of the live candidates (32 bins between a lower end blo and an upper bound hi of all
//       distances, monotone bin function) -> the longest prefix of bins holding <= KS = 64 candidates: the
//       MEMBERS.  Every other candidate of C1 -- and every other point of the cloud -- is then strictly
//       below every member.
//   (2) members -> shared memory {x, y, z, D, ~orig}.
//   (3) all pairs (i, j) of members, spread over the 512 threads (a mask word is one ballot): does j rank BEFORE i (key_j > key_i, key =
//       (D, ~orig): the order in which FPS would pick them if nothing changed), and would picking j LOWER
//       D_i (d(i, j) < D_i)?  -> per member two 64-bit masks bef_i, aff_i = {j before i that lower i}.
//   (4) one warp resolves the pick sequence with bit operations: walking the members in rank order, member
//       i is the next FPS pick with mindist D_i exactly when no ACCEPTED member of aff_i precedes it (its D
//       is then unchanged, every higher-ranked member has been picked or has dropped below it, everything
//       else was below it to begin with).  acc_i = !(aff_i & ACC) is solved by fixed-point iteration over
//       ballots (members with empty aff_i first; typically 2-3 iterations).  A rejected member whose new
//       distance could still be >= the smallest member distance (stop_i) might have to be picked before
//       lower-ranked members: the step is cut at the first such member in rank order.
//   (5) the accepted picks are emitted in rank order and applied to all of C1 by all warps.
// A step yields ~20-35 picks for 4 CTA barriers and a few hundred instructions per thread, where the
// sequential chain costs ~200 cycles per pick.  Exactness: see (4); ties are covered because bef is a strict
// total order on (D, ~orig) and equal distances always share a bin.  If the first bin alone overflows KS
// (many nearly equal distances) the bin range is narrowed to it (twice at most), then the step is a single
// block-wide argmax with the full tie-break.
// ---------------------------------------------------------------------------------------------
constexpr int KS = 64;
struct __align__(16) ParSmem {
    float4 sC[KS];                 // members {x, y, z, D}
    unsigned long long aff[KS];    // members ranked before i whose pick would lower D_i
    unsigned long long bef[KS];    // members ranked before i
    unsigned sO[KS];               // ~orig of the members
    int hist[2][16][32];           // per-warp histograms, double-buffered by step parity
    uint4 wb[16];
    unsigned wmax[16];
    unsigned stop[2];              // bit i: a member of aff_i may leave D_i >= the smallest member distance
    int ncomp;                     // slots handed out by the running compaction
    int nmem;
    unsigned minD;                 // smallest member distance (bits)
    int npk;                       // picks accepted by the step
    unsigned hi;                   // upper bound of every candidate's distance after the step (bits)
};
static_assert(sizeof(ParSmem) <= 3392 + 8 * PB, "smem_layout reserves this much for the local phase");

__device__ __forceinline__ unsigned long long ballot64(bool a, bool b)
{
    return (unsigned long long)__ballot_sync(FULL, a) | ((unsigned long long)__ballot_sync(FULL, b) << 32);
}

template <int CPT1, bool STATS, bool EUC>
__device__ __forceinline__ void local_fps_par(const float *cX, const float *cY, const float *cZ, const float *cD,
                                              const unsigned *cO, float *const cand2, const int cnt, const unsigned taubits, int &j, int &nb,
                                              const int M, ParSmem *ps, float4 *bpick, int *out_idx, float *out_mind,
                                              const int tid, unsigned long long &c_steps, unsigned long long &c_fallback,
                                              long long &t_sel, long long &t_pick, long long &t_upd, long long &t_pairs,
                                              long long &t_publish, const Publisher &pubr)
{
    static_assert(CPT1 % 2 == 0 && BT == 512 && KS == 64, "shape");
    constexpr int H1 = CPT1 / 2;
    const int lane = tid & 31, warp = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const float tau = __uint_as_float(taubits);
    // candidate slots 2t, 2t+1 (then 2*BT + 2t, ...): a buffer that is not full leaves whole warps with padding
    // only, and those warps drop out of the update loop
    f32x2 X[H1], Y[H1], Z[H1];
    float D[CPT1];
    // Euclidean mode: sqrt_rn is monotone, so min_k sqrt_rn(d2_k) == sqrt_rn(min_k d2_k): the picks of a step are
    // applied in the squared domain (M2 = the smallest d2 since the last fold) and folded into D -- which holds
    // distances -- once per step, instead of one correctly rounded square root per (candidate, pick) pair
    float M2[EUC ? CPT1 : 1];
#pragma unroll
    for (int c = 0; c < (EUC ? CPT1 : 1); ++c) M2[c] = __uint_as_float(F32_INF_BITS);
#pragma unroll
    for (int h = 0; h < H1; ++h) {
        const int i0 = h * 2 * BT + 2 * tid, i1 = i0 + 1;
        const bool ok0 = i0 < cnt, ok1 = i1 < cnt;
        X[h] = pack2(ok0 ? cX[i0] : 0.0f, ok1 ? cX[i1] : 0.0f);
        Y[h] = pack2(ok0 ? cY[i0] : 0.0f, ok1 ? cY[i1] : 0.0f);
        Z[h] = pack2(ok0 ? cZ[i0] : 0.0f, ok1 ? cZ[i1] : 0.0f);
        D[2 * h] = ok0 ? cD[i0] : 0.0f;          // padding: D = 0 is never above tau
        D[2 * h + 1] = ok1 ? cD[i1] : 0.0f;
    }
    int jl = j, nbl = 0;
    long long tt0 = 0, tt1 = 0;
    // block maximum: the first upper bound
    auto block_max = [&]() -> unsigned {
        float m = D[0];
#pragma unroll
        for (int c = 1; c < CPT1; ++c) m = fmaxf(m, D[c]);
        const unsigned wm = __reduce_max_sync(FULL, __float_as_uint(m));
        if (lane == 0) ps->wmax[warp] = wm;
        __syncthreads();
        return __reduce_max_sync(FULL, lane < BT / 32 ? ps->wmax[lane] : 0u);
    };
    ps->hist[0][warp][lane] = 0;
    ps->hist[1][warp][lane] = 0;
    if (tid == 0) { ps->nmem = 0; ps->minD = 0xffffffffu; ps->stop[0] = ps->stop[1] = 0u; ps->ncomp = 0; }
    // the candidate buffer in use (cX .. cO) and the spare one the live candidates are compacted into
    constexpr int TCAP = CPT1 * BT;
    float *sX = cand2, *sY = sX ? sX + TCAP : nullptr, *sZ = sX ? sX + 2 * TCAP : nullptr, *sD = sX ? sX + 3 * TCAP : nullptr;
    unsigned *sO = sX ? reinterpret_cast<unsigned *>(sX + 4 * TCAP) : nullptr;
    int cntc = cnt;                      // slots in use
    unsigned hibits = block_max();       // (its barrier also publishes the initialisation above)
    bool hi_exact = true;
    float blo = tau;                     // lower end of the bin range; members are above it
    int refine = 0, hp = 0;
    // one pick applied to this thread's candidates
    auto apply_pick = [&](const float4 s) {
        const f32x2 SX = pack2(s.x, s.x), SY = pack2(s.y, s.y), SZ = pack2(s.z, s.z);
#pragma unroll
        for (int h = 0; h < H1; ++h) {
            const f32x2 dx = sub2(X[h], SX), dy = sub2(Y[h], SY), dz = sub2(Z[h], SZ);
            float x0, x1, y0, y1, z0, z1;
            unpack2(mul2(dx, dx), x0, x1);
            unpack2(mul2(dy, dy), y0, y1);
            unpack2(mul2(dz, dz), z0, z1);
            if (EUC) {       // squared domain; folded into D at the top of the next step (one square root per step)
                M2[2 * h] = fminf(M2[2 * h], __fadd_rn(__fadd_rn(x0, y0), z0));
                M2[2 * h + 1] = fminf(M2[2 * h + 1], __fadd_rn(__fadd_rn(x1, y1), z1));
            } else {
                D[2 * h] = fminf(D[2 * h], __fadd_rn(__fadd_rn(x0, y0), z0));
                D[2 * h + 1] = fminf(D[2 * h + 1], __fadd_rn(__fadd_rn(x1, y1), z1));
            }
        }
    };
    auto apply_range = [&](const int lo, const int hi_) {
        bool live = false;
#pragma unroll
        for (int c = 0; c < CPT1; ++c) live |= D[c] > tau;
        if (__any_sync(FULL, live))
            for (int i = lo; i < hi_; ++i) apply_pick(bpick[i]);
    };
    for (;;) {
        if (!(hibits > taubits)) break;                      // nothing above tau is left: the candidates no longer decide
        if (STATS) tt0 = clock64();
        hp ^= 1;
        if (EUC) {
#pragma unroll
            for (int c = 0; c < CPT1; ++c) {
                D[c] = fminf(D[c], __fsqrt_rn(M2[c]));
                M2[c] = __uint_as_float(F32_INF_BITS);
            }
        }
        const float hi = __uint_as_float(hibits);
        const float scale = fminf(__fdiv_rn(32.0f, __fsub_rn(hi, blo)), FLT_MAX);
        // bin(d): 0 for d = hi, growing as d falls; monotone because fp32 subtraction and multiplication by a
        // positive constant are monotone
#define RFPS_BIN(d) ((int)fminf(fmaxf(__fmul_rn(__fsub_rn(hi, (d)), scale), 0.0f), 31.0f))
        // ---- (1) per-warp histogram of the candidates above blo ----
        int bin[CPT1];
#pragma unroll
        for (int c = 0; c < CPT1; ++c) {
            const bool in = D[c] > blo;
            bin[c] = in ? RFPS_BIN(D[c]) : 32;
            if (in) atomicAdd(&ps->hist[hp][warp][bin[c]], 1);
        }
        __syncthreads();
        ps->hist[hp ^ 1][warp][lane] = 0;                    // the other buffer: every warp is done with it
        int bstar, total;
        {
            int tot = 0;
#pragma unroll
            for (int w = 0; w < BT / 32; ++w) tot += ps->hist[hp][w][lane];
            int incl = tot;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += t;
            }
            total = __shfl_sync(FULL, incl, 31);
            bstar = __popc(__ballot_sync(FULL, incl <= KS));
        }
        // ---- compaction: candidates at or below tau are out of the round for good.  Once fewer than 5/8 of the slots
        // in use are live, the live ones are packed into the first slots of the spare buffer: whole warps then hold
        // padding only and drop out of the update loop (5), which is the largest part of a step.  The histogram
        // just taken stays valid (it is summed over the warps); only this thread's bins are recomputed. ----
        if (sX != nullptr && blo == tau && cntc > 4 * KS && total * 8 < cntc * 5 && total > 0) {
            unsigned bal[CPT1];
            int cw = 0;
#pragma unroll
            for (int c = 0; c < CPT1; ++c) {
                bal[c] = __ballot_sync(FULL, D[c] > tau);
                cw += __popc(bal[c]);
            }
            if (cw) {
                int base = 0;
                if (lane == 0) base = atomicAdd(&ps->ncomp, cw);
                base = __shfl_sync(FULL, base, 0);
#pragma unroll
                for (int c = 0; c < CPT1; ++c) {
                    if (D[c] > tau) {
                        const int sl = base + __popc(bal[c] & lt);
                        float x0, x1, y0, y1, z0, z1;
                        unpack2(X[c >> 1], x0, x1);
                        unpack2(Y[c >> 1], y0, y1);
                        unpack2(Z[c >> 1], z0, z1);
                        sX[sl] = (c & 1) ? x1 : x0; sY[sl] = (c & 1) ? y1 : y0; sZ[sl] = (c & 1) ? z1 : z0;
                        sD[sl] = D[c];
                        sO[sl] = cO[(c >> 1) * 2 * BT + 2 * tid + (c & 1)];
                    }
                    base += __popc(bal[c]);
                }
            }
            __syncthreads();
            cntc = ps->ncomp;
            {   // swap the buffers: the compacted one becomes cX .., the old one the spare
                float *tX = const_cast<float *>(cX), *tY = const_cast<float *>(cY), *tZ = const_cast<float *>(cZ), *tD = const_cast<float *>(cD);
                unsigned *tO = const_cast<unsigned *>(cO);
                cX = sX; cY = sY; cZ = sZ; cD = sD; cO = sO;
                sX = tX; sY = tY; sZ = tZ; sD = tD; sO = tO;
            }
#pragma unroll
            for (int h = 0; h < H1; ++h) {
                const int i0 = h * 2 * BT + 2 * tid, i1 = i0 + 1;
                const bool ok0 = i0 < cntc, ok1 = i1 < cntc;
                X[h] = pack2(ok0 ? cX[i0] : 0.0f, ok1 ? cX[i1] : 0.0f);
                Y[h] = pack2(ok0 ? cY[i0] : 0.0f, ok1 ? cY[i1] : 0.0f);
                Z[h] = pack2(ok0 ? cZ[i0] : 0.0f, ok1 ? cZ[i1] : 0.0f);
                D[2 * h] = ok0 ? cD[i0] : 0.0f;
                D[2 * h + 1] = ok1 ? cD[i1] : 0.0f;
            }
#pragma unroll
            for (int c = 0; c < CPT1; ++c) bin[c] = D[c] > blo ? RFPS_BIN(D[c]) : 32;
            __syncthreads();                                 // everybody has read ncomp
            if (tid == 0) ps->ncomp = 0;
        }
        if (total == 0) {
            if (blo == tau) break;                           // no live candidate (hi was only a bound)
            blo = tau; refine = 0; hi_exact = false;         // cannot happen with an exact hi; start over from the bound
            continue;
        }
        if (bstar == 0) {
            // the first bin alone holds more than KS candidates
            if (!hi_exact) {                                 // the bins hang on a bound: redo them from the true maximum
                hibits = block_max();
                hi_exact = true;
                continue;
            }
            const float nlo = __fsub_rn(hi, __fmul_rn(__fsub_rn(hi, blo), 0x1p-5f));
            if (refine < 2 && nlo > blo && nlo < hi) {       // narrow the bin range to (about) the first bin
                blo = nlo;
                ++refine;
                continue;
            }
            // ---- fallback: one pick by a block-wide argmax with the full tie-break (hi is the true maximum) ----
            float m = D[0];
#pragma unroll
            for (int c = 1; c < CPT1; ++c) m = fmaxf(m, D[c]);
            unsigned o = 0u, oi = 0u;
            if (__float_as_uint(m) == hibits) {
#pragma unroll
                for (int c = 0; c < CPT1; ++c)
                    if (D[c] == m) {
                        const unsigned i = (unsigned)((c >> 1) * 2 * BT + 2 * tid + (c & 1));
                        const unsigned oc = cO[i];
                        if (oc >= o) { o = oc; oi = i; }
                    }
            }
            const unsigned wo = __reduce_max_sync(FULL, o);
            const int wl = __ffs(__ballot_sync(FULL, o == wo)) - 1;
            const unsigned widx = __shfl_sync(FULL, oi, wl);
            if (lane == 0) ps->wb[warp] = make_uint4(wo, widx, 0u, 0u);
            __syncthreads();
            const uint4 v = lane < BT / 32 ? ps->wb[lane] : make_uint4(0u, 0u, 0u, 0u);
            const unsigned go = __reduce_max_sync(FULL, v.x);
            const unsigned gidx = __shfl_sync(FULL, v.y, __ffs(__ballot_sync(FULL, v.x == go)) - 1);
            if (tid == 0) {
                out_idx[jl] = (int)(~go);
                out_mind[jl] = hi;
                bpick[nbl] = make_float4(cX[gidx], cY[gidx], cZ[gidx], 0.0f);
                if (pubr.gpick) pubr.gpick[nbl] = bpick[nbl];
                c_fallback++;
            }
            __syncthreads();
            if (pubr.on() && tid == 0) pubr((unsigned)(nbl + 1));
            apply_range(nbl, nbl + 1);
            ++jl;
            ++nbl;
            c_steps++;
            hi_exact = false;                                // hi stays a valid bound
            blo = tau;
            refine = 0;
            if (jl >= M || nbl >= PB) break;
            continue;
        }
        // ---- (2) members (bin < bstar) -> shared memory ----
        {
            unsigned bal[CPT1];
            int cntw = 0;
#pragma unroll
            for (int c = 0; c < CPT1; ++c) {
                bal[c] = __ballot_sync(FULL, bin[c] < bstar);
                cntw += __popc(bal[c]);
            }
            if (cntw) {
                int base = 0;
                if (lane == 0) base = atomicAdd(&ps->nmem, cntw);
                base = __shfl_sync(FULL, base, 0);
                unsigned mind = 0xffffffffu;
#pragma unroll
                for (int c = 0; c < CPT1; ++c) {
                    if (bin[c] < bstar) {
                        const int sl = base + __popc(bal[c] & lt);
                        float x0, x1, y0, y1, z0, z1;
                        unpack2(X[c >> 1], x0, x1);
                        unpack2(Y[c >> 1], y0, y1);
                        unpack2(Z[c >> 1], z0, z1);
                        ps->sC[sl] = make_float4((c & 1) ? x1 : x0, (c & 1) ? y1 : y0, (c & 1) ? z1 : z0, D[c]);
                        ps->sO[sl] = cO[(c >> 1) * 2 * BT + 2 * tid + (c & 1)];
                        mind = min(mind, __float_as_uint(D[c]));
                    }
                    base += __popc(bal[c]);
                }
                mind = __reduce_min_sync(FULL, mind);
                if (lane == 0) atomicMin(&ps->minD, mind);
            }
        }
        __syncthreads();
        const int n = ps->nmem;
        const unsigned thmbits = ps->minD;
        if (STATS) { tt1 = clock64(); t_sel += tt1 - tt0; tt0 = tt1; }
        // ---- (3) all pairs: warp w takes the members i = 4w .. 4w+3 in turn, its lanes the partners j = lane and
        // lane + 32 (loaded once, consecutive addresses); a mask word is then ONE ballot ----
        {
            const float thm = __uint_as_float(thmbits);
            const int j0 = lane, j1 = lane + 32;
            const bool v0 = j0 < n, v1 = j1 < n;
            const float4 c0 = v0 ? ps->sC[j0] : make_float4(0.f, 0.f, 0.f, 0.f), c1 = v1 ? ps->sC[j1] : make_float4(0.f, 0.f, 0.f, 0.f);
            // rank key (distance bits, ~orig): unsigned order = "larger distance first, ties to the lowest index"; the keys
            // of two different points differ, and an absent partner (key 0) ranks before nobody (members are > tau >= 0)
            const unsigned long long k0 = v0 ? ((unsigned long long)__float_as_uint(c0.w) << 32) | ps->sO[j0] : 0ull;
            const unsigned long long k1 = v1 ? ((unsigned long long)__float_as_uint(c1.w) << 32) | ps->sO[j1] : 0ull;
#pragma unroll
            for (int ii = 0; ii < 4; ++ii) {
                // (no early exit: without a branch between the four members their dependent chains overlap; a member
                // slot beyond n is computed on slot 0 and not stored)
                const bool live = 4 * warp + ii < n;
                const int i = live ? 4 * warp + ii : 0;
                const float4 ci = ps->sC[i];
                const unsigned long long ki = ((unsigned long long)__float_as_uint(ci.w) << 32) | ps->sO[i];
                const float d0 = distf<EUC>(d2_rn(ci.x, ci.y, ci.z, c0.x, c0.y, c0.z));
                const float d1 = distf<EUC>(d2_rn(ci.x, ci.y, ci.z, c1.x, c1.y, c1.z));
                const bool b0 = k0 > ki, b1 = k1 > ki;
                const bool l0 = b0 && d0 < ci.w, l1 = b1 && d1 < ci.w;
                const unsigned bw0 = __ballot_sync(FULL, b0), bw1 = __ballot_sync(FULL, b1);
                const unsigned aw0 = __ballot_sync(FULL, l0), aw1 = __ballot_sync(FULL, l1);
                const bool sany = __any_sync(FULL, (l0 && !(d0 < thm)) || (l1 && !(d1 < thm)));
                if (lane == 0 && live) {
                    ps->aff[i] = ((unsigned long long)aw1 << 32) | aw0;
                    ps->bef[i] = ((unsigned long long)bw1 << 32) | bw0;
                    if (sany) atomicOr(&ps->stop[i >> 5], 1u << (i & 31));
                }
            }
        }
        __syncthreads();
        if (STATS) t_pairs += clock64() - tt0;
        // ---- (4) one warp resolves the pick sequence ----
        if (warp == 0) {
            const int ia = lane, ib = lane + 32;
            const bool va = ia < n, vb = ib < n;
            const unsigned long long affa = va ? ps->aff[ia] : 0ull, affb = vb ? ps->aff[ib] : 0ull;
            const unsigned long long befa = va ? ps->bef[ia] : 0ull, befb = vb ? ps->bef[ib] : 0ull;
            const float4 ca = va ? ps->sC[ia] : make_float4(0.f, 0.f, 0.f, 0.f), cb = vb ? ps->sC[ib] : make_float4(0.f, 0.f, 0.f, 0.f);
            const bool sta = (ps->stop[0] >> lane) & 1u, stb = (ps->stop[1] >> lane) & 1u;
            __syncwarp();
            if (lane == 0) { ps->stop[0] = ps->stop[1] = 0u; ps->nmem = 0; ps->minD = 0xffffffffu; }   // for the next step
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
            const int lim = min(M - jl, PB - nbl);            // >= 1 here
            const int posa = __popcll(A & befa), posb = __popcll(A & befb);
            acca &= posa < lim; accb &= posb < lim;
            A = ballot64(acca, accb);
            if (acca) {
                out_idx[jl + posa] = (int)(~ps->sO[ia]);
                out_mind[jl + posa] = ca.w;
                bpick[nbl + posa] = make_float4(ca.x, ca.y, ca.z, 0.0f);
                if (pubr.gpick) pubr.gpick[nbl + posa] = make_float4(ca.x, ca.y, ca.z, 0.0f);
            }
            if (accb) {
                out_idx[jl + posb] = (int)(~ps->sO[ib]);
                out_mind[jl + posb] = cb.w;
                bpick[nbl + posb] = make_float4(cb.x, cb.y, cb.z, 0.0f);
                if (pubr.gpick) pubr.gpick[nbl + posb] = make_float4(cb.x, cb.y, cb.z, 0.0f);
            }
            // bound of what is left: members neither picked nor surely below every member, else the smallest
            // member distance (everything outside the members is below it)
            const bool la = va && !acca && !(reja && !sta && (unsigned)ranka < rmin), lb = vb && !accb && !(rejb && !stb && (unsigned)rankb < rmin);
            const unsigned hin = __reduce_max_sync(FULL, max(la ? __float_as_uint(ca.w) : 0u, lb ? __float_as_uint(cb.w) : 0u));
            if (lane == 0) { ps->npk = __popcll(A); ps->hi = max(hin, thmbits); }
        }
        __syncthreads();
        const int npk = ps->npk;
        hibits = ps->hi;
        hi_exact = false;
        blo = tau;
        refine = 0;
        c_steps++;
        if (STATS) { tt1 = clock64(); t_pick += tt1 - tt0; tt0 = tt1; }
        // the workers may start applying these picks: they take pieces of >= STREAM_MIN picks, so the count is
        // published when it crosses a multiple of that.  The release is issued by a thread with no global stores of
        // its own in flight (warp 1; warp 0 has just written out_idx / out_mindist): its fence is then short.  The
        // barrier above orders warp 0's writes to bpick before it.
        if (pubr.on() && tid == 32 && (nbl + npk) / STREAM_MIN != nbl / STREAM_MIN) pubr((unsigned)(nbl + npk));
        if (STATS) { tt1 = clock64(); t_publish += tt1 - tt0; tt0 = tt1; }
        // ---- (5) the step's picks -> all of C1 ----
        apply_range(nbl, nbl + npk);
        nbl += npk;
        jl += npk;
        if (STATS) t_upd += clock64() - tt0;
        if (jl >= M || nbl >= PB) break;
#undef RFPS_BIN
    }
    j = jl;
    nb = nbl;
}

// ---------------------------------------------------------------------------------------------
// the kernel: one cluster per cloud.  32 consecutive (Hilbert-ordered) voxels form a group with its
// own bounding sphere; CTA `rank` owns the groups g = rank + C*gl (round-robin, so that dense
// regions of the cloud are spread over the CTAs); local voxel slot kl = 32*gl + l is voxel
// k = 32*g + l.
// ---------------------------------------------------------------------------------------------
static_assert(sizeof(HierSmem) <= 3392 + 8 * PB, "smem_layout reserves this much for HierSmem");

template <int CPT, int LW, bool STATS, bool EUC, bool GRID>
__global__ void __launch_bounds__(BT, 1) k_fps_batched(const BatchParams P, const int flags)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int TC = cand_capacity(CPT, LW);
    constexpr int NW = BT / 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    // the CTAs of one cloud: a thread-block cluster (exchange over DSMEM), or -- GRID -- `ctas_per_cloud`
    // consecutive CTAs of a cooperative launch (exchange through global memory)
    const int C = GRID ? P.ctas_per_cloud : (int)cluster_nctarank();
    const int rank = GRID ? (int)(blockIdx.x % (unsigned)C) : (int)cluster_ctarank();
    const int b = blockIdx.x / C;
    const bool no_prune = flags & FPS_FLAG_NO_PRUNE, no_skip = flags & FPS_FLAG_NO_SKIP;
    const bool no_batch = flags & FPS_FLAG_NO_BATCH;

    const SmemLayout L = smem_layout(P.Kc_cap, TC, LW);
    float4 *sgeom = reinterpret_cast<float4 *>(smem_raw + L.geom);    // [Kc] {cx, cy, cz, R}
    float4 *sggeom = reinterpret_cast<float4 *>(smem_raw + L.ggeom);  // [Gc] group spheres
    unsigned *vdv = reinterpret_cast<unsigned *>(smem_raw + L.vdv);   // [Kc] Dist_v bits = max Dist_p in the voxel (Eq. 30)
    int2 *sseg = reinterpret_cast<int2 *>(smem_raw + L.seg);          // [Kc] {first point, count} of the voxel's segment
    int *sloc = reinterpret_cast<int *>(smem_raw + L.loc);            // [Kc] first point in this CTA's resident copy, or -1
    int *gpre = reinterpret_cast<int *>(smem_raw + L.gpre);           // [Gc+1] resident points before group gl
    float *svthr = reinterpret_cast<float *>(smem_raw + L.vthr);      // [Kc] prune threshold of the voxel (from its key and radius)
    float *sgthr = reinterpret_cast<float *>(smem_raw + L.gthr);      // [Gc] prune threshold of the group (from the largest key in it)
    float4 *bpick = reinterpret_cast<float4 *>(smem_raw + L.bpick);   // [PB] picks of the current batch
    float *cX = reinterpret_cast<float *>(smem_raw + L.cand), *cY = cX + TC, *cZ = cY + TC, *cD = cZ + TC;
    unsigned *cO = reinterpret_cast<unsigned *>(cD + TC);
    Ctl *ctl = reinterpret_cast<Ctl *>(smem_raw + L.ctl);
    uint4 *wbest = reinterpret_cast<uint4 *>(smem_raw + L.wbest);
    uint2 *lslot = reinterpret_cast<uint2 *>(smem_raw + L.lslot);
    HierSmem *hs = reinterpret_cast<HierSmem *>(smem_raw + L.hier);
    int *qkl = reinterpret_cast<int *>(smem_raw + L.qkl);             // [Kc] queued voxel slots
    unsigned *qmask = reinterpret_cast<unsigned *>(smem_raw + L.qmask);   // [Kc][SUBW] surviving picks per voxel slot (zero when not queued)
    unsigned *qbits = reinterpret_cast<unsigned *>(smem_raw + L.qbits);   // [Gc] voxel-slot-already-queued bits
    int *qn = reinterpret_cast<int *>(smem_raw + L.qn);               // [0..1] queue length (double-buffered), [2] pop counter

    // this cloud: points [po, po + Nb), Mb samples from start point startb, outputs at obase
    const size_t po = (size_t)P.poff[b], vo = (size_t)b * P.K_cap;
    const int Nb = P.poff[b + 1] - P.poff[b];
    const int Mb = P.rag ? P.rag[b] : P.M;
    const int startb = P.rag ? P.rag[(P.B + 1) + b] : P.start_idx;
    const size_t obase = P.rag ? (size_t)P.rag[2 * (P.B + 1) + b] : (size_t)b * P.M;
    const float *__restrict__ px = P.px + po;
    const float *__restrict__ py = P.py + po;
    const float *__restrict__ pz = P.pz + po;
    const int *__restrict__ porig = P.porig + po;
    float *Dp = P.Dp + po;
    const float4 *__restrict__ vgeom = P.vgeom + vo;
    const float4 *__restrict__ ggeom = P.ggeom + (size_t)b * P.G_cap;
    const int2 *__restrict__ vseg = P.vseg + vo;
    int *out_idx = P.out_idx + obase;
    float *out_mind = P.out_mind + obase;
    const int K = P.K[b];
    const int G = (K + 31) / 32;
    // roles: with C > 1 CTA 0 is the PICKER (candidate-set FPS, owns no voxel) and CTAs 1..C-1 are the
    // WORKERS (own the voxels; apply the picks WHILE the picker is still producing them).  C == 1: both.
    const bool split = C > 1;
    const int W = split ? C - 1 : 1, wr = split ? rank - 1 : 0;
    const bool worker = !split || rank > 0;
    const int Gc = (worker && G > wr) ? (G - wr + W - 1) / W : 0;   // groups owned by this CTA
    const int Kc = Gc * 32;                                         // voxel slots of this CTA (some may be empty)
#define RFPS_VOXEL_OF(kl) ((wr + W * ((kl) >> 5)) * 32 + ((kl) & 31))

    // ---- a7: state reset.  Thresholds = NaN: nothing can be pruned by the first pick, which therefore
    // performs the paper's "initial update" (Eq. 13-14).  Dist_p = +inf (below, with the resident copy). ----
    for (int kl = tid; kl < Kc; kl += BT) {
        const int k = RFPS_VOXEL_OF(kl);
        sgeom[kl] = k < K ? vgeom[k] : make_float4(0.f, 0.f, 0.f, 0.f);
        sseg[kl] = k < K ? vseg[k] : make_int2(0, 0);
        // not visited yet: Dist_v = NaN, whose prune threshold is NaN ("d2 >= NaN" is false: visit).  Every
        // voxel is visited by the first pick, so no NaN survives round 1.  Empty slot: Dist_v = 0, below
        // every live distance, threshold 0 ("d2 >= 0" always prunes)
        vdv[kl] = k < K ? F32_NAN_BITS : 0u;
        svthr[kl] = k < K ? __uint_as_float(F32_NAN_BITS) : 0.0f;
    }
    for (int gl = tid; gl < Gc; gl += BT) { sggeom[gl] = ggeom[wr + W * gl]; qbits[gl] = 0u; sgthr[gl] = __uint_as_float(F32_NAN_BITS); }
    for (int i = tid; i < Kc * SUBW; i += BT) qmask[i] = 0u;
    // ---- resident points.  The points of a group of 32 consecutive voxels are one contiguous run of the sorted
    // arrays; the runs of the groups this CTA owns are copied one after the other into what is left of its shared
    // memory -- as many whole groups as fit, the rest is read from global memory (L2) as before.  x, y, z and
    // Dist_p only: the original index is needed for candidates and for exact ties of the global maximum, both
    // rare, and stays in global memory. ----
    float *const sPX = reinterpret_cast<float *>(smem_raw + (split ? L.picker : L.pts));
    const int pts_cap = worker ? (int)(((size_t)P.smem_bytes - (split ? L.picker : L.pts)) / 16) : 0;
    float *const sPY = sPX + pts_cap, *const sPZ = sPY + pts_cap, *const sPD = sPZ + pts_cap;
    __syncthreads();
    if (warp == 0) {
        // exclusive prefix of the groups' point counts (a group's run ends where the next group's starts; Gc is small)
        int carry = 0;
        for (int base = 0; base < Gc; base += 32) {
            const int gl = base + lane;
            int len = 0;
            if (gl < Gc) {
                int s = 0;
                for (int l = 0; l < 32; ++l) s += sseg[gl * 32 + l].y;
                len = s;
            }
            int incl = len;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(FULL, incl, o);
                if (lane >= o) incl += t;
            }
            if (gl < Gc) gpre[gl] = carry + incl - len;
            carry += __shfl_sync(FULL, incl, 31);
        }
        if (lane == 0) gpre[Gc] = carry;
    }
    __syncthreads();
    // groups 0 .. Gres-1 are resident (the prefix is monotone; Gc < BT because the voxel state has to fit as well)
    const int Gres = __syncthreads_count(tid < Gc && gpre[tid + 1] <= pts_cap);
    for (int kl = tid; kl < Kc; kl += BT) {
        const int gl = kl >> 5;
        sloc[kl] = gl < Gres ? gpre[gl] + (sseg[kl].x - sseg[gl * 32].x) : -1;
    }
    {
        const int nres = Gres > 0 ? gpre[Gres] : 0;
        const float inf = __uint_as_float(F32_INF_BITS);
        int gl = 0;
        for (int q = tid; q < nres; q += BT) {          // coalesced: consecutive q are consecutive sorted points
            while (q >= gpre[gl + 1]) ++gl;
            const int p = sseg[gl * 32].x + (q - gpre[gl]);
            sPX[q] = px[p];
            sPY[q] = py[p];
            sPZ[q] = pz[p];
            sPD[q] = inf;
        }
        // Dist_p of the groups that stay in global memory: only this CTA ever touches them
        for (int gl2 = Gres; gl2 < Gc; ++gl2) {
            const int p0 = sseg[gl2 * 32].x, len = gpre[gl2 + 1] - gpre[gl2];
            for (int q = tid; q < len; q += BT) Dp[p0 + q] = inf;
        }
    }
    // exchange block of this cloud as seen from here (sample_batched_shapes.h)
    unsigned char *const gxb = GRID ? P.gx + (size_t)b * gx_bytes(TC) : nullptr;
    float4 *const gpick = GRID ? reinterpret_cast<float4 *>(gxb + GX_PICK) : nullptr;
    float *const gcand = GRID ? reinterpret_cast<float *>(gxb + gx_cand()) : nullptr;
    const unsigned ctl0 = GRID ? 0u : mapa(smem_u32(ctl), 0u);          // cluster: the picker's control block
    if (tid == 0) {
        qn[0] = qn[1] = qn[2] = qn[3] = 0;
        ctl->pub = 0u; ctl->cmd = 0u; ctl->cmd_tb = 0u; ctl->ack = 0u;
#pragma unroll
        for (int a = 0; a < 8; ++a) ctl->ccount[a] = 0u;
        ctl->cmd_after = 0u; ctl->best_lo = 0u;
        const int p = P.pinv[po + startb];
        bpick[0] = make_float4(px[p], py[p], pz[p], 0.0f);     // s_0 = the caller's start point
        if (rank == 0) {
            out_idx[0] = startb;
            out_mind[0] = __uint_as_float(F32_INF_BITS);
        }
    }
    int nb = 1, j = 1;
    unsigned qpar = 0u, prev_taubits = 0u;
    bool prev_tau_valid = false;
    float g = 0.25f;                 // tau = Dmax * (1 - g); adapted from the candidate counts
    float gt = GTARGET;              // fraction of the candidate buffer the next extraction aims at; follows the overflow rate
    unsigned long long c_vtest = 0, c_vvisit = 0, c_pvisit = 0, c_pcomp = 0, c_eff = 0, c_rounds = 0, c_retries = 0,
                       c_singles = 0, c_cands = 0, c_xvox = 0, c_xpts = 0, c_gtest = 0, c_subrounds = 0, c_fallback = 0;
    long long t_apply = 0, t_max = 0, t_extract = 0, t_local = 0, t0 = 0, t1 = 0;   // CTA 0 / thread 0, SM cycles
    long long t_lpairs = 0, t_lpub = 0;                                      // parallel resolution: all-pairs part of the pick time / publishing
    long long t_lsel = 0, t_lpick = 0, t_lupd = 0;                          // local phase: selection / pick loop / update after it
    long long t_a = 0, t_b = 0, ta0 = 0, n_subs = 0;                        // every CTA / thread 0
    long long t_wtail = 0, t_wx = 0, t_widle = 0, tw0 = 0;                  // workers / thread 0: applying what is left when a batch is
                                                                            // declared complete, extraction scans, waiting for messages
    // Dist_p = +inf and the control blocks are in place before any message is sent (grid mode: the global exchange
    // block was zeroed by the host, and nothing a CTA writes before its first message is read by another CTA)
    if (GRID) {
        __syncthreads();
    } else cluster_sync_all();

    // =====================================================================================
    // APPLY: the picks bpick[lo, hi), SUBP (= 128) at a time (whole CTA; contains CTA barriers).
        //   phase A  one warp per group of 32 voxels: lane i tests picks i, i+32, .. against the group
        //            sphere (Dist_v := max over the group's voxels), then lane l tests voxel l against
        //            the survivors; voxels with survivors are queued with their pick mask
        //   phase B  warps pop queued voxels (dynamic) and walk their points once for all surviving picks
        // =====================================================================================
    // ---- a10-a12 for one voxel: point skip, update, voxel key + thresholds.  Called by a whole warp; vmask =
    // the picks bpick[sub + 32*w + i] whose bit i of word w is set ----
    auto visit = [&](const int kl, const unsigned (&vmask)[SUBW], const int sub) {
            const int2 sg = sseg[kl];
            const int lo = sloc[kl];
            // the voxel's points: this CTA's resident copy, or the sorted global arrays (generic pointers)
            const float *X = lo >= 0 ? sPX + lo : px + sg.x, *Y = lo >= 0 ? sPY + lo : py + sg.x, *Z = lo >= 0 ? sPZ + lo : pz + sg.x;
            float *Dq = lo >= 0 ? sPD + lo : Dp + sg.x;
            float bestD = -1.0f;
            int npk = 0;
#pragma unroll
            for (int w = 0; w < SUBW; ++w) npk += __popc(vmask[w]);
            // two chunks of 32 points per step: both chunks' loads are in flight together
            for (int pb = 0; pb < sg.y; pb += 64) {
                const int pA = pb + lane, pB = pb + 32 + lane;
                const bool inA = pA < sg.y, inB = pB < sg.y;
                float xA = 0.f, yA = 0.f, zA = 0.f, DA0 = -1.0f, xB = 0.f, yB = 0.f, zB = 0.f, DB0 = -1.0f;
                if (inA) { xA = X[pA]; yA = Y[pA]; zA = Z[pA]; DA0 = Dq[pA]; }
                if (inB) { xB = X[pB]; yB = Y[pB]; zB = Z[pB]; DB0 = Dq[pB]; }
                float DA = DA0, DB = DB0;
#pragma unroll
                for (int w = 0; w < SUBW; ++w) {
                    unsigned m = vmask[w];
                    while (m) {
                        const int i = __ffs(m) - 1;
                        m &= m - 1u;
                        const float4 s = bpick[sub + 32 * w + i];
                        {
                            const float dx = __fsub_rn(xA, s.x), dy = __fsub_rn(yA, s.y), dz = __fsub_rn(zA, s.z);
                            const float dx2 = __fmul_rn(dx, dx), dy2 = __fmul_rn(dy, dy), dz2 = __fmul_rn(dz, dz);
                            // Eq. 28: squared domain, or literally |dx| >= D in the Euclidean mode (sqrt_rn(fl(dx*dx)) == |dx|)
                            if (no_skip || !(EUC ? (fabsf(dx) >= DA || fabsf(dy) >= DA || fabsf(dz) >= DA) : (dx2 >= DA || dy2 >= DA || dz2 >= DA))) {
                                const float d = distf<EUC>(__fadd_rn(__fadd_rn(dx2, dy2), dz2));
                                if (STATS && inA) c_pcomp++;
                                if (d < DA) {                                          // Eq. 29 / Eq. 2 (strict)
                                    DA = d;
                                    if (STATS) c_eff++;
                                }
                            }
                        }
                        {
                            const float dx = __fsub_rn(xB, s.x), dy = __fsub_rn(yB, s.y), dz = __fsub_rn(zB, s.z);
                            const float dx2 = __fmul_rn(dx, dx), dy2 = __fmul_rn(dy, dy), dz2 = __fmul_rn(dz, dz);
                            if (no_skip || !(EUC ? (fabsf(dx) >= DB || fabsf(dy) >= DB || fabsf(dz) >= DB) : (dx2 >= DB || dy2 >= DB || dz2 >= DB))) {
                                const float d = distf<EUC>(__fadd_rn(__fadd_rn(dx2, dy2), dz2));
                                if (STATS && inB) c_pcomp++;
                                if (d < DB) {
                                    DB = d;
                                    if (STATS) c_eff++;
                                }
                            }
                        }
                    }
                }
                if (DA < DA0) Dq[pA] = DA;
                if (DB < DB0) Dq[pB] = DB;
                if (STATS) c_pvisit += (inA ? npk : 0) + (inB ? npk : 0);
                // absent lanes carry D = -1 (< every real distance)
                bestD = fmaxf(bestD, fmaxf(DA, DB));
            }
            // a12: Dist_v = max Dist_p of the voxel (Eq. 30).  Which point attains it -- the lowest original index
            // among them, PAPER.md:179 -- is only needed when the voxel holds the global maximum in a round without
            // candidates; compute_max looks it up then
            const unsigned mhi = __reduce_max_sync(FULL, bestD >= 0.0f ? __float_as_uint(bestD) : 0u);
            if (lane == 0) {
                vdv[kl] = mhi;
                svthr[kl] = EUC ? prune_threshold_euc(mhi, sgeom[kl].w) : prune_threshold(mhi, sgeom[kl].w);
                if (STATS) c_vvisit++;
            }
            __syncwarp();
            // refresh the group threshold.  A concurrent visit to another voxel of the group may make this
            // read one stale (larger) Dist_v: the threshold then errs on the conservative side
            {
                const int gl = kl >> 5;
                const unsigned dvg = __reduce_max_sync(FULL, vdv[gl * 32 + lane]);
                if (lane == 0) sgthr[gl] = EUC ? prune_threshold_euc(dvg, sggeom[gl].w) : prune_threshold(dvg, sggeom[gl].w);
            }
    };

    auto apply_range = [&](const int lo, const int hi) {
        for (int sub = lo; sub < hi; sub += SUBP) {
            const int nsub = min(SUBP, hi - sub);
            if (STATS && tid == 0) { ta0 = clock64(); n_subs++; }
            // ---- a9: radius prune (Eq. 25), two levels.  Work unit = (group, word of 32 picks), spread over
            // the warps so that a group whose sphere prunes badly does not serialise on one warp ----
            const int nw = (nsub + 31) >> 5;
            for (int u = warp; u < Gc * nw; u += NW) {
                const int gl = u / nw, w = u - gl * nw;
                const int kl = gl * 32 + lane;
                const bool valid = RFPS_VOXEL_OF(kl) < K;
                const int n = min(32, nsub - 32 * w);
                unsigned mask = 0u;
                if (no_prune) {
                    mask = valid ? (n == 32 ? FULL : ((1u << n) - 1u)) : 0u;
                    if (STATS && valid) c_vtest += n;
                } else {
                    // thresholds are kept current by the visits (phase B): group threshold from Dist_v := max
                    // over the group, voxel threshold from its own Dist_v (NaN = not visited yet: never pruned)
                    const float4 gg = sggeom[gl];
                    const float thr_g = sgthr[gl];
                    bool gs = false;
                    if (lane < n) {
                        const float4 s = bpick[sub + 32 * w + lane];
                        gs = !(d2_rn(gg.x, gg.y, gg.z, s.x, s.y, s.z) >= thr_g);
                    }
                    unsigned gmask = __ballot_sync(FULL, gs);
                    if (STATS && lane == 0) c_gtest += n;
                    if (gmask) {
                        const float4 gm = sgeom[kl];
                        const float thr = svthr[kl];
                        if (STATS && valid) c_vtest += __popc(gmask);
                        while (gmask) {
                            const int i = __ffs(gmask) - 1;
                            gmask &= gmask - 1u;
                            const float4 s = bpick[sub + 32 * w + i];
                            if (!(d2_rn(gm.x, gm.y, gm.z, s.x, s.y, s.z) >= thr)) mask |= 1u << i;
                        }
                    }
                }
                const unsigned bal = __ballot_sync(FULL, mask != 0u);
                if (bal) {
                    if (mask) qmask[kl * SUBW + w] = mask;
                    // the first unit that finds survivors for a voxel queues it (one bit per voxel slot)
                    unsigned old = 0u;
                    if (lane == 0) old = atomicOr(&qbits[gl], bal);
                    old = __shfl_sync(FULL, old, 0);
                    const unsigned fresh = bal & ~old;
                    if (fresh) {
                        int qb = 0;
                        if (lane == 0) qb = atomicAdd(&qn[qpar], __popc(fresh));
                        qb = __shfl_sync(FULL, qb, 0);
                        if (fresh & (1u << lane)) qkl[qb + __popc(fresh & lt)] = kl;
                    }
                }
            }
            __syncthreads();
            const int nq = qn[qpar];
            if (tid == 0) { qn[qpar ^ 1u] = 0; qn[2] = 0; }
            for (int gl = tid; gl < Gc; gl += BT) qbits[gl] = 0u;
            if (STATS && tid == 0) { const long long t = clock64(); t_a += t - ta0; ta0 = t; }
            __syncthreads();
            // ---- a10-a12: point skip, update, voxel key + threshold; one warp per queued voxel ----
            for (;;) {
                int qi = 0;
                if (lane == 0) qi = atomicAdd(&qn[2], 1);
                qi = __shfl_sync(FULL, qi, 0);
                if (qi >= nq) break;
                const int kl = qkl[qi];
                unsigned vmask[SUBW];
                {
                    const uint4 qm = *reinterpret_cast<const uint4 *>(&qmask[kl * SUBW]);
                    vmask[0] = qm.x; vmask[1] = qm.y; vmask[2] = qm.z; vmask[3] = qm.w;
                    __syncwarp();
                    if (lane == 0) *reinterpret_cast<uint4 *>(&qmask[kl * SUBW]) = make_uint4(0u, 0u, 0u, 0u);   // leave it clean
                }
                visit(kl, vmask, sub);
            }
            __syncthreads();
            qpar ^= 1u;
            if (STATS && tid == 0) t_b += clock64() - ta0;
        }
    };

    // ---- a8 on this CTA's voxels: max Dist_v and, among the points attaining it, the lowest original index
    // (PAPER.md:179), as one 64-bit key (Dist_v bits << 32 | ~orig).  The voxels keep Dist_v only; the index is
    // looked up here, in the voxels that hold the maximum (normally one) -- also when the maximum is +0
    // (duplicates exhausted, reading A7: every point ties and the lowest index is the answer; empty slots hold
    // Dist_v = 0 too, with no points).  Whole CTA; the result is valid in thread 0. ----
    auto cta_best_key = [&]() -> unsigned long long {
        {
            unsigned bhi = 0u;
            for (int kl = tid; kl < Kc; kl += BT) bhi = max(bhi, vdv[kl]);
            bhi = __reduce_max_sync(FULL, bhi);
            if (lane == 0) wbest[warp].x = bhi;
            if (tid == 0) ctl->best_lo = 0u;
        }
        __syncthreads();
        const unsigned chi = __reduce_max_sync(FULL, lane < NW ? wbest[lane].x : 0u);
        unsigned bo = 0u;
        for (int kl = warp; kl < Kc; kl += NW) {
            if (vdv[kl] != chi) continue;                                 // warp-uniform
            const int2 sg = sseg[kl];
            const int lo = sloc[kl];
            const float *Dq = lo >= 0 ? sPD + lo : Dp + sg.x;
            for (int p = lane; p < sg.y; p += 32)
                if (__float_as_uint(Dq[p]) == chi) bo = max(bo, ~(unsigned)porig[sg.x + p]);
        }
        bo = __reduce_max_sync(FULL, bo);
        if (lane == 0 && bo) atomicMax(&ctl->best_lo, bo);
        __syncthreads();
        return ((unsigned long long)chi << 32) | ctl->best_lo;
    };

    // ---- candidates {p : Dist_p > tb} of this CTA's voxels -> the cloud's candidate buffer.  reserve(n) hands out
    // n consecutive slots (it may run past the buffer: the count then says "too many"); store(slot, ...) writes one
    // candidate.  Whole CTA. ----
    auto extract_scan = [&](const unsigned tb, auto reserve, auto store) {
        for (int base = 0; base < Kc; base += BT) {
            const int kl = base + tid;
            const bool hit = kl < Kc && vdv[kl] > tb;                     // empty slots hold 0
            const unsigned bal = __ballot_sync(FULL, hit);
            if (bal) {
                int qb = 0;
                if (lane == 0) qb = atomicAdd(&qn[qpar], __popc(bal));
                qb = __shfl_sync(FULL, qb, 0);
                if (hit) qkl[qb + __popc(bal & lt)] = kl;
            }
        }
        __syncthreads();
        const int nq = qn[qpar];
        if (tid == 0) { qn[qpar ^ 1u] = 0; qn[2] = 0; }
        __syncthreads();
        for (;;) {
            int qi = 0;
            if (lane == 0) qi = atomicAdd(&qn[2], 1);
            qi = __shfl_sync(FULL, qi, 0);
            if (qi >= nq) break;
            const int kq = qkl[qi];
            const int2 sg = sseg[kq];
            const int lo = sloc[kq];
            const float *X = lo >= 0 ? sPX + lo : px + sg.x, *Y = lo >= 0 ? sPY + lo : py + sg.x, *Z = lo >= 0 ? sPZ + lo : pz + sg.x;
            const float *Dq = lo >= 0 ? sPD + lo : Dp + sg.x;
            if (STATS && lane == 0) c_xvox++;
            // two chunks of 32 points per step, everything loaded up front, one slot reservation per step; the
            // original index (global memory) is fetched for the hits only
            for (int pb = 0; pb < sg.y; pb += 64) {
                const int pA = pb + lane, pB = pb + 32 + lane;
                const bool inA = pA < sg.y, inB = pB < sg.y;
                unsigned dA = 0u, dB = 0u, oA = 0u, oB = 0u;
                float xA = 0.f, yA = 0.f, zA = 0.f, xB = 0.f, yB = 0.f, zB = 0.f;
                if (inA) { dA = __float_as_uint(Dq[pA]); xA = X[pA]; yA = Y[pA]; zA = Z[pA]; }
                if (inB) { dB = __float_as_uint(Dq[pB]); xB = X[pB]; yB = Y[pB]; zB = Z[pB]; }
                const bool isA = dA > tb, isB = dB > tb;
                if (isA) oA = ~(unsigned)porig[sg.x + pA];
                if (isB) oB = ~(unsigned)porig[sg.x + pB];
                const unsigned balA = __ballot_sync(FULL, isA), balB = __ballot_sync(FULL, isB);
                if (STATS) c_xpts += (inA ? 1 : 0) + (inB ? 1 : 0);
                if (balA | balB) {
                    unsigned cb = 0u;
                    if (lane == 0) cb = reserve((unsigned)(__popc(balA) + __popc(balB)));
                    cb = __shfl_sync(FULL, cb, 0);
                    const unsigned slotA = cb + (unsigned)__popc(balA & lt);
                    const unsigned slotB = cb + (unsigned)__popc(balA) + (unsigned)__popc(balB & lt);
                    if (isA && slotA < (unsigned)TC) store(slotA, xA, yA, zA, dA, oA);
                    if (isB && slotB < (unsigned)TC) store(slotB, xB, yB, zB, dB, oB);
                }
            }
        }
        qpar ^= 1u;
        __syncthreads();
    };

    // ---- threshold control shared by the solo and the picker loop: tau = Dmax * (1 - g), g follows the counts ----
    auto next_threshold = [&](const unsigned gref, const int attempt) -> unsigned {
        // a cloud that fits the candidate buffer whole is taken whole (tau = 0: every point that can still be
        // picked at a positive distance); the local phase then runs without global rounds
        return (attempt == 0 && Nb <= TC) ? 0u : __float_as_uint(__fmul_rn(__uint_as_float(gref), __fsub_rn(1.0f, g)));
    };
    auto adapt_fit = [&](const unsigned found) {          // aim the next round at ~5/8 of the buffer; move by at most 2x
        const float ratio = fminf(2.0f, fmaxf(0.5f, (gt * TC) / (float)max(found, 1u)));
        g = fminf(0.75f, fmaxf(0x1p-22f, g * ratio));
        gt = fminf(GT_MAX, gt * GT_UP);
    };
    auto adapt_overflow = [&](const unsigned found) {
        g = fmaxf(0x1p-22f, g * fmaxf(0.125f, (0.5f * TC) / (float)found));
        gt = fmaxf(GT_MIN, gt * GT_DOWN);
    };
    // ---- LOCAL: FPS restricted to the candidates (whole CTA); returns through j / nb ----
    auto run_local = [&](const int cnt, const unsigned taubits, int &lj, int &lnb, const Publisher &pubr) {
        if constexpr (LW == LW_PAR) {
            local_fps_par<CPT, STATS, EUC>(cX, cY, cZ, cD, cO, (TC <= 2048 ? reinterpret_cast<float *>(smem_raw + L.cand2) : nullptr), cnt, taubits, lj,
                                           lnb, Mb, reinterpret_cast<ParSmem *>(hs), bpick, out_idx,
                                           out_mind, tid, c_subrounds, c_fallback, t_lsel, t_lpick, t_lupd, t_lpairs, t_lpub, pubr);
        } else if constexpr (LW == LW_HIER) {
            local_fps_hier<CPT, CPT2, STATS, EUC>(cX, cY, cZ, cD, cO, cnt, taubits, lj, lnb, Mb, hs, bpick, out_idx, out_mind, tid,
                                                  c_subrounds, c_fallback, t_lsel, t_lpick, t_lupd, pubr);
        } else if constexpr (!EUC) {
            if (warp < LW) local_fps<CPT, LW>(cX, cY, cZ, cD, cO, cnt, taubits, lj, lnb, Mb, lslot, bpick, out_idx, out_mind, tid);
            if (tid == 0) { ctl->scratch[0] = lj; ctl->scratch[1] = lnb; }      // the other warps learn the outcome
            __syncthreads();
            lj = ctl->scratch[0];
            lnb = ctl->scratch[1];
            __syncthreads();
        }
        if (STATS && tid == 0) c_cands += (unsigned long long)cnt;
    };

    if (!split) {
        // =====================================================================================
        // ONE CTA per cloud: apply, argmax, extract and local phase in turn
        // =====================================================================================
        apply_range(0, 1);      // the start point: every voxel is visited (the paper's initial update, Eq. 13-14)
        while (j < Mb) {
            if (STATS && tid == 0) { c_rounds++; t0 = clock64(); }
            unsigned ghi = 0u, glo = 0u;
            bool have_max = false;
            int cnt = 0;
            unsigned taubits = 0u;
            // A batch that ended on its threshold leaves every point of the cloud <= tau_prev, and the true maximum
            // just below it: tau is hung on tau_prev and the argmax is only computed when that fails -- no candidate
            // above the new tau, or too many -- or when there is no such threshold (first round, batch cut short)
            for (int pass = prev_tau_valid ? 0 : 1; pass < 2 && cnt == 0; ++pass) {
                if (pass == 1) {
                    const unsigned long long key = cta_best_key();
                    if (tid == 0) { ctl->scratch[0] = (int)(unsigned)(key >> 32); ctl->scratch[1] = (int)(unsigned)key; }
                    __syncthreads();
                    ghi = (unsigned)ctl->scratch[0]; glo = (unsigned)ctl->scratch[1];
                    have_max = true;
                    __syncthreads();
                }
                const unsigned gref = have_max ? ghi : prev_taubits;
                taubits = gref;
                if (no_batch || !(gref > 0u && gref < F32_INF_BITS)) continue;
                for (int a = 0; a < MAX_ATTEMPTS; ++a) {
                    const unsigned tb = next_threshold(gref, a);
                    if (!(tb < gref)) break;                     // g too small to separate tau from Dmax
                    if (tid == 0) ctl->ccount[0] = 0u;
                    __syncthreads();
                    extract_scan(tb, [&](unsigned n) { return atomicAdd(&ctl->ccount[0], n); },
                                 [&](unsigned sl, float x, float y, float z, unsigned dbits, unsigned o) {
                                     cX[sl] = x; cY[sl] = y; cZ[sl] = z; cD[sl] = __uint_as_float(dbits); cO[sl] = o;
                                 });
                    const unsigned found = ctl->ccount[0];
                    __syncthreads();
                    if (found <= (unsigned)TC) { cnt = (int)found; taubits = tb; adapt_fit(found); break; }
                    if (STATS && tid == 0) c_retries++;
                    adapt_overflow(found);
                }
            }
            if (STATS && tid == 0) { t1 = clock64(); t_extract += t1 - t0; t0 = t1; }
            if (cnt == 0) {                              // the single global argmax = the paper's own iteration
                if (tid == 0) {
                    out_idx[j] = (int)(~glo);
                    out_mind[j] = __uint_as_float(ghi);
                    const int gpos = P.pinv[po + (size_t)(~glo)];
                    bpick[0] = make_float4(px[gpos], py[gpos], pz[gpos], 0.0f);
                    if (STATS) c_singles++;
                }
                nb = 1;
                j += 1;
            } else {
                int lj = j, lnb = 0;
                run_local(cnt, taubits, lj, lnb, Publisher());
                j = lj;
                nb = lnb;
            }
            __syncthreads();
            if (STATS && tid == 0) { t1 = clock64(); t_local += t1 - t0; t0 = t1; }
            prev_tau_valid = cnt > 0 && nb < PB && j < Mb && !no_batch;
            prev_taubits = taubits;
            if (j < Mb) {
                apply_range(0, nb);
                if (STATS && tid == 0) t_apply += clock64() - t0;
            }
        }
    } else if (rank == 0) {
        // =====================================================================================
        // PICKER: decides the rounds.  Between two batches it sends commands (argmax, candidate extraction at a
        // threshold) and waits for every worker's acknowledgement; then it runs the local phase, publishing the
        // picks as they are produced.  It never waits for a batch to be applied: the workers answer the next
        // command only after they have applied the whole batch before it.
        // =====================================================================================
        unsigned ncmd = 0u, batch = 0u, cur_cmd = 0u, cur_pub = 0u;
        unsigned long long *const gpc = reinterpret_cast<unsigned long long *>(gxb + GX_PC), *const gctb = reinterpret_cast<unsigned long long *>(gxb + GX_CTB),
                           *const gac = reinterpret_cast<unsigned long long *>(gxb + GX_AC);
        auto pub_word = [&](const unsigned v) {            // thread 0
            cur_pub = v;
            if (GRID) st_release_gpu_u64(gpc, ((unsigned long long)cur_cmd << 32) | v);
            else st_release_cluster_u32(smem_u32(&ctl->pub), v);
        };
        // one command: send (thread 0), wait for W acknowledgements, fetch the result, broadcast
        auto send = [&](const unsigned type, const unsigned tb) {
            ++ncmd;
            cur_cmd = (ncmd << 2) | type;
            if (tid == 0) {
                if (GRID) {
                    // nobody touches the count / acknowledgement word between two commands: a plain store resets the count
                    *reinterpret_cast<volatile unsigned long long *>(gac) = (unsigned long long)((ncmd - 1u) * (unsigned)W) << 32;
                    *reinterpret_cast<volatile unsigned long long *>(gctb) =
                        ((unsigned long long)(((batch & 0xffffu) << 16) | (ncmd & 0xffffu)) << 32) | tb;
                    st_release_gpu_u64(gpc, ((unsigned long long)cur_cmd << 32) | cur_pub);
                } else {
                    ctl->ccount[ncmd & 7u] = 0u;
                    ctl->cmd_tb = tb;
                    ctl->cmd_after = batch;
                    st_release_cluster_u32(smem_u32(&ctl->cmd), cur_cmd);
                }
            }
        };
        auto wait = [&](const unsigned type, unsigned &r0, unsigned &r1) {
            if (tid == 0) {
                const unsigned want = ncmd * (unsigned)W;
                if (GRID) {
                    unsigned long long ac;
                    while ((unsigned)((ac = ld_acquire_gpu_u64(gac)) >> 32) != want) __nanosleep(20);
                    if (type == CMD_EXTRACT) ctl->scratch[0] = (int)(unsigned)ac;
                } else {
                    while (ld_acquire_cluster_local_u32(smem_u32(&ctl->ack)) != want) __nanosleep(20);
                    if (type == CMD_EXTRACT) ctl->scratch[0] = (int)*reinterpret_cast<volatile unsigned *>(&ctl->ccount[ncmd & 7u]);
                }
            }
            __syncthreads();                               // thread 0's acquire now covers the whole CTA
            if (type == CMD_MAX && warp == 0) {            // argmax over the workers' slots (Eq. 15-18, last level)
                unsigned khi = 0u, klo = 0u;
                for (int r = 1 + lane; r < C; r += 32) {
                    const uint2 k = GRID ? __ldcg(reinterpret_cast<const uint2 *>(gxb + GX_SLOT) + r) : ctl->slot[r];
                    if (k.x > khi || (k.x == khi && k.y > klo)) { khi = k.x; klo = k.y; }
                }
                unsigned mhi, mlo;
                warp_argmax_key(khi, klo, mhi, mlo);
                if (lane == 0) { ctl->scratch[0] = (int)mhi; ctl->scratch[1] = (int)mlo; }
            }
            if (type == CMD_MAX) __syncthreads();
            r0 = (unsigned)ctl->scratch[0]; r1 = (unsigned)ctl->scratch[1];
            __syncthreads();
        };
        auto command = [&](const unsigned type, const unsigned tb, unsigned &r0, unsigned &r1) {
            send(type, tb);
            wait(type, r0, r1);
        };
        if (tid == 0) {                                    // batch 0 = the start point: every voxel is visited
            if (GRID) gpick[0] = bpick[0];
            pub_word(1u | PUB_DONE | (Mb <= 1 ? PUB_FINAL : 0u));
        }
        while (j < Mb) {
            if (STATS && tid == 0) { c_rounds++; t0 = clock64(); }
            unsigned ghi = 0u, glo = 0u;
            bool have_max = false;
            int cnt = 0;
            unsigned taubits = 0u;
            for (int pass = prev_tau_valid ? 0 : 1; pass < 2 && cnt == 0; ++pass) {
                if (pass == 1) {
                    command(CMD_MAX, 0u, ghi, glo);
                    have_max = true;
                    if (STATS && tid == 0) { t1 = clock64(); t_max += t1 - t0; t0 = t1; }
                }
                const unsigned gref = have_max ? ghi : prev_taubits;
                taubits = gref;
                if (no_batch || !(gref > 0u && gref < F32_INF_BITS)) continue;
                for (int a = 0; a < MAX_ATTEMPTS; ++a) {
                    const unsigned tb = next_threshold(gref, a);
                    if (!(tb < gref)) break;
                    unsigned found, dummy;
                    command(CMD_EXTRACT, tb, found, dummy);
                    if (found <= (unsigned)TC) { cnt = (int)found; taubits = tb; adapt_fit(found); break; }
                    if (STATS && tid == 0) c_retries++;
                    adapt_overflow(found);
                }
            }
            if (GRID && cnt > 0) {                         // candidates: global exchange block -> shared memory
                for (int i = tid; i < cnt; i += BT) {
                    cX[i] = __ldcg(gcand + i); cY[i] = __ldcg(gcand + TC + i); cZ[i] = __ldcg(gcand + 2 * TC + i);
                    cD[i] = __ldcg(gcand + 3 * TC + i); cO[i] = __float_as_uint(__ldcg(gcand + 4 * TC + i));
                }
                __syncthreads();
            }
            if (STATS && tid == 0) { t1 = clock64(); t_extract += t1 - t0; t0 = t1; }
            ++batch;
            Publisher pubr;
            pubr.base = (batch & 0x7ffffu) << PUB_SHIFT;
            if (GRID) { pubr.gptr = gpc; pubr.cmd_hi = cur_cmd; pubr.gpick = gpick; }
            else pubr.local_addr = smem_u32(&ctl->pub);
            if (cnt == 0) {                              // the single global argmax = the paper's own iteration
                if (tid == 0) {
                    out_idx[j] = (int)(~glo);
                    out_mind[j] = __uint_as_float(ghi);
                    const int gpos = P.pinv[po + (size_t)(~glo)];
                    bpick[0] = make_float4(px[gpos], py[gpos], pz[gpos], 0.0f);
                    if (GRID) gpick[0] = bpick[0];
                    if (STATS) c_singles++;
                }
                nb = 1;
                j += 1;
            } else {
                int lj = j, lnb = 0;
                run_local(cnt, taubits, lj, lnb, pubr);
                j = lj;
                nb = lnb;
            }
            __syncthreads();                               // the last picks are written
            prev_tau_valid = cnt > 0 && nb < PB && j < Mb && !no_batch;
            prev_taubits = taubits;
            cur_pub = pubr.base | (unsigned)nb | PUB_DONE | (j >= Mb ? PUB_FINAL : 0u);
            if (tid == 0) pubr((unsigned)nb | PUB_DONE | (j >= Mb ? PUB_FINAL : 0u));
            if (STATS && tid == 0) { t1 = clock64(); t_local += t1 - t0; }
        }
    } else {
        // =====================================================================================
        // WORKER: owns voxels.  Applies every batch while the picker is still producing it (pieces of >=
        // STREAM_MIN picks), then answers the picker's commands -- always after the whole batch before them.
        // =====================================================================================
        unsigned next_batch = 0u, next_cmd = 1u;
        int applied = 0;
        bool in_batch = true;                              // batch `next_batch` is not completely applied yet
        const unsigned pick_rc = GRID ? 0u : mapa(smem_u32(bpick), 0u);
        const unsigned cX0 = GRID ? 0u : mapa(smem_u32(cX), 0u), cY0 = GRID ? 0u : mapa(smem_u32(cY), 0u), cZ0 = GRID ? 0u : mapa(smem_u32(cZ), 0u),
                       cD0 = GRID ? 0u : mapa(smem_u32(cD), 0u), cO0 = GRID ? 0u : mapa(smem_u32(cO), 0u);
        unsigned long long *const gpc = reinterpret_cast<unsigned long long *>(gxb + GX_PC), *const gctb = reinterpret_cast<unsigned long long *>(gxb + GX_CTB),
                           *const gac = reinterpret_cast<unsigned long long *>(gxb + GX_AC);
        auto ack = [&]() {                                 // after a barrier that follows the command's last store
            if (tid == 0) {
                if (GRID) red_release_gpu_add_u64(gac, 1ull << 32);
                else red_release_cluster_add_u32(ctl0 + (unsigned)offsetof(Ctl, ack), 1u);
            }
        };
        for (;;) {
            // ---- wait for the next message (thread 0 polls, the CTA sleeps at the barrier) ----
            if (tid == 0) {
                if (STATS) tw0 = clock64();
                unsigned v, c, tbv = 0u;
                for (;;) {
                    // The command word is read BEFORE (cluster mode) or TOGETHER WITH (grid mode: one 64-bit word) the
                    // batch word: the picker finishes a batch (pub: DONE) and only then sends the next command, so a
                    // worker that sees the new command is guaranteed (acquire) to see the batch it has to apply
                    // first.  Reading pub first has a window in which the command is seen and the batch is not.
                    unsigned long long pay = 0ull;
                    if (GRID) {
                        pay = *reinterpret_cast<volatile unsigned long long *>(gctb);      // in flight together with the next load
                        const unsigned long long pc = ld_acquire_gpu_u64(gpc);
                        v = (unsigned)pc;
                        c = in_batch ? 0u : (unsigned)(pc >> 32);
                    } else {
                        c = in_batch ? 0u : ld_acquire_cluster_u32(ctl0 + (unsigned)offsetof(Ctl, cmd));
                        v = ld_acquire_cluster_u32(ctl0 + (unsigned)offsetof(Ctl, pub));
                    }
                    const bool mine = (v >> PUB_SHIFT) == (next_batch & 0x7ffffu);
                    if (mine && ((v & (PUB_DONE | PUB_FINAL)) || (int)(v & PUB_COUNT) - applied >= STREAM_MIN)) { c = 0u; break; }
                    if (!in_batch && !mine && (c >> 2) == next_cmd) {
                        // answered only when the batch it follows has been applied (it may have been sent early)
                        if (GRID) {
                            // the payload was loaded before the acquire: if its tag is not this command's, read it again
                            if ((unsigned)((pay >> 32) & 0xffffull) != (next_cmd & 0xffffu)) pay = *reinterpret_cast<volatile unsigned long long *>(gctb);
                            const unsigned after = (unsigned)(pay >> 48);
                            tbv = (unsigned)pay;
                            if (((after + 1u) & 0xffffu) == (next_batch & 0xffffu)) { v = 0u; break; }
                        } else {
                            const unsigned after = ld_dsmem_u32(ctl0 + (unsigned)offsetof(Ctl, cmd_after));
                            if (after + 1u == next_batch) { tbv = ld_dsmem_u32(ctl0 + (unsigned)offsetof(Ctl, cmd_tb)); v = 0u; break; }
                        }
                    }
                    __nanosleep(40);
                }
                if (STATS) t_widle += clock64() - tw0;
                ctl->scratch[0] = (int)v;
                ctl->scratch[1] = (int)c;
                ctl->scratch[2] = (int)tbv;
            }
            __syncthreads();
            const unsigned v = (unsigned)ctl->scratch[0], c = (unsigned)ctl->scratch[1], ctb = (unsigned)ctl->scratch[2];
            __syncthreads();
            if (c) {
                // ---- a command; the batch before it has been applied completely ----
                if ((c & 3u) == CMD_MAX) {
                    const unsigned long long key = cta_best_key();
                    if (tid == 0) {
                        const uint2 k = make_uint2((unsigned)(key >> 32), (unsigned)key);
                        if (GRID) {
                            reinterpret_cast<uint2 *>(gxb + GX_SLOT)[rank] = k;
                        } else {
                            st_dsmem_u32(ctl0 + (unsigned)offsetof(Ctl, slot) + 8u * (unsigned)rank, k.x);
                            st_dsmem_u32(ctl0 + (unsigned)offsetof(Ctl, slot) + 8u * (unsigned)rank + 4u, k.y);
                        }
                    }
                    __syncthreads();
                } else {
                    const unsigned slot = next_cmd & 7u;
                    if (STATS && tid == 0) tw0 = clock64();
                    if (GRID) {
                        extract_scan(ctb, [&](unsigned n) { return (unsigned)atomicAdd(gac, (unsigned long long)n); },
                                     [&](unsigned sl, float x, float y, float z, unsigned dbits, unsigned o) {
                                         gcand[sl] = x; gcand[TC + sl] = y; gcand[2 * TC + sl] = z;
                                         gcand[3 * TC + sl] = __uint_as_float(dbits); gcand[4 * TC + sl] = __uint_as_float(o);
                                     });
                    } else {
                        const unsigned cnt_addr = ctl0 + (unsigned)offsetof(Ctl, ccount) + 4u * slot;
                        extract_scan(ctb, [&](unsigned n) { return atom_add_dsmem_u32(cnt_addr, n); },
                                     [&](unsigned sl, float x, float y, float z, unsigned dbits, unsigned o) {
                                         st_dsmem_u32(cX0 + 4u * sl, __float_as_uint(x));
                                         st_dsmem_u32(cY0 + 4u * sl, __float_as_uint(y));
                                         st_dsmem_u32(cZ0 + 4u * sl, __float_as_uint(z));
                                         st_dsmem_u32(cD0 + 4u * sl, dbits);
                                         st_dsmem_u32(cO0 + 4u * sl, o);
                                     });
                    }
                }
                if (STATS && tid == 0 && (c & 3u) == CMD_EXTRACT) t_wx += clock64() - tw0;
                ack();                                     // (both branches end with a CTA barrier)
                ++next_cmd;
                continue;
            }
            // ---- progress of batch `next_batch` ----
            if (v & PUB_FINAL) break;                      // M reached: nothing needs these picks applied
            const int n = (int)(v & PUB_COUNT);
            const bool done = v & PUB_DONE;
            in_batch = true;
            // whole words of 32 picks, at least STREAM_MIN at a time, until the batch is complete
            const int hi = done ? n : applied + ((n - applied) & ~31);
            if (hi > applied) {
                if (STATS && tid == 0) tw0 = clock64();
                for (int i = applied + tid; i < hi; i += BT) {
                    if (GRID) {
                        bpick[i] = __ldcg(gpick + i);
                    } else {
                        const uint4 q = ld_dsmem_v4(pick_rc + 16u * (unsigned)i);
                        bpick[i] = make_float4(__uint_as_float(q.x), __uint_as_float(q.y), __uint_as_float(q.z), 0.0f);
                    }
                }
                __syncthreads();
                apply_range(applied, hi);
                applied = hi;
                if (STATS && tid == 0 && done) t_wtail += clock64() - tw0;
            }
            if (done && applied == n) { ++next_batch; applied = 0; in_batch = false; }
        }
    }

    if (STATS) {
        atomicAdd(P.counters + CNT_VTEST, c_vtest);
        atomicAdd(P.counters + CNT_VVISIT, c_vvisit);
        atomicAdd(P.counters + CNT_PVISIT, c_pvisit);
        atomicAdd(P.counters + CNT_PCOMP, c_pcomp);
        atomicAdd(P.counters + CNT_EFF, c_eff);
        atomicAdd(P.counters + CNT_XVOX, c_xvox);
        atomicAdd(P.counters + CNT_XPTS, c_xpts);
        atomicAdd(P.counters + CNT_GTEST, c_gtest);
        if (tid == 0) {
            atomicAdd(P.counters + CNT_CYC_A_SUM, (unsigned long long)t_a);
            atomicAdd(P.counters + CNT_CYC_B_SUM, (unsigned long long)t_b);
            atomicMax(P.counters + CNT_CYC_A_MAX, (unsigned long long)t_a);
            atomicMax(P.counters + CNT_CYC_B_MAX, (unsigned long long)t_b);
            atomicAdd(P.counters + CNT_W_TAIL, (unsigned long long)t_wtail);
            atomicAdd(P.counters + CNT_W_XSCAN, (unsigned long long)t_wx);
            atomicAdd(P.counters + CNT_W_IDLE, (unsigned long long)t_widle);
            if (split && rank > 0) atomicAdd(P.counters + CNT_W_PIECES, (unsigned long long)n_subs);
        }
        if (tid == 0 && rank == 0) {
            atomicAdd(P.counters + CNT_SUBS, (unsigned long long)n_subs);
            atomicAdd(P.counters + CNT_SUBROUNDS, c_subrounds);
            atomicAdd(P.counters + CNT_FALLBACK, c_fallback);
            atomicAdd(P.counters + CNT_LSEL, (unsigned long long)t_lsel);
            atomicAdd(P.counters + CNT_LPICK, (unsigned long long)t_lpick);
            atomicAdd(P.counters + CNT_LUPD, (unsigned long long)t_lupd);
            atomicAdd(P.counters + CNT_LPAIRS, (unsigned long long)t_lpairs);
            atomicAdd(P.counters + CNT_LPUB, (unsigned long long)t_lpub);
            atomicAdd(P.counters + CNT_ROUNDS, c_rounds);
            atomicAdd(P.counters + CNT_RETRIES, c_retries);
            atomicAdd(P.counters + CNT_SINGLES, c_singles);
            atomicAdd(P.counters + CNT_CANDS, c_cands);
            atomicAdd(P.counters + CNT_CYC_APPLY, (unsigned long long)t_apply);
            atomicAdd(P.counters + CNT_CYC_MAX, (unsigned long long)t_max);
            atomicAdd(P.counters + CNT_CYC_EXTRACT, (unsigned long long)t_extract);
            atomicAdd(P.counters + CNT_CYC_LOCAL, (unsigned long long)t_local);
        }
    }
    if (!GRID) cluster_sync_all();   // no CTA may exit while a peer can still read its shared memory
#undef RFPS_VOXEL_OF
}

template <int CPT, int LW, bool STATS, bool EUC, bool GRID>
static int launch_batched_one(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st)
{
    auto kern = k_fps_batched<CPT, LW, STATS, EUC, GRID>;
    // the voxel state and the picker's regions are the minimum; everything else up to the device limit holds
    // resident points (sample_batched_shapes.h)
    const size_t smem = (size_t)bp.smem_bytes;
    RFPS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (!GRID && ix.cluster_size > 8) RFPS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)(ix.B * (GRID ? ix.grid_ctas : ix.cluster_size)));
    cfg.blockDim = dim3(BT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    if (GRID) {
        // the CTAs of a cloud wait for one another's messages: all of them must be resident (checked when the
        // shape was chosen; a cooperative launch fails instead of deadlocking if they are not)
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
    } else {
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)ix.cluster_size;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
    }
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    RFPS_CUDA(cudaLaunchKernelEx(&cfg, kern, bp, ix.flags));
    return FPS_OK;
}

template <int CPT, int LW>
static int launch_batched_s(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st)
{
    const bool stats = ix.flags & FPS_FLAG_STATS;
    if constexpr (LW == LW_PAR) {           // the grid-wide exchange is built for the default local phase only
        if (ix.grid_ctas > 0) {
            if (ix.flags & FPS_FLAG_EUCLIDEAN)
                return stats ? launch_batched_one<CPT, LW, true, true, true>(bp, ix, st) : launch_batched_one<CPT, LW, false, true, true>(bp, ix, st);
            return stats ? launch_batched_one<CPT, LW, true, false, true>(bp, ix, st) : launch_batched_one<CPT, LW, false, false, true>(bp, ix, st);
        }
    }
    if constexpr (LW >= LW_HIER) {          // the Euclidean mode is built for the 16-warp local phases only
        if (ix.flags & FPS_FLAG_EUCLIDEAN)
            return stats ? launch_batched_one<CPT, LW, true, true, false>(bp, ix, st) : launch_batched_one<CPT, LW, false, true, false>(bp, ix, st);
    }
    return stats ? launch_batched_one<CPT, LW, true, false, false>(bp, ix, st) : launch_batched_one<CPT, LW, false, false, false>(bp, ix, st);
}

}  // namespace rfps
