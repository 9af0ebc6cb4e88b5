// sample_kernel.cu -- steps a7-a13 of the hot path: ONE persistent kernel runs all M-1 iterations
// of {select s_j, radius prune, point skip, fp32 min-distance update, per-voxel max, global argmax}.
//
// Paper: section 3.4 (Eq. 15-30) and the RadiusFPS-G kernels of section 4.2-4.3
// (Fusion Kernel 1 / Alg. 3; Fusion Kernel 2 / Alg. 4).  The
// paper launches two kernels per sample on an RTX 6000 Ada; here one launch covers the whole
// sequence and nothing crosses the host.
//
// Mapping (B200): one thread-block CLUSTER of C CTAs per cloud (C = 1 for small clouds: the
// "one cloud per CTA" batched mode).  CTA `rank` owns the contiguous voxel range
// [rank*Kc, (rank+1)*Kc) and the points of those voxels; only its own SM ever touches their
// Dist_p / voxel state, so they stay in that SM's L1 and the only cross-CTA traffic is one
// 32-byte candidate message per CTA per iteration.
//
// One iteration, CTA view:
//   A  every thread tests the voxels it owns (geometry + threshold in registers) against s_j:
//        pruned  iff  d2(s_j, c_k) >= thr_k                                   [Eq. 25, squared form]
//      survivors are pushed to a shared-memory queue                          -- __syncthreads
//   B  warps pull queue entries; one warp walks one voxel's points with coalesced SoA loads:
//        skip  iff  dx*dx >= D or dy*dy >= D or dz*dz >= D                     [Eq. 28, squared form]
//        d = ((dx*dx + dy*dy) + dz*dz);  if (d < D) Dist_p = d                 [Eq. 29 / Eq. 2]
//      warp-shuffle argmax of (Dist_p, lowest original index) -> voxel state   [Eq. 30, Alg. 3]
//                                                                             -- __syncthreads
//   C  owners reload the state of the voxels they pushed; per-warp best key via redux.sync;
//      one slot per warp in shared memory                                     -- __syncthreads
//      every warp reduces the <=32 slots -> CTA best                          [Eq. 15-18]
//   X  (C > 1) lanes 0..C-1 of warp 0 send {key, x, y, z} to every CTA of the cluster with
//      st.async (...mbarrier::complete_tx); every thread waits on its CTA's mbarrier, reads the C
//      slots and takes the max.  Slots and mbarriers are double-buffered by iteration parity, so
//      no cluster-wide barrier is needed in the loop.
//
// Arithmetic: d2 is evaluated with __fsub_rn/__fmul_rn/__fadd_rn only (never contracted to FMA).
// Keys: (fp32 bits of d2) as the high word, 0xFFFFFFFF - original index as the low word; an
// unsigned lexicographic max of the pair is "largest distance, ties to the lowest original index"
// (Alg. 3's (d, -i_orig) pair).
#include <cfloat>
#include <cstring>

#include "device_utils.cuh"
#include "internal.h"

namespace rfps {

constexpr int MAX_CLUSTER = 16;

struct SampleParams {
    const float *px, *py, *pz;
    const int *porig, *pinv;
    float *Dp;
    const float4 *vgeom;
    const int2 *vseg;
    uint4 *vstate;
    const int *K;
    const int *poff;              // [B+1] first point of every cloud
    const int *rag;               // ragged call: [3][B+1] = M_b, start_b, output offsets; else null
    int B, K_cap, M, start_idx;
    int *out_idx;
    float *out_mind;
    unsigned long long *counters;
};

struct __align__(16) XMsg {   // one candidate: 32 bytes = two st.async.v4.b32
    unsigned hi, lo;           // key
    float x, y, z;             // coordinates of the candidate point
    unsigned pad0, pad1, pad2;
};

enum { CNT_VTEST = 0, CNT_VVISIT, CNT_PVISIT, CNT_PCOMP, CNT_EFF };

template <int VPT, int TB, bool CL, bool STATS>
__global__ void __launch_bounds__(TB, 1) k_fps_sample(const SampleParams P, const int flags)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int T = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = T >> 5;
    const int C = CL ? (int)cluster_nctarank() : 1;
    const int rank = CL ? (int)cluster_ctarank() : 0;
    const int b = blockIdx.x / C;
    const bool no_prune = flags & FPS_FLAG_NO_PRUNE, no_skip = flags & FPS_FLAG_NO_SKIP;

    // ---- shared memory carve-up ----
    XMsg *xslot = reinterpret_cast<XMsg *>(smem_raw);                         // [2][MAX_CLUSTER]
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(xslot + 2 * MAX_CLUSTER);   // [2]
    uint4 *wbest = reinterpret_cast<uint4 *>(mbar + 2);                       // [32] {hi, lo, pos, -}
    int *qn = reinterpret_cast<int *>(wbest + 32);                            // [4]
    int *queue = qn + 4;                                                      // [VPT * T]

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
    const int2 *__restrict__ vseg = P.vseg + vo;
    uint4 *vstate = P.vstate + vo;
    const int K = P.K[b];
    const int Kc = (K + C - 1) / C;
    const int k0 = min(K, rank * Kc), k1 = min(K, k0 + Kc);

    if (tid < 32) wbest[tid] = make_uint4(0u, 0u, 0u, 0u);
    if (tid == 0) {
        qn[0] = 0;
        if (CL) {
            mbar_init(smem_u32(&mbar[0]), 1);
            mbar_init(smem_u32(&mbar[1]), 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }

    // ---- a7: state reset.  Dist_p = +inf for the points this CTA owns; thresholds = NaN (nothing can
    // be pruned in iteration 1, which therefore performs the paper's "initial update", Eq. 13-14). ----
    {
        const int p0 = k0 < K ? vseg[k0].x : Nb;
        const int p1 = k1 < K ? vseg[k1].x : Nb;
        const float inf = __uint_as_float(0x7f800000u);
        for (int p = p0 + tid; p < p1; p += T) Dp[p] = inf;
    }
    float cx[VPT], cy[VPT], cz[VPT], thr[VPT];
    unsigned khi[VPT], klo[VPT], kpos[VPT];
#pragma unroll
    for (int v = 0; v < VPT; ++v) {
        const int k = k0 + v * T + tid;
        if (k < k1) {
            const float4 g = vgeom[k];
            cx[v] = g.x; cy[v] = g.y; cz[v] = g.z;
            thr[v] = __uint_as_float(0x7fc00000u);   // NaN: "d2c >= thr" is false -> visit
        } else {
            cx[v] = cy[v] = cz[v] = 0.0f;
            thr[v] = 0.0f;                           // empty slot: always pruned
        }
        khi[v] = klo[v] = kpos[v] = 0u;              // below every real key (real keys have lo >= 2^31)
    }
    unsigned bhi = 0u, blo = 0u, bpos = 0u;          // this thread's best key over its slots

    // ---- s_0 = the caller's start point ----
    float sx, sy, sz;
    {
        const int p = P.pinv[po + startb];
        sx = px[p]; sy = py[p]; sz = pz[p];
    }
    if (rank == 0 && tid == 0) {
        P.out_idx[obase] = startb;
        P.out_mind[obase] = __uint_as_float(0x7f800000u);
    }
    if (CL) {
        if (tid == 0) {
            mbar_arrive_expect_tx(smem_u32(&mbar[0]), (unsigned)(C * sizeof(XMsg)));
            mbar_arrive_expect_tx(smem_u32(&mbar[1]), (unsigned)(C * sizeof(XMsg)));
        }
        cluster_sync_all();    // every CTA's mbarriers are initialised before any remote store can land
    } else {
        __syncthreads();
    }

    unsigned long long c_vtest = 0, c_vvisit = 0, c_pvisit = 0, c_pcomp = 0, c_eff = 0;

    for (int j = 1; j < Mb; ++j) {
        // ================= phase A: radius prune (Eq. 25) over the voxels this thread owns =================
        unsigned pushed = 0u;
#pragma unroll
        for (int v = 0; v < VPT; ++v) {
            const float dx = __fsub_rn(cx[v], sx), dy = __fsub_rn(cy[v], sy), dz = __fsub_rn(cz[v], sz);
            const float d2c = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
            const int k = k0 + v * T + tid;
            bool visit = !(d2c >= thr[v]);
            if (no_prune) visit = k < k1;
            if (STATS && k < k1) c_vtest++;
            const unsigned m = __ballot_sync(FULL, visit);
            if (m) {
                int base = 0;
                if (lane == 0) base = atomicAdd(qn, __popc(m));
                base = __shfl_sync(FULL, base, 0);
                if (visit) {
                    queue[base + __popc(m & ((1u << lane) - 1u))] = k;
                    pushed |= 1u << v;
                }
            }
        }
        __syncthreads();
        const int nq = qn[0];

        // ================= phase B: point skip + update + voxel max (Eq. 28-30), one warp per voxel =========
        for (int qi = warp; qi < nq; qi += nwarps) {
            const int k = queue[qi];
            const int2 sg = vseg[k];
            const float R = vgeom[k].w;
            float bestD = -1.0f;
            unsigned bestO = 0u;      // ~orig of this lane's best
            int bestP = 0;
            for (int p = sg.x + lane; p < sg.x + sg.y; p += 32) {
                const float x = px[p], y = py[p], z = pz[p];
                const unsigned o = ~(unsigned)porig[p];
                float D = Dp[p];
                const float dx = __fsub_rn(x, sx), dy = __fsub_rn(y, sy), dz = __fsub_rn(z, sz);
                const float dx2 = __fmul_rn(dx, dx), dy2 = __fmul_rn(dy, dy), dz2 = __fmul_rn(dz, dz);
                if (no_skip || !(dx2 >= D || dy2 >= D || dz2 >= D)) {
                    const float d = __fadd_rn(__fadd_rn(dx2, dy2), dz2);
                    if (STATS) c_pcomp++;
                    if (d < D) {
                        D = d;
                        Dp[p] = d;
                        if (STATS) c_eff++;
                    }
                }
                if (D > bestD || (D == bestD && o > bestO)) { bestD = D; bestO = o; bestP = p; }
            }
            if (STATS) { c_pvisit += (sg.x + lane < sg.x + sg.y) ? ((sg.y - lane + 31) / 32) : 0; }
            // lanes without a point carry key (0,0); a real key has lo >= 2^31 so it always wins
            const unsigned hi = bestD >= 0.0f ? __float_as_uint(bestD) : 0u;
            unsigned mhi, mlo;
            const int win = warp_argmax_key(hi, bestD >= 0.0f ? bestO : 0u, mhi, mlo);
            const int wpos = __shfl_sync(FULL, bestP, win);
            if (lane == 0) {
                vstate[k] = make_uint4(mhi, mlo, (unsigned)wpos, __float_as_uint(prune_threshold(mhi, R)));
                if (STATS) c_vvisit++;
            }
        }
        __syncthreads();
        if (tid == 0) qn[0] = 0;

        // ================= phase C: argmax over voxel keys (Eq. 15-18) =================
        if (pushed) {
#pragma unroll
            for (int v = 0; v < VPT; ++v)
                if (pushed & (1u << v)) {
                    const uint4 s = vstate[k0 + v * T + tid];
                    khi[v] = s.x; klo[v] = s.y; kpos[v] = s.z;
                    thr[v] = __uint_as_float(s.w);
                }
            bhi = khi[0]; blo = klo[0]; bpos = kpos[0];
#pragma unroll
            for (int v = 1; v < VPT; ++v)
                if (khi[v] > bhi || (khi[v] == bhi && klo[v] > blo)) { bhi = khi[v]; blo = klo[v]; bpos = kpos[v]; }
        }
        if (__any_sync(FULL, pushed != 0u)) {
            unsigned mhi, mlo;
            const int win = warp_argmax_key(bhi, blo, mhi, mlo);
            const unsigned wpos = __shfl_sync(FULL, bpos, win);
            if (lane == 0) wbest[warp] = make_uint4(mhi, mlo, wpos, 0u);
        }
        __syncthreads();
        unsigned ghi, glo, gpos;
        {
            const uint4 wb = lane < nwarps ? wbest[lane] : make_uint4(0u, 0u, 0u, 0u);
            const int win = warp_argmax_key(wb.x, wb.y, ghi, glo);
            gpos = __shfl_sync(FULL, wb.z, win);
        }

        if (!CL) {
            sx = px[gpos]; sy = py[gpos]; sz = pz[gpos];
        } else {
            // ================= phase X: all-gather of the C CTA candidates over DSMEM =================
            const unsigned par = (unsigned)j & 1u;
            if (warp == 0 && lane < C) {
                const float x = px[gpos], y = py[gpos], z = pz[gpos];
                const unsigned dst = mapa(smem_u32(&xslot[par * MAX_CLUSTER + rank]), (unsigned)lane);
                const unsigned bar = mapa(smem_u32(&mbar[par]), (unsigned)lane);
                st_async_v4(dst, ghi, glo, __float_as_uint(x), __float_as_uint(y), bar);
                st_async_v4(dst + 16, __float_as_uint(z), 0u, 0u, 0u, bar);
            }
            mbar_wait(smem_u32(&mbar[par]), ((unsigned)(j - 1) >> 1) & 1u);
            XMsg m;
            if (lane < C) m = xslot[par * MAX_CLUSTER + lane];
            else { m.hi = 0u; m.lo = 0u; m.x = m.y = m.z = 0.0f; }
            const int win = warp_argmax_key(m.hi, m.lo, ghi, glo);
            sx = __shfl_sync(FULL, m.x, win);
            sy = __shfl_sync(FULL, m.y, win);
            sz = __shfl_sync(FULL, m.z, win);
            // re-arm this parity's mbarrier for iteration j+2 (its phase j has completed)
            if (tid == 0) mbar_arrive_expect_tx(smem_u32(&mbar[par]), (unsigned)(C * sizeof(XMsg)));
        }
        if (rank == 0 && tid == 0) {
            P.out_idx[obase + j] = (int)(~glo);
            P.out_mind[obase + j] = __uint_as_float(ghi);
        }
    }

    if (STATS) {
        atomicAdd(P.counters + CNT_VTEST, c_vtest);
        atomicAdd(P.counters + CNT_VVISIT, c_vvisit);
        atomicAdd(P.counters + CNT_PVISIT, c_pvisit);
        atomicAdd(P.counters + CNT_PCOMP, c_pcomp);
        atomicAdd(P.counters + CNT_EFF, c_eff);
    }
    if (CL) cluster_sync_all();   // no CTA may exit while a peer can still store into its shared memory
}

// ---------------------------------------------------------------------------------------------
// host side: launch shape and launch
// ---------------------------------------------------------------------------------------------
static size_t sample_smem_bytes(int vpt, int threads)
{
    return sizeof(XMsg) * 2 * MAX_CLUSTER + 2 * sizeof(unsigned long long) + 32 * sizeof(uint4) + 4 * sizeof(int) +
           (size_t)vpt * threads * sizeof(int);
}

int choose_launch_shape(DeviceIndex &ix, const fps_build_opts &o)
{
    int T = o.block_threads > 0 ? o.block_threads : 512;
    if (T < 32 || T > 1024 || (T & 31)) { set_error("block_threads=%d must be a multiple of 32 in [32,1024]", T); return FPS_ERR_INVALID; }
    int C = o.cluster_size;
    if (C != 0 && C != 1 && C != 2 && C != 4 && C != 8 && C != 16) { set_error("cluster_size=%d must be 0,1,2,4,8 or 16", C); return FPS_ERR_INVALID; }
    const int K = ix.K_max > 0 ? ix.K_max : 1;
    if (C == 0) {
        // one cloud per CTA while the voxel list fits a few slots per thread and the cloud is small;
        // otherwise a cluster, capped so that all B clusters are co-resident on the device's SMs.
        if (K <= 2 * T && ix.N <= 32768) C = 1;
        else {
            C = 2;
            while (C < 16 && (long long)C * T * 2 < K) C *= 2;
            while (C < 16 && (long long)C * 16384 < ix.N) C *= 2;
            while (C > 1 && (long long)C * ix.B > device_props().sm_count) C /= 2;
        }
    }
    const int maxvpt = T <= 512 ? 8 : 4;
    int vpt = 1;
    while (vpt < maxvpt && (long long)C * T * vpt < K) vpt *= 2;
    if (o.cluster_size == 0)
        while ((long long)C * T * vpt < K && C < 16) C *= 2;
    if (o.block_threads == 0)
        while ((long long)C * T * vpt < K && T < 1024) { T *= 2; if (T > 512 && vpt > 4) vpt = 4; }
    if ((long long)C * T * vpt < K) {
        set_error("K_max=%d voxels do not fit cluster_size=%d x block_threads=%d x %d slots; use a smaller n_vox or a larger tile_points",
                  K, C, T, vpt);
        return FPS_ERR_INVALID;
    }
    ix.cluster_size = C;
    ix.block_threads = T;
    ix.vpt = vpt;
    return FPS_OK;
}

template <int VPT, int TB, bool CL, bool STATS>
static int launch_one(const SampleParams &sp, const DeviceIndex &ix, cudaStream_t st)
{
    auto kern = k_fps_sample<VPT, TB, CL, STATS>;
    const size_t smem = sample_smem_bytes(VPT, ix.block_threads);
    RFPS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)(ix.B * ix.cluster_size));
    cfg.blockDim = dim3((unsigned)ix.block_threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    if (CL) {
        if (ix.cluster_size > 8) RFPS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)ix.cluster_size;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
    }
    RFPS_CUDA(cudaLaunchKernelEx(&cfg, kern, sp, ix.flags));
    return FPS_OK;
}

template <int VPT, int TB>
static int launch_vt(const SampleParams &sp, const DeviceIndex &ix, cudaStream_t st)
{
    const bool cl = ix.cluster_size > 1, stats = ix.flags & FPS_FLAG_STATS;
    if (cl) return stats ? launch_one<VPT, TB, true, true>(sp, ix, st) : launch_one<VPT, TB, true, false>(sp, ix, st);
    return stats ? launch_one<VPT, TB, false, true>(sp, ix, st) : launch_one<VPT, TB, false, false>(sp, ix, st);
}

int launch_sample(DeviceIndex &ix, int32_t M, int32_t start_idx, const int32_t *rag_dev, int64_t iterations,
                  int32_t *out_idx, float *out_mindist, cudaStream_t st)
{
    SampleParams sp;
    sp.px = ix.px; sp.py = ix.py; sp.pz = ix.pz;
    sp.porig = ix.porig; sp.pinv = ix.pinv;
    sp.Dp = ix.Dp;
    sp.vgeom = ix.vgeom; sp.vseg = ix.vseg; sp.vstate = ix.vstate;
    sp.K = ix.K_dev;
    sp.poff = ix.poff_dev; sp.rag = rag_dev; sp.B = ix.B;
    sp.K_cap = ix.K_cap; sp.M = M; sp.start_idx = start_idx;
    sp.out_idx = out_idx; sp.out_mind = out_mindist;
    sp.counters = ix.counters;
    if (ix.flags & FPS_FLAG_STATS) RFPS_CUDA(cudaMemsetAsync(ix.counters, 0, NUM_COUNTERS * sizeof(unsigned long long), st));
    ix.last_iterations = iterations;
    ix.last_stream = st;
    const bool big = ix.block_threads > 512;
    switch (ix.vpt) {
        case 1: return big ? launch_vt<1, 1024>(sp, ix, st) : launch_vt<1, 512>(sp, ix, st);
        case 2: return big ? launch_vt<2, 1024>(sp, ix, st) : launch_vt<2, 512>(sp, ix, st);
        case 4: return big ? launch_vt<4, 1024>(sp, ix, st) : launch_vt<4, 512>(sp, ix, st);
        case 8: if (!big) return launch_vt<8, 512>(sp, ix, st);
    }
    set_error("unsupported launch shape vpt=%d threads=%d", ix.vpt, ix.block_threads);
    return FPS_ERR_INVALID;
}

// ---------------------------------------------------------------------------------------------
// gathered coordinates of the samples (out_xyz).  One thread per sample: original
// index -> sorted position (pinv) -> SoA coordinates.  rag: layout of the last fps_sample_ragged call.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_gather_xyz(const float *__restrict__ px, const float *__restrict__ py,
                                                     const float *__restrict__ pz, const int *__restrict__ pinv,
                                                     const int *__restrict__ poff, const int *__restrict__ rag, int B, int M,
                                                     const int *__restrict__ idx, float *__restrict__ out_xyz)
{
    const int b = blockIdx.y;
    const int Mb = rag ? rag[b] : M;
    const size_t obase = rag ? (size_t)rag[2 * (B + 1) + b] : (size_t)b * M;
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Mb) return;
    const int Nb = poff[b + 1] - poff[b];
    const int i = idx[obase + j];
    float x = __uint_as_float(F32_NAN_BITS), y = x, z = x;       // an index outside the cloud gives NaN
    if (i >= 0 && i < Nb) {
        const size_t p = (size_t)poff[b] + pinv[(size_t)poff[b] + i];
        x = px[p]; y = py[p]; z = pz[p];
    }
    float *o = out_xyz + 3 * (obase + j);
    o[0] = x; o[1] = y; o[2] = z;
}

int launch_gather_xyz(DeviceIndex &ix, const int32_t *idx, int32_t M, int32_t M_max, const int32_t *rag_dev, float *out_xyz,
                      cudaStream_t st)
{
    k_gather_xyz<<<dim3((unsigned)((M_max + 255) / 256), (unsigned)ix.B), 256, 0, st>>>(ix.px, ix.py, ix.pz, ix.pinv, ix.poff_dev,
                                                                                      rag_dev, ix.B, M, idx, out_xyz);
    RFPS_CUDA(cudaGetLastError());
    ix.last_stream = st;      // fps_index_destroy releases the arena stream-ordered behind this kernel
    return FPS_OK;
}

}  // namespace rfps
