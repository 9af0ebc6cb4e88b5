// sample_batched.cu -- host side of exact batched picking: launch shape, dispatch to the instantiations of
// k_fps_batched (sample_batched.cuh; one translation unit per local-phase shape, sb_inst_*.cu, so that they
// compile in parallel), and the pick-chain latency-floor measurement.
#include <cfloat>
#include <algorithm>
#include <cstring>

#include "device_utils.cuh"
#include "internal.h"
#include "sample_batched_shapes.h"

namespace rfps {

// ---------------------------------------------------------------------------------------------
// host side: launch shape and launch
// ---------------------------------------------------------------------------------------------

int choose_batched_shape(DeviceIndex &ix, const fps_build_opts &o)
{
    // Local phase.  Clouds of <= 8 192 points are held whole in the registers of one CTA (2 points
    // per thread up to 1 024 points, 4 up to 2 048, 8 up to 4 096, 16 up to 8 192: k_fps_whole, sample_whole.cu -- one
    // CTA per cloud, no workers); larger clouds work on the top ~1 024 candidates per round.  Both resolve the picks of
    // a step in parallel (local_warps = 32) by default.  An explicit cluster size, the flat / hierarchical local phases
    // and FPS_FLAG_NO_BATCH keep the general kernel for small clouds too
    int LW = o.local_warps > 0 ? o.local_warps : LW_PAR;
    int C = o.cluster_size;
    const bool whole_ok = LW == LW_PAR && C == 0 && !(o.flags & FPS_FLAG_NO_BATCH);
    int CPT = o.cand_per_thread > 0 ? o.cand_per_thread
              : (LW >= LW_HIER ? (ix.N <= 1024 ? 2 : (ix.N <= 2048 ? 4 : (ix.N <= 4096 ? 8 : (ix.N <= 8192 && whole_ok ? 16 : 2)))) : (LW == 8 ? 16 : 8));
    ix.whole = whole_ok && CPT <= 16 && ix.N <= cand_capacity(CPT, LW);
    bool ok_shape = ix.whole && (CPT == 2 || CPT == 4 || CPT == 8 || CPT == 16);
#define RFPS_OK(C_, L_) ok_shape |= (CPT == C_ && LW == L_);
    RFPS_BATCHED_SHAPES(RFPS_OK)
#undef RFPS_OK
    if ((o.flags & FPS_FLAG_EUCLIDEAN) && LW < LW_HIER) {
        set_error("FPS_FLAG_EUCLIDEAN needs a 16-warp local phase (local_warps = 0, 16 or 32)");
        return FPS_ERR_INVALID;
    }
    if (!ok_shape) {
        set_error("local_warps=%d / cand_per_thread=%d: use 32 (parallel resolution) or 16 (hierarchical) with 2, 4 or 8 (32 with 16 "
                  "for clouds of <= 8192 points), or the flat shapes 4 x 8, 1 x 8, 8 x 16", LW, CPT);
        return FPS_ERR_INVALID;
    }
    if (ix.whole) C = 1;
    const int sms = device_props().sm_count;
    if (C < -sms || C > 16) { set_error("cluster_size=%d must be 0 (choose), 1..16 (CTAs per cluster) or -2..-%d (CTAs per cloud, grid mode)", C, sms); return FPS_ERR_INVALID; }
    if (o.block_threads != 0 && o.block_threads != BT) { set_error("block_threads=%d: the batched kernel runs %d threads per CTA", o.block_threads, BT); return FPS_ERR_INVALID; }
    const int K = ix.K_max > 0 ? ix.K_max : 1;
    const int TC = cand_capacity(CPT, LW);
    const int G = (K + 31) / 32;
    auto slots = [&](int c) { const int w = c > 1 ? c - 1 : 1; return 32 * ((G + w - 1) / w); };   // voxel slots per worker CTA
    const size_t max_smem = (size_t)device_props().max_smem_optin;
    auto fits = [&](int c) { return smem_layout(slots(c), TC, LW).total <= max_smem; };
    int grid = 0;
    if (C < 0) {
        // grid mode asked for: -C CTAs per cloud, all clouds resident at once (the CTAs of a cloud wait for one another)
        grid = -C;
        if (grid < 2 || LW != LW_PAR) { set_error("cluster_size=%d: grid mode takes >= 2 CTAs per cloud and the default local phase", C); return FPS_ERR_INVALID; }
        if ((long long)grid * ix.B > batched_max_resident_ctas(max_smem)) {
            set_error("cluster_size=%d: %d clouds x %d CTAs cannot all be resident on this device", C, ix.B, grid);
            return FPS_ERR_INVALID;
        }
        C = grid;
    } else if (C == 0) {
        // the largest cluster that (a) leaves every CTA >= 1 024 points, (b) holds the voxel state in
        // shared memory and (c) lets all B clusters be resident at once (a cluster lives inside one
        // GPC, so fewer clusters fit than SMs / C suggests: 15 of 8, 22 of 6, 7 of 16 on B200's 148 SMs);
        // otherwise the clouds would run in waves
        const int want = std::min(ix.B, sms);
        C = 1;
        for (int c = 16; c > 1; --c) {
            if ((long long)ix.N < 1024ll * c || !fits(c)) continue;
            if (batched_max_resident_clusters(c, max_smem) >= std::min(want, sms / c)) { C = c; break; }   // the launch takes all shared memory
        }
        while (C < 16 && !fits(C)) ++C;
        // Clusters leave part of the GPU idle (a cluster lives inside one GPC and holds <= 16 CTAs): where spreading each
        // cloud over the grid gives it at least a third more CTAs -- one picker CTA and up to sms / B - 1 workers, every
        // worker >= 1 group of voxels and >= ~1 000 points -- that is what runs (measured: C5 9.3 -> 7.7 ms with 148
        // CTAs instead of 16, C3 4.0 -> 3.9 ms with 119, C4 3.69 -> 3.55 ms with 4 x 37, C2 1.07 -> 1.04 ms with 16 x 9
        // instead of 16 x 6)
        if (LW == LW_PAR && C > 1 && ix.B * 2 <= sms) {
            int p = std::min(sms / ix.B, std::min(G + 1, ix.N / 1024 + 1));
            while (p > C && !fits(p)) --p;
            if (p >= C + std::max(2, C / 3) && (long long)p * ix.B <= batched_max_resident_ctas(max_smem)) { grid = p; C = p; }
        }
    }
    if (!ix.whole && !fits(C)) {
        set_error("K_max=%d voxels do not fit the shared memory of %d CTAs; use a smaller n_vox or a larger tile_points", K, C);
        return FPS_ERR_INVALID;
    }
    ix.grid_ctas = grid;
    ix.cluster_size = C;
    ix.block_threads = BT;
    ix.vpt = 0;
    ix.local_warps = LW;
    ix.cand_per_thread = CPT;
    ix.Kc_cap = slots(C);
    return FPS_OK;
}

int launch_sample_batched(DeviceIndex &ix, int32_t M, int32_t start_idx, const int32_t *rag_dev, int64_t iterations,
                          int32_t *out_idx, float *out_mindist, cudaStream_t st)
{
    BatchParams bp;
    bp.px = ix.px; bp.py = ix.py; bp.pz = ix.pz;
    bp.porig = ix.porig; bp.pinv = ix.pinv;
    bp.Dp = ix.Dp;
    bp.vgeom = ix.vgeom; bp.ggeom = ix.ggeom; bp.vseg = ix.vseg;
    bp.K = ix.K_dev;
    bp.poff = ix.poff_dev; bp.rag = rag_dev; bp.B = ix.B;
    bp.K_cap = ix.K_cap; bp.G_cap = ix.G_cap; bp.Kc_cap = ix.Kc_cap; bp.M = M; bp.start_idx = start_idx;
    bp.ctas_per_cloud = ix.grid_ctas > 0 ? ix.grid_ctas : ix.cluster_size;
    bp.gx = nullptr;
    if (ix.grid_ctas > 0) {
        // the clouds' exchange blocks: allocated once per handle, control words zeroed before every launch
        const size_t pitch = gx_bytes(cand_capacity(ix.cand_per_thread, ix.local_warps));
        if (!ix.gx) {
            if (dev_alloc_async(&ix.gx, pitch * (size_t)ix.B, st) != cudaSuccess) {
                cudaGetLastError();
                ix.gx = nullptr;
                set_error("device allocation of the exchange blocks failed");
                return FPS_ERR_NOMEM;
            }
            ix.gx_pitch = pitch;
        }
        RFPS_CUDA(cudaMemset2DAsync(ix.gx, pitch, 0, GX_PICK, (size_t)ix.B, st));
        bp.gx = (unsigned char *)ix.gx;
    }
    bp.smem_bytes = std::max((int)smem_layout(ix.Kc_cap, cand_capacity(ix.cand_per_thread, ix.local_warps), ix.local_warps).total,
                             device_props().max_smem_optin);
    bp.out_idx = out_idx; bp.out_mind = out_mindist;
    bp.counters = ix.counters;
    if (ix.flags & FPS_FLAG_STATS) RFPS_CUDA(cudaMemsetAsync(ix.counters, 0, NUM_COUNTERS * sizeof(unsigned long long), st));
    ix.last_iterations = iterations;
    ix.last_stream = st;
    if (ix.whole) return launch_sample_whole(bp, ix, st);
#define RFPS_CASE(CPT, LW) if (ix.cand_per_thread == CPT && ix.local_warps == LW) return launch_batched_##CPT##_##LW(bp, ix, st);
    RFPS_BATCHED_SHAPES(RFPS_CASE)
#undef RFPS_CASE
    set_error("unsupported local shape cand_per_thread=%d local_warps=%d", ix.cand_per_thread, ix.local_warps);
    return FPS_ERR_INVALID;
}

// ---------------------------------------------------------------------------------------------
// Latency floor of one pick (bench.py "latency": the roofline that actually binds this path).  One warp,
// 32*CPL candidates in registers, the bare dependent chain of a pick and nothing else:
//   update (d2, min) -> lane max -> redux.max(D bits) -> redux.max(slot id) -> 3 broadcast shared loads.
// No tie detection, no termination test, no pick log, no candidate selection, no global round.  A unique
// per-slot floor is added to the distances so that they never collapse to ties; the arithmetic per pick
// is that of the real loop.  Returns SM cycles per pick.
// ---------------------------------------------------------------------------------------------
template <int CPL>
__global__ void __launch_bounds__(32, 1) k_pick_chain_floor(const int iters, float *out)
{
    __shared__ float sX[32 * CPL], sY[32 * CPL], sZ[32 * CPL];
    const int lane = threadIdx.x;
    float x[CPL], y[CPL], z[CPL], d[CPL], fl[CPL];
#pragma unroll
    for (int c = 0; c < CPL; ++c) {
        const int i = c * 32 + lane;
        x[c] = sX[i] = (float)((i * 37) % 101) * 0.01f;
        y[c] = sY[i] = (float)((i * 53) % 103) * 0.01f;
        z[c] = sZ[i] = (float)((i * 71) % 107) * 0.01f;
        fl[c] = 1.0f + (float)i * 0x1p-10f;
        d[c] = 4.0f + fl[c];
    }
    __syncwarp();
    unsigned acc = 0u;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        float bm = d[0];
#pragma unroll
        for (int c = 1; c < CPL; ++c) bm = fmaxf(bm, d[c]);
        unsigned id = 0u;
#pragma unroll
        for (int c = 0; c < CPL; ++c)
            if (d[c] == bm) id = (unsigned)(c * 32 + lane + 1);
        const unsigned hi = __float_as_uint(bm);
        const unsigned ghi = __reduce_max_sync(FULL, hi);
        const unsigned wid = __reduce_max_sync(FULL, hi == ghi ? id : 0u) - 1u;
        const float sx = sX[wid], sy = sY[wid], sz = sZ[wid];
        acc += wid;
#pragma unroll
        for (int c = 0; c < CPL; ++c) d[c] = fminf(d[c], __fadd_rn(d2_rn(x[c], y[c], z[c], sx, sy, sz), fl[c]));
    }
    const long long t1 = clock64();
    if (lane == 0) { out[0] = (float)(t1 - t0) / (float)iters; out[1] = (float)acc; }
}

int measure_pick_chain(int cand_per_lane, int iters, float *cycles_per_pick)
{
    float *d = nullptr, h[2] = {0.f, 0.f};
    RFPS_CUDA(cudaMalloc(&d, 2 * sizeof(float)));
    for (int rep = 0; rep < 2; ++rep) {      // the first launch warms the instruction cache
        switch (cand_per_lane) {
            case 1: k_pick_chain_floor<1><<<1, 32>>>(iters, d); break;
            case 2: k_pick_chain_floor<2><<<1, 32>>>(iters, d); break;
            case 4: k_pick_chain_floor<4><<<1, 32>>>(iters, d); break;
            default: cudaFree(d); set_error("cand_per_lane=%d must be 1, 2 or 4", cand_per_lane); return FPS_ERR_INVALID;
        }
    }
    cudaError_t e = cudaMemcpy(h, d, sizeof h, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) { set_error("pick-chain measurement failed: %s", cudaGetErrorString(e)); return FPS_ERR_CUDA; }
    *cycles_per_pick = h[0];
    return FPS_OK;
}

}  // namespace rfps
