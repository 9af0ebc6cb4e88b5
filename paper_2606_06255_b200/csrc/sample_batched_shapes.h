// sample_batched_shapes.h -- what the host side (sample_batched.cu) and the kernel (sample_batched.cuh) of exact
// batched picking share: constants, kernel parameters, the shared-memory carve-up, and the per-shape launchers
// (one translation unit each, sb_inst_*.cu).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#include "internal.h"

namespace rfps {

constexpr int BT = 512;        // threads per CTA
constexpr int PB = 1024;       // picks per batch (capacity of the batch buffer)
constexpr int MAX_ATTEMPTS = 4;
constexpr int STREAM_MIN = 64;    // workers start on a piece of the running batch once it has this many picks
constexpr unsigned PUB_DONE = 1u << 31, PUB_FINAL = 1u << 30, PUB_COUNT = 0xffffu;
// extraction control: the next extraction aims at the fraction `gt` of the candidate buffer; gt starts at GTARGET,
// creeps up after an extraction that fitted and drops after one that overflowed (all measured on C1-C5)
constexpr float GTARGET = 0.625f, GT_MAX = 0.7f, GT_UP = 1.03f, GT_MIN = 0.35f, GT_DOWN = 0.85f;
constexpr int POLL_NS = 32;       // back-off of the warps that follow the pick warp's published count
constexpr int CPT2 = 3;           // candidates per lane of the pick warp (hierarchical local phase)
constexpr int KCH = 16;           // picks the pick warp runs speculatively between two exit tests
// local-phase shapes (fps_build_opts.local_warps): 1..8 = flat FPS on that many warps; LW_HIER = all 16 warps hold
// candidates, one warp picks sequentially from the top of them; LW_PAR = all 16 warps hold candidates, the top <= 64
// are resolved in parallel per step (the default)
constexpr int LW_HIER = 16, LW_PAR = 32;
__host__ __device__ constexpr int cand_capacity(int cpt, int lw) { return cpt * 32 * (lw < 16 ? lw : 16); }
constexpr int SUBW = 4;        // 32-bit mask words per queued voxel
constexpr int SUBP = 32 * SUBW;   // picks applied between two CTA barriers

struct BatchParams {
    const float *px, *py, *pz;
    const int *porig, *pinv;
    float *Dp;
    const float4 *vgeom, *ggeom;
    const int2 *vseg;
    const int *K;
    const int *poff;                               // [B+1] first point of every cloud
    const int *rag;                                // ragged call: [3][B+1] = M_b, start_b, output offsets; else null
    int B, K_cap, G_cap, Kc_cap, M, start_idx;     // Kc_cap: voxel slots per CTA (a multiple of 32); M, start_idx: uniform call
    int smem_bytes;                                // dynamic shared memory of the launch (what is left of it holds resident points)
    int *out_idx;
    float *out_mind;
    unsigned long long *counters;
};

struct __align__(16) Ctl {          // per-CTA control block; CTA 0's copy is the cluster's
    unsigned ccount[4 * MAX_ATTEMPTS];  // candidates found by an extraction attempt (may exceed TC):
                                        // [round parity][pass: hung on the previous tau / on the true maximum][attempt]
    unsigned best_hi, best_lo, pad3, pad0;       // this CTA's best voxel key
    int nb, j, pad1, pad2;          // (CTA 0) size of the batch just produced, samples emitted so far
    unsigned pub, pad4, pad5, pad6; // (CTA 0) picks of the running batch published so far | PUB_DONE | PUB_FINAL
};

// shared-memory carve-up (host and device must agree).  The picker-only regions (candidates, local-phase
// scratch) come last: a worker CTA of a cluster with a separate picker never touches them, and its RESIDENT
// POINTS -- x, y, z, Dist_p of the voxels it owns, copied once per fps_sample so that the visits of a9-a12 and
// the candidate extraction run at shared-memory instead of L2 latency -- start at `picker` and use everything
// up to the end of the allocation; a single-CTA cloud (picker and worker in one) starts them at `pts`.
struct SmemLayout {
    size_t geom, ggeom, vdv, seg, loc, vthr, gthr, bpick, ctl, wbest, qkl, qmask, qbits, qn, gpre, picker, cand, lslot, hier, pts, total;
};
__host__ __device__ inline SmemLayout smem_layout(int Kc_cap, int TC, int LW)
{
    SmemLayout L;
    size_t o = 0;
    L.geom = o;  o += sizeof(float4) * (size_t)Kc_cap;
    L.ggeom = o; o += sizeof(float4) * (size_t)(Kc_cap / 32);
    L.seg = o;   o += sizeof(int2) * (size_t)Kc_cap;
    L.vdv = o;   o += sizeof(unsigned) * (size_t)Kc_cap;
    L.loc = o;   o += sizeof(int) * (size_t)Kc_cap;
    L.vthr = o;  o += sizeof(float) * (size_t)Kc_cap;
    L.gthr = o;  o += (sizeof(float) * (size_t)(Kc_cap / 32) + 15) & ~(size_t)15;
    L.gpre = o;  o += (sizeof(int) * (size_t)(Kc_cap / 32 + 1) + 15) & ~(size_t)15;
    L.bpick = o; o += sizeof(float4) * PB;
    L.ctl = o;   o += sizeof(Ctl);
    L.wbest = o; o += sizeof(uint4) * 32;
    L.qmask = o; o += sizeof(unsigned) * SUBW * (size_t)Kc_cap;
    L.qkl = o;   o += sizeof(int) * (size_t)Kc_cap;
    L.qbits = o; o += (sizeof(unsigned) * (size_t)(Kc_cap / 32) + 15) & ~(size_t)15;
    L.qn = o;    o += sizeof(int) * 4;
    L.picker = o;
    L.cand = o;  o += sizeof(float) * 5 * (size_t)TC;
    L.lslot = o; o += sizeof(uint2) * 2 * 8;
    L.hier = o;  o += 3392 + 8 * PB;     // local-phase scratch (HierSmem / ParSmem), checked in sample_batched.cuh
    L.pts = o;
    L.total = o;                          // + 16 B per resident point (the launch asks for the device maximum)
    (void)LW;
    return L;
}

// per-shape launchers (sb_inst_*.cu): cand_per_thread x local_warps
#define RFPS_BATCHED_SHAPES(X) X(2, 32) X(4, 32) X(8, 32) X(2, 16) X(4, 16) X(8, 16) X(8, 4) X(8, 1) X(16, 8)
#define RFPS_DECL_LAUNCH(CPT, LW) int launch_batched_##CPT##_##LW(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st);
RFPS_BATCHED_SHAPES(RFPS_DECL_LAUNCH)
#undef RFPS_DECL_LAUNCH
// how many clusters of `c` CTAs of the default kernel can be resident at once (0 on error)
int batched_max_resident_clusters(int c, size_t smem);

}  // namespace rfps
