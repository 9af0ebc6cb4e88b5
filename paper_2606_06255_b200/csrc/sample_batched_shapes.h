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
    int ctas_per_cloud;                            // grid mode: CTAs per cloud (1 picker + workers); cluster mode: the cluster size
    unsigned char *gx;                             // grid mode: [B] exchange blocks of gx_bytes(candidate capacity) each, zeroed
    int *out_idx;
    float *out_mind;
    unsigned long long *counters;
};

// Exchange block of one cloud: how its picker CTA and its worker CTAs talk.  It lives in the picker's shared
// memory when the cloud's CTAs form a thread-block cluster (the workers reach it over DSMEM), and in global
// memory when they are spread over the whole grid (cooperative launch; then followed by the pick and candidate
// buffers, see GX_* below).  All traffic is one-way messages with release / acquire at cluster or gpu scope;
// there is no barrier between the CTAs of a cloud while it is sampled.
//   pub    picker -> workers: the batch being produced: (batch id << PUB_SHIFT) | flags | picks published so far
//   cmd    picker -> workers: (command id << 2) | type, issued between two batches; cmd_tb = its threshold,
//          cmd_after = the batch that has to be applied completely before the command is answered (a command may
//          be sent before that batch is declared complete)
//   ack    workers -> picker: counts completed commands (every worker adds 1 per command)
//   ccount workers -> picker: candidates found by extraction command id & 7 (may exceed the buffer)
//   slot   workers -> picker: worker `rank`'s best key (Dist_v bits, ~orig) for a MAX command, one slot per worker
//          (plain stores, reduced by the picker; a red.max.u64 on the picker's shared memory lost updates when
//          several workers arrived together -- measured on B200);
//          cluster mode: in this block; grid mode: GX_SLOT bytes into the cloud's global block
struct __align__(16) Ctl {
    unsigned ccount[8];
    unsigned pub, cmd, cmd_tb, ack;
    unsigned cmd_after, best_lo;    // (best_lo: this CTA's tie-break index while its best key is being computed)
    int scratch[6];                 // CTA-local broadcast of what thread 0 read
    uint2 slot[16];
};
constexpr unsigned PUB_COUNT = 0x7ffu, PUB_DONE = 1u << 11, PUB_FINAL = 1u << 12;
constexpr int PUB_SHIFT = 13;       // batch id above the flags (compared modulo 2^19)
constexpr unsigned CMD_MAX = 1u, CMD_EXTRACT = 2u;
// grid mode: byte offsets inside a cloud's global exchange block; tc = candidate capacity
constexpr size_t GX_SLOT = 256, GX_PICK = 2048;      // the header (control words + one slot per CTA) is zeroed before a launch
// Grid mode packs the control words into three 64-bit words so that a poll is ONE L2 round trip (every message
// latency is on the critical path of a round):
//   GX_PC  = cmd << 32 | pub            written whole by the picker (release), read whole by the workers (acquire)
//   GX_CTB = the current command's payload: (cmd_after & 0xffff) << 48 | (command id & 0xffff) << 32 | cmd_tb, written
//            before GX_PC; a worker loads it together with GX_PC and re-reads it if the id tag is not the command's
//   GX_AC  = acknowledgements (cumulative) << 32 | candidates found by the running extraction: the workers reserve
//            candidate slots and acknowledge on the same word, the picker reads both with one acquire
constexpr size_t GX_PC = 216, GX_CTB = 224, GX_AC = 232;
static_assert(sizeof(Ctl) <= GX_PC && GX_AC + 8 <= GX_SLOT, "packed control words sit between the control block and the slots");
__host__ __device__ constexpr size_t gx_cand(void) { return GX_PICK + sizeof(float4) * 1024; }
__host__ __device__ constexpr size_t gx_bytes(int tc) { return gx_cand() + sizeof(float) * 5 * (size_t)tc; }

// shared-memory carve-up (host and device must agree).  The picker-only regions (candidates, local-phase
// scratch) come last: a worker CTA of a cluster with a separate picker never touches them, and its RESIDENT
// POINTS -- x, y, z, Dist_p of the voxels it owns, copied once per fps_sample so that the visits of a9-a12 and
// the candidate extraction run at shared-memory instead of L2 latency -- start at `picker` and use everything
// up to the end of the allocation; a single-CTA cloud (picker and worker in one) starts them at `pts`.
struct SmemLayout {
    size_t geom, ggeom, vdv, seg, loc, vthr, gthr, bpick, ctl, wbest, qkl, qmask, qbits, qn, gpre, picker, cand, cand2, lslot, hier, pts, total;
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
    // second candidate buffer: the parallel-resolution local phase compacts the live candidates into it as the
    // round proceeds (buffers of <= 2 048 candidates; larger ones hold a whole small cloud, where nothing dies)
    L.cand2 = o; o += (LW == LW_PAR && TC <= 2048) ? sizeof(float) * 5 * (size_t)TC : 0;
    L.lslot = o; o += sizeof(uint2) * 2 * 8;
    L.hier = o;  o += 3392 + 8 * PB;     // local-phase scratch (HierSmem / ParSmem), checked in sample_batched.cuh
    L.pts = o;
    L.total = o;                          // + 16 B per resident point (the launch asks for the device maximum)
    return L;
}

// per-shape launchers (sb_inst_*.cu): cand_per_thread x local_warps
#define RFPS_BATCHED_SHAPES(X) X(2, 32) X(4, 32) X(8, 32) X(2, 16) X(4, 16) X(8, 16) X(8, 4) X(8, 1) X(16, 8)
#define RFPS_DECL_LAUNCH(CPT, LW) int launch_batched_##CPT##_##LW(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st);
RFPS_BATCHED_SHAPES(RFPS_DECL_LAUNCH)
#undef RFPS_DECL_LAUNCH
// small clouds, one CTA per cloud (sample_whole.cu); cand_per_thread 2, 4 or 8
int launch_sample_whole(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st);
// how many clusters of `c` CTAs of the default kernel can be resident at once (0 on error)
int batched_max_resident_clusters(int c, size_t smem);
// grid mode: how many CTAs of the default kernel fit the device at once
int batched_max_resident_ctas(size_t smem);

}  // namespace rfps
