// internal.h -- shared declarations of the radiusfps CUDA library (not installed; the public
// interface is include/radiusfps.h).  Nothing here is used by, or taken from, oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdarg>
#include <cstdio>

#include "radiusfps.h"

namespace rfps {

// ---------------------------------------------------------------------------------------------
// error plumbing: thread-local message + status
// ---------------------------------------------------------------------------------------------
void set_error(const char *fmt, ...);

#define RFPS_CUDA(call)                                                                          \
    do {                                                                                         \
        cudaError_t e__ = (call);                                                                \
        if (e__ != cudaSuccess) {                                                                \
            ::rfps::set_error("%s:%d: %s failed: %s", __FILE__, __LINE__, #call,                 \
                              cudaGetErrorString(e__));                                          \
            return FPS_ERR_CUDA;                                                                 \
        }                                                                                        \
    } while (0)

// ---------------------------------------------------------------------------------------------
// per-voxel records (one "voxel" = one segment of the sorted SoA arrays with its own bounding
// sphere; with tiling a grid voxel of Eq. 8 may be split into several of them)
// ---------------------------------------------------------------------------------------------
// VoxelGeom  (constant after build)   {cx, cy, cz, R}   R >= max_p ||p - c||  (rounded up, A9)
// VoxelSeg   (constant after build)   {off, cnt}        segment [off, off+cnt) of the cloud's arrays
// VoxelState (rewritten on every visit) {dv_bits, ~orig, pos, thr_bits}:
//     dv_bits  fp32 bits of Dist_v[k] = max Dist_p in the voxel            (Eq. 30)
//     ~orig    0xFFFFFFFF - (lowest original index attaining it)           (tie-break)
//     pos      sorted position of that point
//     thr_bits fp32 bits of the prune threshold: the voxel is pruned iff d2(s_j, c_k) >= thr
//              (sqrt-free squared-domain form of Eq. 25 with fp32 safety margins)

constexpr int NUM_COUNTERS = 32;

// what the launch-shape logic needs to know about the current device (queried once per device)
struct DeviceProps {
    int sm_count = 0;          // multiprocessors
    int max_smem_optin = 0;    // largest dynamic shared memory per block (opt-in), bytes
};
const DeviceProps &device_props();

struct DeviceIndex {
    int32_t B = 0, N = 0;               // clouds; points of the LARGEST cloud (all clouds, if uniform)
    bool ragged = false;                // built by fps_index_build_ragged
    int32_t *poff_host = nullptr;       // [B+1] first point of every cloud in the concatenated arrays (malloc)
    int32_t *poff_dev = nullptr;        // the same on the device
    int32_t *rag_dev = nullptr;         // [3][B+1] per-call arguments of fps_sample_ragged
    int32_t *rag_host = nullptr;        // host staging for them (malloc)
    int32_t rag_M_max = 0;              // largest M_b of the last fps_sample_ragged call (0 = none yet)
    int32_t n_vox = 0, tile_points = 0;
    int32_t K_max = 0, K_cap = 0;       // largest per-cloud K; per-cloud stride of the voxel arrays
    int32_t G_cap = 0;                  // per-cloud stride of the group array (K_cap / 32)
    void *arena = nullptr;              // the ONE device allocation behind every pointer below
    bool arena_pooled = false;          // allocated from the library's stream-ordered pool
    int64_t K_total = 0;
    int32_t max_voxel_points = 0;
    int32_t cluster_size = 0, block_threads = 0, vpt = 0;   // sampling-kernel launch shape
    int32_t local_warps = 0, cand_per_thread = 0, Kc_cap = 0;   // batched kernel: local-phase shape, voxels per CTA
    int32_t grid_ctas = 0;              // batched kernel: > 0 = CTAs per cloud spread over the grid (cooperative launch,
                                        // exchange through global memory); 0 = one cluster of cluster_size CTAs per cloud
    bool whole = false;                 // every cloud fits one CTA's registers: k_fps_whole (sample_whole.cu) samples it
    void *gx = nullptr;                 // grid mode: the clouds' exchange blocks (allocated by the first fps_sample)
    size_t gx_pitch = 0;
    int32_t flags = 0;
    int32_t build_launches = 0;         // kernels launched by fps_index_build (a1-a6)
    // point arrays, [B][N], sorted by voxel
    float *px = nullptr, *py = nullptr, *pz = nullptr;
    int32_t *porig = nullptr;           // sorted position -> original index
    int32_t *pinv = nullptr;            // original index  -> sorted position
    float *Dp = nullptr;                // Dist_p
    // voxel arrays, [B][K_cap]
    float4 *vgeom = nullptr;
    float4 *ggeom = nullptr;            // [B][G_cap] spheres around groups of 32 consecutive voxels
    int2 *vseg = nullptr;
    uint4 *vstate = nullptr;
    int32_t *K_dev = nullptr;           // [B]
    int32_t *K_host = nullptr;          // [B] (malloc)
    unsigned long long *counters = nullptr;   // [NUM_COUNTERS] device, FPS_FLAG_STATS
    int64_t device_bytes = 0;
    int64_t last_iterations = 0;
    cudaStream_t last_stream = nullptr;
};

int build_index(DeviceIndex &ix, const float *points, const fps_build_opts &o);
void free_index(DeviceIndex &ix);
void trim_pool();   // return the library pool's unused memory to the driver (fps_trim)
// stream-ordered device memory from the library's private pool (falls back to cudaMalloc/cudaFree)
cudaError_t dev_alloc_async(void **p, size_t bytes, cudaStream_t stream);
void dev_free_async(void *p, cudaStream_t stream);
// rag_dev: null for a uniform call (M, start_idx apply to every cloud), else device [3][B+1] =
// {M_b}, {start_b}, {output offset of cloud b}.  iterations = sum over clouds of (M_b - 1), for the stats.
int launch_sample(DeviceIndex &ix, int32_t M, int32_t start_idx, const int32_t *rag_dev, int64_t iterations,
                  int32_t *out_idx, float *out_mindist, cudaStream_t stream);
int choose_launch_shape(DeviceIndex &ix, const fps_build_opts &o);
int launch_gather_xyz(DeviceIndex &ix, const int32_t *idx, int32_t M, int32_t M_max, const int32_t *rag_dev, float *out_xyz,
                      cudaStream_t stream);
// exact batched picking (sample_batched.cu)
int launch_sample_batched(DeviceIndex &ix, int32_t M, int32_t start_idx, const int32_t *rag_dev, int64_t iterations,
                          int32_t *out_idx, float *out_mindist, cudaStream_t stream);
int choose_batched_shape(DeviceIndex &ix, const fps_build_opts &o);
int measure_pick_chain(int cand_per_lane, int iters, float *cycles_per_pick);
// fps_sample_noalloc: index in the static device array of index_build.cu, no device allocation anywhere
int sample_noalloc(const float *points, int32_t N, int32_t M, int32_t start_idx, int32_t flags, int32_t *out_idx, float *out_mindist,
                   cudaStream_t stream);

}  // namespace rfps

struct fps_index {
    rfps::DeviceIndex ix;
};
