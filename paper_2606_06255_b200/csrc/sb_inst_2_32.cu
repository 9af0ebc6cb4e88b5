// sb_inst_2_32.cu -- k_fps_batched with 2 candidates per thread and local-phase shape 32 (one translation
// unit per shape so that the shapes compile in parallel; the kernel is sample_batched.cuh)
#include <mutex>

#include "sample_batched.cuh"

namespace rfps {

int launch_batched_2_32(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st) { return launch_batched_s<2, 32>(bp, ix, st); }

// (asked for every index build; the answer depends on the device, the cluster size and the shared memory only)
static int resident_clusters_uncached(int c, size_t smem);
int batched_max_resident_clusters(int c, size_t smem)
{
    static std::mutex mu;
    static int cache[64][17];
    static size_t cache_smem[64][17];
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64 || c < 1 || c > 16) return resident_clusters_uncached(c, smem);
    std::lock_guard<std::mutex> lock(mu);
    if (cache_smem[dev][c] != smem || cache[dev][c] == 0) { cache[dev][c] = resident_clusters_uncached(c, smem); cache_smem[dev][c] = smem; }
    return cache[dev][c];
}
static int resident_clusters_uncached(int c, size_t smem)
{
    auto kern = k_fps_batched<2, 32, false, false, false>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    if (c > 8 && cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) { cudaGetLastError(); return 0; }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)(c * device_props().sm_count));
    cfg.blockDim = dim3(BT);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)c;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
    return n;
}

int batched_max_resident_ctas(size_t smem)
{
    auto kern = k_fps_batched<2, 32, false, false, true>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, BT, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    return per_sm * device_props().sm_count;
}

}  // namespace rfps
