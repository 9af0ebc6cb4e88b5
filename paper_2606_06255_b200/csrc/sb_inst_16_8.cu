// sb_inst_16_8.cu -- k_fps_batched with 16 candidates per thread and local-phase shape 8 (one translation
// unit per shape so that the shapes compile in parallel; the kernel is sample_batched.cuh)
#include "sample_batched.cuh"

namespace rfps {

int launch_batched_16_8(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st) { return launch_batched_s<16, 8>(bp, ix, st); }

}  // namespace rfps
