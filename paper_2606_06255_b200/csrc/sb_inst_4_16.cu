// sb_inst_4_16.cu -- k_fps_batched with 4 candidates per thread and local-phase shape 16 (one translation
// unit per shape so that the shapes compile in parallel; the kernel is sample_batched.cuh)
#include "sample_batched.cuh"

namespace rfps {

int launch_batched_4_16(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st) { return launch_batched_s<4, 16>(bp, ix, st); }

}  // namespace rfps
