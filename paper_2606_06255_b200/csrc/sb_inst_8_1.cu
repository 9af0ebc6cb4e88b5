// sb_inst_8_1.cu -- k_fps_batched with 8 candidates per thread and local-phase shape 1 (one translation
// unit per shape so that the shapes compile in parallel; the kernel is sample_batched.cuh)
#include "sample_batched.cuh"

namespace rfps {

int launch_batched_8_1(const BatchParams &bp, const DeviceIndex &ix, cudaStream_t st) { return launch_batched_s<8, 1>(bp, ix, st); }

}  // namespace rfps
