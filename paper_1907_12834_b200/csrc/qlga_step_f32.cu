// qlga_step_f32.cu -- fp32 instantiation of the fused pass kernels (qlga_pass.cuh): QLGA_F32,
// fp32 storage and fp32 (packed two-wide) arithmetic.
#include "qlga_pass.cuh"

namespace qlga {

cudaError_t launch_pass_f32(const Launch& L, int dir, const PassParams& P, int threads, int cxw) {
    return launch_pass_t<float, float>(L, dir, P, threads, cxw);
}

}  // namespace qlga
