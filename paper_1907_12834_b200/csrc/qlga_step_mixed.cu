// qlga_step_mixed.cu -- QLGA_F32X: the state is stored in fp32 (80 B per site) and every pass does its
// arithmetic in fp64 registers: one rounding to fp32 per amplitude per pass instead of one
// per floating-point operation.  Same kernels as QLGA_F64 with float2 loads and stores (qlga_pass.cuh).
#include "qlga_pass.cuh"

namespace qlga {

cudaError_t launch_pass_mixed(const Launch& L, int dir, const PassParams& P, int threads, int cxw) {
    return launch_pass_t<double, float>(L, dir, P, threads, cxw);
}

}  // namespace qlga
