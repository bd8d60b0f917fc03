// matsubara3d_moment_plain.cu -- specialised moment kernels (mats3d_moment_kernel, matsubara3d_kernels.cuh) with the
// plain moment loop; see matsubara3d.cu for the call site.
#include "matsubara3d_kernels.cuh"

namespace dfrg {
#define DFRG_M3_SYM_TU false
#define DFRG_M3_LAUNCH_NAME mats3d_moment_launch_plain
#include "matsubara3d_moment_inst.inc"
}  // namespace dfrg
