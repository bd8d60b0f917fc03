// matsubara3d_anyshape.cu -- instantiations and dispatch of mats3d_gmoment_kernel (any n_max, n_jext <= 32); see
// matsubara3d_kernels.cuh for the kernel and matsubara3d.cu for the call site.
#include "matsubara3d_kernels.cuh"

namespace dfrg {

// generic-shape moment kernel: NJ = the smallest compiled value >= n_jext
template <int NJ, bool SYM>
static int mats3d_gmoment_go(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream) {
#define DFRG_M3_GGO(MF)                                                                                              \
  {                                                                                                                  \
    auto kern = P.mode == 2 ? mats3d_gmoment_kernel<NJ, MF, 256, true, SYM>                                          \
                            : mats3d_gmoment_kernel<NJ, MF, 256, false, SYM>;                                        \
    const int rca = opt_in_max_smem(kern);                                                                           \
    if (rca != DFRG_OK) return rca;                                                                                  \
    kern<<<pl.grid, 256, pl.smem, stream>>>(P);                                                                      \
  }
  if constexpr (NJ <= 16) {
    if (pl.variant == 0) { DFRG_M3_GGO(2) } else { DFRG_M3_GGO(1) }
  } else {
    DFRG_M3_GGO(1)
  }
#undef DFRG_M3_GGO
  return check_cuda(cudaGetLastError());
}
int mats3d_gmoment_dispatch(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream) {
#define X(NJ)                                                                      \
  if (P.n_jext <= NJ) {                                                            \
    if (P.sym_try) {                                                               \
      const int rc = mats3d_gmoment_go<NJ, true>(P, pl, stream);                   \
      if (rc != DFRG_OK) return rc;                                                \
    }                                                                              \
    return mats3d_gmoment_go<NJ, false>(P, pl, stream);                            \
  }
  X(2) X(4) X(8) X(16) X(32)
#undef X
  return DFRG_EUNSUPPORTED;
}


// complex (mu != 0) moment kernel: one field point per thread, NJ = the smallest compiled value >= n_jext
template <int NJ, bool SYM>
static int mats3d_cmoment_go(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream) {
  auto kern = P.mode == 2 ? mats3d_cmoment_kernel<NJ, SYM, true> : mats3d_cmoment_kernel<NJ, SYM, false>;
  if constexpr (NJ == 16) {   // BASELINE config 4's shape: pair code enumerated at compile time
    if (P.n_max == 11 && P.n_jext == 16 && !pl.any_shape_forced)
      kern = P.mode == 2 ? mats3d_cmoment_kernel<16, SYM, true, 11> : mats3d_cmoment_kernel<16, SYM, false, 11>;
  }
  const int rca = opt_in_max_smem(kern);
  if (rca != DFRG_OK) return rca;
  kern<<<pl.grid, 256, pl.smem, stream>>>(P);
  return check_cuda(cudaGetLastError());
}
int mats3d_cmoment_dispatch(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream) {
#define X(NJ)                                                                      \
  if (P.n_jext <= NJ) {                                                            \
    if (P.sym_try) {                                                               \
      const int rc = mats3d_cmoment_go<NJ, true>(P, pl, stream);                   \
      if (rc != DFRG_OK) return rc;                                                \
    }                                                                              \
    return mats3d_cmoment_go<NJ, false>(P, pl, stream);                            \
  }
  X(2) X(4) X(8) X(16) X(32)
#undef X
  return DFRG_EUNSUPPORTED;
}
}  // namespace dfrg
