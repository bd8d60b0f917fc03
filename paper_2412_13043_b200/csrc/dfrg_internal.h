// dfrg_internal.h -- host-side helpers shared by the C-ABI translation units (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#include "../../include/dfrg.h"

namespace dfrg {

void set_last_cuda_error(int e);

// Records the error and returns DFRG_ECUDA if e != cudaSuccess, else DFRG_OK.
inline int check_cuda(cudaError_t e) {
  if (e == cudaSuccess) return DFRG_OK;
  set_last_cuda_error((int)e);
  return DFRG_ECUDA;
}

// DFRG_EUNSUPPORTED unless the current device is compute capability 10.x.  The device's attributes are queried once
// per device and cached (one cudaGetDevice per call afterwards).
int require_sm100(int* sm_count);

// Largest dynamic shared memory the library asks for: the 227 KB a CTA may opt into on sm_100 minus 1 KB for the
// kernels' static shared memory (barriers, reduction scratch).  Every kernel that needs more than the 48 KB default is
// raised to its own limit (opt-in maximum - its static part) ONCE per device (kernel attributes are per device) --
// never per call and never to a per-call size, so concurrent callers cannot lower each other's limit between the set
// and the launch.
// A kernel with more than 1 KB of static shared memory (the LPA kernels' reduction scratch: 3-6 KB) has a smaller limit
// than kMaxDynSmem: its launcher asks for the exact figure (`limit`) and compares before it launches.
constexpr size_t kMaxDynSmem = 226 * 1024;
int opt_in_max_smem_impl(const void* kernel, size_t* limit);   // DFRG_OK / DFRG_ECUDA; thread-safe, cached per (device, kernel)
template <typename K>
inline int opt_in_max_smem(K kernel, size_t* limit = nullptr) {   // *limit: the most dynamic shared memory `kernel` may be launched with
  return opt_in_max_smem_impl(reinterpret_cast<const void*>(kernel), limit);
}

inline bool valid_regulator(const dfrg_regulator& r) {
  if (!(r.k > 0.0) || !(r.zk > 0.0) || !(r.eta == r.eta)) return false;
  if (r.kind == DFRG_REG_LITIM) return true;
  return r.kind == DFRG_REG_EXP_POLY && r.order >= 1 && r.order <= 16;
}
inline bool valid_rule(const dfrg_rule& r) { return r.n >= 1 && r.x && r.w; }
inline bool valid_table(const dfrg_table& t, int min_rows) {
  if (!t.v || t.n_freq < min_rows || !(t.lnq_hi > t.lnq_lo)) return false;
  if (t.interp == 3) return t.n_q >= 4;
  if (t.interp == 1) return t.n_q >= 2;
  return false;
}

// Stream-ordered scratch for intermediate tables (S3 pre-pass outputs): allocated from a library-owned
// cudaMemPool per device (created lazily, release threshold = max so that blocks are reused across calls
// without touching the OS allocator), freed in stream order right after the consuming kernel.  No
// synchronisation; dfrg_shutdown() destroys the pools.
int scratch_alloc(void** ptr, size_t bytes, cudaStream_t stream);  // DFRG_OK / DFRG_ENOMEM / DFRG_ECUDA
void scratch_free(void* ptr, cudaStream_t stream);
void scratch_shutdown();

// Per-thread device arena used by the *_host entry points: one growing cudaMalloc block plus a
// private stream.  reset() rewinds; put() copies a host array in (async on the arena stream) and
// returns the device address; get() reserves device space for an output.
class Arena {
 public:
  int begin(size_t bytes_needed);  // DFRG_OK / DFRG_ENOMEM / DFRG_ECUDA
  double* put(const double* host, size_t n);   // small arrays are gathered in a pinned staging block (see upload())
  double* reserve(size_t n);
  int upload();                                // one H2D copy of everything put() gathered; call before the launch
  int fetch(double* host, const double* dev, size_t n);  // async D2H
  int finish();                                          // synchronise the arena stream
  cudaStream_t stream() const { return stream_; }
  void release();
  int status() const { return status_; }

 private:
  char* base_ = nullptr;
  size_t cap_ = 0, off_ = 0;
  char* hstage_ = nullptr;                     // pinned mirror of the first hcap_ bytes of the arena
  size_t hcap_ = 0, up_lo_ = 0, up_hi_ = 0;
  cudaStream_t stream_ = nullptr;
  int status_ = DFRG_OK;
};
Arena& thread_arena();

}  // namespace dfrg
