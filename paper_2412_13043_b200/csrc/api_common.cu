// api_common.cu -- status strings, error slot, device check, Gauss-Legendre nodes (S1, host) and
// the host-entry-point arena.
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <map>
#include <mutex>
#include <utility>

#include "dfrg_internal.h"

namespace dfrg {

static thread_local int g_last_cuda_error = 0;
void set_last_cuda_error(int e) { g_last_cuda_error = e; }

// Per-device cache of (compute capability major, SM count): filled on first use of a device.
static std::mutex g_dev_mutex;
static int g_dev_major[64] = {}, g_dev_sms[64] = {};
int require_sm100(int* sm_count) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { set_last_cuda_error((int)e); return DFRG_ECUDA; }
  if (dev < 0 || dev >= 64) return DFRG_EUNSUPPORTED;
  int major, sms;
  {
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    if (g_dev_major[dev] == 0) {
      int mj = 0, sm = 0;
      e = cudaDeviceGetAttribute(&mj, cudaDevAttrComputeCapabilityMajor, dev);
      if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev);
      if (e != cudaSuccess) { set_last_cuda_error((int)e); return DFRG_ECUDA; }
      g_dev_major[dev] = mj;
      g_dev_sms[dev] = sm;
    }
    major = g_dev_major[dev];
    sms = g_dev_sms[dev];
  }
  if (major != 10) return DFRG_EUNSUPPORTED;
  if (sm_count) *sm_count = sms;
  return DFRG_OK;
}

static std::mutex g_attr_mutex;
static std::map<std::pair<int, const void*>, size_t> g_attr_done;   // (device, kernel) -> its dynamic shared-memory limit
int opt_in_max_smem_impl(const void* kernel, size_t* limit) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return check_cuda(e);
  std::lock_guard<std::mutex> lock(g_attr_mutex);
  const std::pair<int, const void*> key(dev, kernel);
  const auto it = g_attr_done.find(key);
  if (it != g_attr_done.end()) {
    if (limit) *limit = it->second;
    return DFRG_OK;
  }
  // the opt-in limit covers static + dynamic shared memory: leave room for the kernel's own static part
  cudaFuncAttributes fa;
  e = cudaFuncGetAttributes(&fa, kernel);
  if (e != cudaSuccess) return check_cuda(e);
  int optin = 0;
  e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (e != cudaSuccess) return check_cuda(e);
  const int dyn = optin - (int)fa.sharedSizeBytes;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn);
  if (e != cudaSuccess) return check_cuda(e);
  g_attr_done[key] = (size_t)dyn;
  if (limit) *limit = (size_t)dyn;
  return DFRG_OK;
}

// ---- stream-ordered scratch pool ---------------------------------------------------------------------
static std::mutex g_pool_mutex;
static cudaMemPool_t g_pools[64] = {};

static int get_pool(cudaMemPool_t* pool) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return check_cuda(e);
  if (dev < 0 || dev >= 64) return DFRG_EUNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  if (!g_pools[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    e = cudaMemPoolCreate(&g_pools[dev], &props);
    if (e != cudaSuccess) { g_pools[dev] = nullptr; return check_cuda(e); }
    unsigned long long threshold = ~0ull;
    cudaMemPoolSetAttribute(g_pools[dev], cudaMemPoolAttrReleaseThreshold, &threshold);
  }
  *pool = g_pools[dev];
  return DFRG_OK;
}

int scratch_alloc(void** ptr, size_t bytes, cudaStream_t stream) {
  cudaMemPool_t pool;
  int rc = get_pool(&pool);
  if (rc != DFRG_OK) return rc;
  cudaError_t e = cudaMallocFromPoolAsync(ptr, bytes, pool, stream);
  if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); set_last_cuda_error((int)e); return DFRG_ENOMEM; }
  return check_cuda(e);
}
void scratch_free(void* ptr, cudaStream_t stream) {
  if (ptr) cudaFreeAsync(ptr, stream);
}
void scratch_shutdown() {
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  for (int d = 0; d < 64; ++d)
    if (g_pools[d]) { cudaMemPoolDestroy(g_pools[d]); g_pools[d] = nullptr; }
}

// ---- arena ---------------------------------------------------------------------------------------
static size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

// Host arrays of up to ARENA_STAGE_MAX bytes are gathered in a pinned staging block that mirrors the start of the device
// arena and go up in ONE copy (a call has ~10 small inputs: nodes, weights, tables, coefficients, field and momentum
// grids; ten separate cudaMemcpyAsync cost ~50 us of host time); larger arrays are copied directly.
static const size_t ARENA_STAGE_MAX = 256 * 1024, ARENA_STAGE_CAP = 2 * 1024 * 1024;

int Arena::begin(size_t bytes_needed) {
  status_ = DFRG_OK;
  off_ = 0;
  up_lo_ = up_hi_ = 0;
  if (!hstage_) {
    if (cudaHostAlloc((void**)&hstage_, ARENA_STAGE_CAP, cudaHostAllocDefault) == cudaSuccess) hcap_ = ARENA_STAGE_CAP;
    else { hstage_ = nullptr; hcap_ = 0; cudaGetLastError(); }   // no staging: put() copies directly
  }
  if (!stream_) {
    cudaError_t e = cudaStreamCreateWithFlags(&stream_, cudaStreamNonBlocking);
    if (e != cudaSuccess) { set_last_cuda_error((int)e); return status_ = DFRG_ECUDA; }
  }
  if (bytes_needed > cap_) {
    if (base_) cudaFree(base_);
    base_ = nullptr;
    cap_ = 0;
    const size_t want = align256(bytes_needed + (bytes_needed >> 2));
    cudaError_t e = cudaMalloc((void**)&base_, want);
    if (e != cudaSuccess) { set_last_cuda_error((int)e); cudaGetLastError(); return status_ = DFRG_ENOMEM; }
    cap_ = want;
  }
  return DFRG_OK;
}
double* Arena::reserve(size_t n) {
  const size_t b = align256(n * sizeof(double));
  if (off_ + b > cap_) { status_ = DFRG_ENOMEM; return nullptr; }
  double* p = (double*)(base_ + off_);
  off_ += b;
  return p;
}
double* Arena::put(const double* host, size_t n) {
  const size_t at = off_;
  double* p = reserve(n);
  if (!p) return nullptr;
  const size_t bytes = n * sizeof(double);
  if (bytes <= ARENA_STAGE_MAX && off_ <= hcap_ && (up_hi_ == 0 || at == up_hi_)) {   // contiguous with what is staged
    memcpy(hstage_ + at, host, bytes);
    if (up_hi_ == 0) up_lo_ = at;
    up_hi_ = off_;
    return p;
  }
  cudaError_t e = cudaMemcpyAsync(p, host, bytes, cudaMemcpyHostToDevice, stream_);
  if (e != cudaSuccess) { set_last_cuda_error((int)e); status_ = DFRG_ECUDA; return nullptr; }
  return p;
}
int Arena::upload() {
  if (up_hi_ > up_lo_) {
    cudaError_t e = cudaMemcpyAsync(base_ + up_lo_, hstage_ + up_lo_, up_hi_ - up_lo_, cudaMemcpyHostToDevice, stream_);
    up_lo_ = up_hi_ = 0;
    if (e != cudaSuccess) { set_last_cuda_error((int)e); return status_ = DFRG_ECUDA; }
  }
  return status_;
}
int Arena::fetch(double* host, const double* dev, size_t n) {
  cudaError_t e = cudaMemcpyAsync(host, dev, n * sizeof(double), cudaMemcpyDeviceToHost, stream_);
  if (e != cudaSuccess) { set_last_cuda_error((int)e); return status_ = DFRG_ECUDA; }
  return DFRG_OK;
}
int Arena::finish() {
  cudaError_t e = cudaStreamSynchronize(stream_);
  if (e != cudaSuccess) { set_last_cuda_error((int)e); return status_ = DFRG_ECUDA; }
  return status_;
}
void Arena::release() {
  if (base_) cudaFree(base_);
  if (hstage_) cudaFreeHost(hstage_);
  if (stream_) cudaStreamDestroy(stream_);
  base_ = nullptr; cap_ = off_ = 0; stream_ = nullptr; hstage_ = nullptr; hcap_ = 0; up_lo_ = up_hi_ = 0;
}
Arena& thread_arena() {
  static thread_local Arena a;
  return a;
}

}  // namespace dfrg

using namespace dfrg;

extern "C" {

const char* dfrg_strerror(int status) {
  switch (status) {
    case DFRG_OK: return "ok";
    case DFRG_EINVAL: return "invalid argument";
    case DFRG_EUNSUPPORTED: return "unsupported size, dimension or device";
    case DFRG_ECUDA: return "CUDA runtime error (see dfrg_last_cuda_error)";
    case DFRG_ENOMEM: return "device arena allocation failed";
    case DFRG_ESCRATCH: return "call needs more scratch than the fixed array of the no-allocation entry point holds";
    default: return "unknown status";
  }
}
int dfrg_last_cuda_error(void) { return g_last_cuda_error; }
int dfrg_version(void) { return 100; }
void dfrg_shutdown(void) {
  thread_arena().release();
  scratch_shutdown();
  std::lock_guard<std::mutex> lock(g_attr_mutex);
  g_attr_done.clear();   // kernel attributes do not survive a device reset: set them again on the next call
}

// S1: Gauss-Legendre nodes.  Half the roots from the Tricomi initial guess, Newton on P_n with the
// three-term recurrence in long double, mirrored; derivative from P_n' = n (P_{n-1} - x P_n)/(1 - x^2).
int dfrg_matsubara_n_max(int domain, double T, double k, double extent) {
  if (!(T > 0.0) || !(k > 0.0) || !(extent >= 0.0) || !isfinite(extent)) return DFRG_EINVAL;
  if (domain != DFRG_DOMAIN_X0 && domain != DFRG_DOMAIN_Q0) return DFRG_EINVAL;
  const double cut = domain == DFRG_DOMAIN_X0 ? extent * k : extent;
  const double n = ceil(cut / (2.0 * 3.14159265358979323846 * T));
  if (!(n <= 1073741824.0)) return DFRG_EINVAL;
  return (int)n;
}

// Gauss-Legendre rule: roots of P_n by Newton on the three-term recurrence
//   P_j = x P_{j-1} + c_j (x P_{j-1} - P_{j-2}),  c_j = (j-1)/j      (= ((2j-1) x P_{j-1} - (j-1) P_{j-2})/j, no division)
// (1) Tricomi's initial guesses;  (2) three Newton iterations in double, eight roots side by side (independent chains:
// the recurrence is latency bound);  (3) per root two passes in long double: one Newton correction at the double root
// (d ~ 1e-16, so the corrected root is converged in long double), one evaluation of P_n' at the corrected root for the
// weight 2/((1-x^2) P_n'^2).  Only the non-negative half is computed; the rule is mirrored, hence exactly symmetric.
int dfrg_quad_nodes(int rule_kind, int n, double a, double b, double* x_host, double* w_host) {
  if (rule_kind != DFRG_RULE_GAUSS_LEGENDRE || n < 1 || n > 4096 || !x_host || !w_host) return DFRG_EINVAL;
  if (!(b > a) || !isfinite(a) || !isfinite(b)) return DFRG_EINVAL;
  const double PI_D = 3.14159265358979323846;
  const long double hw = ((long double)b - (long double)a) / 2.0L, mid = ((long double)b + (long double)a) / 2.0L;
  const int half = (n + 1) / 2;
  const long double nn = (long double)n;
  static thread_local long double cj[4097];
  static thread_local double cjd[4097], xr[2048 + 8];
  for (int j = 2; j <= n; ++j) { cj[j] = ((long double)j - 1.0L) / (long double)j; cjd[j] = (double)cj[j]; }
  {  // (1) r-th largest root
    const double nd = (double)n;
    for (int r = 0; r < half; ++r) {
      const double theta = PI_D * (4.0 * r + 3.0) / (4.0 * nd + 2.0);
      const double sn = sin(theta);
      xr[r] = (1.0 - (nd - 1.0) / (8.0 * nd * nd * nd) - (39.0 - 28.0 / (sn * sn)) / (384.0 * nd * nd * nd * nd)) * cos(theta);
    }
    for (int r = half; r < half + 8; ++r) xr[r] = 0.5;  // padding of the last block
  }
  constexpr int NB = 8;
  for (int r0 = 0; r0 < half && n > 1; r0 += NB) {  // (2)
    for (int it = 0; it < 3; ++it) {
      double x[NB], qm[NB], qn[NB];
      for (int t = 0; t < NB; ++t) { x[t] = xr[r0 + t]; qm[t] = 1.0; qn[t] = x[t]; }
      for (int j = 2; j <= n; ++j) {
        const double c = cjd[j];
        for (int t = 0; t < NB; ++t) {
          const double xq = x[t] * qn[t];
          const double qj = xq + c * (xq - qm[t]);
          qm[t] = qn[t];
          qn[t] = qj;
        }
      }
      for (int t = 0; t < NB; ++t) {
        const double dq = (double)n * (qm[t] - x[t] * qn[t]) / ((1.0 - x[t]) * (1.0 + x[t]));
        xr[r0 + t] = x[t] - qn[t] / dq;
      }
    }
  }
  constexpr int LB = 4;   // (3) four roots side by side (independent long-double chains)
  for (int r0 = 0; r0 < half; r0 += LB) {
    long double x[LB], pm[LB], pn[LB], dp[LB];
    for (int t = 0; t < LB; ++t) {
      x[t] = (long double)xr[r0 + t];
      if (n % 2 == 1 && r0 + t == half - 1) x[t] = 0.0L;   // the middle root of an odd rule is 0 exactly
    }
    for (int pass = 0; pass < 2; ++pass) {   // pass 0: Newton correction at the double root; pass 1: P_n' at the final root
      for (int t = 0; t < LB; ++t) { pm[t] = 1.0L; pn[t] = x[t]; }
      for (int j = 2; j <= n; ++j) {
        const long double c = cj[j];
        for (int t = 0; t < LB; ++t) {
          const long double xp = x[t] * pn[t];
          const long double pj = xp + c * (xp - pm[t]);
          pm[t] = pn[t];
          pn[t] = pj;
        }
      }
      for (int t = 0; t < LB; ++t) {
        if (n == 1) pm[t] = 1.0L;
        dp[t] = nn * (pm[t] - x[t] * pn[t]) / ((1.0L - x[t]) * (1.0L + x[t]));
        if (pass == 0 && !(n % 2 == 1 && r0 + t == half - 1)) x[t] -= pn[t] / dp[t];
      }
    }
    for (int t = 0; t < LB && r0 + t < half; ++t) {
      const int r = r0 + t;
      const long double w = 2.0L / ((1.0L - x[t]) * (1.0L + x[t]) * dp[t] * dp[t]);
      x_host[n - 1 - r] = (double)(mid + hw * x[t]);
      w_host[n - 1 - r] = (double)(hw * w);
      x_host[r] = (double)(mid - hw * x[t]);
      w_host[r] = (double)(hw * w);
    }
  }
  return DFRG_OK;
}

}  // extern "C"
