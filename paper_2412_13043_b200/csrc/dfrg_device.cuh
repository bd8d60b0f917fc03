// dfrg_device.cuh -- device-side building blocks shared by the integration kernels (sm_100a).
//   * FP64 reciprocal from the hardware seed (MUFU.RCP64H) + one cubic Newton step
//   * regulators (eq. 14)
//   * log-grid cubic / linear interpolation reading shared-memory tables
//   * TMA 1-D bulk copies global -> shared with an mbarrier (cp.async.bulk; SASS: UBLKCP)
//   * deterministic block reductions (fixed shuffle tree, fixed warp order)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dfrg {

// ---- FP64 reciprocal ---------------------------------------------------------------------------
// rcp.approx.ftz.f64 is the MUFU.RCP64H seed (relative error < 2^-20).  With e = 1 - d r0 the
// cubic step r = r0 (1 + e + e^2) leaves e^3 < 2^-60 plus the rounding of three FMAs: <= ~1 ulp.
// Cost: 1 MUFU + 3 DFMA, no branches.  d = 0, inf, NaN or a subnormal d return NaN/0 -- the
// callers' dmin output flags such nodes (include/dfrg.h, "numerical special cases").
__device__ __forceinline__ double rcp_seed(double d) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
  return r;
}
__device__ __forceinline__ double fast_rcp(double d) {
  const double r0 = rcp_seed(d);
  const double e = fma(-d, r0, 1.0);
  const double t = fma(e, e, e);
  return fma(r0, t, r0);
}

// ---- regulators --------------------------------------------------------------------------------
struct RegParams {
  int kind;   // 0 Litim, 1 EXP_POLY
  int order;
  double k2;      // k^2
  double inv_k2;  // 1/k^2
};

__device__ __forceinline__ void regulator(const RegParams& rp, double s, double& R, double& Rdot) {
  if (rp.kind == 0) {
    const bool in = s < rp.k2;
    R = in ? rp.k2 - s : 0.0;
    Rdot = in ? 2.0 * rp.k2 : 0.0;
    return;
  }
  const double x = s * rp.inv_k2;
  double r;
  double geo;
  if (rp.order == 1) {
    r = rp.k2 * exp(-x);
    geo = x;
  } else {
    double expo = 0.0, xi = 1.0;
    geo = 0.0;
    for (int i = 1; i <= rp.order; ++i) {
      xi *= x;
      expo += xi / (double)i;
      geo += xi;
    }
    r = rp.k2 * exp(-expo);
  }
  R = r;
  Rdot = 2.0 * r * (1.0 + geo);
}

// ---- log-grid table look-up --------------------------------------------------------------------
struct GridParams {
  double lo;     // ln q_0
  double inv_h;  // (n-1)/(hi-lo)
  int n;
  int interp;    // 1 or 3
};

// Value of the table row `v` (shared or global memory) at squared momentum s.
__device__ __forceinline__ double table_lookup(const double* __restrict__ v, const GridParams& g, double s) {
  const double l = 0.5 * log(s);  // s == 0 -> -inf -> clamps to the first entry
  double t = (l - g.lo) * g.inv_h;
  t = (t > 0.0) ? t : 0.0;  // NaN -> 0
  const double tmax = (double)(g.n - 1);
  t = (t < tmax) ? t : tmax;
  if (g.interp == 3) {
    int i0 = (int)t - 1;  // t >= 0: truncation == floor
    i0 = max(i0, 0);
    i0 = min(i0, g.n - 4);
    const double sg = t - (double)i0;
    const double a0 = sg, a1 = sg - 1.0, a2 = sg - 2.0, a3 = sg - 3.0;
    const double L0 = -(a1 * a2 * a3) * (1.0 / 6.0);
    const double L1 = (a0 * a2 * a3) * 0.5;
    const double L2 = -(a0 * a1 * a3) * 0.5;
    const double L3 = (a0 * a1 * a2) * (1.0 / 6.0);
    return fma(v[i0], L0, fma(v[i0 + 1], L1, fma(v[i0 + 2], L2, v[i0 + 3] * L3)));
  }
  int i = (int)t;
  i = min(i, g.n - 2);
  const double tau = t - (double)i;
  return fma(v[i + 1], tau, v[i] * (1.0 - tau));
}

__device__ __forceinline__ double ipow(double x, int e) {
  double r = 1.0;
  for (int i = 0; i < e; ++i) r *= x;
  return r;
}

// ---- TMA 1-D bulk copy + mbarrier ----------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx_only(uint64_t* bar, uint32_t bytes) {  // no arrival
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int n_threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n_threads) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

__device__ __forceinline__ bool tma_ok(const void* p, size_t bytes) {
  return ((reinterpret_cast<uintptr_t>(p) & 15) == 0) && ((bytes & 15) == 0) && bytes > 0;
}

// Stages up to 8 arrays of doubles into shared memory.  Thread 0 issues one TMA bulk copy per
// aligned array and arms the mbarrier with the byte total; unaligned arrays are copied with plain
// loads by all threads.  Ends with a block-wide barrier: on return all data is visible to all threads.
struct StageList {
  const double* src[8];
  double* dst[8];
  int n[8];
  int count;
  __device__ StageList() : count(0) {}
  __device__ void add(double* d, const double* s, int n_) {
    src[count] = s; dst[count] = d; n[count] = n_; ++count;
  }
};

__device__ __forceinline__ void stage_to_smem(const StageList& L, uint64_t* bar, uint32_t parity) {
  // bar must have been initialised (count 1) and fenced before the first call
  if (threadIdx.x == 0) {
    uint32_t total = 0;
    for (int a = 0; a < L.count; ++a)
      if (tma_ok(L.src[a], (size_t)L.n[a] * 8) && tma_ok(L.dst[a], 16)) total += (uint32_t)L.n[a] * 8u;
    mbar_expect_tx(bar, total);
    for (int a = 0; a < L.count; ++a)
      if (tma_ok(L.src[a], (size_t)L.n[a] * 8) && tma_ok(L.dst[a], 16))
        tma_bulk_g2s(L.dst[a], L.src[a], (uint32_t)L.n[a] * 8u, bar);
  }
  for (int a = 0; a < L.count; ++a) {
    if (!(tma_ok(L.src[a], (size_t)L.n[a] * 8) && tma_ok(L.dst[a], 16)))
      for (int i = threadIdx.x; i < L.n[a]; i += blockDim.x) L.dst[a][i] = L.src[a][i];
  }
  mbar_wait(bar, parity);
  __syncthreads();
}

// ---- deterministic reductions ----------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// Sum over the block; result valid in thread 0.  scratch: >= 32 doubles of shared memory.
__device__ __forceinline__ double block_sum(double v, double* scratch) {
  v = warp_sum(v);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (lane == 0) scratch[wid] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x == 0)
    for (int w = 0; w < nw; ++w) r += scratch[w];
  return r;
}
__device__ __forceinline__ double block_min(double v, double* scratch) {
  v = warp_min(v);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (lane == 0) scratch[wid] = v;
  __syncthreads();
  double r = scratch[0];
  for (int w = 1; w < nw; ++w) r = fmin(r, scratch[w]);
  return r;  // valid in every thread
}

}  // namespace dfrg
