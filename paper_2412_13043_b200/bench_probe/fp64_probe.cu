// fp64_probe.cu -- measurement aid of bench.py, NOT part of the library: the denominator of the FP64 roofline.
// Built into its own shared object (libdfrg_probe.so) by paper_2412_13043_b200/build.py; the product ABI
// (include/dfrg.h, libdfrg.so) does not contain it.
//
//   int dfrg_probe_fp64_peak(int n_iter, int ctas_per_sm, double* sink_dev, double* flops_out_host, void* cuda_stream)
// runs a register-only kernel of 8 independent DFMA chains per thread (n_iter x 64 DFMA per thread, one CTA of 512
// threads per SM x ctas_per_sm) on cuda_stream; *flops_out_host receives the FP64 flops it executes (2 per DFMA).
// Returns 0, -1 (bad argument) or -3 (CUDA error).
#include <cuda_runtime.h>

namespace {
__global__ void __launch_bounds__(512) fp64_peak_kernel(int n_iter, double* sink) {
  double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 0.1, a2 = a0 + 0.2, a3 = a0 + 0.3;
  double a4 = a0 + 0.4, a5 = a0 + 0.5, a6 = a0 + 0.6, a7 = a0 + 0.7;
  const double m = 0.999999, c = 1e-7;
  for (int it = 0; it < n_iter; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
  }
  const double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (s == 123456.789) sink[0] = s;  // never true; keeps the chains alive
}

// Issue model: the same 8 DFMA chains with K independent instructions of another pipe interleaved per 8 DFMA (volatile
// inline PTX: one SASS instruction each, never merged or removed):
//   KIND 0: 32-bit integer add (ALU)      KIND 1: I2F.F64 / F2I.F64 conversions (XU)      KIND 2: 16-byte shared-memory load (LSU)
//   KIND 3: rcp.approx.ftz.f64 = MUFU.RCP64H (XU)
// If an FP64 warp instruction held its scheduler's issue port for two cycles, the time would grow as (16 + K)/16 with K
// integer adds; if the port is free in the second cycle, K <= 8 adds cost nothing.  The XU and LSU variants show whether
// those pipes run beside the FP64 pipe (ratio 1 while their own throughput is not exceeded) or in turn with it.
template <int KIND, int K>
__global__ void __launch_bounds__(512) fp64_issue_kernel(int n_iter, double* sink) {
  __shared__ double2 sh[64];
  if (threadIdx.x < 64) sh[threadIdx.x] = make_double2(1.0, 2.0);
  __syncthreads();
  double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 0.1, a2 = a0 + 0.2, a3 = a0 + 0.3;
  double a4 = a0 + 0.4, a5 = a0 + 0.5, a6 = a0 + 0.6, a7 = a0 + 0.7;
  int x[8];
  double y[8];
  double2 v[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x + i; y[i] = 1.5 + i; v[i] = make_double2(0.0, 0.0); }
  const unsigned saddr = (unsigned)__cvta_generic_to_shared(sh) + 16u * (threadIdx.x & 7);
  const double m = 0.999999, c = 1e-7;
  auto other = [&](int i) {
    // (ptxas folds a chain of adds of a constant and hoists a conversion of an unchanged register: every instruction below
    // depends on the one before it in its own chain, by a value the assembler cannot know)
    if (KIND == 0) asm volatile("add.s32 %0, %0, %1;" : "+r"(x[i]) : "r"(x[(i + 1) & 7]));
    else if (KIND == 1) {
      if (i & 1) asm volatile("cvt.rzi.s32.f64 %0, %1;" : "=r"(x[i >> 1]) : "d"(y[i >> 1]));
      else asm volatile("cvt.rn.f64.s32 %0, %1;" : "=d"(y[i >> 1]) : "r"(x[i >> 1]));
    } else if (KIND == 3) asm volatile("rcp.approx.ftz.f64 %0, %0;" : "+d"(y[i]));   // MUFU.RCP64H: y -> 1/y -> y ...
    else asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v[i].x), "=d"(v[i].y) : "r"(saddr));
  };
  for (int it = 0; it < n_iter; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
#pragma unroll
      for (int i = 0; i < K / 2; ++i) other(i);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
#pragma unroll
      for (int i = K / 2; i < K; ++i) other(i);
    }
  }
  double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  int xs = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) { xs ^= x[i]; s += y[i] + v[i].x + v[i].y; }
  if (s == 123456.789 || xs == 0x7fffffff) sink[0] = s;
}
}  // namespace

//   int dfrg_probe_fp64_issue(int n_iter, int kind, int k, double* sink_dev, void* cuda_stream)
// launches the issue-model kernel (one CTA of 512 threads per SM): k in {0, 1, 2, 4, 8} instructions of `kind` per 8 DFMA.
extern "C" int dfrg_probe_fp64_issue(int n_iter, int kind, int k, double* sink, void* cuda_stream) {
  if (n_iter < 1 || !sink) return -1;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -3;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  void (*kern)(int, double*) = nullptr;
#define DFRG_PROBE_PICK(KD, KK) if (kind == KD && k == KK) kern = fp64_issue_kernel<KD, KK>;
  DFRG_PROBE_PICK(0, 0) DFRG_PROBE_PICK(0, 4) DFRG_PROBE_PICK(0, 8)
  DFRG_PROBE_PICK(1, 2) DFRG_PROBE_PICK(1, 4) DFRG_PROBE_PICK(1, 8)
  DFRG_PROBE_PICK(2, 2) DFRG_PROBE_PICK(2, 4) DFRG_PROBE_PICK(2, 8)
  DFRG_PROBE_PICK(3, 1) DFRG_PROBE_PICK(3, 2) DFRG_PROBE_PICK(3, 4)
#undef DFRG_PROBE_PICK
  if (!kern) return -1;
  kern<<<sms, 512, 0, st>>>(n_iter, sink);
  return cudaGetLastError() == cudaSuccess ? 0 : -3;
}

extern "C" int dfrg_probe_fp64_peak(int n_iter, int ctas_per_sm, double* sink, double* flops_out, void* cuda_stream) {
  if (n_iter < 1 || ctas_per_sm < 1 || ctas_per_sm > 4 || !sink) return -1;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -3;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
  const int grid = sms * ctas_per_sm;
  fp64_peak_kernel<<<grid, 512, 0, (cudaStream_t)cuda_stream>>>(n_iter, sink);
  if (flops_out) *flops_out = 2.0 * 64.0 * (double)n_iter * 512.0 * (double)grid;
  return cudaGetLastError() == cudaSuccess ? 0 : -3;
}
