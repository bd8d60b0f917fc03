// lpa.cu -- dfrg_integrate_lpa: LPA O(N) flow right-hand side (BASELINE.json configs 0, 1).
//
// One CTA per tile of 32 field points.  Prologue (S2/S3): the radial rule is staged into shared
// memory with a TMA bulk copy; the block builds the field-independent table of (D0, W) pairs,
//     D0 = s + R(sR),  W = fold * w_i q_i^(d-1) Rdot(sR),
// over (Matsubara index n >= 0) x (radial node i); the terms are even in n, so n and -n are folded
// (fold = 2 for n > 0).  Hot loop (S4): lane = field point, warp = (channel, node slice); every lane
// of a warp reads the same (D0, W) pair (shared-memory broadcast) and does add -> reciprocal -> FMA
// into four independent accumulators.  S5: fixed-order combination of the slices through shared
// memory.  dmin needs no work in the hot loop: fl(D0 + m2) is monotone in D0, so
// min_nodes fl(D0 + m2) = fl(min_nodes D0 + m2) exactly.
#include "dfrg_device.cuh"
#include "dfrg_internal.h"

namespace dfrg {

constexpr int LPA_THREADS = 256;   // 8 warps: 2 channels x 4 node slices
constexpr int LPA_SLICES = 4;
constexpr int LPA_FTILE = 32;
constexpr int LPA_MAX_PAIRS = 12288;
constexpr int LPA_MAX_T = 16;      // temperatures per launch (dfrg_integrate_lpa_batch)

struct LpaParams {
  int d, reg_arg4d, nq, n_field, fermion_reg;
  double N, prefactor, mu;
  double Tv[LPA_MAX_T];     // temperature of batch entry blockIdx.y (a single call is a batch of one)
  int nmaxv[LPA_MAX_T];     // its Matsubara cut-off
  RegParams reg;
  FastMathConsts fmc;
  const double *xq, *wq, *rho, *u, *du;
  double *flow, *chan, *dmin, *dchan;
};

// WANT_D: also dI/dm2 = -sum W / D^2 per channel (two more FP64 instructions per evaluation)
template <bool WANT_D>
__global__ void __launch_bounds__(LPA_THREADS) lpa_kernel(const LpaParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double red[32];
  __shared__ double part[2][LPA_SLICES][LPA_FTILE];
  __shared__ double dpart[WANT_D ? 2 : 1][LPA_SLICES][LPA_FTILE];

  const int it = blockIdx.y;                      // batch entry: its own (T, n_max) and output planes
  const double T = P.Tv[it];
  const int n_terms = (T > 0.0) ? P.nmaxv[it] + 1 : 1;
  const int n_pairs = n_terms * P.nq;
  double2* tab = reinterpret_cast<double2*>(smem_raw);                 // [n_pairs] (D0, W)
  double* sx = reinterpret_cast<double*>(smem_raw + (size_t)n_pairs * 16);  // [nq]
  double* sw = sx + ((P.nq + 1) & ~1);                                      // [nq]

  if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  __syncthreads();
  StageList L;
  L.add(sx, P.xq, P.nq);
  L.add(sw, P.wq, P.nq);
  const FastMath fm = fm_stage(L, sw + ((P.nq + 1) & ~1), P.fmc);                  // [FM_DOUBLES]
  stage_to_smem(L, &bar, 0);

  // ---- S3: field-independent table ----
  const double two_pi_T = 2.0 * 3.14159265358979323846 * T;
  double dmin0 = __longlong_as_double(0x7ff0000000000000LL);
  for (int t = threadIdx.x; t < n_pairs; t += LPA_THREADS) {
    const int n = t / P.nq, i = t - n * P.nq;
    const double q = sx[i];
    const double wn = two_pi_T * (double)n;
    const double s = wn * wn + q * q;
    const double sR = P.reg_arg4d ? s : q * q;
    double R, Rd;
    regulator(P.reg, fm, sR, R, Rd);
    const double D0 = s + R;
    const double fold = (n > 0) ? 2.0 : 1.0;
    tab[t] = make_double2(D0, fold * (sw[i] * ipow(q, P.d - 1) * Rd));
    dmin0 = fmin(dmin0, D0);
  }
  dmin0 = block_min(dmin0, red);  // includes the barriers that publish tab[]

  // ---- S4: hot loop ----
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int ch = wid & 1, slice = wid >> 1;
  const int f = blockIdx.x * LPA_FTILE + lane;
  const bool live = f < P.n_field;
  double m2 = 1.0, m2pi = 1.0, m2sig = 1.0;
  if (live) {
    m2pi = P.u[f];
    m2sig = m2pi + 2.0 * P.rho[f] * P.du[f];
    m2 = ch ? m2sig : m2pi;
  }
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  double d0 = 0.0, d1 = 0.0, d2 = 0.0, d3 = 0.0;
  int t = slice;
  if constexpr (!WANT_D) {
    for (; t + 3 * LPA_SLICES < n_pairs; t += 4 * LPA_SLICES) {
      const double2 p0 = tab[t], p1 = tab[t + LPA_SLICES], p2 = tab[t + 2 * LPA_SLICES], p3 = tab[t + 3 * LPA_SLICES];
      a0 = fma(p0.y, fast_rcp(p0.x + m2), a0);
      a1 = fma(p1.y, fast_rcp(p1.x + m2), a1);
      a2 = fma(p2.y, fast_rcp(p2.x + m2), a2);
      a3 = fma(p3.y, fast_rcp(p3.x + m2), a3);
    }
    for (; t < n_pairs; t += LPA_SLICES) {
      const double2 p0 = tab[t];
      a0 = fma(p0.y, fast_rcp(p0.x + m2), a0);
    }
  } else {
    for (; t + 3 * LPA_SLICES < n_pairs; t += 4 * LPA_SLICES) {
      const double2 p0 = tab[t], p1 = tab[t + LPA_SLICES], p2 = tab[t + 2 * LPA_SLICES], p3 = tab[t + 3 * LPA_SLICES];
      const double r0 = fast_rcp(p0.x + m2), r1 = fast_rcp(p1.x + m2), r2 = fast_rcp(p2.x + m2), r3 = fast_rcp(p3.x + m2);
      const double w0 = p0.y * r0, w1 = p1.y * r1, w2 = p2.y * r2, w3 = p3.y * r3;
      a0 = fma(p0.y, r0, a0); a1 = fma(p1.y, r1, a1); a2 = fma(p2.y, r2, a2); a3 = fma(p3.y, r3, a3);  // as without WANT_D
      d0 = fma(w0, r0, d0); d1 = fma(w1, r1, d1); d2 = fma(w2, r2, d2); d3 = fma(w3, r3, d3);
    }
    for (; t < n_pairs; t += LPA_SLICES) {
      const double2 p0 = tab[t];
      const double r0 = fast_rcp(p0.x + m2);
      const double w0 = p0.y * r0;
      a0 = fma(p0.y, r0, a0);
      d0 = fma(w0, r0, d0);
    }
    dpart[ch][slice][lane] = (d0 + d1) + (d2 + d3);
  }
  part[ch][slice][lane] = (a0 + a1) + (a2 + a3);
  __syncthreads();

  // ---- S5/S6 ----
  if (wid == 0 && live) {
    const double scale = (T > 0.0) ? P.prefactor * T : P.prefactor;
    const size_t o1 = (size_t)it * P.n_field, o2 = 2 * o1;
    double I[2];
#pragma unroll
    for (int c = 0; c < 2; ++c)
      I[c] = scale * ((part[c][0][lane] + part[c][1][lane]) + (part[c][2][lane] + part[c][3][lane]));
    P.flow[o1 + f] = (P.N - 1.0) * I[0] + I[1];
    if (P.chan) { P.chan[o2 + f] = I[0]; P.chan[o2 + P.n_field + f] = I[1]; }
    if (P.dmin) P.dmin[o1 + f] = fmin(dmin0 + m2pi, dmin0 + m2sig) * P.reg.inv_k2;
    if constexpr (WANT_D) {
#pragma unroll
      for (int c = 0; c < 2; ++c)
        P.dchan[o2 + c * P.n_field + f] =
            -scale * ((dpart[c][0][lane] + dpart[c][1][lane]) + (dpart[c][2][lane] + dpart[c][3][lane]));
    }
  }
}

// ---- fermionic statistics at chemical potential mu (dfrg_lpa_desc::statistics == 1; include/dfrg.h) ----
// nu_n = (2n+1) pi T, p0 = nu_n + i mu, spatial regulator:  D = a + i b,  a = nu^2 - mu^2 + q^2 + R(q^2) + m2,  b = 2 nu mu,
//   I_F(m2) = C T sum_{n=-n_max-1..n_max} sum_i w q^(d-1) Rdot(q^2) Re(1/D),   Re 1/D = a/(a^2+b^2),  Re 1/D^2 = (a^2-b^2)/(a^2+b^2)^2.
// The terms are even in nu, so n and -n-1 are folded (weight 2).  Same mapping as lpa_kernel; the field-independent
// table holds (a - m2, W, b^2) per (n >= 0, radial node).  dmin = min over nodes of |D|/k^2, tracked in the hot loop.
template <bool WANT_D>
__global__ void __launch_bounds__(LPA_THREADS) lpa_fermion_kernel(const LpaParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double part[2][LPA_SLICES][LPA_FTILE];
  __shared__ double dpart[2][LPA_SLICES][LPA_FTILE];
  __shared__ double mpart[2][LPA_SLICES][LPA_FTILE];

  const int it = blockIdx.y;
  const double T = P.Tv[it];
  const int n_pairs = (P.nmaxv[it] + 1) * P.nq;
  double4* tab = reinterpret_cast<double4*>(smem_raw);                      // [n_pairs] (a0, W, b^2, -)
  double* sx = reinterpret_cast<double*>(smem_raw + (size_t)n_pairs * 32);  // [nq]
  double* sw = sx + ((P.nq + 1) & ~1);

  if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  __syncthreads();
  StageList L;
  L.add(sx, P.xq, P.nq);
  L.add(sw, P.wq, P.nq);
  const FastMath fm = fm_stage(L, sw + ((P.nq + 1) & ~1), P.fmc);
  stage_to_smem(L, &bar, 0);

  const double pi_T = 3.14159265358979323846 * T;
  for (int t = threadIdx.x; t < n_pairs; t += LPA_THREADS) {
    const int n = t / P.nq, i = t - n * P.nq;
    const double q = sx[i];
    const double nu = (2.0 * (double)n + 1.0) * pi_T;
    double K, Rd;   // K = q^2 + R(q^2), or (q + RF(q^2))^2 with the fermionic regulator (reading A25)
    if (P.fermion_reg) {
      const double A = fermion_kinetic(P.reg, fm, 1.0, q * q, Rd);
      K = A * A;
    } else {
      regulator(P.reg, fm, q * q, K, Rd);
      K += q * q;
    }
    const double b = 2.0 * nu * P.mu;
    tab[t] = make_double4(nu * nu - P.mu * P.mu + K, 2.0 * (sw[i] * ipow(q, P.d - 1) * Rd), b * b, 0.0);
  }
  __syncthreads();

  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int ch = wid & 1, slice = wid >> 1;
  const int f = blockIdx.x * LPA_FTILE + lane;
  const bool live = f < P.n_field;
  double m2 = 1.0;
  if (live) m2 = ch ? P.u[f] + 2.0 * P.rho[f] * P.du[f] : P.u[f];
  const bool want_dmin = P.dmin != nullptr;
  double acc = 0.0, accd = 0.0, den_min = __longlong_as_double(0x7ff0000000000000LL);
#pragma unroll 4
  for (int t = slice; t < n_pairs; t += LPA_SLICES) {
    const double4 e = tab[t];
    const double a = e.x + m2;
    const double den = fma(a, a, e.z);
    const double r = fast_rcp(den);
    const double wr = e.y * r;
    acc = fma(wr, a, acc);
    if constexpr (WANT_D) accd = fma(wr * r, fma(a, a, -e.z), accd);
    if (want_dmin) den_min = fmin(den_min, den);
  }
  part[ch][slice][lane] = acc;
  dpart[ch][slice][lane] = accd;
  mpart[ch][slice][lane] = den_min;
  __syncthreads();
  if (wid == 0 && live) {
    const double scale = P.prefactor * T;
    const size_t o1 = (size_t)it * P.n_field, o2 = 2 * o1;
    double I[2];
#pragma unroll
    for (int c = 0; c < 2; ++c)
      I[c] = scale * ((part[c][0][lane] + part[c][1][lane]) + (part[c][2][lane] + part[c][3][lane]));
    P.flow[o1 + f] = (P.N - 1.0) * I[0] + I[1];
    if (P.chan) { P.chan[o2 + f] = I[0]; P.chan[o2 + P.n_field + f] = I[1]; }
    if (want_dmin) {
      double dm = mpart[0][0][lane];
#pragma unroll
      for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int sl = 0; sl < LPA_SLICES; ++sl) dm = fmin(dm, mpart[c][sl][lane]);
      P.dmin[o1 + f] = sqrt(dm) * P.reg.inv_k2;
    }
    if constexpr (WANT_D) {
#pragma unroll
      for (int c = 0; c < 2; ++c)
        P.dchan[o2 + c * P.n_field + f] =
            -scale * ((dpart[c][0][lane] + dpart[c][1][lane]) + (dpart[c][2][lane] + dpart[c][3][lane]));
    }
  }
}

// dynamic shared memory of one CTA: the (D0, W) table over (n >= 0, q) plus the staged rule and the log/exp tables
static size_t lpa_smem(const dfrg_lpa_desc* D) {
  const size_t n_terms = (D->T > 0.0) ? (size_t)D->n_max + 1 : 1;
  const bool fermi = D->statistics == DFRG_STAT_FERMION;
  return n_terms * D->q.n * (fermi ? 32 : 16) + (2 * (size_t)((D->q.n + 1) & ~1) + FM_DOUBLES) * 8;
}

// n_T batch entries (Tv, nmaxv; a single call is a batch of one): grid.y = n_T, outputs with a leading [n_T] axis
static int lpa_launch(const dfrg_lpa_desc* D, int n_T, const double* Tv, const int* nmaxv, int n_field, const double* rho,
                      const double* u, const double* du, double* flow, double* chan, double* dmin, cudaStream_t stream) {
  LpaParams P;
  P.d = D->d; P.reg_arg4d = D->reg_arg4d; P.nq = D->q.n; P.n_field = n_field;
  P.fermion_reg = D->fermion_reg;
  P.N = D->N; P.prefactor = D->prefactor; P.mu = D->mu;
  size_t smem = 0;
  for (int t = 0; t < LPA_MAX_T; ++t) {
    P.Tv[t] = t < n_T ? Tv[t] : 0.0;
    P.nmaxv[t] = t < n_T ? nmaxv[t] : 0;
    if (t < n_T) {
      dfrg_lpa_desc Dt = *D;
      Dt.T = Tv[t]; Dt.n_max = nmaxv[t];
      const size_t st = lpa_smem(&Dt);
      smem = st > smem ? st : smem;
    }
  }
  P.reg = reg_params(D->reg.kind, D->reg.order, D->reg.k, D->reg.zk, D->reg.eta);
  P.fmc = fm_consts();
  P.xq = D->q.x; P.wq = D->q.w; P.rho = rho; P.u = u; P.du = du;
  P.flow = flow; P.chan = chan; P.dmin = dmin; P.dchan = D->dchan;
  const bool fermi = D->statistics == DFRG_STAT_FERMION;
  auto kern = fermi ? (D->dchan ? lpa_fermion_kernel<true> : lpa_fermion_kernel<false>)
                    : (D->dchan ? lpa_kernel<true> : lpa_kernel<false>);
  if (smem > kMaxDynSmem) return DFRG_EUNSUPPORTED;   // (lpa_validate bounds the table; this is the exact size)
  size_t smem_limit = 0;   // 227 KB minus this kernel's static shared memory (3-6 KB of reduction scratch)
  const int rca = opt_in_max_smem(kern, &smem_limit);
  if (rca != DFRG_OK) return rca;
  if (smem > smem_limit) return DFRG_EUNSUPPORTED;    // nothing enqueued
  const dim3 grid((n_field + LPA_FTILE - 1) / LPA_FTILE, n_T);
  kern<<<grid, LPA_THREADS, smem, stream>>>(P);
  return check_cuda(cudaGetLastError());
}

static int lpa_validate(const dfrg_lpa_desc* D, int n_field, const double* rho, const double* u, const double* du,
                        double* flow) {
  if (!D || !rho || !u || !du || !flow || n_field < 1) return DFRG_EINVAL;
  if (!valid_regulator(D->reg) || !valid_rule(D->q)) return DFRG_EINVAL;
  if (!(D->T >= 0.0) || D->n_max < 0 || !(D->N == D->N)) return DFRG_EINVAL;
  if (D->d < 1 || D->d > 8) return DFRG_EUNSUPPORTED;
  const long long n_terms = (D->T > 0.0) ? (long long)D->n_max + 1 : 1;
  if (D->statistics != DFRG_STAT_BOSON && D->statistics != DFRG_STAT_FERMION) return DFRG_EINVAL;
  if (D->statistics == DFRG_STAT_FERMION) {
    // fermionic frequencies need T > 0; with a chemical potential the time component is complex: spatial regulator only
    if (!(D->T > 0.0) || D->reg_arg4d != 0 || !(D->mu == D->mu)) return DFRG_EINVAL;
    if (n_terms * D->q.n > LPA_MAX_PAIRS / 2) return DFRG_EUNSUPPORTED;
    if (D->fermion_reg != 0 && D->fermion_reg != 1) return DFRG_EINVAL;
  } else if (D->mu != 0.0 || D->fermion_reg != 0) {
    return DFRG_EINVAL;
  }
  if (n_terms * D->q.n > LPA_MAX_PAIRS) return DFRG_EUNSUPPORTED;
  if (lpa_smem(D) > kMaxDynSmem) return DFRG_EUNSUPPORTED;   // the table, the rule and the log/exp tables must fit one CTA
  return DFRG_OK;
}

static int lpa_validate_batch(const dfrg_lpa_desc* D, int n_T, const double* T, const int* n_max, int n_field,
                              const double* rho, const double* u, const double* du, double* flow) {
  if (!D || !T || !n_max || n_T < 1) return DFRG_EINVAL;
  if (n_T > LPA_MAX_T) return DFRG_EUNSUPPORTED;
  for (int t = 0; t < n_T; ++t) {
    dfrg_lpa_desc Dt = *D;
    Dt.T = T[t]; Dt.n_max = n_max[t];
    const int rc = lpa_validate(&Dt, n_field, rho, u, du, flow);
    if (rc != DFRG_OK) return rc;
  }
  return DFRG_OK;
}

}  // namespace dfrg

using namespace dfrg;

extern "C" int dfrg_integrate_lpa_batch(const dfrg_lpa_desc* D, int n_T, const double* T_host, const int* n_max_host,
                                        int n_field, const double* rho, const double* u, const double* du, double* flow,
                                        double* chan, double* dmin, void* cuda_stream) {
  int rc = lpa_validate_batch(D, n_T, T_host, n_max_host, n_field, rho, u, du, flow);
  if (rc != DFRG_OK) return rc;
  rc = require_sm100(nullptr);
  if (rc != DFRG_OK) return rc;
  return lpa_launch(D, n_T, T_host, n_max_host, n_field, rho, u, du, flow, chan, dmin, (cudaStream_t)cuda_stream);
}

extern "C" int dfrg_integrate_lpa(const dfrg_lpa_desc* D, int n_field, const double* rho, const double* u,
                                  const double* du, double* flow, double* chan, double* dmin, void* cuda_stream) {
  int rc = lpa_validate(D, n_field, rho, u, du, flow);
  if (rc != DFRG_OK) return rc;
  rc = require_sm100(nullptr);
  if (rc != DFRG_OK) return rc;
  return lpa_launch(D, 1, &D->T, &D->n_max, n_field, rho, u, du, flow, chan, dmin, (cudaStream_t)cuda_stream);
}

extern "C" int dfrg_integrate_lpa_batch_host(const dfrg_lpa_desc* D, int n_T, const double* T_host, const int* n_max_host,
                                             int n_field, const double* rho, const double* u, const double* du,
                                             double* flow, double* chan, double* dmin) {
  int rc = lpa_validate_batch(D, n_T, T_host, n_max_host, n_field, rho, u, du, flow);
  if (rc != DFRG_OK) return rc;
  rc = require_sm100(nullptr);
  if (rc != DFRG_OK) return rc;
  Arena& A = thread_arena();
  const size_t nf = (size_t)n_field, nq = (size_t)D->q.n, nt = (size_t)n_T;
  rc = A.begin((2 * nq + 3 * nf + 6 * nf * nt) * sizeof(double) + 16 * 256);
  if (rc != DFRG_OK) return rc;
  dfrg_lpa_desc Dd = *D;
  Dd.q.x = A.put(D->q.x, nq);
  Dd.q.w = A.put(D->q.w, nq);
  const double* d_rho = A.put(rho, nf);
  const double* d_u = A.put(u, nf);
  const double* d_du = A.put(du, nf);
  double* d_flow = A.reserve(nt * nf);
  double* d_chan = chan ? A.reserve(2 * nt * nf) : nullptr;
  double* d_dmin = dmin ? A.reserve(nt * nf) : nullptr;
  Dd.dchan = D->dchan ? A.reserve(2 * nt * nf) : nullptr;
  if (A.upload() != DFRG_OK) return A.status();
  rc = lpa_launch(&Dd, n_T, T_host, n_max_host, n_field, d_rho, d_u, d_du, d_flow, d_chan, d_dmin, A.stream());
  if (rc != DFRG_OK) return rc;
  A.fetch(flow, d_flow, nt * nf);
  if (chan) A.fetch(chan, d_chan, 2 * nt * nf);
  if (dmin) A.fetch(dmin, d_dmin, nt * nf);
  if (D->dchan) A.fetch(D->dchan, Dd.dchan, 2 * nt * nf);
  return A.finish();
}

extern "C" int dfrg_integrate_lpa_host(const dfrg_lpa_desc* D, int n_field, const double* rho, const double* u,
                                       const double* du, double* flow, double* chan, double* dmin) {
  int rc = lpa_validate(D, n_field, rho, u, du, flow);
  if (rc != DFRG_OK) return rc;
  rc = require_sm100(nullptr);
  if (rc != DFRG_OK) return rc;
  Arena& A = thread_arena();
  const size_t nf = (size_t)n_field, nq = (size_t)D->q.n;
  rc = A.begin((2 * nq + 3 * nf + 6 * nf) * sizeof(double) + 16 * 256);
  if (rc != DFRG_OK) return rc;
  dfrg_lpa_desc Dd = *D;
  Dd.q.x = A.put(D->q.x, nq);
  Dd.q.w = A.put(D->q.w, nq);
  const double* d_rho = A.put(rho, nf);
  const double* d_u = A.put(u, nf);
  const double* d_du = A.put(du, nf);
  double* d_flow = A.reserve(nf);
  double* d_chan = chan ? A.reserve(2 * nf) : nullptr;
  double* d_dmin = dmin ? A.reserve(nf) : nullptr;
  Dd.dchan = D->dchan ? A.reserve(2 * nf) : nullptr;
  if (A.upload() != DFRG_OK) return A.status();
  rc = lpa_launch(&Dd, 1, &Dd.T, &Dd.n_max, n_field, d_rho, d_u, d_du, d_flow, d_chan, d_dmin, A.stream());
  if (rc != DFRG_OK) return rc;
  A.fetch(flow, d_flow, nf);
  if (chan) A.fetch(chan, d_chan, 2 * nf);
  if (dmin) A.fetch(dmin, d_dmin, nf);
  if (D->dchan) A.fetch(D->dchan, Dd.dchan, 2 * nf);
  return A.finish();
}
