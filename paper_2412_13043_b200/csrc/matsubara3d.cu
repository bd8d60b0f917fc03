// matsubara3d.cu -- dfrg_integrate_matsubara3d: 3-D spatial loop + Matsubara sum (BASELINE.json config 4).
//
// CTA = (external momentum p, external fermion index j, tile of field points); it walks the loop
// Matsubara index n = -n_max..n_max.  Per n:
//   S2: the two table rows it needs (Z_phi row |j-n|, Z_psi row nbar) arrive by TMA bulk copy.
//   S3: the block builds the field-independent node tables in shared memory,
//         inner[i][c] = (D0phi, Nw),  D0phi = Z_phi(r^2) s_phi + R(s_phi),  Nw = wc_c P(y1, y2, y3)
//         outer[i]    = (D0psi, Wpsi), D0psi = Z_psi(q_i^2) s_psi + R(s_psi), Wpsi = wq_i q_i^2 Rdot(s_psi)
//       with P evaluated as a cubic in y2 = p q c/k^2 whose four coefficients depend on (n, i) only.
//   S4: thread = MF field points; per radial node the angular sum A_f = sum_c Nw / (D0phi + m2phi_f)
//       (add -> reciprocal -> FMA; every lane reads the same table entry: shared-memory broadcast),
//       then acc_f += Wpsi G_psi(f)^2 A_f.
//   S5/S6: each thread owns its outputs; sums are sequential in (n, i, c) order per field point.
// dmin: min over nodes of D0 is field independent (fl(D0 + m2) is monotone in D0).
#include "dfrg_device.cuh"
#include "dfrg_internal.h"

namespace dfrg {

constexpr int M3_THREADS = 256;
constexpr int M3_MAX_PAIRS = 6144;

struct Mats3dParams {
  int nq, nc, n_field, n_p, n_jext, n_max;
  double T, prefactor;
  RegParams reg;
  GridParams grid;
  const double *xq, *wq, *xc, *wc, *Zpsi, *Zphi, *coef, *m2psi, *m2phi, *pext;
  double *out, *dmin;
};

template <int MF>
__global__ void __launch_bounds__(M3_THREADS) mats3d_kernel(const Mats3dParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double red[32];
  __shared__ double skap[20];

  const int nq = P.nq, nc = P.nc, npairs = nq * nc, nt = P.grid.n;
  double2* inner = reinterpret_cast<double2*>(smem_raw);  // [nq*nc]
  double2* outer = inner + npairs;                         // [nq]
  double* beta = reinterpret_cast<double*>(outer + nq);    // [nq][4]
  double* sxq = beta + 4 * nq;
  double* swq = sxq + ((nq + 1) & ~1);
  double* sxc = swq + ((nq + 1) & ~1);
  double* swc = sxc + ((nc + 1) & ~1);
  double* rowpsi = swc + ((nc + 1) & ~1);
  double* rowphi = rowpsi + ((nt + 1) & ~1);

  if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  if (threadIdx.x < 20) skap[threadIdx.x] = P.coef[threadIdx.x];
  __syncthreads();
  uint32_t parity = 0;
  {
    StageList L;
    L.add(sxq, P.xq, nq); L.add(swq, P.wq, nq);
    L.add(sxc, P.xc, nc); L.add(swc, P.wc, nc);
    stage_to_smem(L, &bar, parity);
    parity ^= 1;
  }

  const int e = blockIdx.x / P.n_jext, j = blockIdx.x - e * P.n_jext;
  const double p = P.pext[e];
  const double pi = 3.14159265358979323846;
  const double nuj = (2.0 * j + 1.0) * pi * P.T;
  const double ik2 = P.reg.inv_k2;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);

  const int f0 = blockIdx.y * (M3_THREADS * MF) + threadIdx.x;
  double m2psi[MF], m2phi[MF], acc[MF];
#pragma unroll
  for (int m = 0; m < MF; ++m) {
    const int f = f0 + m * M3_THREADS;
    m2psi[m] = (f < P.n_field) ? P.m2psi[f] : 1.0;
    m2phi[m] = (f < P.n_field) ? P.m2phi[f] : 1.0;
    acc[m] = 0.0;
  }
  double dmin_psi = inf, dmin_phi = inf;

  for (int n = -P.n_max; n <= P.n_max; ++n) {
    const int nbar = n >= 0 ? n : -n - 1;
    const int mm = j - n;
    const int mabs = mm >= 0 ? mm : -mm;
    const double nun = (2.0 * n + 1.0) * pi * P.T;
    const double om = 2.0 * pi * (double)mm * P.T;
    const double y1 = nun * nuj * ik2;

    __syncthreads();  // previous hot loop done with inner/outer/rows
    {
      StageList L;
      L.add(rowpsi, P.Zpsi + (size_t)nbar * nt, nt);
      L.add(rowphi, P.Zphi + (size_t)mabs * nt, nt);
      stage_to_smem(L, &bar, parity);
      parity ^= 1;
    }
    // ---- S3a: per radial node ----
    for (int i = threadIdx.x; i < nq; i += M3_THREADS) {
      const double q = sxq[i];
      const double spsi = nun * nun + q * q;
      double R, Rd;
      regulator(P.reg, spsi, R, Rd);
      const double D0 = table_lookup(rowpsi, P.grid, q * q) * spsi + R;
      outer[i] = make_double2(D0, swq[i] * q * q * Rd);
      dmin_psi = fmin(dmin_psi, D0);
      // P = sum_b y2^b beta_b,  beta_b = sum_{a+c<=3-b} kap_abc y1^a y3^c   (idx: a outermost, then b, then c)
      const double y3 = spsi * ik2;
      double be[4] = {0.0, 0.0, 0.0, 0.0};
      int idx = 0;
      double y1a = 1.0;
#pragma unroll
      for (int a = 0; a <= 3; ++a) {
#pragma unroll
        for (int b = 0; b <= 3 - a; ++b) {
          double y3c = y1a;
#pragma unroll
          for (int c = 0; c <= 3 - a - b; ++c) {
            be[b] = fma(skap[idx++], y3c, be[b]);
            y3c *= y3;
          }
        }
        y1a *= y1;
      }
      beta[4 * i + 0] = be[0]; beta[4 * i + 1] = be[1]; beta[4 * i + 2] = be[2]; beta[4 * i + 3] = be[3];
    }
    __syncthreads();
    // ---- S3b: per (radial, angular) node ----
    for (int t = threadIdx.x; t < npairs; t += M3_THREADS) {
      const int i = t / nc, jc = t - i * nc;
      const double q = sxq[i], c = sxc[jc];
      double r2 = p * p + q * q - 2.0 * p * q * c;
      r2 = r2 > 0.0 ? r2 : 0.0;
      const double sphi = om * om + r2;
      double R, Rd;
      regulator(P.reg, sphi, R, Rd);
      const double D0 = table_lookup(rowphi, P.grid, r2) * sphi + R;
      const double y2 = p * q * c * ik2;
      const double poly = fma(fma(fma(beta[4 * i + 3], y2, beta[4 * i + 2]), y2, beta[4 * i + 1]), y2, beta[4 * i]);
      inner[t] = make_double2(D0, swc[jc] * poly);
      dmin_phi = fmin(dmin_phi, D0);
    }
    __syncthreads();

    // ---- S4 ----
    for (int i = 0; i < nq; ++i) {
      const double2* row = inner + i * nc;
      double a[MF];
#pragma unroll
      for (int m = 0; m < MF; ++m) a[m] = 0.0;
#pragma unroll 4
      for (int jc = 0; jc < nc; ++jc) {
        const double2 pr = row[jc];
#pragma unroll
        for (int m = 0; m < MF; ++m) a[m] = fma(pr.y, fast_rcp(pr.x + m2phi[m]), a[m]);
      }
      const double2 o = outer[i];
#pragma unroll
      for (int m = 0; m < MF; ++m) {
        const double g = fast_rcp(o.x + m2psi[m]);
        acc[m] = fma(o.y * (g * g), a[m], acc[m]);
      }
    }
  }

  const double scale = P.prefactor * P.T;
  double dpsi = 0.0, dphi = 0.0;
  if (P.dmin) {
    dpsi = block_min(dmin_psi, red);
    dphi = block_min(dmin_phi, red);
  }
#pragma unroll
  for (int m = 0; m < MF; ++m) {
    const int f = f0 + m * M3_THREADS;
    if (f < P.n_field) {
      const size_t o = (size_t)blockIdx.x * P.n_field + f;
      P.out[o] = scale * acc[m];
      if (P.dmin) P.dmin[o] = fmin(dpsi + m2psi[m], dphi + m2phi[m]) * ik2;
    }
  }
}

static size_t mats3d_smem(int nq, int nc, int nt) {
  return (size_t)nq * nc * 16 + (size_t)nq * 16 +
         8 * (size_t)(4 * nq + 2 * ((nq + 1) & ~1) + 2 * ((nc + 1) & ~1) + 2 * ((nt + 1) & ~1));
}

static int mats3d_validate(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi, const double* m2_phi, int n_p,
                           const double* p, int n_jext, double* out) {
  if (!D || !m2_psi || !m2_phi || !p || !out || n_field < 1 || n_p < 1 || n_jext < 1) return DFRG_EINVAL;
  if (!valid_regulator(D->reg) || !valid_rule(D->q) || !valid_rule(D->cos1) || !D->coef || D->n_coef != 20)
    return DFRG_EINVAL;
  if (!(D->T > 0.0) || D->n_max < 0) return DFRG_EINVAL;
  if (!valid_table(D->tab_psi, D->n_max + 1) || !valid_table(D->tab_phi, n_jext + D->n_max)) return DFRG_EINVAL;
  if (D->tab_psi.n_q != D->tab_phi.n_q || D->tab_psi.lnq_lo != D->tab_phi.lnq_lo ||
      D->tab_psi.lnq_hi != D->tab_phi.lnq_hi || D->tab_psi.interp != D->tab_phi.interp)
    return DFRG_EINVAL;
  if ((long long)D->q.n * D->cos1.n > M3_MAX_PAIRS || D->tab_psi.n_q > 1024) return DFRG_EUNSUPPORTED;
  if ((long long)n_p * n_jext > 2147483647LL) return DFRG_EUNSUPPORTED;
  return DFRG_OK;
}

static int mats3d_launch(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi, const double* m2_phi, int n_p,
                         const double* p, int n_jext, double* out, double* dmin, cudaStream_t stream) {
  Mats3dParams P;
  P.nq = D->q.n; P.nc = D->cos1.n; P.n_field = n_field; P.n_p = n_p; P.n_jext = n_jext; P.n_max = D->n_max;
  P.T = D->T; P.prefactor = D->prefactor;
  P.reg.kind = D->reg.kind; P.reg.order = D->reg.order; P.reg.k2 = D->reg.k * D->reg.k; P.reg.inv_k2 = 1.0 / P.reg.k2;
  P.grid.lo = D->tab_psi.lnq_lo; P.grid.n = D->tab_psi.n_q; P.grid.interp = D->tab_psi.interp;
  P.grid.inv_h = (double)(P.grid.n - 1) / (D->tab_psi.lnq_hi - D->tab_psi.lnq_lo);
  P.xq = D->q.x; P.wq = D->q.w; P.xc = D->cos1.x; P.wc = D->cos1.w;
  P.Zpsi = D->tab_psi.v; P.Zphi = D->tab_phi.v; P.coef = D->coef;
  P.m2psi = m2_psi; P.m2phi = m2_phi; P.pext = p; P.out = out; P.dmin = dmin;
  const size_t smem = mats3d_smem(P.nq, P.nc, P.grid.n);
  const int mf = (n_field > M3_THREADS) ? 2 : 1;
  dim3 grid(n_p * n_jext, (n_field + M3_THREADS * mf - 1) / (M3_THREADS * mf));
  if (grid.y > 65535) return DFRG_EUNSUPPORTED;
  cudaError_t e;
  if (mf == 2) {
    e = cudaFuncSetAttribute(mats3d_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return check_cuda(e);
    mats3d_kernel<2><<<grid, M3_THREADS, smem, stream>>>(P);
  } else {
    e = cudaFuncSetAttribute(mats3d_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return check_cuda(e);
    mats3d_kernel<1><<<grid, M3_THREADS, smem, stream>>>(P);
  }
  return check_cuda(cudaGetLastError());
}

}  // namespace dfrg

using namespace dfrg;

extern "C" int dfrg_integrate_matsubara3d(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi,
                                          const double* m2_phi, int n_p, const double* p, int n_jext, double* out,
                                          double* dmin, void* cuda_stream) {
  int rc = mats3d_validate(D, n_field, m2_psi, m2_phi, n_p, p, n_jext, out);
  if (rc != DFRG_OK) return rc;
  rc = require_sm100(nullptr);
  if (rc != DFRG_OK) return rc;
  return mats3d_launch(D, n_field, m2_psi, m2_phi, n_p, p, n_jext, out, dmin, (cudaStream_t)cuda_stream);
}

extern "C" int dfrg_integrate_matsubara3d_host(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi,
                                               const double* m2_phi, int n_p, const double* p, int n_jext,
                                               double* out, double* dmin) {
  int rc = mats3d_validate(D, n_field, m2_psi, m2_phi, n_p, p, n_jext, out);
  if (rc != DFRG_OK) return rc;
  rc = require_sm100(nullptr);
  if (rc != DFRG_OK) return rc;
  Arena& A = thread_arena();
  const size_t nf = (size_t)n_field, n_out = (size_t)n_p * n_jext * nf;
  const size_t rows_psi = (size_t)D->n_max + 1, rows_phi = (size_t)n_jext + D->n_max, nt = (size_t)D->tab_psi.n_q;
  const size_t need = 2 * ((size_t)D->q.n + D->cos1.n) + (rows_psi + rows_phi) * nt + 20 + 2 * nf + n_p + 2 * n_out;
  rc = A.begin(need * sizeof(double) + 32 * 256);
  if (rc != DFRG_OK) return rc;
  dfrg_mats3d_desc Dd = *D;
  Dd.q.x = A.put(D->q.x, D->q.n); Dd.q.w = A.put(D->q.w, D->q.n);
  Dd.cos1.x = A.put(D->cos1.x, D->cos1.n); Dd.cos1.w = A.put(D->cos1.w, D->cos1.n);
  Dd.tab_psi.v = A.put(D->tab_psi.v, rows_psi * nt);  // only the rows the sum touches
  Dd.tab_phi.v = A.put(D->tab_phi.v, rows_phi * nt);
  Dd.coef = A.put(D->coef, 20);
  const double* d_mpsi = A.put(m2_psi, nf);
  const double* d_mphi = A.put(m2_phi, nf);
  const double* d_p = A.put(p, n_p);
  double* d_out = A.reserve(n_out);
  double* d_dmin = dmin ? A.reserve(n_out) : nullptr;
  if (A.status() != DFRG_OK) return A.status();
  rc = mats3d_launch(&Dd, n_field, d_mpsi, d_mphi, n_p, d_p, n_jext, d_out, d_dmin, A.stream());
  if (rc != DFRG_OK) return rc;
  A.fetch(out, d_out, n_out);
  if (dmin) A.fetch(dmin, d_dmin, n_out);
  return A.finish();
}
