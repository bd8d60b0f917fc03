// matsubara3d.cu -- dfrg_integrate_matsubara3d: 3-D spatial loop + Matsubara sum (BASELINE.json config 4): host side
// (validation, plan, scratch, launches) and the C entry points.  Kernels: matsubara3d_kernels.cuh.
//
// Launches per call, all on the caller's stream:
//  (1) mats3d_phi_rows_kernel  (S3, field independent)   D0phi[p][i][m][c] = Z_phi(r^2; row m) s_phi + R,  m = 0 .. n_jext-1+n_max
//      The boson denominator depends on the external and loop Matsubara indices only through |j - n|: the 16 x 23 (j, n)
//      combinations of config 4 share 27 rows per momentum p.  Also checks whether the cos rule is exactly symmetric.
//  (2) mats3d_psi_kernel       (S3)   psi[n][i] = (D0psi, Wpsi)  (+ Im D0psi at mu != 0)
//  (3) one moment kernel per requested output (value, d/dm2_psi, d/dm2_phi), chosen by the plan below:
//        mats3d_moment_kernel   specialised (n_max, n_jext) = (11,16), (3,3): compile-time pair code behind a jump table
//        mats3d_gmoment_kernel  any (n_max, n_jext <= 32)
//        mats3d_cmoment_kernel  mu != 0: complex fermion line
//        mats3d_main_kernel     n_jext > 32: row-streaming kernel without the moment factorisation
//      The symmetric-pair and the plain instantiation of a moment kernel are both enqueued; the one that does not match
//      the device-side symmetry flag returns at once.
//  (4) mats3d_fixup_kernel     (S5/S6) adds the per-CTA partial sums in slot order, writes out (and out_im), dmin.
// dmin: fl(D0 + m2) is monotone in D0, so the minimum over nodes is (min D0) + m2: no hot-loop work (|D_psi| per field
// point at mu != 0: mats3d_psimin_cplx_kernel).
#include "matsubara3d_kernels.cuh"

namespace dfrg {

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
  if ((long long)n_p * n_jext > 2147483647LL || n_p > 65535) return DFRG_EUNSUPPORTED;
  if ((D->reg_arg4d != 0 && D->reg_arg4d != 1) || !(D->mu == D->mu)) return DFRG_EINVAL;
  if (D->fermion_reg != 0 && D->fermion_reg != 1) return DFRG_EINVAL;
  if (D->path < 0 || D->path > 63) return DFRG_EINVAL;
  if (D->mu != 0.0) {
    if (D->reg_arg4d != 0 || !D->out_im) return DFRG_EINVAL;   // complex time component: spatial regulators only
    if ((D->dout_dm2_psi && !D->dout_dm2_psi_im) || (D->dout_dm2_phi && !D->dout_dm2_phi_im)) return DFRG_EINVAL;
    if (n_jext > 32) return DFRG_EUNSUPPORTED;
  }
  return DFRG_OK;
}

template <int GROUPS, int MF>
static int mats3d_launch_main(const Mats3dParams& P, int sm_count, cudaStream_t stream) {
  const size_t smem = mats3d_main_smem(P.nq, P.nc, P.row_stride, P.psi_stride, GROUPS, MF);
  if (smem > kMaxDynSmem) return DFRG_EUNSUPPORTED;
  auto kern = P.mode == 2 ? mats3d_main_kernel<GROUPS, MF, true> : mats3d_main_kernel<GROUPS, MF, false>;
  const int rca = opt_in_max_smem(kern);
  if (rca != DFRG_OK) return rca;
  const long long n_ftiles = (P.n_field + M3_FT * MF - 1) / (M3_FT * MF);
  const long long n_items = (long long)P.n_p * P.n_jext * n_ftiles;
  const int grid = (int)(n_items < sm_count ? n_items : sm_count);
  kern<<<grid, GROUPS * M3_FT + 32, smem, stream>>>(P);
  return check_cuda(cudaGetLastError());
}

// ---- moment-path dispatch: (n_max, n_jext) pairs with a compiled (specialised) instantiation --------------------
// The instantiations live in matsubara3d_moment_sym.cu / matsubara3d_moment_plain.cu (symmetric-pair and plain moment
// loops; separate translation units so that nvcc builds them side by side); DFRG_M3_SHAPES is in the kernel header.
int mats3d_moment_launch_sym(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream);
int mats3d_moment_launch_plain(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream);

static bool mats3d_moment_shape(int n_max, int n_jext) {
#define X(a, b) if (n_max == a && n_jext == b) return true;
  DFRG_M3_SHAPES(X)
#undef X
  return false;
}
static int mats3d_moment_dispatch(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream) {
  // symmetric-pair instantiation first (runs iff the pre-pass found the cos rule symmetric), then the plain one
  if (P.sym_try) {
    const int rc = mats3d_moment_launch_sym(P, pl, stream);
    if (rc != DFRG_OK) return rc;
  }
  return mats3d_moment_launch_plain(P, pl, stream);
}

// any-shape moment kernel: compiled in matsubara3d_anyshape.cu (its own translation unit: the two sets of kernel
// instantiations build side by side)
int mats3d_gmoment_dispatch(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream);
int mats3d_cmoment_dispatch(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream);   // mu != 0 (complex fermion line)

static int mats3d_launch(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi, const double* m2_phi, int n_p,
                         const double* p, int n_jext, double* out, double* dmin, int sm_count, cudaStream_t stream) {
  Mats3dParams P;
  P.nq = D->q.n; P.nc = D->cos1.n; P.n_field = n_field; P.n_p = n_p; P.n_jext = n_jext; P.n_max = D->n_max;
  P.n_rows = n_jext + D->n_max;
  const int npairs = P.nq * P.nc;
  P.row_stride = (npairs + 1) & ~1;  // TMA bulk copies move multiples of 16 bytes
  P.chunk_stride = (P.n_rows * P.nc + 1) & ~1;
  P.psi_stride = P.nq;
  P.T = D->T; P.prefactor = D->prefactor;
  P.reg = reg_params(D->reg.kind, D->reg.order, D->reg.k, D->reg.zk, D->reg.eta);
  P.grid.lo = D->tab_psi.lnq_lo; P.grid.n = D->tab_psi.n_q; P.grid.interp = D->tab_psi.interp;
  P.grid.inv_h = (double)(P.grid.n - 1) / (D->tab_psi.lnq_hi - D->tab_psi.lnq_lo);
  P.fmc = fm_consts();
  P.xq = D->q.x; P.wq = D->q.w; P.xc = D->cos1.x; P.wc = D->cos1.w;
  P.Zpsi = D->tab_psi.v; P.Zphi = D->tab_phi.v; P.coef = D->coef;
  P.m2psi = m2_psi; P.m2phi = m2_phi; P.pext = p; P.out = out; P.dmin = dmin;
  P.part = nullptr; P.tile_fields = 0; P.max_slots = 0; P.grid_main = 0; P.mode = 0; P.sym_try = 0; P.symflag = nullptr;
  P.reg_arg4d = D->reg_arg4d; P.mu = D->mu; P.fermion_reg = D->fermion_reg;
  P.psi_im = nullptr; P.psimin_f = nullptr; P.out_im = nullptr; P.part_im = nullptr;
  const bool cplx = D->mu != 0.0;

  // ---- path: moment factorisation wherever it applies; dfrg_mats3d_desc::path overrides (testing / tuning) ----
  const int path = D->path;
  bool moment = n_jext <= 32 && (cplx || !(path & DFRG_M3_ROW_STREAMING));
  MomentPlan pl = {};
  pl.any_shape_forced = (path & DFRG_M3_ANY_SHAPE) != 0;
  if (moment) {
    pl.generic = !mats3d_moment_shape(D->n_max, n_jext) || (path & DFRG_M3_ANY_SHAPE);
    pl.variant = n_field <= 256 ? 2 : ((path & DFRG_M3_ONE_FIELD) ? 1 : 0);   // MF 2 x 256, MF 1 x 512, MF 1 x 256 threads
    if (pl.generic && (n_jext > 16 || pl.variant == 1)) pl.variant = 2;  // any-shape kernel: 256 threads only
    if (cplx) { pl.generic = true; pl.variant = 2; }                     // complex kernel: one field point per thread
    pl.tile = pl.variant == 2 ? 256 : 512;
    const int n_ftiles = (n_field + pl.tile - 1) / pl.tile;
    const long long upp = (long long)n_p * P.nq, U = (long long)n_ftiles * upp;
    pl.grid = (int)(U < sm_count ? U : sm_count);
    pl.max_slots = 1;
    for (long long seg = 0; seg < (long long)n_ftiles * n_p; ++seg) {
      const long long ufirst = seg * P.nq, ulast = ufirst + P.nq - 1;
      const int c0 = (int)(((ufirst + 1) * pl.grid - 1) / U), c1 = (int)(((ulast + 1) * pl.grid - 1) / U);
      if (c1 - c0 + 1 > pl.max_slots) pl.max_slots = c1 - c0 + 1;
    }
    pl.smem = 8 * (size_t)(2 * P.chunk_stride + 2 * n_jext * (2 * D->n_max + 1) * 4 + 4 * (D->n_max + 1) + 4 * P.nc + P.nq);
    if (pl.generic)   // + the thread-private columns of H
      pl.smem += 8 * ((size_t)(D->n_max + 1) * 256 * (pl.variant == 0 ? 2 : 1) + 2);
    if (cplx)         // beta' and H are complex: twice the shared memory for both
      pl.smem = 8 * (size_t)(2 * P.chunk_stride + 2 * n_jext * (2 * D->n_max + 1) * 8 + 4 * (D->n_max + 1) + 4 * P.nc +
                             ((P.nq + 1) & ~1) + 2 * (size_t)(D->n_max + 1) * 256 + 2);
    if (pl.smem > 220 * 1024) {
      if (cplx) return DFRG_EUNSUPPORTED;
      moment = false;
    }
  }
  P.phi_layout = moment ? 1 : 0;
  P.sym_try = (moment && (P.nc % (2 * M3_NBAT)) == 0 && !(path & DFRG_M3_PLAIN_MOMENTS)) ? 1 : 0;
  P.tile_fields = pl.tile; P.max_slots = pl.max_slots; P.grid_main = pl.grid;

  const int n_terms = 2 * D->n_max + 1;
  const size_t n_d0 = moment ? (size_t)n_p * P.nq * P.chunk_stride : (size_t)n_p * P.n_rows * P.row_stride;
  const size_t n_rowmin = ((size_t)n_p * P.n_rows + 1) & ~(size_t)1;
  const size_t n_psi = (size_t)n_terms * P.psi_stride * 2;
  const size_t n_psimin = ((size_t)n_terms + 1) & ~(size_t)1;
  const size_t n_part = moment ? (size_t)pl.max_slots * n_p * n_jext * n_field : 0;
  const size_t n_cplx = cplx ? n_part + (size_t)n_terms * P.psi_stride + (((size_t)n_field + 1) & ~(size_t)1) : 0;
  void* scratch = nullptr;
  int rc = scratch_alloc(&scratch, (n_d0 + n_rowmin + n_psi + n_psimin + n_part + 2 + n_cplx) * sizeof(double), stream);
  if (rc != DFRG_OK) return rc;
  P.d0phi = (double*)scratch;
  P.psi = (double2*)(P.d0phi + n_d0);
  P.rowmin = (double*)(P.psi) + n_psi;
  P.psimin = P.rowmin + n_rowmin;
  P.part = P.psimin + n_psimin;
  P.symflag = (int*)(P.part + n_part);
  if (cplx) {
    P.part_im = P.part + n_part + 2;
    P.psi_im = P.part_im + n_part;
    P.psimin_f = P.psi_im + (size_t)n_terms * P.psi_stride;
    P.out_im = D->out_im;
  } else {   // real results: the imaginary parts are zero
    double* const zero_fill[3] = {D->out_im, D->dout_dm2_psi ? D->dout_dm2_psi_im : nullptr,
                                  D->dout_dm2_phi ? D->dout_dm2_phi_im : nullptr};
    for (int z = 0; z < 3 && rc == DFRG_OK; ++z)
      if (zero_fill[z])
        rc = check_cuda(cudaMemsetAsync(zero_fill[z], 0, (size_t)n_p * n_jext * n_field * sizeof(double), stream));
    if (rc != DFRG_OK) { scratch_free(scratch, stream); return rc; }
  }

  mats3d_phi_rows_kernel<<<dim3(P.n_rows, n_p), M3_PRE_THREADS, 0, stream>>>(P);
  rc = check_cuda(cudaGetLastError());
  if (rc == DFRG_OK) {
    mats3d_psi_kernel<<<n_terms, 128, 0, stream>>>(P);
    rc = check_cuda(cudaGetLastError());
  }
  if (rc == DFRG_OK && cplx && dmin) {
    mats3d_psimin_cplx_kernel<<<(n_field + 127) / 128, 128, 0, stream>>>(P);
    rc = check_cuda(cudaGetLastError());
  }
  // one pass for the values, one more for each requested mass derivative (same kernels, mode 1 / 2)
  double* const pass_out[3] = {out, D->dout_dm2_psi, D->dout_dm2_phi};
  double* const pass_out_im[3] = {D->out_im, D->dout_dm2_psi_im, D->dout_dm2_phi_im};
  for (int mode = 0; mode < 3 && rc == DFRG_OK; ++mode) {
    if (!pass_out[mode]) continue;
    P.mode = mode;
    P.out = pass_out[mode];
    P.out_im = cplx ? pass_out_im[mode] : nullptr;
    P.dmin = mode == 0 ? dmin : nullptr;
    if (moment) {
      rc = cplx ? mats3d_cmoment_dispatch(P, pl, stream)
                : (pl.generic ? mats3d_gmoment_dispatch(P, pl, stream) : mats3d_moment_dispatch(P, pl, stream));
      if (rc == DFRG_OK) {
        const long long n_out = (long long)n_p * n_jext * n_field;
        mats3d_fixup_kernel<<<(unsigned)((n_out + 255) / 256), 256, 0, stream>>>(P);
        rc = check_cuda(cudaGetLastError());
      }
    } else {
      // row-streaming path: consumer groups per CTA (radial nodes are dealt round-robin to the groups) and field points
      // per thread; dfrg_mats3d_desc::path overrides the defaults
      int mf = n_field > 2 * M3_FT ? 4 : (n_field > M3_FT ? 2 : 1);
      if (path & DFRG_M3_ONE_FIELD) mf = 1;
      const int groups = (path & DFRG_M3_GROUPS_7) ? 7 : ((path & DFRG_M3_GROUPS_4) ? 4 : 6);
      if (mf == 4) {
        if (groups == 7) rc = mats3d_launch_main<7, 4>(P, sm_count, stream);
        else if (groups == 4) rc = mats3d_launch_main<4, 4>(P, sm_count, stream);
        else rc = mats3d_launch_main<6, 4>(P, sm_count, stream);
      } else if (mf == 2) {
        if (groups == 7) rc = mats3d_launch_main<7, 2>(P, sm_count, stream);
        else if (groups == 4) rc = mats3d_launch_main<4, 2>(P, sm_count, stream);
        else rc = mats3d_launch_main<6, 2>(P, sm_count, stream);
      } else {
        rc = mats3d_launch_main<4, 1>(P, sm_count, stream);
      }
    }
  }
  scratch_free(scratch, stream);
  return rc;
}

}  // namespace dfrg

using namespace dfrg;

extern "C" int dfrg_integrate_matsubara3d(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi,
                                          const double* m2_phi, int n_p, const double* p, int n_jext, double* out,
                                          double* dmin, void* cuda_stream) {
  int rc = mats3d_validate(D, n_field, m2_psi, m2_phi, n_p, p, n_jext, out);
  if (rc != DFRG_OK) return rc;
  int sms = 0;
  rc = require_sm100(&sms);
  if (rc != DFRG_OK) return rc;
  return mats3d_launch(D, n_field, m2_psi, m2_phi, n_p, p, n_jext, out, dmin, sms, (cudaStream_t)cuda_stream);
}

extern "C" int dfrg_integrate_matsubara3d_host(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi,
                                               const double* m2_phi, int n_p, const double* p, int n_jext,
                                               double* out, double* dmin) {
  int rc = mats3d_validate(D, n_field, m2_psi, m2_phi, n_p, p, n_jext, out);
  if (rc != DFRG_OK) return rc;
  int sms = 0;
  rc = require_sm100(&sms);
  if (rc != DFRG_OK) return rc;
  Arena& A = thread_arena();
  const size_t nf = (size_t)n_field, n_out = (size_t)n_p * n_jext * nf;
  const size_t rows_psi = (size_t)D->n_max + 1, rows_phi = (size_t)n_jext + D->n_max, nt = (size_t)D->tab_psi.n_q;
  const size_t need = 2 * ((size_t)D->q.n + D->cos1.n) + (rows_psi + rows_phi) * nt + 20 + 2 * nf + n_p + 7 * n_out;
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
  Dd.dout_dm2_psi = D->dout_dm2_psi ? A.reserve(n_out) : nullptr;
  Dd.dout_dm2_phi = D->dout_dm2_phi ? A.reserve(n_out) : nullptr;
  Dd.out_im = D->out_im ? A.reserve(n_out) : nullptr;
  Dd.dout_dm2_psi_im = D->dout_dm2_psi_im ? A.reserve(n_out) : nullptr;
  Dd.dout_dm2_phi_im = D->dout_dm2_phi_im ? A.reserve(n_out) : nullptr;
  if (A.upload() != DFRG_OK) return A.status();
  rc = mats3d_launch(&Dd, n_field, d_mpsi, d_mphi, n_p, d_p, n_jext, d_out, d_dmin, sms, A.stream());
  if (rc != DFRG_OK) return rc;
  A.fetch(out, d_out, n_out);
  if (dmin) A.fetch(dmin, d_dmin, n_out);
  if (D->dout_dm2_psi) A.fetch(D->dout_dm2_psi, Dd.dout_dm2_psi, n_out);
  if (D->dout_dm2_phi) A.fetch(D->dout_dm2_phi, Dd.dout_dm2_phi, n_out);
  if (D->out_im) A.fetch(D->out_im, Dd.out_im, n_out);
  if (D->dout_dm2_psi && D->dout_dm2_psi_im) A.fetch(D->dout_dm2_psi_im, Dd.dout_dm2_psi_im, n_out);
  if (D->dout_dm2_phi && D->dout_dm2_phi_im) A.fetch(D->dout_dm2_phi_im, Dd.dout_dm2_phi_im, n_out);
  return A.finish();
}
