// loop4d.cu -- dfrg_integrate_loop4d: 4-D vacuum loops (BASELINE.json configs 2 and 3, and the SURVEY 8(f) families).
//
// Two-point family.  One persistent warp-specialised kernel: producer warps build the field-independent (D0, W') of
//   the next chunk of radial nodes while the consumers do add -> reciprocal -> FMA over (field point x node), two
//   field points per reciprocal; a fix-up kernel adds the per-CTA partial sums in fixed order.
//
// Three-point family.  No field axis: S3 is the evaluation.  Two paths (see the comments at the kernels):
//   general  -- any list of external configurations (|p1|, |p2|, alpha): persistent CTAs walk the list; thread =
//               (q, c1) pairs, c2 loop inside; the c2-independent part (s_a, G_A(s_a), first vertex factor, the five
//               coefficients of P as a quartic in q.p2) is hoisted out of the c2 loop.
//   product grid -- ext[a S + r] = (|p1|_a, |p2|_r, alpha_r) (dfrg_loop4d_desc::ext_outer): what depends on |p1| alone
//               comes from a pre-pass table, what depends on (|p2|, alpha) alone is built once per work unit in shared
//               memory; one look-up and one Horner evaluation remain per (a, r, node).
//   The integrand has no phi dependence: the phi axis contributes sum_phi w.  Fixed-order sums.
//   With a 3-D vertex table lambda3(S0, a, s) (DFRG_LOOP_THREEPOINT_TAB3D): the same two paths (t3d_kernel for a general
//   list, the product-grid kernels instantiated with TAB3D), the table in shared memory, trilinear look-ups.
//
// Four-point family (DFRG_LOOP_FOURPOINT).  Genuine three-angle kinematics + ghost box: fp4_main_kernel, thread =
//   (q, c1, c2) triple with the phi loop inside (see the comment at the kernel).
#include "loop4d_kernels.cuh"

namespace dfrg {

static int loop4d_validate(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext, const double* ext,
                           double* out) {
  if (!D || !ext || !out || n_ext < 1) return DFRG_EINVAL;
  if (!valid_regulator(D->reg) || !valid_rule(D->q) || !valid_rule(D->cos1) || !D->coef) return DFRG_EINVAL;
  if (D->family == DFRG_LOOP_TWOPOINT) {
    if (n_field < 1 || !m2 || D->n_coef != 2 || !valid_table(D->tab[0], 1)) return DFRG_EINVAL;
    if ((long long)D->q.n * D->cos1.n > TP_MAX_PAIRS || D->cos1.n > TP_CHUNK_NODES || D->tab[0].n_q > 1024)
      return DFRG_EUNSUPPORTED;
    return DFRG_OK;
  }
  if (D->family == DFRG_LOOP_THREEPOINT_TAB3D) {
    if (n_field != 0 || D->n_coef != 35 || !valid_rule(D->cos2) || !valid_rule(D->phi) || D->dout_dm2) return DFRG_EINVAL;
    if (!valid_table(D->tab[0], 1) || !D->tab3d.v) return DFRG_EINVAL;
    long long ntab3 = 1;
    for (int a = 0; a < 3; ++a) {
      if (D->tab3d.n[a] < 2 || !(D->tab3d.hi[a] > D->tab3d.lo[a]) || (D->tab3d.is_log[a] != 0 && D->tab3d.is_log[a] != 1))
        return DFRG_EINVAL;
      ntab3 *= D->tab3d.n[a];
      if (ntab3 > T3D_MAX_TABLE) return DFRG_EUNSUPPORTED;
    }
    if ((long long)D->q.n * D->cos1.n > 65536 || D->tab[0].n_q > 1024 || D->q.n > 4096 || D->cos1.n > 4096 ||
        D->cos2.n > 4096)
      return DFRG_EUNSUPPORTED;
    return DFRG_OK;
  }
  if (D->family == DFRG_LOOP_THREEPOINT || D->family == DFRG_LOOP_FOURPOINT) {
    const bool four = D->family == DFRG_LOOP_FOURPOINT;
    if (n_field != 0 || D->n_coef != (four ? 70 : 35) || !valid_rule(D->cos2) || !valid_rule(D->phi) || D->dout_dm2)
      return DFRG_EINVAL;
    for (int t = 0; t < 3; ++t)
      if (!valid_table(D->tab[t], 1)) return DFRG_EINVAL;
    for (int t = 1; t < 3; ++t)
      if (D->tab[t].n_q != D->tab[0].n_q || D->tab[t].lnq_lo != D->tab[0].lnq_lo ||
          D->tab[t].lnq_hi != D->tab[0].lnq_hi || D->tab[t].interp != D->tab[0].interp)
        return DFRG_EINVAL;
    if ((long long)D->q.n * D->cos1.n > 65536 || D->tab[0].n_q > 1024 || D->q.n > 4096 || D->cos1.n > 4096 ||
        D->cos2.n > 4096)
      return DFRG_EUNSUPPORTED;
    if (four && (D->cos2.n > FP4_THREADS || D->phi.n > 4096)) return DFRG_EUNSUPPORTED;
    return DFRG_OK;
  }
  return DFRG_EINVAL;
}


static int loop4d_launch(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext, const double* ext,
                         double* out, double* dmin, int sm_count, cudaStream_t stream) {
  if (D->family == DFRG_LOOP_TWOPOINT) return twopoint_launch(D, n_field, m2, n_ext, ext, out, dmin, sm_count, stream);
  if (D->family == DFRG_LOOP_FOURPOINT) return fourpoint_launch(D, n_ext, ext, out, dmin, sm_count, stream);
  ThreePointParams P;
  P.nq = D->q.n; P.n1 = D->cos1.n; P.n2 = D->cos2.n; P.nphi = D->phi.n; P.n_ext = n_ext;
  P.prefactor = D->prefactor;
  fill_common(D->reg, D->tab[0], &P.reg, &P.grid);
  P.fmc = fm_consts();
  P.xq = D->q.x; P.wq = D->q.w; P.x1 = D->cos1.x; P.w1 = D->cos1.w; P.x2 = D->cos2.x; P.w2 = D->cos2.w; P.wphi = D->phi.w;
  P.ZA = D->tab[0].v; P.L3 = D->tab[2].v; P.coef = D->coef; P.ext = ext; P.out = out; P.dmin = dmin;
  P.skip_flag = nullptr;
  const int regk = regulator_variant(D->reg);
  void* scratch = nullptr;
  int rc;
  if (D->family == DFRG_LOOP_THREEPOINT_TAB3D) {
    ThreePoint3DParams Q3;
    Q3.v3 = D->tab3d.v;
    int ntab3 = 1;
    for (int a = 0; a < 3; ++a) {
      Q3.T.n[a] = D->tab3d.n[a]; Q3.T.is_log[a] = D->tab3d.is_log[a]; Q3.T.lo[a] = D->tab3d.lo[a];
      Q3.T.inv_h[a] = (double)(D->tab3d.n[a] - 1) / (D->tab3d.hi[a] - D->tab3d.lo[a]);
      ntab3 *= D->tab3d.n[a];
    }
    if (threepoint3d_general_smem(P.nq, P.n1, P.n2, P.grid.n, ntab3) > kMaxDynSmem) return DFRG_EUNSUPPORTED;
    // product grid promised (ext_outer): share the |p1|-only and (|p2|, alpha)-only vertices as the 1-D family does
    rc = t3g_launch(P, D->ext_outer, regk, &Q3.T, Q3.v3, ntab3, sm_count, stream, &scratch);
    if (rc != DFRG_OK) return rc;
    Q3.B = P;   // with skip_flag as t3g_launch left it
    rc = threepoint3d_general_launch(Q3, regk, sm_count, stream);
  } else {
    if (threepoint_general_smem(P.nq, P.n1, P.n2, P.grid.n) > kMaxDynSmem) return DFRG_EUNSUPPORTED;   // before anything is enqueued
    // product-grid path (ext_outer = G promised by the caller, checked on the device)
    rc = t3g_launch(P, D->ext_outer, regk, nullptr, nullptr, 0, sm_count, stream, &scratch);
    if (rc != DFRG_OK) return rc;   // P.skip_flag is set if the product-grid kernels were enqueued
    rc = threepoint_general_launch(P, regk, sm_count, stream);
  }
  scratch_free(scratch, stream);
  return rc;
}

}  // namespace dfrg

using namespace dfrg;

extern "C" int dfrg_integrate_loop4d(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext,
                                     const double* ext, double* out, double* dmin, void* cuda_stream) {
  int rc = loop4d_validate(D, n_field, m2, n_ext, ext, out);
  if (rc != DFRG_OK) return rc;
  int sms = 0;
  rc = require_sm100(&sms);
  if (rc != DFRG_OK) return rc;
  return loop4d_launch(D, n_field, m2, n_ext, ext, out, dmin, sms, (cudaStream_t)cuda_stream);
}

extern "C" int dfrg_integrate_loop4d_host(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext,
                                          const double* ext, double* out, double* dmin) {
  int rc = loop4d_validate(D, n_field, m2, n_ext, ext, out);
  if (rc != DFRG_OK) return rc;
  int sms = 0;
  rc = require_sm100(&sms);
  if (rc != DFRG_OK) return rc;
  Arena& A = thread_arena();
  const bool two = D->family == DFRG_LOOP_TWOPOINT;
  const size_t nf = two ? (size_t)n_field : 1, ne = (size_t)n_ext,
               next_d = two ? ne : (D->family == DFRG_LOOP_FOURPOINT ? 6 * ne : 3 * ne);
  // the two-point family does not use (and loop4d_validate does not look at) the cos2 / phi axes
  size_t need = 2 * ((size_t)D->q.n + D->cos1.n + (two ? 0 : (size_t)D->cos2.n + D->phi.n)) + 3 * (size_t)D->tab[0].n_q + 128 +
                nf + next_d +
                (D->family == DFRG_LOOP_THREEPOINT_TAB3D ? (size_t)T3D_MAX_TABLE + 16 : 0) +
                3 * ne * nf;
  rc = A.begin(need * sizeof(double) + 32 * 256);
  if (rc != DFRG_OK) return rc;
  dfrg_loop4d_desc Dd = *D;
  Dd.q.x = A.put(D->q.x, D->q.n); Dd.q.w = A.put(D->q.w, D->q.n);
  Dd.cos1.x = A.put(D->cos1.x, D->cos1.n); Dd.cos1.w = A.put(D->cos1.w, D->cos1.n);
  if (!two) {
    Dd.cos2.x = A.put(D->cos2.x, D->cos2.n); Dd.cos2.w = A.put(D->cos2.w, D->cos2.n);
    Dd.phi.x = A.put(D->phi.x, D->phi.n); Dd.phi.w = A.put(D->phi.w, D->phi.n);
  }
  const bool tab3d = D->family == DFRG_LOOP_THREEPOINT_TAB3D;
  for (int t = 0; t < ((two || tab3d) ? 1 : 3); ++t) Dd.tab[t].v = A.put(D->tab[t].v, D->tab[t].n_q);
  if (tab3d) Dd.tab3d.v = A.put(D->tab3d.v, (size_t)D->tab3d.n[0] * D->tab3d.n[1] * D->tab3d.n[2]);
  Dd.coef = A.put(D->coef, D->n_coef);
  const double* d_m2 = two ? A.put(m2, nf) : nullptr;
  const double* d_ext = A.put(ext, next_d);
  double* d_out = A.reserve(ne * nf);
  double* d_dmin = dmin ? A.reserve(ne * nf) : nullptr;
  Dd.dout_dm2 = D->dout_dm2 ? A.reserve(ne * nf) : nullptr;
  if (A.upload() != DFRG_OK) return A.status();
  rc = loop4d_launch(&Dd, n_field, d_m2, n_ext, d_ext, d_out, d_dmin, sms, A.stream());
  if (rc != DFRG_OK) return rc;
  A.fetch(out, d_out, ne * nf);
  if (dmin) A.fetch(dmin, d_dmin, ne * nf);
  if (D->dout_dm2) A.fetch(D->dout_dm2, Dd.dout_dm2, ne * nf);
  return A.finish();
}

