// loop4d_fourpoint.cu -- four-point box family of dfrg_integrate_loop4d (DFRG_LOOP_FOURPOINT, reading A21).
#include "loop4d_kernels.cuh"

namespace dfrg {

// =====================================================================================================
// four-point box: genuine three-angle kinematics + ghost loop (include/dfrg.h, DFRG_LOOP_FOURPOINT)
// =====================================================================================================
// Every node of the (q, c1, c2, phi) grid is a distinct evaluation.  Persistent CTAs; work unit = (external
// configuration e, chunk of KP (q, c1) pairs); thread = one (q, c1, c2) triple of the unit, phi loop inside.
// Per triple (outside the phi loop): s_a, s_b and everything that hangs on them -- G_A, G_c at q^2, s_a, s_b, the
// vertex factors l3(l1) l3(l2) -- folded into the four coefficients of each polynomial as a cubic in
// x3 = q.p3/k^2 = X3c + X3s cos(phi).  Per node: s_d, e^-x, one log-grid coordinate serving Z_A and Z_c, two more
// look-ups for l3(l3) l3(l4), ONE reciprocal 1/(D_A D_c) serving both boxes, two Horner cubics.  All tables are the
// conflict-free replicated shared-memory tables of the three-point kernels.  Fixed-order sums: per-thread sequential,
// block tree per (CTA, e), per-CTA partial sums added in slot order by fp4_fixup_kernel.

static size_t fp4_smem(int nq, int n1, int n2, int nphi, int nt) {
  return 8 * (size_t)(2 * ((nq + 1) & ~1) + 2 * ((n1 + 1) & ~1) + 2 * ((n2 + 1) & ~1) + 3 * ((nt + 1) & ~1) + 72 +
                      FM_DOUBLES + FX_DOUBLES + LG_DOUBLES + 3 * cells_guarded_size(nt) * 2 + 4 * nq + 2 * nphi + 16);
}

template <int REGK, bool WANT_DMIN>
__global__ void __launch_bounds__(FP4_THREADS, 1) fp4_main_kernel(const FourPointParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double red[32];
  const int nq = P.nq, n1 = P.n1, n2 = P.n2, nphi = P.nphi, nt = P.grid.n, KP = P.KP, NCH = P.NCH;
  const int npairs = nq * n1;
  const int tid = threadIdx.x;
  double* sxq = reinterpret_cast<double*>(smem_raw);
  double* swq = sxq + ((nq + 1) & ~1);
  double* sx1 = swq + ((nq + 1) & ~1);
  double* sw1 = sx1 + ((n1 + 1) & ~1);
  double* sx2 = sw1 + ((n1 + 1) & ~1);
  double* sw2 = sx2 + ((n2 + 1) & ~1);
  double* sZA = sw2 + ((n2 + 1) & ~1);
  double* sZc = sZA + ((nt + 1) & ~1);
  double* sL3 = sZc + ((nt + 1) & ~1);
  double* skap = sL3 + ((nt + 1) & ~1);   // 70 (+2)
  double* fmmem = skap + 72;
  double* fxmem = fmmem + FM_DOUBLES;
  double* lgmem = fxmem + FX_DOUBLES;
  double2* cA_all = reinterpret_cast<double2*>(lgmem + LG_DOUBLES);
  double2* cC_all = cA_all + cells_guarded_size(nt);
  double2* cL_all = cC_all + cells_guarded_size(nt);
  double4* qtab = reinterpret_cast<double4*>(cL_all + cells_guarded_size(nt));  // [nq] (W G_A(q^2), W G_c(q^2), D_A, D_c)
  double2* phitab = reinterpret_cast<double2*>(qtab + nq);                       // [nphi] (cos phi, w)
  double* ec = reinterpret_cast<double*>(phitab + nphi);                         // [16] per-e constants

  if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  __syncthreads();
  {
    StageList L;
    L.add(sxq, P.xq, nq); L.add(swq, P.wq, nq);
    L.add(sx1, P.x1, n1); L.add(sw1, P.w1, n1);
    L.add(sx2, P.x2, n2); L.add(sw2, P.w2, n2);
    stage_to_smem(L, &bar, 0);
  }
  {
    StageList L;
    L.add(sZA, P.ZA, nt); L.add(sZc, P.Zc, nt); L.add(sL3, P.L3, nt);
    stage_to_smem(L, &bar, 1);
  }
  const FastMath fm = fm_build(fmmem, P.fmc);
  const double* fxtab = fx_build(fxmem, P.reg.zk * P.reg.k2);
  const LogGrid lg = lg_build(lgmem, P.grid.lo, P.grid.inv_h, nt);
  const double* kc = P.fmc.c;
  const double2* cA = cells_build_guarded(cA_all, sZA, nt, P.grid.interp);
  const double2* cC = cells_build_guarded(cC_all, sZc, nt, P.grid.interp);
  const double2* cL = cells_build_guarded(cL_all, sL3, nt, P.grid.interp);
  for (int j = tid; j < 70; j += FP4_THREADS) skap[j] = P.coef[j];
  for (int j = tid; j < nphi; j += FP4_THREADS) phitab[j] = make_double2(cos(P.xphi[j]), P.wphi[j]);
  __syncthreads();

  const double ik2 = P.reg.inv_k2, k2 = P.reg.k2, third = 1.0 / 3.0;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  // radial table: what depends on q alone
  double dmq = inf;
  for (int i = tid; i < nq; i += FP4_THREADS) {
    const double q = sxq[i], sq = q * q;
    double Rq, Rdq;
    regulator(P.reg, fm, sq, Rq, Rdq);
    const double t = lg_coord(lg, kc, sq);
    const double DA = fma(lg_cell_eval(cA, lg, t), sq, Rq), DC = fma(lg_cell_eval(cC, lg, t), sq, Rq);
    const double W = swq[i] * q * q * q * Rdq;
    qtab[i] = make_double4(W * fast_rcp(DA), W * fast_rcp(DC), DA, DC);
    dmq = fmin(dmq, fmin(DA, DC));
  }
  dmq = block_min(dmq, red);  // also publishes qtab

  const long long U = (long long)P.n_ext * NCH;
  const long long u0 = (long long)blockIdx.x * U / gridDim.x, u1 = (long long)(blockIdx.x + 1) * U / gridDim.x;
  int cur_e = -1;
  double acc = 0.0, dm = dmq;
  for (long long u = u0; u < u1; ++u) {
    const int e = (int)(u / NCH), ch = (int)(u - (long long)e * NCH);
    if (e != cur_e) {
      cur_e = e;
      __syncthreads();   // everybody is done with the previous e's constants
      if (tid == 0) {
        const double p1 = P.ext[6 * e], p2 = P.ext[6 * e + 1], p3 = P.ext[6 * e + 2];
        double sa_, ca_, sb_, cb_, sg_, cg_;
        sincos(P.ext[6 * e + 3], &sa_, &ca_);
        sincos(P.ext[6 * e + 4], &sb_, &cb_);
        sincos(P.ext[6 * e + 5], &sg_, &cg_);
        const double p1p2 = p1 * p2 * ca_, p1p3 = p1 * p3 * cb_, p2p3 = p2 * p3 * (ca_ * cb_ + sa_ * sb_ * cg_);
        double s12 = p1 * p1 + p2 * p2 + 2.0 * p1p2;
        double s123 = p1 * p1 + p2 * p2 + p3 * p3 + 2.0 * (p1p2 + p1p3 + p2p3);
        s12 = s12 > 0.0 ? s12 : 0.0;
        s123 = s123 > 0.0 ? s123 : 0.0;
        ec[0] = p1; ec[1] = p2; ec[2] = p3; ec[3] = ca_; ec[4] = sa_; ec[5] = cb_; ec[6] = sb_ * cg_; ec[7] = sb_ * sg_;
        ec[8] = s12; ec[9] = s123;
      }
      __syncthreads();
    }
    const int pair0 = ch * KP;
    const int npl = min(KP, npairs - pair0);
    if (tid < npl * n2) {
      const int pl = tid / n2, j2 = tid - pl * n2;
      const int pair = pair0 + pl;
      const int i = pair / n1, j1 = pair - i * n1;
      const double p1 = ec[0], p2 = ec[1], p3 = ec[2], ca_ = ec[3], sa_ = ec[4], cb_ = ec[5], sbcg = ec[6], sbsg = ec[7];
      const double s12 = ec[8], s123 = ec[9];
      const double q = sxq[i], c1 = sx1[j1], c2 = sx2[j2];
      const double sq = q * q;
      const double sin1 = sqrt((1.0 - c1) * (1.0 + c1)), sin2 = sqrt((1.0 - c2) * (1.0 + c2));
      const double4 qt = qtab[i];
      const double wnode = (sw1[j1] * sin1) * sw2[j2];
      // ---- the (q, c1) and (q, c1, c2) levels ----
      const double u1v = q * p1 * c1;
      const double u2v = q * p2 * (ca_ * c1 + sa_ * sin1 * c2);
      double s_a = sq + p1 * p1 + 2.0 * u1v;
      s_a = clamp_lo(s_a, 0.0);
      double s_b = sq + s12 + 2.0 * (u1v + u2v);
      s_b = clamp_lo(s_b, 0.0);
      const double Ra = t3_reg_R<REGK>(P.reg, fxtab, kc, s_a), Rb = t3_reg_R<REGK>(P.reg, fxtab, kc, s_b);
      const double ta = lg_coord(lg, kc, s_a), tb = lg_coord(lg, kc, s_b);
      const double DaA = fma(lg_cell_eval(cA, lg, ta), s_a, Ra), Dac = fma(lg_cell_eval(cC, lg, ta), s_a, Ra);
      const double DbA = fma(lg_cell_eval(cA, lg, tb), s_b, Rb), Dbc = fma(lg_cell_eval(cC, lg, tb), s_b, Rb);
      if (WANT_DMIN) dm = fmin(fmin(dm, fmin(DaA, Dac)), fmin(DbA, Dbc));
      const double lam12 = lg_lookup(cL, lg, kc, (sq + p1 * p1 + s_a) * third) *
                           lg_lookup(cL, lg, kc, (s_a + p2 * p2 + s_b) * third);
      const double CA = (qt.x * wnode) * (fast_rcp(DaA * DbA) * lam12);
      const double CC = (qt.y * wnode) * fast_rcp(Dac * Dbc);
      // both polynomials as cubics in x3: g[d] = sum_{a+b+c<=3-d} kap_abcd x0^a x1^b x2^c  (a outermost, then b, c, d)
      const double x0 = sq * ik2, x1 = u1v * ik2, x2 = u2v * ik2;
      double gA[4] = {0.0, 0.0, 0.0, 0.0}, gC[4] = {0.0, 0.0, 0.0, 0.0};
      {
        int idx = 0;
        double xa = 1.0;
#pragma unroll
        for (int a = 0; a <= 3; ++a) {
          double xab = xa;
#pragma unroll
          for (int b = 0; b <= 3 - a; ++b) {
            double xabc = xab;
#pragma unroll
            for (int c = 0; c <= 3 - a - b; ++c) {
#pragma unroll
              for (int d = 0; d <= 3 - a - b - c; ++d) {
                gA[d] = fma(skap[idx], xabc, gA[d]);
                gC[d] = fma(skap[35 + idx], xabc, gC[d]);
                ++idx;
              }
              xabc *= x2;
            }
            xab *= x1;
          }
          xa *= x0;
        }
      }
#pragma unroll
      for (int d = 0; d < 4; ++d) { gA[d] *= CA; gC[d] *= CC; }
      const double qp3 = q * p3 * ik2;
      const double X3c = qp3 * (cb_ * c1 + sbcg * sin1 * c2);
      const double X3s = qp3 * (sbsg * sin1 * sin2);
      const double sd0 = sq + s123 + 2.0 * (u1v + u2v);
      const double twok2 = 2.0 * k2;
      const double l3_0 = (s_b + p3 * p3) * third, l4_0 = (s123 + sq) * third;
      // ---- phi loop: one distinct evaluation per node ----
      double acc_phi = 0.0;
#pragma unroll 2
      for (int jp = 0; jp < nphi; ++jp) {
        const double2 cw = phitab[jp];
        const double x3 = fma(X3s, cw.x, X3c);
        double s_d = fma(twok2, x3, sd0);
        s_d = clamp_lo(s_d, 0.0);
        const double Rd = t3_reg_R<REGK>(P.reg, fxtab, kc, s_d);
        const double td = lg_coord(lg, kc, s_d);
        const double DdA = fma(lg_cell_eval(cA, lg, td), s_d, Rd), Ddc = fma(lg_cell_eval(cC, lg, td), s_d, Rd);
        if (WANT_DMIN) dm = fmin(dm, fmin(DdA, Ddc));
        const double rinv = fast_rcp(DdA * Ddc);
        const double lam34 = lg_lookup(cL, lg, kc, fma(s_d, third, l3_0)) * lg_lookup(cL, lg, kc, fma(s_d, third, l4_0));
        const double PA = fma(fma(fma(gA[3], x3, gA[2]), x3, gA[1]), x3, gA[0]);
        const double PC = fma(fma(fma(gC[3], x3, gC[2]), x3, gC[1]), x3, gC[0]);
        const double tA = (rinv * Ddc) * lam34 * PA;          // G_A(s_d) = D_c / (D_A D_c)
        acc_phi = fma(cw.y, fma(rinv * DdA, PC, tA), acc_phi);
      }
      acc += acc_phi;
    }
    const bool last_of_e = (u + 1 == u1) || ((u + 1) / NCH != e);
    if (last_of_e) {
      const long long ufirst = (long long)e * NCH;
      const int c_first = (int)(((ufirst + 1) * gridDim.x - 1) / U);
      const int slot = (int)blockIdx.x - c_first;
      const double total = block_sum(acc, red);
      const double dmb = WANT_DMIN ? block_min(dm, red) : 0.0;
      if (tid == 0) {
        P.part[(size_t)slot * P.n_ext + e] = total;
        if (WANT_DMIN) P.partD[(size_t)slot * P.n_ext + e] = dmb;
      }
      acc = 0.0;
      dm = dmq;
    }
  }
}

__global__ void __launch_bounds__(256) fp4_fixup_kernel(const FourPointParams P) {
  const long long e = (long long)blockIdx.x * 256 + threadIdx.x;
  if (e >= P.n_ext) return;
  const long long U = (long long)P.n_ext * P.NCH;
  const long long ufirst = e * P.NCH, ulast = ufirst + P.NCH - 1;
  const int c_first = (int)(((ufirst + 1) * P.grid_main - 1) / U), c_last = (int)(((ulast + 1) * P.grid_main - 1) / U);
  CompSum t(P.part[e]);
  for (int s = 1; s <= c_last - c_first; ++s) t.add(P.part[(size_t)s * P.n_ext + e]);
  P.out[e] = P.prefactor * t.value();
  if (P.dmin) {
    double dm = P.partD[e];
    for (int s = 1; s <= c_last - c_first; ++s) dm = fmin(dm, P.partD[(size_t)s * P.n_ext + e]);
    P.dmin[e] = dm * P.reg.inv_k2;
  }
}


int fourpoint_launch(const dfrg_loop4d_desc* D, int n_ext, const double* ext, double* out, double* dmin, int sm_count,
                     cudaStream_t stream) {
  FourPointParams P;
  P.nq = D->q.n; P.n1 = D->cos1.n; P.n2 = D->cos2.n; P.nphi = D->phi.n; P.n_ext = n_ext;
  P.prefactor = D->prefactor;
  fill_common(D->reg, D->tab[0], &P.reg, &P.grid);
  P.fmc = fm_consts();
  P.xq = D->q.x; P.wq = D->q.w; P.x1 = D->cos1.x; P.w1 = D->cos1.w; P.x2 = D->cos2.x; P.w2 = D->cos2.w;
  P.xphi = D->phi.x; P.wphi = D->phi.w;
  P.ZA = D->tab[0].v; P.Zc = D->tab[1].v; P.L3 = D->tab[2].v; P.coef = D->coef; P.ext = ext; P.out = out; P.dmin = dmin;
  const int npairs = P.nq * P.n1;
  P.KP = FP4_THREADS / P.n2 < npairs ? FP4_THREADS / P.n2 : npairs;
  P.NCH = (npairs + P.KP - 1) / P.KP;
  const long long U = (long long)n_ext * P.NCH;
  P.grid_main = (int)(U < sm_count ? U : sm_count);
  P.max_slots = 1;
  for (int e = 0; e < n_ext; ++e) {
    const long long ufirst = (long long)e * P.NCH, ulast = ufirst + P.NCH - 1;
    const int c0 = (int)(((ufirst + 1) * P.grid_main - 1) / U), c1 = (int)(((ulast + 1) * P.grid_main - 1) / U);
    if (c1 - c0 + 1 > P.max_slots) P.max_slots = c1 - c0 + 1;
  }
  const size_t n_part = (size_t)P.max_slots * n_ext;
  void* scratch4 = nullptr;
  int rc = scratch_alloc(&scratch4, 2 * n_part * sizeof(double), stream);
  if (rc != DFRG_OK) return rc;
  P.part = (double*)scratch4;
  P.partD = P.part + n_part;
  const size_t smem4 = fp4_smem(P.nq, P.n1, P.n2, P.nphi, P.grid.n);
  const int regk4 = D->reg.kind == DFRG_REG_LITIM ? 0 : (D->reg.order == 1 ? 1 : 2);
  void (*k4)(const FourPointParams) = nullptr;
#define DFRG_FP4_PICK(K) if (regk4 == K) k4 = dmin ? fp4_main_kernel<K, true> : fp4_main_kernel<K, false>;
  DFRG_FP4_PICK(0) DFRG_FP4_PICK(1) DFRG_FP4_PICK(2)
#undef DFRG_FP4_PICK
  if (smem4 > kMaxDynSmem) { scratch_free(scratch4, stream); return DFRG_EUNSUPPORTED; }
  rc = opt_in_max_smem(k4);
  if (rc != DFRG_OK) { scratch_free(scratch4, stream); return rc; }
  k4<<<P.grid_main, FP4_THREADS, smem4, stream>>>(P);
  fp4_fixup_kernel<<<(n_ext + 255) / 256, 256, 0, stream>>>(P);
  rc = check_cuda(cudaGetLastError());
  scratch_free(scratch4, stream);
  return rc;
}

}  // namespace dfrg
