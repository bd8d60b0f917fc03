// loop4d_threepoint.cu -- three-point family of dfrg_integrate_loop4d, general list of external configurations
// (BASELINE.json config 3 without a layout promise; DFRG_LOOP_THREEPOINT and DFRG_LOOP_THREEPOINT_TAB3D).
#include "loop4d_kernels.cuh"

namespace dfrg {

// ---- three-point, general kernel (any list of external configurations) ----
// Persistent CTAs, thread = (q, c1) pairs, c2 loop inside.  The three table look-ups of a node go through lg_coord /
// lg_cell_eval (no separate logarithm, no FP64 clamps), e^-x through the replicated 64-entry table, every affine
// step is a single FMA, and the regulator kind is a template parameter.
template <int REGK, bool WANT_DMIN, int T3V2_THREADS, int UNR>
__global__ void __launch_bounds__(T3V2_THREADS, 1) threepoint_kernel_v2(const ThreePointParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double red[32];

  if (P.skip_flag && *P.skip_flag == 0) return;
  const int nq = P.nq, n1 = P.n1, n2 = P.n2, nt = P.grid.n;
  double* sxq = reinterpret_cast<double*>(smem_raw);
  double* swq = sxq + ((nq + 1) & ~1);
  double* sx1 = swq + ((nq + 1) & ~1);
  double* sw1 = sx1 + ((n1 + 1) & ~1);
  double* sx2 = sw1 + ((n1 + 1) & ~1);
  double* sw2 = sx2 + ((n2 + 1) & ~1);
  double* sZA = sw2 + ((n2 + 1) & ~1);
  double* sL3 = sZA + ((nt + 1) & ~1);
  double* skap = sL3 + ((nt + 1) & ~1);  // 36
  double* fmmem = skap + 36;             // [FM_DOUBLES]  (regulator() of the once-per-CTA radial table)
  double* fxmem = fmmem + FM_DOUBLES;    // [FX_DOUBLES]
  double* lgmem = fxmem + FX_DOUBLES;    // [LG_DOUBLES]
  double2* cZA_all = reinterpret_cast<double2*>(lgmem + LG_DOUBLES);  // guarded cells, replicated
  double2* cL3_all = cZA_all + cells_guarded_size(nt);
  double2* qtab = cL3_all + cells_guarded_size(nt);                   // [nq] (wq q^3 Rdot(q^2) G_A(q^2), D(q^2))
  double2* xw2 = qtab + nq;                                           // [n2] (c2 node, weight)

  if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  __syncthreads();
  {
    StageList L;
    L.add(sxq, P.xq, nq); L.add(swq, P.wq, nq);
    L.add(sx1, P.x1, n1); L.add(sw1, P.w1, n1);
    L.add(sx2, P.x2, n2); L.add(sw2, P.w2, n2);
    L.add(sZA, P.ZA, nt); L.add(sL3, P.L3, nt);
    stage_to_smem(L, &bar, 0);
  }
  const FastMath fm = fm_build(fmmem, P.fmc);
  const double* fxtab = fx_build(fxmem, P.reg.zk * P.reg.k2);
  const LogGrid lg = lg_build(lgmem, P.grid.lo, P.grid.inv_h, nt);
  const double* kc = P.fmc.c;
  const double2* cZA = cells_build_guarded(cZA_all, sZA, nt, P.grid.interp);
  const double2* cL3 = cells_build_guarded(cL3_all, sL3, nt, P.grid.interp);
  if (threadIdx.x < 35) skap[threadIdx.x] = P.coef[threadIdx.x];
  for (int j = threadIdx.x; j < n2; j += T3V2_THREADS) xw2[j] = make_double2(sx2[j], sw2[j]);
  __syncthreads();

  const double ik2 = P.reg.inv_k2;
  const double third = 1.0 / 3.0;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  // ---- S3, once per CTA: the part that depends on the radial node only (not on the external point) ----
  double dmq = inf;
  for (int i = threadIdx.x; i < nq; i += T3V2_THREADS) {
    const double q = sxq[i], sq = q * q;
    double Rq, Rdq;
    regulator(P.reg, fm, sq, Rq, Rdq);
    const double Dq = lg_lookup(cZA, lg, kc, sq) * sq + Rq;
    qtab[i] = make_double2((swq[i] * q * q * q * Rdq) * fast_rcp(Dq), Dq);
    dmq = fmin(dmq, Dq);
  }
  dmq = block_min(dmq, red);  // also publishes qtab
  double sum_wphi = 0.0;      // the integrand has no phi dependence: the axis contributes sum_phi w
  for (int jp = 0; jp < P.nphi; ++jp) sum_wphi += P.wphi[jp];

  const int npairs = nq * n1;
  // persistent: this CTA owns the external points e = blockIdx.x, blockIdx.x + gridDim.x, ...
  for (int e = blockIdx.x; e < P.n_ext; e += gridDim.x) {
    const double p1 = P.ext[3 * e], p2 = P.ext[3 * e + 1], al = P.ext[3 * e + 2];
    double sa_, ca_;
    sincos(al, &sa_, &ca_);
    double scc = p1 * p1 + p2 * p2 + 2.0 * p1 * p2 * ca_;
    scc = scc > 0.0 ? scc : 0.0;
    double dm = dmq;
    double acc = 0.0;
    for (int t = threadIdx.x; t < npairs; t += T3V2_THREADS) {
      const int i = t / n1, j1 = t - i * n1;
      const double q = sxq[i], c1 = sx1[j1];
      const double sq = q * q;
      const double sin1 = sqrt((1.0 - c1) * (1.0 + c1));
      const double wpair = qtab[i].x * (sw1[j1] * sin1);
      // (q, c1) pieces
      const double qp1 = q * p1 * c1;
      double s_a = sq + p1 * p1 + 2.0 * qp1;
      s_a = clamp_lo(s_a, 0.0);
      const double Da = fma(lg_lookup(cZA, lg, kc, s_a), s_a, t3_reg_R<REGK>(P.reg, fxtab, kc, s_a));
      if (WANT_DMIN) dm = fmin(dm, Da);
      const double Ga = fast_rcp(Da);
      const double lam1 = lg_lookup(cL3, lg, kc, (p1 * p1 + sq + s_a) * third);
      // P as a quartic in z = q.p2/k^2: gam[c] = sum_{a+b<=4-c} kap_abc X^a Y^b
      const double X = sq * ik2, Y = qp1 * ik2;
      double gam[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      {
        int idx = 0;
        double Xa = 1.0;
#pragma unroll
        for (int a = 0; a <= 4; ++a) {
          double XaYb = Xa;
#pragma unroll
          for (int b = 0; b <= 4 - a; ++b) {
#pragma unroll
            for (int c = 0; c <= 4 - a - b; ++c) gam[c] = fma(skap[idx++], XaYb, gam[c]);
            XaYb *= Y;
          }
          Xa *= X;
        }
      }
      // q.p2/k^2 = zc + zs c2 (in units of k^2, so that Horner runs on it directly);  s_b = sb0 - 2 k^2 z
      const double zc = q * p2 * ca_ * c1 * ik2;
      const double zs = q * p2 * sa_ * sin1 * ik2;
      const double sb0 = sq + p2 * p2;
      const double m2k2 = -2.0 * P.reg.k2;
      const double l20 = (p2 * p2 + sq) * third, l30 = (scc + s_a) * third;
      const double w0 = wpair * (Ga * lam1);
      double acc2 = 0.0;
#pragma unroll UNR
      for (int j2 = 0; j2 < n2; ++j2) {
        const double2 xw = xw2[j2];
        const double z = fma(zs, xw.x, zc);
        double s_b = fma(m2k2, z, sb0);
        s_b = clamp_lo(s_b, 0.0);
        const double Rb = t3_reg_R<REGK>(P.reg, fxtab, kc, s_b);
        const double Db = fma(lg_lookup(cZA, lg, kc, s_b), s_b, Rb);
        if (WANT_DMIN) dm = fmin(dm, Db);
        const double lam2 = lg_lookup(cL3, lg, kc, fma(s_b, third, l20));
        const double lam3 = lg_lookup(cL3, lg, kc, fma(s_b, third, l30));
        const double poly = fma(fma(fma(fma(gam[4], z, gam[3]), z, gam[2]), z, gam[1]), z, gam[0]);
        acc2 = fma(xw.y * poly, fast_rcp(Db) * (lam2 * lam3), acc2);
      }
      acc = fma(w0, acc2, acc);
    }
    const double total = block_sum(acc, red);
    const double dmin_b = WANT_DMIN ? block_min(dm, red) : 0.0;
    if (threadIdx.x == 0) {
      P.out[e] = P.prefactor * sum_wphi * total;
      if (WANT_DMIN) P.dmin[e] = dmin_b * ik2;
    }
  }
}

static size_t threepoint_v2_smem(int nq, int n1, int n2, int nt) {
  return 8 * (size_t)(2 * ((nq + 1) & ~1) + 2 * ((n1 + 1) & ~1) + 2 * ((n2 + 1) & ~1) + 2 * ((nt + 1) & ~1) + 36 +
                      FM_DOUBLES + FX_DOUBLES + LG_DOUBLES + 2 * cells_guarded_size(nt) * 2 + 2 * nq + 2 * n2);
}

// =====================================================================================================
// three-point with a 3-D vertex dressing table (include/dfrg.h, DFRG_LOOP_THREEPOINT_TAB3D)
// =====================================================================================================
// The kinematics, propagators, polynomial and mapping of the general three-point kernel (thread = (q, c1) pairs, c2 loop
// inside, persistent CTAs over the external configurations); every vertex factor is a trilinear look-up in
// lambda3(S0^2, a, s) (the paper's 96 x 8 x 7 vertex grids): the whole table sits in
// shared memory (43 KB for 96 x 8 x 7), a look-up gathers its 8 corners with plain 64-bit loads -- the first family
// whose table traffic competes with the arithmetic.  The vertex at (p1, q, q+p1) is hoisted out of the c2 loop.
static size_t t3d_smem(int nq, int n1, int n2, int nt, int ntab3) {
  return 8 * (size_t)(2 * ((nq + 1) & ~1) + 2 * ((n1 + 1) & ~1) + 2 * ((n2 + 1) & ~1) + ((nt + 1) & ~1) + 36 +
                      FM_DOUBLES + FX_DOUBLES + LG_DOUBLES + cells_guarded_size(nt) * 2 + 2 * nq + 2 * n2 +
                      ((ntab3 + 1) & ~1));
}

template <int REGK, bool WANT_DMIN>
__global__ void __launch_bounds__(256, 1) t3d_kernel(const ThreePoint3DParams Q) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double red[32];
  constexpr int NT = 256;
  const ThreePointParams& P = Q.B;
  const Tab3DParams& T = Q.T;
  if (P.skip_flag && *P.skip_flag == 0) return;   // the product-grid kernels did the work
  const int nq = P.nq, n1 = P.n1, n2 = P.n2, nt = P.grid.n;
  const int ntab3 = T.n[0] * T.n[1] * T.n[2];
  double* sxq = reinterpret_cast<double*>(smem_raw);
  double* swq = sxq + ((nq + 1) & ~1);
  double* sx1 = swq + ((nq + 1) & ~1);
  double* sw1 = sx1 + ((n1 + 1) & ~1);
  double* sx2 = sw1 + ((n1 + 1) & ~1);
  double* sw2 = sx2 + ((n2 + 1) & ~1);
  double* sZA = sw2 + ((n2 + 1) & ~1);
  double* skap = sZA + ((nt + 1) & ~1);  // 36
  double* fmmem = skap + 36;
  double* fxmem = fmmem + FM_DOUBLES;
  double* lgmem = fxmem + FX_DOUBLES;
  double2* cZA_all = reinterpret_cast<double2*>(lgmem + LG_DOUBLES);
  double2* qtab = cZA_all + cells_guarded_size(nt);                   // [nq]
  double2* xw2 = qtab + nq;                                           // [n2]
  double* stab3 = reinterpret_cast<double*>(xw2 + n2);                // [ntab3]

  if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  __syncthreads();
  {
    StageList L;
    L.add(sxq, P.xq, nq); L.add(swq, P.wq, nq);
    L.add(sx1, P.x1, n1); L.add(sw1, P.w1, n1);
    L.add(sx2, P.x2, n2); L.add(sw2, P.w2, n2);
    L.add(sZA, P.ZA, nt); L.add(stab3, Q.v3, ntab3);   // the whole 3-D table: one TMA bulk copy
    stage_to_smem(L, &bar, 0);
  }
  const FastMath fm = fm_build(fmmem, P.fmc);
  const double* fxtab = fx_build(fxmem, P.reg.zk * P.reg.k2);
  const LogGrid lg = lg_build(lgmem, P.grid.lo, P.grid.inv_h, nt);
  const double* kc = P.fmc.c;
  const double2* cZA = cells_build_guarded(cZA_all, sZA, nt, P.grid.interp);
  if (threadIdx.x < 35) skap[threadIdx.x] = P.coef[threadIdx.x];
  for (int j = threadIdx.x; j < n2; j += NT) xw2[j] = make_double2(sx2[j], sw2[j]);
  __syncthreads();

  const double ik2 = P.reg.inv_k2;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  double dmq = inf;
  for (int i = threadIdx.x; i < nq; i += NT) {
    const double q = sxq[i], sq = q * q;
    double Rq, Rdq;
    regulator(P.reg, fm, sq, Rq, Rdq);
    const double Dq = lg_lookup(cZA, lg, kc, sq) * sq + Rq;
    qtab[i] = make_double2((swq[i] * q * q * q * Rdq) * fast_rcp(Dq), Dq);
    dmq = fmin(dmq, Dq);
  }
  dmq = block_min(dmq, red);  // also publishes qtab
  double sum_wphi = 0.0;
  for (int jp = 0; jp < P.nphi; ++jp) sum_wphi += P.wphi[jp];

  const int npairs = nq * n1;
  for (int e = blockIdx.x; e < P.n_ext; e += gridDim.x) {
    const double p1 = P.ext[3 * e], p2 = P.ext[3 * e + 1], al = P.ext[3 * e + 2];
    double sa_, ca_;
    sincos(al, &sa_, &ca_);
    double scc = p1 * p1 + p2 * p2 + 2.0 * p1 * p2 * ca_;
    scc = scc > 0.0 ? scc : 0.0;
    double dm = dmq;
    double acc = 0.0;
    for (int t = threadIdx.x; t < npairs; t += NT) {
      const int i = t / n1, j1 = t - i * n1;
      const double q = sxq[i], c1 = sx1[j1];
      const double sq = q * q;
      const double sin1 = sqrt((1.0 - c1) * (1.0 + c1));
      const double wpair = qtab[i].x * (sw1[j1] * sin1);
      const double qp1 = q * p1 * c1;
      double s_a = sq + p1 * p1 + 2.0 * qp1;
      s_a = clamp_lo(s_a, 0.0);
      const double Da = fma(lg_lookup(cZA, lg, kc, s_a), s_a, t3_reg_R<REGK>(P.reg, fxtab, kc, s_a));
      if (WANT_DMIN) dm = fmin(dm, Da);
      const double lam1 = tab3d_vertex(stab3, T, fm, p1 * p1, sq, s_a);
      const double X = sq * ik2, Y = qp1 * ik2;
      double gam[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      {
        int idx = 0;
        double Xa = 1.0;
#pragma unroll
        for (int a = 0; a <= 4; ++a) {
          double XaYb = Xa;
#pragma unroll
          for (int b = 0; b <= 4 - a; ++b) {
#pragma unroll
            for (int c = 0; c <= 4 - a - b; ++c) gam[c] = fma(skap[idx++], XaYb, gam[c]);
            XaYb *= Y;
          }
          Xa *= X;
        }
      }
      const double zc = q * p2 * ca_ * c1 * ik2;
      const double zs = q * p2 * sa_ * sin1 * ik2;
      const double sb0 = sq + p2 * p2;
      const double m2k2 = -2.0 * P.reg.k2;
      const double w0 = wpair * (fast_rcp(Da) * lam1);
      double acc2 = 0.0;
      for (int j2 = 0; j2 < n2; ++j2) {
        const double2 xw = xw2[j2];
        const double z = fma(zs, xw.x, zc);
        double s_b = fma(m2k2, z, sb0);
        s_b = clamp_lo(s_b, 0.0);
        const double Db = fma(lg_lookup(cZA, lg, kc, s_b), s_b, t3_reg_R<REGK>(P.reg, fxtab, kc, s_b));
        if (WANT_DMIN) dm = fmin(dm, Db);
        const double lam2 = tab3d_vertex(stab3, T, fm, p2 * p2, sq, s_b);
        const double lam3 = tab3d_vertex(stab3, T, fm, scc, s_a, s_b);
        const double poly = fma(fma(fma(fma(gam[4], z, gam[3]), z, gam[2]), z, gam[1]), z, gam[0]);
        acc2 = fma(xw.y * poly, fast_rcp(Db) * (lam2 * lam3), acc2);
      }
      acc = fma(w0, acc2, acc);
    }
    const double total = block_sum(acc, red);
    const double dmin_b = WANT_DMIN ? block_min(dm, red) : 0.0;
    if (threadIdx.x == 0) {
      P.out[e] = P.prefactor * sum_wphi * total;
      if (WANT_DMIN) P.dmin[e] = dmin_b * ik2;
    }
  }
}


size_t threepoint_general_smem(int nq, int n1, int n2, int nt) { return threepoint_v2_smem(nq, n1, n2, nt); }
size_t threepoint3d_general_smem(int nq, int n1, int n2, int nt, int ntab3) { return t3d_smem(nq, n1, n2, nt, ntab3); }

int threepoint_general_launch(const ThreePointParams& P, int regk, int sm_count, cudaStream_t stream) {
  const size_t smem = threepoint_v2_smem(P.nq, P.n1, P.n2, P.grid.n);
  if (smem > kMaxDynSmem) return DFRG_EUNSUPPORTED;
  void (*kern)(const ThreePointParams) = nullptr;
#define DFRG_T3_PICK(K) if (regk == K) kern = P.dmin ? threepoint_kernel_v2<K, true, 256, 8> : threepoint_kernel_v2<K, false, 256, 8>;
  DFRG_T3_PICK(0) DFRG_T3_PICK(1) DFRG_T3_PICK(2)
#undef DFRG_T3_PICK
  const int rca = opt_in_max_smem(kern);
  if (rca != DFRG_OK) return rca;
  const int grid = P.n_ext < sm_count ? P.n_ext : sm_count;  // persistent: 1 CTA of 256 threads x 240 registers per SM
  kern<<<grid, 256, smem, stream>>>(P);
  return check_cuda(cudaGetLastError());
}

int threepoint3d_general_launch(const ThreePoint3DParams& Q3, int regk, int sm_count, cudaStream_t stream) {
  const ThreePointParams& P = Q3.B;
  const size_t smem3 = t3d_smem(P.nq, P.n1, P.n2, P.grid.n, Q3.T.n[0] * Q3.T.n[1] * Q3.T.n[2]);
  if (smem3 > kMaxDynSmem) return DFRG_EUNSUPPORTED;
  void (*k3)(const ThreePoint3DParams) = nullptr;
#define DFRG_T3D_PICK(K) if (regk == K) k3 = P.dmin ? t3d_kernel<K, true> : t3d_kernel<K, false>;
  DFRG_T3D_PICK(0) DFRG_T3D_PICK(1) DFRG_T3D_PICK(2)
#undef DFRG_T3D_PICK
  const int rca = opt_in_max_smem(k3);
  if (rca != DFRG_OK) return rca;
  const int grid3 = P.n_ext < sm_count ? P.n_ext : sm_count;
  k3<<<grid3, 256, smem3, stream>>>(Q3);
  return check_cuda(cudaGetLastError());
}

}  // namespace dfrg
