// loop4d_grid.cu -- three-point family of dfrg_integrate_loop4d on a product grid of external momenta
// (dfrg_loop4d_desc::ext_outer; BASELINE.json config 3 as bench.py runs it), 1-D and 3-D vertex tables.
#include "loop4d_kernels.cuh"

namespace dfrg {

// =====================================================================================================
// three-point on a product grid of external momenta
// =====================================================================================================
// When the external configurations form a product  ext[a S + r] = (|p1|_a, |p2|_r, alpha_r),  a < G, r < S
// (BASELINE.json config 3: 32 |p1| x (32 |p2| x 8 alpha); the paper's vertex grids are of this kind,
// PAPER.md:336), almost everything in a node is shared:
//   depends on (|p2|, alpha) only -- shared by the G values of |p1|:   s_b, G_A(s_b), lambda3((p2^2+q^2+s_b)/3), z = q.p2/k^2
//   depends on |p1| only          -- shared by the S pairs (|p2|, alpha): s_a, G_A(s_a), lambda3((p1^2+q^2+s_a)/3), the five
//                                                                       coefficients of P as a quartic in z
// and only  lambda3((s_c + s_a + s_b)/3)  and the Horner evaluation of P are left per (a, r, node): 19 FP64 instructions
// instead of 66.  The caller promises the layout through dfrg_loop4d_desc::ext_outer = G; the pre-pass kernel checks it
// on the device and, if it does not hold, the product-grid kernels return at once and the general kernel runs instead
// (both are enqueued; the one that is not needed exits after reading one flag).
//
//  (1) t3g_prepass_kernel: promise check; tabR[r] = (|p2|, cos alpha, sin alpha); tabA[pair][a][0..7] for every (q, c1) pair:
//        s_a/3,  the five quartic coefficients times w0 = wq q^3 Rdot(q^2) G_A(q^2) w1 sqrt(1-c1^2) G_A(s_a) lambda3(.),  D_a.
//  (2) t3g_main_kernel: persistent, one CTA per SM.  Work unit = (r, chunk of KP pairs); the units are dealt to the
//      CTAs in contiguous ranges.  Phase 0 (two units ahead): the unit's pair data (q.p2 split into its c2-independent and
//      c2-proportional parts, q^2).  Phase 1 (all threads, one unit ahead, double buffered): the shared node data
//      (w2 G_A(s_b) lambda3(.), z) of the unit's KP x n2 nodes into shared memory.  Phase 2: thread = (a, pair slot); per
//      node one coordinate, the cell of lambda3 cached in registers, one Horner, two multiply-adds; the shared node data
//      are warp-uniform broadcasts.  A thread keeps the running sum of its a while the CTA stays inside one r; the partial
//      sums of an output are written per CTA ("slot") and added in fixed order by
//  (3) t3g_fixup_kernel (deterministic: the ownership of units is a pure function of the grid size).

// common shared-memory carve-up of the two product-grid kernels
struct T3GShared {
  double *sxq, *swq, *sx1, *sw1, *sx2, *sw2, *sZA, *sL3, *skap, *fmmem, *fxmem, *lgmem;
  double2 *cZA_all, *cL3_all, *qtab, *xw2, *nodeA;
  double *nodeZ, *red, *stab3;
};
__device__ __forceinline__ T3GShared t3g_carve(unsigned char* raw, int nq, int n1, int n2, int nt) {
  T3GShared s;
  s.sxq = reinterpret_cast<double*>(raw);
  s.swq = s.sxq + ((nq + 1) & ~1);
  s.sx1 = s.swq + ((nq + 1) & ~1);
  s.sw1 = s.sx1 + ((n1 + 1) & ~1);
  s.sx2 = s.sw1 + ((n1 + 1) & ~1);
  s.sw2 = s.sx2 + ((n2 + 1) & ~1);
  s.sZA = s.sw2 + ((n2 + 1) & ~1);
  s.sL3 = s.sZA + ((nt + 1) & ~1);
  s.skap = s.sL3 + ((nt + 1) & ~1);  // 36
  s.fmmem = s.skap + 36;
  s.fxmem = s.fmmem + FM_DOUBLES;
  s.lgmem = s.fxmem + FX_DOUBLES;
  s.cZA_all = reinterpret_cast<double2*>(s.lgmem + LG_DOUBLES);
  s.cL3_all = s.cZA_all + cells_guarded_size(nt);
  s.qtab = s.cL3_all + cells_guarded_size(nt);
  s.xw2 = s.qtab + nq;
  s.nodeA = s.xw2 + n2;                                          // [2][T3G_NODES]
  s.nodeZ = reinterpret_cast<double*>(s.nodeA + 2 * T3G_NODES);  // [2][T3G_NODES]
  s.red = s.nodeZ + 2 * T3G_NODES;                               // [T3G_MAXT]
  s.stab3 = s.red + T3G_MAXT;                                    // [ntab3]  (TAB3D only)
  return s;
}
static size_t t3g_smem(int nq, int n1, int n2, int nt, int ntab3 = 0) {
  return 8 * (size_t)(2 * ((nq + 1) & ~1) + 2 * ((n1 + 1) & ~1) + 2 * ((n2 + 1) & ~1) + 2 * ((nt + 1) & ~1) + 36 +
                      FM_DOUBLES + FX_DOUBLES + LG_DOUBLES + 2 * cells_guarded_size(nt) * 2 + 2 * nq + 2 * n2 +
                      2 * 2 * T3G_NODES + 2 * T3G_NODES + T3G_MAXT + ((ntab3 + 1) & ~1));
}

template <int REGK, bool TAB3D>
__global__ void __launch_bounds__(T3G_THREADS, 1) t3g_prepass_kernel(const ThreeGridParams Q) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double red[32];
  const ThreePointParams& P = Q.B;
  const int nq = P.nq, n1 = P.n1, n2 = P.n2, nt = P.grid.n, G = Q.G, S = Q.S;
  const T3GShared sm = t3g_carve(smem_raw, nq, n1, n2, nt);

  if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  __syncthreads();
  {
    StageList L;
    L.add(sm.sxq, P.xq, nq); L.add(sm.swq, P.wq, nq);
    L.add(sm.sx1, P.x1, n1); L.add(sm.sw1, P.w1, n1);
    L.add(sm.sZA, P.ZA, nt);
    if (TAB3D) L.add(sm.stab3, Q.v3, Q.ntab3); else L.add(sm.sL3, P.L3, nt);
    stage_to_smem(L, &bar, 0);
  }
  const FastMath fm = fm_build(sm.fmmem, P.fmc);
  const double* fxtab = fx_build(sm.fxmem, P.reg.zk * P.reg.k2);
  const LogGrid lg = lg_build(sm.lgmem, P.grid.lo, P.grid.inv_h, nt);
  const double* kc = P.fmc.c;
  const double2* cZA = cells_build_guarded(sm.cZA_all, sm.sZA, nt, P.grid.interp);
  const double2* cL3 = TAB3D ? nullptr : cells_build_guarded(sm.cL3_all, sm.sL3, nt, P.grid.interp);
  if (threadIdx.x < 35) sm.skap[threadIdx.x] = P.coef[threadIdx.x];
  __syncthreads();

  const double ik2 = P.reg.inv_k2, third = 1.0 / 3.0;
  const long long gtid = (long long)blockIdx.x * T3G_THREADS + threadIdx.x, gstride = (long long)gridDim.x * T3G_THREADS;
  // promise check
  for (long long e = gtid; e < P.n_ext; e += gstride) {
    const long long a = e / S, r = e - a * S;
    const bool ok = P.ext[3 * e] == P.ext[3 * (a * S)] && P.ext[3 * e + 1] == P.ext[3 * r + 1] &&
                    P.ext[3 * e + 2] == P.ext[3 * r + 2];
    if (!ok) *Q.flag = 1;
  }
  for (long long r = gtid; r < S; r += gstride) {
    double sa_, ca_;
    sincos(P.ext[3 * r + 2], &sa_, &ca_);
    Q.tabR[4 * r] = P.ext[3 * r + 1]; Q.tabR[4 * r + 1] = ca_; Q.tabR[4 * r + 2] = sa_; Q.tabR[4 * r + 3] = 0.0;
  }
  // radial table (every CTA builds its own copy)
  double dmq = __longlong_as_double(0x7ff0000000000000LL);
  for (int i = threadIdx.x; i < nq; i += T3G_THREADS) {
    const double q = sm.sxq[i], sq = q * q;
    double Rq, Rdq;
    regulator(P.reg, fm, sq, Rq, Rdq);
    const double Dq = lg_lookup(cZA, lg, kc, sq) * sq + Rq;
    sm.qtab[i] = make_double2((sm.swq[i] * q * q * q * Rdq) * fast_rcp(Dq), Dq);
    dmq = fmin(dmq, Dq);
  }
  dmq = block_min(dmq, red);  // also publishes qtab
  if (blockIdx.x == 0 && threadIdx.x == 0) *Q.qmin = dmq;

  const long long n_items = (long long)nq * n1 * G;
  for (long long it = gtid; it < n_items; it += gstride) {
    const int pair = (int)(it / G), a = (int)(it - (long long)pair * G);
    const int i = pair / n1, j1 = pair - i * n1;
    const double p1 = P.ext[3 * ((long long)a * S)];
    const double q = sm.sxq[i], c1 = sm.sx1[j1];
    const double sq = q * q;
    const double sin1 = sqrt((1.0 - c1) * (1.0 + c1));
    const double wpair = sm.qtab[i].x * (sm.sw1[j1] * sin1);
    const double qp1 = q * p1 * c1;
    double s_a = sq + p1 * p1 + 2.0 * qp1;
    s_a = clamp_lo(s_a, 0.0);
    const double Da = fma(lg_lookup(cZA, lg, kc, s_a), s_a, t3_reg_R<REGK>(P.reg, fxtab, kc, s_a));
    const double Ga = fast_rcp(Da);
    const double lam1 = TAB3D ? tab3d_vertex(sm.stab3, Q.T3, fm, p1 * p1, sq, s_a)
                              : lg_lookup(cL3, lg, kc, (p1 * p1 + sq + s_a) * third);
    const double X = sq * ik2, Y = qp1 * ik2;
    double gam[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    {
      int idx = 0;
      double Xa = 1.0;
#pragma unroll
      for (int aa = 0; aa <= 4; ++aa) {
        double XaYb = Xa;
#pragma unroll
        for (int b = 0; b <= 4 - aa; ++b) {
#pragma unroll
          for (int c = 0; c <= 4 - aa - b; ++c) gam[c] = fma(sm.skap[idx++], XaYb, gam[c]);
          XaYb *= Y;
        }
        Xa *= X;
      }
    }
    double2* ta = reinterpret_cast<double2*>(Q.tabA + ((size_t)pair * G + a) * 8);
    const double w0 = wpair * (Ga * lam1);
    ta[0] = make_double2(TAB3D ? s_a : s_a * third, w0 * gam[0]);
    ta[1] = make_double2(w0 * gam[1], w0 * gam[2]);
    ta[2] = make_double2(w0 * gam[3], w0 * gam[4]);
    ta[3] = make_double2(0.0, Da);
  }
}

// ---- main kernel: shared-memory layout (hot tables first, at compile-time offsets) ----
//   [0, 64 KB)  replicated mantissa table of lg2_coord;  then the guarded cells of lambda3 (the one table the hot loop
//   reads), the guarded cells of Z_A, the exp table, and everything whose size depends on the call.
struct T3MShared {
  double* lgmem;
  double4 *cL3, *cZA;
  double *fxmem, *fmmem, *sxq, *sx1, *ssin1, *sx2, *sw2, *sZA, *sL3;
  double2 *xw2, *nodeA;
  double4* ptab;
  double *rowc, *nodeS, *red, *stab3;
};
__device__ __forceinline__ T3MShared t3m_carve(unsigned char* raw, int nq, int n1, int n2, int nt, int nodes, int kp,
                                               int nt_thr) {
  T3MShared s;
  s.lgmem = reinterpret_cast<double*>(raw);
  s.cL3 = reinterpret_cast<double4*>(s.lgmem + LG_DOUBLES);
  s.cZA = s.cL3 + (nt + 1);
  s.fxmem = reinterpret_cast<double*>(s.cZA + (nt + 1));
  s.fmmem = s.fxmem + FX_DOUBLES;
  s.sxq = s.fmmem + FM_DOUBLES;
  s.sx1 = s.sxq + ((nq + 1) & ~1);
  s.ssin1 = s.sx1 + ((n1 + 1) & ~1);
  s.sx2 = s.ssin1 + ((n1 + 1) & ~1);
  s.sw2 = s.sx2 + ((n2 + 1) & ~1);
  s.sZA = s.sw2 + ((n2 + 1) & ~1);
  s.sL3 = s.sZA + ((nt + 1) & ~1);
  s.xw2 = reinterpret_cast<double2*>(s.sL3 + ((nt + 1) & ~1));
  s.nodeA = s.xw2 + n2;                                       // [2][nodes] (w2 G_A(s_b) lambda3(.), z)
  s.ptab = reinterpret_cast<double4*>(s.nodeA + 2 * nodes);   // [2][kp]    (zc, zs, q^2, -) of a pair
  s.rowc = reinterpret_cast<double*>(s.ptab + 2 * kp);        // [2][kp]    (q^2 + p2^2)/3 of the row (one per pair)
  s.nodeS = s.rowc + 2 * kp;                                  // [2][nodes] s_b        (TAB3D only)
  s.red = s.nodeS + 2 * nodes;                                // [threads]
  s.stab3 = s.red + nt_thr;                                   // [ntab3]               (TAB3D only)
  return s;
}
static size_t t3m_smem(int nq, int n1, int n2, int nt, int nodes, int kp, int threads, int ntab3) {
  return 8 * (size_t)(LG_DOUBLES + 2 * 4 * (nt + 1) + FX_DOUBLES + FM_DOUBLES + ((nq + 1) & ~1) + 2 * ((n1 + 1) & ~1) +
                      2 * ((n2 + 1) & ~1) + 2 * ((nt + 1) & ~1) + 2 * n2 + 2 * 2 * nodes + 2 * 4 * kp + 2 * kp +
                      2 * nodes + threads + ((ntab3 + 1) & ~1));
}

// Hot loop (1-D vertex table), per (a, r, node):  x = (s_c + s_a + s_b)/3 = up + m2k23 z  with  up = (s_c + s_a + q^2 + p2^2)/3
// per row and z the node's q.p2/k^2 (so the node record is one 16-byte broadcast (w, z)); t' = lg2_coord(x); the cell of
// lambda3 lives in registers (cc.k, cc.Fd) and is reloaded only when t' leaves it: tau = t' - Fd lies in [0, 1) exactly when
// the high word of tau, read as an unsigned integer, is below that of 1.0 (negative, >= 1 and NaN all fail), so the test is
// one integer compare off the FP64 pipe; cubic in tau; quartic Horner in z; two multiply-adds.  17 FP64 instructions.
// Along a row x is monotone in the c2 node (s_b is affine in c2) and a cell is 25 % wide in x, so 9 nodes in 10 stay in
// the cell of their predecessor.  Whether the cell is reloaded or not, tau = t' - floor(t') (clamped) is the same number.
struct CellCache {
  double4 k;
  double Fd;
};
__device__ __forceinline__ double t3m_node(const double2 b, const double up, const double m2k23, const LogGrid2& lg,
                                           const double4* __restrict__ cL3, CellCache& cc, const double (&cur)[6],
                                           const double acc2) {
  const double tq = lg2_coord(lg, fma(b.y, m2k23, up));
  double tau = tq - cc.Fd;
  if ((unsigned)__double2hiint(tau) >= 0x3ff00000u) {   // (predicated: a branch per node costs more than it saves)
    const unsigned F = lg2_cell(lg, tq);
    cc.Fd = (double)F;
    cc.k = cL3[F];
    tau = tq - cc.Fd;
  }
  const double lam3 = fma(fma(fma(cc.k.w, tau, cc.k.z), tau, cc.k.y), tau, cc.k.x);
  const double poly = fma(fma(fma(fma(cur[5], b.y, cur[4]), b.y, cur[3]), b.y, cur[2]), b.y, cur[1]);
  return fma(b.x * poly, lam3, acc2);
}

template <int REGK, int NT, int N2, bool TAB3D>   // N2: compile-time cos2 order (full unroll), 0 = run time
__global__ void __launch_bounds__(NT, 1) t3g_main_kernel(const ThreeGridParams Q) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double red32[32];
  if (*Q.flag != 0) return;  // the layout promise does not hold: the general kernel does the work
  const ThreePointParams& P = Q.B;
  const int nq = P.nq, n1 = P.n1, n2 = N2 ? N2 : P.n2, nt = P.grid.n, G = Q.G, S = Q.S, KP = Q.KP, NCH = Q.NCH;
  const int NODES = Q.NODES;
  const int npairs = nq * n1;
  const T3MShared sm = t3m_carve(smem_raw, nq, n1, n2, nt, NODES, KP, NT);
  const int tid = threadIdx.x;

  if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  __syncthreads();
  {
    StageList L;
    L.add(sm.sxq, P.xq, nq);
    L.add(sm.sx1, P.x1, n1);
    L.add(sm.sx2, P.x2, n2); L.add(sm.sw2, P.w2, n2);
    L.add(sm.sZA, P.ZA, nt);
    if (TAB3D) L.add(sm.stab3, Q.v3, Q.ntab3); else L.add(sm.sL3, P.L3, nt);
    // the shifted copy for the paired look-up of the hot loop (source not 16-byte aligned: plain loads)
    if (TAB3D && Q.paired3) L.add(sm.stab3 + ((Q.ntab3 + 1) & ~1), Q.v3 + 1, Q.ntab3 - 1);
    stage_to_smem(L, &bar, 0);
  }
  const double* stab3B = sm.stab3 + ((Q.ntab3 + 1) & ~1);
  const FastMath fm = fm_build(sm.fmmem, P.fmc);   // the S0 axis of the 3-D table (TAB3D)
  const double* fxtab = fx_build(sm.fxmem, P.reg.zk * P.reg.k2);
  const LogGrid2 lg = lg2_build(sm.lgmem, Q.lgc, nt);
  const double* kc = P.fmc.c;
  cells2_build(sm.cZA, sm.sZA, nt, P.grid.interp);
  if (!TAB3D) cells2_build(sm.cL3, sm.sL3, nt, P.grid.interp);
  for (int j = tid; j < n2; j += NT) sm.xw2[j] = make_double2(sm.sx2[j], sm.sw2[j]);
  for (int j = tid; j < n1; j += NT) {
    const double c1 = sm.sx1[j];
    sm.ssin1[j] = sqrt((1.0 - c1) * (1.0 + c1));
  }
  __syncthreads();   // publishes the tables

  const double ik2 = P.reg.inv_k2, third = 1.0 / 3.0, m2k2 = -2.0 * P.reg.k2;
  const double& m2k23 = Q.m2k23;   // straight from the kernel parameters: a constant-bank operand of the hot loop
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  const long long U = (long long)S * NCH;
  const long long u0 = (long long)blockIdx.x * U / gridDim.x, u1 = (long long)(blockIdx.x + 1) * U / gridDim.x;
  const int nw = NT / G;                 // pair slots
  const bool active = tid < nw * G;
  const int a = tid % G, w = tid / G;
  const double p1 = P.ext[3 * ((long long)a * S)];

  double dmB_cur = inf, dmB_nxt = inf;
  // Phase 0 (two units ahead): the pair data of unit u -- z = zc + zs c2,  s_b = q^2 + p2^2 - 2 k^2 z
  auto phase0 = [&](const int r, const int ch, const int b) {
    const int pair0 = ch * KP;
    const int npl = min(KP, npairs - pair0);
    const double p2 = Q.tabR[4 * r], ca_ = Q.tabR[4 * r + 1], sa_ = Q.tabR[4 * r + 2];
    const double pc = p2 * ca_ * ik2, ps = p2 * sa_ * ik2;
    double4* pt = sm.ptab + b * KP;
    for (int pl = tid; pl < npl; pl += NT) {
      const int pair = pair0 + pl;
      const int i = pair / n1, j1 = pair - i * n1;
      const double q = sm.sxq[i];
      pt[pl] = make_double4(q * sm.sx1[j1] * pc, q * sm.ssin1[j1] * ps, q * q, 0.0);
    }
  };
  // Phase 1 (one unit ahead): shared node data of unit u into buffer b
  auto phase1 = [&](const int r, const int ch, const int b, double& dmB) {
    const int pair0 = ch * KP;
    const int npl = min(KP, npairs - pair0);
    const double p2sq = Q.tabR[4 * r] * Q.tabR[4 * r];
    const double4* pt = sm.ptab + b * KP;
    double2* nA = sm.nodeA + b * NODES;
    double* rc = sm.rowc + b * KP;
    double* nS = sm.nodeS + b * NODES;
    for (int n = tid; n < npl * n2; n += NT) {
      const int pl = n / n2, j2 = n - pl * n2;
      const double4 pd = pt[pl];
      const double2 xw = sm.xw2[j2];
      const double z = fma(pd.y, xw.x, pd.x);
      const double sb0 = pd.z + p2sq, sb03 = sb0 * third;
      double s_b = fma(m2k2, z, sb0);
      s_b = clamp_lo(s_b, 0.0);
      const double Db = fma(lg2_lookup(sm.cZA, lg, s_b), s_b, t3_reg_R<REGK>(P.reg, fxtab, kc, s_b));
      dmB = fmin(dmB, Db);
      const double lam2 = TAB3D ? tab3d_vertex(sm.stab3, Q.T3, fm, p2sq, pd.z, s_b)
                                : lg2_lookup(sm.cL3, lg, fma(s_b, third, sb03));
      nA[n] = make_double2(xw.y * (fast_rcp(Db) * lam2), z);
      if (TAB3D) nS[n] = s_b;
      if (j2 == 0) rc[pl] = sb03;
    }
  };

  double acc = 0.0;
  Tab3Cell cell3;
  cell3.o = -1;
  CellCache cc;
  cc.Fd = inf; cc.k = make_double4(0.0, 0.0, 0.0, 0.0);   // tau = t' - inf fails the range test: the first node loads its cell
  // (r, ch) of the units u, u + 1, u + 2, advanced without divisions
  int r = (int)(u0 / NCH), ch = (int)(u0 - (long long)r * NCH);
  auto next_unit = [&](int& rr, int& cc_) { if (++cc_ == NCH) { cc_ = 0; ++rr; } };
  int r1 = r, ch1 = ch;
  next_unit(r1, ch1);
  int r2 = r1, ch2 = ch1;
  next_unit(r2, ch2);
  const int nu = (int)(u1 - u0);
  if (nu > 0) phase0(r, ch, 0);
  __syncthreads();
  if (nu > 0) phase1(r, ch, 0, dmB_cur);
  if (nu > 1) phase0(r1, ch1, 1);
  __syncthreads();
  for (int iu = 0; iu < nu; ++iu) {
    const int b = iu & 1;
    const bool last_of_r = (iu + 1 == nu) || (r1 != r);
    const int pair0 = ch * KP;
    const int npl = min(KP, npairs - pair0);
    // the first row's coefficients: on their way into L1 while phase 1 runs
    if (active && w < npl)
      asm volatile("prefetch.global.L1 [%0];" ::"l"(Q.tabA + ((size_t)(pair0 + w) * G + a) * 8));
    if (iu + 1 < nu) phase1(r1, ch1, b ^ 1, last_of_r ? dmB_nxt : dmB_cur);
    // ---- phase 2 ----
    {
      const double p2 = Q.tabR[4 * r], ca_ = Q.tabR[4 * r + 1];
      double scc = p1 * p1 + p2 * p2 + 2.0 * p1 * p2 * ca_;
      scc = scc > 0.0 ? scc : 0.0;
      const double scc3 = scc * third;
      const double2* nA = sm.nodeA + b * NODES;
      const double* rc = sm.rowc + b * KP;
      const double* nS = sm.nodeS + b * NODES;
      const double2* ta = reinterpret_cast<const double2*>(Q.tabA) + ((size_t)(pair0 + w) * G + a) * 4;
      const size_t ta_step = (size_t)nw * G * 4;
      double2 c01 = make_double2(0.0, 0.0), c23 = c01, c45 = c01;
      if (active && w < npl) { c01 = ta[0]; c23 = ta[1]; c45 = ta[2]; }   // (idle threads and pair slots beyond the chunk: ta points past tabA)
      for (int pl = w; pl < npl; pl += nw) {
        if (active) {
          const double cur[6] = {c01.x, c01.y, c23.x, c23.y, c45.x, c45.y};
          ta += ta_step;
          if (pl + nw < npl) { c01 = ta[0]; c23 = ta[1]; c45 = ta[2]; }
          const double2* na = nA + pl * n2;
          double acc2 = acc;      // (w0 is folded into the quartic coefficients: the row adds straight into the running sum)
          if constexpr (TAB3D) {
            const double* ns = nS + pl * n2;
            if (Q.paired3) {
#pragma unroll 4
              for (int j2 = 0; j2 < n2; ++j2) {
                const double2 bs = na[j2];
                const double lam3 = tab3d_vertex_cached(sm.stab3, stab3B, Q.T3, fm, cell3, scc, cur[0], ns[j2]);
                const double poly = fma(fma(fma(fma(cur[5], bs.y, cur[4]), bs.y, cur[3]), bs.y, cur[2]), bs.y, cur[1]);
                acc2 = fma(bs.x * poly, lam3, acc2);
              }
            } else {
#pragma unroll 4
              for (int j2 = 0; j2 < n2; ++j2) {
                const double2 bs = na[j2];
                const double lam3 = tab3d_vertex(sm.stab3, Q.T3, fm, scc, cur[0], ns[j2]);
                const double poly = fma(fma(fma(fma(cur[5], bs.y, cur[4]), bs.y, cur[3]), bs.y, cur[2]), bs.y, cur[1]);
                acc2 = fma(bs.x * poly, lam3, acc2);
              }
            }
          } else {
            const double up = (cur[0] + scc3) + rc[pl];
            if constexpr (N2 > 0) {
#pragma unroll
              for (int j2 = 0; j2 < N2; ++j2) acc2 = t3m_node(na[j2], up, m2k23, lg, sm.cL3, cc, cur, acc2);
            } else {
#pragma unroll 4
              for (int j2 = 0; j2 < n2; ++j2) acc2 = t3m_node(na[j2], up, m2k23, lg, sm.cL3, cc, cur, acc2);
            }
          }
          acc = acc2;
        }
      }
    }
    if (iu + 2 < nu) phase0(r2, ch2, b);
    if (last_of_r) {
      // partial sums of this CTA for r: slot = rank of this CTA among the owners of r's units
      const long long ufirst = (long long)r * NCH;
      const int c_first = (int)(((ufirst + 1) * gridDim.x - 1) / U);
      const int slot = (int)blockIdx.x - c_first;
      sm.red[tid] = active ? acc : 0.0;
      const double dB = block_min(dmB_cur, red32);  // two barriers: also publishes sm.red
      if (tid < G) {
        double t = sm.red[tid];
        for (int ww = 1; ww < nw; ++ww) t += sm.red[tid + ww * G];
        Q.part[(size_t)slot * P.n_ext + (size_t)tid * S + r] = t;
      }
      if (tid == 0) Q.partB[(size_t)slot * S + r] = dB;
      acc = 0.0;
      dmB_cur = dmB_nxt;
      dmB_nxt = inf;
    }
    __syncthreads();  // unit u is drained: its buffer may be refilled; the stage of unit u+1 is complete
    r = r1; ch = ch1; r1 = r2; ch1 = ch2;
    next_unit(r2, ch2);
  }
}

__global__ void __launch_bounds__(256) t3g_fixup_kernel(const ThreeGridParams Q) {
  if (*Q.flag != 0) return;
  const ThreePointParams& P = Q.B;
  const long long e = (long long)blockIdx.x * 256 + threadIdx.x;
  if (e >= P.n_ext) return;
  const int S = Q.S, G = Q.G, NCH = Q.NCH;
  const int a = (int)(e / S), r = (int)(e - (long long)a * S);
  const long long U = (long long)S * NCH;
  const long long ufirst = (long long)r * NCH, ulast = ufirst + NCH - 1;
  const int c_first = (int)(((ufirst + 1) * Q.grid_main - 1) / U), c_last = (int)(((ulast + 1) * Q.grid_main - 1) / U);
  CompSum ts(Q.part[e]);
  for (int s = 1; s <= c_last - c_first; ++s) ts.add(Q.part[(size_t)s * P.n_ext + e]);
  const double t = ts.value();
  double sum_wphi = 0.0;
  for (int jp = 0; jp < P.nphi; ++jp) sum_wphi += P.wphi[jp];
  P.out[e] = P.prefactor * sum_wphi * t;
  if (P.dmin) {
    double dm = *Q.qmin;
    for (int s = 0; s <= c_last - c_first; ++s) dm = fmin(dm, Q.partB[(size_t)s * S + r]);
    const int npairs = P.nq * P.n1;
    for (int pair = 0; pair < npairs; ++pair) dm = fmin(dm, Q.tabA[((size_t)pair * G + a) * 8 + 7]);
    P.dmin[e] = dm * P.reg.inv_k2;
  }
}


int t3g_launch(ThreePointParams& P, int G, int regk, const Tab3DParams* T3, const double* v3, int ntab3,
                      int sm_count, cudaStream_t stream, void** scratch_out) {
  const int n_ext = P.n_ext;
  if (!(G >= 2 && G <= 256 && n_ext % G == 0 && P.n2 <= T3G_NODES)) return DFRG_OK;
  const size_t smem_pre = t3g_smem(P.nq, P.n1, P.n2, P.grid.n, T3 ? ntab3 : 0);
  if (smem_pre > kMaxDynSmem) return DFRG_OK;   // (large 3-D tables: the general kernel)
  // node buffer of the main kernel: the largest of 2048 / 1024 / 512 nodes that fits (fewer, longer work units)
  const int npairs = P.nq * P.n1;
  const int nw = T3G_MAXT / G;   // pair slots of the main kernel
  auto pairs_per_unit = [&](int nodes_) {
    int kp = nodes_ / P.n2 < npairs ? nodes_ / P.n2 : npairs;
    if (kp > nw) kp -= kp % nw;   // whole rounds of the pair slots
    return kp;
  };
  int nodes = 2048;
  while (nodes > T3G_NODES && (nodes / 2 >= P.n2) &&
         t3m_smem(P.nq, P.n1, P.n2, P.grid.n, nodes, pairs_per_unit(nodes), T3G_MAXT, T3 ? ntab3 : 0) > 176 * 1024)
    nodes /= 2;
  if (nodes < P.n2) nodes = T3G_NODES;
  const int kp = pairs_per_unit(nodes);
  size_t smem_main = t3m_smem(P.nq, P.n1, P.n2, P.grid.n, nodes, kp, T3G_MAXT, T3 ? ntab3 : 0);
  if (smem_main > kMaxDynSmem) return DFRG_OK;
  // a second, shifted copy of the 3-D table for the paired look-up of the hot loop, if it fits (n[2] >= 2 always holds)
  const size_t smem_copy = 8 * (size_t)((ntab3 + 1) & ~1);
  const bool paired3 = T3 != nullptr && smem_main + smem_copy <= kMaxDynSmem;
  if (paired3) smem_main += smem_copy;
  ThreeGridParams Q;
  Q.B = P;
  Q.G = G; Q.S = n_ext / G;
  Q.v3 = v3; Q.ntab3 = ntab3; Q.paired3 = paired3 ? 1 : 0;
  if (T3) Q.T3 = *T3;
  Q.NODES = nodes;
  Q.lgc = lg2_consts(P.grid.lo, P.grid.inv_h);
  Q.m2k23 = -2.0 * P.reg.k2 * (1.0 / 3.0);
  Q.KP = kp;
  Q.NCH = (npairs + Q.KP - 1) / Q.KP;
  const long long U = (long long)Q.S * Q.NCH;
  Q.grid_main = (int)(U < sm_count ? U : sm_count);
  Q.max_slots = 1;
  for (int r = 0; r < Q.S; ++r) {
    const long long ufirst = (long long)r * Q.NCH, ulast = ufirst + Q.NCH - 1;
    const int c0 = (int)(((ufirst + 1) * Q.grid_main - 1) / U), c1 = (int)(((ulast + 1) * Q.grid_main - 1) / U);
    if (c1 - c0 + 1 > Q.max_slots) Q.max_slots = c1 - c0 + 1;
  }
  const size_t n_tabA = (size_t)npairs * 8 * G, n_tabR = 4 * (size_t)Q.S, n_part = (size_t)Q.max_slots * n_ext,
               n_partB = (size_t)Q.max_slots * Q.S;
  void* scratch = nullptr;
  int rc = scratch_alloc(&scratch, (n_tabA + n_tabR + n_part + n_partB + 4) * sizeof(double), stream);
  if (rc != DFRG_OK) return rc;
  *scratch_out = scratch;
  Q.tabA = (double*)scratch;
  Q.tabR = Q.tabA + n_tabA;
  Q.part = Q.tabR + n_tabR;
  Q.partB = Q.part + n_part;
  Q.qmin = Q.partB + n_partB;
  Q.flag = (int*)(Q.qmin + 2);
  cudaError_t e = cudaMemsetAsync(Q.flag, 0, sizeof(int), stream);
  void (*kpre)(const ThreeGridParams) = nullptr;
  void (*kmain)(const ThreeGridParams) = nullptr;
  const bool n2_16 = P.n2 == 16;   // BASELINE config 3's cos2 order: fully unrolled rows
#define DFRG_T3G_PICK(K)                                                                                  \
  if (regk == K) {                                                                                        \
    kpre = T3 ? t3g_prepass_kernel<K, true> : t3g_prepass_kernel<K, false>;                               \
    kmain = T3 ? t3g_main_kernel<K, T3G_MAXT, 0, true>                                                    \
               : (n2_16 ? t3g_main_kernel<K, T3G_MAXT, 16, false> : t3g_main_kernel<K, T3G_MAXT, 0, false>); \
  }
  DFRG_T3G_PICK(0) DFRG_T3G_PICK(1) DFRG_T3G_PICK(2)
#undef DFRG_T3G_PICK
  int rca = e == cudaSuccess ? DFRG_OK : check_cuda(e);
  if (rca == DFRG_OK) rca = opt_in_max_smem(kpre);
  if (rca == DFRG_OK) rca = opt_in_max_smem(kmain);
  if (rca != DFRG_OK) { scratch_free(scratch, stream); *scratch_out = nullptr; return rca; }
  kpre<<<sm_count, T3G_THREADS, smem_pre, stream>>>(Q);
  kmain<<<Q.grid_main, T3G_MAXT, smem_main, stream>>>(Q);
  t3g_fixup_kernel<<<(n_ext + 255) / 256, 256, 0, stream>>>(Q);
  rc = check_cuda(cudaGetLastError());
  if (rc != DFRG_OK) { scratch_free(scratch, stream); *scratch_out = nullptr; return rc; }
  P.skip_flag = Q.flag;
  return DFRG_OK;
}

}  // namespace dfrg
