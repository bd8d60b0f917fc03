// dfrg_device.cuh -- device-side building blocks shared by the integration kernels (sm_100a).
//   * FP64 reciprocal from the hardware seed (MUFU.RCP64H) + one cubic Newton step
//   * table-driven FP64 log / exp (shared-memory tables), regulators (eq. 14)
//   * log-grid cubic / linear interpolation reading per-cell cubics in shared memory
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

// ---- table-driven FP64 log and exp --------------------------------------------------------------------------
// The S3 pre-computation is dominated by log (table coordinate) and exp (regulator).  libdevice's versions
// cost ~100 SASS instructions each, two thirds of them integer/constant traffic.  These versions keep two small
// tables in shared memory (copied per CTA from the correctly rounded literals of fm_tables.inc, fm_build / TMA) and need ~10 FP64 instructions:
//   fm_log(s):  s = 2^e m, m in [1,2); j = top 7 mantissa bits; r = m * (1/c_j) - 1, |r| <= 2^-8;
//               ln s = e ln2 + ln c_j + (r - r^2/2 + ... - r^6/6)          abs. error <~ 3e-16 for |e| < 64
//   fm_exp_neg(x) = e^-x, 0 <= x: n = rint(-64 x / ln2), r = -x - n ln2/64, |r| <= ln2/128;
//               e^-x = 2^(n>>6) 2^((n&63)/64) (1 + r + ... + r^5/120)       rel. error <~ 2 ulp; exactly 0 where libm's
//               e^-x is 0 (x >= 745.1332191019412) and, flushed, where libm's is a subnormal (x >= 708.4).
// fm_log(0) = -709.8 (exponent field 0): every table coordinate derived from it clamps to the first grid point.
struct FastMath {
  const double2* logtab;  // [128] (1/c_j, ln c_j)
  const double* exptab;   // [64]  2^(j/64)
  const double* k;        // FastMathConsts::c inside the kernel parameters
};
// Polynomial coefficients travel inside the kernel parameter struct (constant bank c[0x0]) so that DFMA reads
// them as constant operands; as compile-time literals the compiler rebuilds each 64-bit immediate in uniform
// registers (two UMOV) before every use.
struct FastMathConsts {
  double c[20];
};
inline FastMathConsts fm_consts() {
  FastMathConsts k = {{
      -1.0 / 6.0, 1.0 / 5.0, -0.25, 1.0 / 3.0, -0.5,  // 0-4  ln(1+r) = r + r^2 (-1/2 + r/3 - r^2/4 + r^3/5 - r^4/6)
      0.6931471805592082, 7.371002565167799e-13,      // 5,6  ln2 hi / lo (40-bit split)
      -92.33248261689366, 6755399441055744.0,         // 7,8  -64/ln2, 1.5 * 2^52
      -0.01083042469326756, -2.9815858269852933e-12,  // 9,10 -(ln2/64) hi / lo (32-bit split)
      1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0, 0.5, 1.0,   // 11-15 exp series
      -369.3299304675746,                             // 16    -256/ln2                  (fx_exp_neg, 256-entry table)
      -0.01083042469326756 / 4.0, -2.9815858269852933e-12 / 4.0,  // 17,18 -(ln2/256) hi / lo
      0.0}};
  return k;
}
// Branch-free clamps as one DSETP + two SEL (CUDA's fmin/fmax add NaN fix-ups: seven instructions each).
__device__ __forceinline__ double clamp_lo(double x, double lo) {  // x > lo ? x : lo   (NaN -> lo)
  double r;
  asm("{\n.reg .pred p;\nsetp.gt.f64 p, %1, %2;\nselp.f64 %0, %1, %2, p;\n}" : "=d"(r) : "d"(x), "d"(lo));
  return r;
}
__device__ __forceinline__ double clamp_hi(double x, double hi) {  // x < hi ? x : hi   (NaN -> hi)
  double r;
  asm("{\n.reg .pred p;\nsetp.lt.f64 p, %1, %2;\nselp.f64 %0, %1, %2, p;\n}" : "=d"(r) : "d"(x), "d"(hi));
  return r;
}
constexpr int FM_DOUBLES = 2 * 128 + 64;
#include "fm_tables.inc"   // kFmLog, kFmExp, kLg2Log: correctly rounded constants (gen_fm_tables.py)

// All threads of the CTA; the caller synchronises before first use.  mem: FM_DOUBLES doubles, 16-byte aligned.
// The tables are constants of the library (fm_tables.inc): a CTA copies them from global memory (L2 resident after the
// first CTA) instead of computing 128 divisions + logarithms and 64 exp2 in its set-up.
__device__ __forceinline__ FastMath fm_build(double* mem, const FastMathConsts& consts) {
  double2* lt = reinterpret_cast<double2*>(mem);
  double* et = mem + 256;
  for (int j = threadIdx.x; j < 128; j += blockDim.x)
    lt[j] = make_double2(kFmLog[2 * j], kFmLog[2 * j + 1]);  // (1/c_j rounded, ln of the centre the rounded reciprocal stands for)
  for (int j = threadIdx.x; j < 64; j += blockDim.x) et[j] = kFmExp[j];
  FastMath fm;
  fm.logtab = lt;
  fm.exptab = et;
  fm.k = consts.c;
  return fm;
}

// The same tables through a stage list (TMA bulk copies from the constant arrays: no instructions in the CTA's set-up).
// Declared after StageList below; mem: FM_DOUBLES doubles, 16-byte aligned.
struct StageList;
__device__ __forceinline__ FastMath fm_stage(StageList& L, double* mem, const FastMathConsts& consts);

__device__ __forceinline__ double fm_log(const FastMath& fm, double s) {
  const int hi = __double2hiint(s);
  const int e = (hi >> 20) - 1023;
  const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(s));
  const double2 T = fm.logtab[(hi >> 13) & 127];
  const double r = fma(m, T.x, -1.0);
  double q = fma(r, fm.k[0], fm.k[1]);
  q = fma(r, q, fm.k[2]);
  q = fma(r, q, fm.k[3]);
  q = fma(r, q, fm.k[4]);
  const double lm = fma(r * r, q, r);  // ln(1 + r)
  const double ed = (double)e;
  return fma(ed, fm.k[5], T.y) + fma(ed, fm.k[6], lm);
}

// libm's e^-x is exactly 0 from x = 745.1332191019412 on (reading A17: 0 on both sides).  Here the argument is clamped to 746
// and the scaling by 2^(n >> 6) -- an integer add into the exponent field -- returns exactly 0 whenever the result would not
// be a normal number: e^-x = 0 for x >= 708.4 (libm returns subnormals, < 2.3e-308, between 708.4 and 745.13).  One integer
// compare and two selects on the result; a test on the bits of x itself (a 64-bit compare with x kept alive across the
// series) cost the three- and four-point kernels 8-20 % of their time.
__device__ __forceinline__ double exp_scale_flush(const double v, const int n) {
  const int hi = __double2hiint(v) + ((n >> 6) << 20);
  const bool sub = hi < 0x00100000;                 // exponent field <= 0 (or wrapped below it)
  return __hiloint2double(sub ? 0 : hi, sub ? 0 : __double2loint(v));
}
__device__ __forceinline__ double fm_exp_neg(const FastMath& fm, double x) {
  x = clamp_hi(x, 746.0);   // (NaN -> 746 -> 0)
  const double MAGIC = fm.k[8];  // 1.5 * 2^52: the low word of y holds rint(-x * 64/ln2)
  const double y = fma(x, fm.k[7], MAGIC);
  const int n = __double2loint(y);
  const double nd = y - MAGIC;
  double r = fma(nd, fm.k[9], -x);
  r = fma(nd, fm.k[10], r);
  double p = fma(r, fm.k[11], fm.k[12]);
  p = fma(r, p, fm.k[13]);
  p = fma(r, p, fm.k[14]);
  p = fma(r, p, fm.k[15]);
  p = fma(r, p, fm.k[15]);
  const double v = fm.exptab[n & 63] * p;
  return exp_scale_flush(v, n);
}

// ---- regulators --------------------------------------------------------------------------------
struct RegParams {
  int kind;   // 0 Litim, 1 EXP_POLY
  int order;
  double k2;      // k^2
  double inv_k2;  // 1/k^2
  double zk;      // wave-function renormalisation: R = zk R_shape
  double eta;     // anomalous dimension: Rdot = zk (Rdot_shape - eta R_shape)
};
// host side: RegParams from the ABI struct
inline RegParams reg_params(int kind, int order, double k, double zk, double eta) {
  RegParams rp;
  rp.kind = kind; rp.order = order; rp.k2 = k * k; rp.inv_k2 = 1.0 / rp.k2; rp.zk = zk; rp.eta = eta;
  return rp;
}

__device__ __forceinline__ void regulator(const RegParams& rp, const FastMath& fm, double s, double& R, double& Rdot) {
  if (rp.kind == 0) {
    const bool in = s < rp.k2;
    const double Rs = in ? rp.k2 - s : 0.0;
    R = rp.zk * Rs;
    Rdot = rp.zk * ((in ? 2.0 * rp.k2 : 0.0) - rp.eta * Rs);
    return;
  }
  const double x = s * rp.inv_k2;
  double expo = x, geo = x;
  if (rp.order > 1) {
    double xi = x;
    for (int i = 2; i <= rp.order; ++i) {
      xi *= x;
      expo += xi / (double)i;
      geo += xi;
    }
  }
  const double r = rp.k2 * fm_exp_neg(fm, expo);
  R = rp.zk * r;
  Rdot = rp.zk * (2.0 * r * (1.0 + geo) - rp.eta * r);
}

// Fermion line regulated with the fermionic regulator RF / RFdot (reading A25):
//   (sqrt(s) + R_F)^2 = s + R_B  =>  R_F = R_B/(sqrt(s + R_B) + sqrt(s)),  k dR_F/dk = RBdot/(2 sqrt(s + R_B)),
//   RF = zk R_F,  RFdot = zk (k dR_F/dk - eta R_F);  kinetic term A = Z sqrt(sR) + RF(sR) at the regulator argument sR.
// Returns A; ins = 2 A RFdot (what replaces Rdot in the insertion).  The line's denominator is Z^2 (s - sR) + A^2 + m^2.
__device__ __forceinline__ double fermion_kinetic(const RegParams& rp, const FastMath& fm, const double Z, const double sR,
                                                  double& ins) {
  RegParams shape = rp;
  shape.zk = 1.0; shape.eta = 0.0;
  double Rb, Rbd;
  regulator(shape, fm, sR, Rb, Rbd);
  const double root = sqrt(sR + Rb), sq = sqrt(sR);
  const double rf = Rb / (root + sq);
  const double rfd = Rbd / (2.0 * root);
  const double A = fma(Z, sq, rp.zk * rf);
  ins = 2.0 * A * (rp.zk * (rfd - rp.eta * rf));
  return A;
}

// ---- log-grid table look-up --------------------------------------------------------------------
// A table row v[0..n-1] on ln q_i = lo + i h is turned, once per CTA, into per-cell cubics in shared memory:
//   cubic mode (interp 3): cell c = stencil i0 = c, anchored at node c+1:  p(tau) = v[c+1] + tau (d1 + tau (d2 + tau d3)),
//     the 4-point Lagrange interpolant through v[c..c+3] written in tau = t - (c+1)   (n-3 cells)
//   linear mode (interp 1): cell c anchored at node c: p(tau) = v[c] + tau (v[c+1] - v[c])          (n-1 cells)
// so a look-up is fm_log, one FMA, two clamps, an index, two LDS.128 and three FMAs.
struct GridParams {
  double lo;     // ln q_0
  double inv_h;  // (n-1)/(hi-lo)
  int n;
  int interp;    // 1 or 3
  __device__ __forceinline__ int ncell() const { return interp == 3 ? n - 3 : n - 1; }
  __device__ __forceinline__ int off() const { return interp == 3 ? 1 : 0; }
};

// cells: ncell() double4, 32-byte aligned; v may live in shared or global memory.  All threads; caller synchronises.
__device__ __forceinline__ void cells_build(double4* cells, const double* __restrict__ v, const GridParams& g) {
  const int nc_ = g.ncell();
  for (int c = threadIdx.x; c < nc_; c += blockDim.x) {
    if (g.interp == 3) {
      const double v0 = v[c], v1 = v[c + 1], v2 = v[c + 2], v3 = v[c + 3];
      const double d1 = (-2.0 * v0 - 3.0 * v1 + 6.0 * v2 - v3) * (1.0 / 6.0);
      const double d2 = (v0 - 2.0 * v1 + v2) * 0.5;
      const double d3 = ((v3 - v0) + 3.0 * (v1 - v2)) * (1.0 / 6.0);
      cells[c] = make_double4(v1, d1, d2, d3);
    } else {
      cells[c] = make_double4(v[c], v[c + 1] - v[c], 0.0, 0.0);
    }
  }
}

// Value of the table at squared momentum s.
__device__ __forceinline__ double table_lookup(const double4* __restrict__ cells, const GridParams& g,
                                               const FastMath& fm, double s) {
  const double l = 0.5 * fm_log(fm, s);
  double t = (l - g.lo) * g.inv_h;
  t = clamp_lo(t, 0.0);  // NaN -> 0
  t = clamp_hi(t, (double)(g.n - 1));
  int c = (int)t - g.off();  // t >= 0: truncation == floor
  c = max(c, 0);
  c = min(c, g.ncell() - 1);
  const double tau = t - (double)(c + g.off());
  const double4 k = cells[c];
  return fma(fma(fma(k.w, tau, k.z), tau, k.y), tau, k.x);
}

// ---- fused log-grid coordinate and guarded cells (the S3 look-up of the hot three-point loop) -----------------
// t(s) = (ln(s)/2 - lo)/h = A ln s + B straight from the bits of s, without a separate logarithm:
//   s = 2^e m,  j = top 9 mantissa bits,  r = m inv_j - 1 (|r| <= 2^-10),  ln(1+r) = r - r^2/2 + r^3/3 - r^4/4
//   (truncation r^5/5 < 1.8e-16 absolute in ln s: far below the rounding of t itself, ulp(127) = 1.4e-14)
//   t = e A ln2 + (A ln(1+r) + mant[j].y),   mant[j] = (A inv_j, A ln c_j + B),  everything in r' = A r
// E = the exponent field of s >= 0 (callers clamp s at 0): zero and subnormal s land far below the grid (the table's
// first value, as log(0) = -inf would give), inf/NaN far above.  6 FP64 instructions, one conversion, one LDS.128.
// The cells carry guards: index F + 1 with F = clamp(floor(t), -1, n-1); F = -1 and F = n-1 are constant cells
// (clamp-to-edge), the others hold the interpolant of SURVEY 8(c) (4-point Lagrange on the stencil
// i0 = clamp(F-1, 0, n-4), or the linear one) re-expanded in tau = t - F.  Integer clamps replace the FP64 ones.
// Threads of a warp look up unrelated entries, so both tables are replicated LG_REP = 8 times, one copy per
// lane-slot (lane & 7) confined to its own 16-byte bank group: a 128-bit shared-memory load is served in
// quarter-warps of 8 consecutive lanes, hence every look-up is conflict free (4 wavefronts) wherever it points.
constexpr int LG_NM = 512, LG_REP = 8;
constexpr int LG_DOUBLES = 2 * LG_NM * LG_REP;  // 64 KB
struct LogGrid {
  const double2* mant;   // this thread's copy: entry j at mant[j * LG_REP] = (A inv_j, A ln c_j + B)
  double negA, ex1;      // -A, A ln2         (A = 1/(2h))
  double c1, c2, c3;     // -1/(2A), 1/(3A^2), -1/(4A^3): ln(1+r) = r (1 + r'(c1 + r'(c2 + r' c3))) / ... in r' = A r
  int nm1;               // n - 1
};
// All threads of the CTA; the caller synchronises before first use.  mem: LG_DOUBLES doubles, 16-byte aligned.
__device__ __forceinline__ LogGrid lg_build(double* mem, const double lo, const double inv_h, const int n) {
  double2* mt = reinterpret_cast<double2*>(mem);
  const double A = 0.5 * inv_h, B = -lo * inv_h;
  const double ex1 = A * 0.6931471805599453;
  for (int j = threadIdx.x; j < LG_NM; j += blockDim.x) {
    // c_j = 1/inv_j with inv_j = fl(1/(1 + (j + 1/2)/512)) from the constant table; A inv_j is rounded once more, which moves
    // the centre it stands for by < 1.2e-16 relative (5e-16 in t, against ulp(t) = 1.4e-14 at the top of the grid)
    const double2 ent = make_double2(A * kLg2Log[2 * j], fma(-A, kLg2Log[2 * j + 1], B));
#pragma unroll
    for (int r = 0; r < LG_REP; ++r) mt[j * LG_REP + r] = ent;
  }
  LogGrid L;
  L.mant = mt + (threadIdx.x & (LG_REP - 1));
  L.negA = -A;
  L.ex1 = ex1;
  L.c1 = -0.5 / A;
  L.c2 = 1.0 / (3.0 * A * A);
  L.c3 = -0.25 / (A * A * A);
  L.nm1 = n - 1;
  return L;
}
// t(s): six FP64 instructions (r' = A r;  A ln(1+r) = r' (1 + r' (c1 + r' (c2 + r' c3)));  exponent term by FMA).
__device__ __forceinline__ double lg_coord(const LogGrid& L, const double* __restrict__, const double s) {
  const unsigned hi = (unsigned)__double2hiint(s);
  const double m = __hiloint2double((int)((hi & 0x000fffffu) | 0x3ff00000u), __double2loint(s));
  const double2 T = L.mant[((hi >> 11) & (LG_NM - 1)) * LG_REP];
  const double rp = fma(m, T.x, L.negA);
  const double P = fma(rp, fma(rp, fma(rp, L.c3, L.c2), L.c1), 1.0);
  return fma((double)((int)(hi >> 20) - 1023), L.ex1, fma(rp, P, T.y));
}
// Guarded cells of one table row, replicated: n + 1 cells x 2 halves x LG_REP double2.  cells_guarded_size(n) double2.
// v may live in shared or global memory.  All threads; caller synchronises.  Returns this thread's copy.
__device__ __host__ constexpr int cells_guarded_size(int n) { return (n + 1) * 2 * LG_REP; }
__device__ __forceinline__ const double2* cells_build_guarded(double2* cells, const double* __restrict__ v,
                                                              const int n, const int interp) {
  for (int c = threadIdx.x; c <= n; c += blockDim.x) {
    const int F = c - 1;
    double4 k;
    if (F < 0) k = make_double4(v[0], 0.0, 0.0, 0.0);
    else if (F >= n - 1) k = make_double4(v[n - 1], 0.0, 0.0, 0.0);
    else if (interp == 3) {
      int i0 = F - 1;
      i0 = i0 < 0 ? 0 : i0;
      i0 = i0 > n - 4 ? n - 4 : i0;
      const int dl = F - i0;  // anchor node inside the stencil: 0, 1 or 2
      const double v0 = v[i0], v1 = v[i0 + 1], v2 = v[i0 + 2], v3 = v[i0 + 3];
      const double d3 = ((v3 - v0) + 3.0 * (v1 - v2)) * (1.0 / 6.0);
      if (dl == 0)
        k = make_double4(v0, (-11.0 * v0 + 18.0 * v1 - 9.0 * v2 + 2.0 * v3) * (1.0 / 6.0),
                         (2.0 * v0 - 5.0 * v1 + 4.0 * v2 - v3) * 0.5, d3);
      else if (dl == 1)
        k = make_double4(v1, (-2.0 * v0 - 3.0 * v1 + 6.0 * v2 - v3) * (1.0 / 6.0), (v0 - 2.0 * v1 + v2) * 0.5, d3);
      else
        k = make_double4(v2, (v0 - 6.0 * v1 + 3.0 * v2 + 2.0 * v3) * (1.0 / 6.0), (v1 - 2.0 * v2 + v3) * 0.5, d3);
    } else {
      k = make_double4(v[F], v[F + 1] - v[F], 0.0, 0.0);
    }
#pragma unroll
    for (int r = 0; r < LG_REP; ++r) {
      cells[(2 * c) * LG_REP + r] = make_double2(k.x, k.y);
      cells[(2 * c + 1) * LG_REP + r] = make_double2(k.z, k.w);
    }
  }
  return cells + (threadIdx.x & (LG_REP - 1));
}
// cells: this thread's copy (the pointer cells_build_guarded returns)
__device__ __forceinline__ double lg_cell_eval(const double2* __restrict__ cells, const LogGrid& L, const double t) {
  int F = __double2int_rd(t);  // F2I.FLOOR: saturates, NaN -> 0
  F = max(F, -1);
  F = min(F, L.nm1);
  const double tau = t - (double)F;
  const double2* cp = cells + (F + 1) * (2 * LG_REP);
  const double2 k0 = cp[0], k1 = cp[LG_REP];
  return fma(fma(fma(k1.y, tau, k1.x), tau, k0.y), tau, k0.x);
}
__device__ __forceinline__ double lg_lookup(const double2* __restrict__ cells, const LogGrid& L,
                                            const double* __restrict__ kc, const double s) {
  return lg_cell_eval(cells, L, lg_coord(L, kc, s));
}

// ---- second-generation coordinate / cells for the hot product-grid loop (t3g_main_kernel) ---------------------
// Same mathematics as lg_coord / lg_cell_eval, arranged for the fewest issue slots per look-up:
//   * mant[j] = (inv_j, A ln c_j + B + 1): the reciprocal is NOT pre-multiplied by A, so 2^-e can be folded into its
//     exponent field with one integer multiply-add (inv' = inv_j 2^-e; r = fma(x, inv', -1) is the same exact residual as
//     m inv_j - 1 without building the mantissa m), and A moves into the series coefficients a1..a4;
//   * the coordinate comes out as t' = t + 1 >= 0 for every s on or above the first grid point, so that one
//     saturating float-to-unsigned conversion is floor AND the lower clamp: F' = min(cvt.rmi.u32(t'), n) in [0, n];
//   * guarded cells are NOT replicated (32 bytes each, cell F' at byte 32 F'): the hot loop keeps the current cell in
//     registers and reloads it only when F' changes (x is monotone along the c2 row, so this is rare).
// x = 0 and subnormal x give t' << 0 -> cell 0 (the table's first value); valid for x < 2^1023.
// The series coefficients travel in the kernel parameters (constant bank), so that every DFMA of the coordinate reads
// its constant as an operand and no register holds them.
struct LogGrid2Consts {
  double a1, a2, a3, a4;  // A, -A/2, A/3, -A/4   (A = 1/(2h)):  A ln(1+r) = r (a1 + r (a2 + r (a3 + r a4)))
  double ex1;             // A ln2
  double bq;              // B + 1 = 1 - lo/h
};
inline LogGrid2Consts lg2_consts(const double lo, const double inv_h) {   // host side
  const double A = 0.5 * inv_h;
  LogGrid2Consts K;
  K.a1 = A; K.a2 = -0.5 * A; K.a3 = A * (1.0 / 3.0); K.a4 = -0.25 * A;
  K.ex1 = A * 0.6931471805599453;
  K.bq = -lo * inv_h + 1.0;
  return K;
}
struct LogGrid2 {
  const char* mant;      // the table: entry j, replica r at byte 128 j + 16 r
  unsigned rep16;        // 16 * (this thread's replica): OR-ed into the byte offset (the index bits start at bit 7)
  unsigned n;            // grid points = index of the upper guard cell
  const LogGrid2Consts* K;   // inside the kernel parameters
};
__device__ __forceinline__ LogGrid2 lg2_build(double* mem, const LogGrid2Consts& K, const int n) {
  double2* mt = reinterpret_cast<double2*>(mem);
  for (int j = threadIdx.x; j < LG_NM; j += blockDim.x) {
    static_assert(LG_NM == 512, "kLg2Log holds 512 entries");
    const double inv = kLg2Log[2 * j];               // fl(1/c_j), c_j = 1 + (j + 1/2)/512; the rounded value defines the centre
    const double2 ent = make_double2(inv, fma(-K.a1, kLg2Log[2 * j + 1], K.bq));
#pragma unroll
    for (int r = 0; r < LG_REP; ++r) mt[j * LG_REP + r] = ent;
  }
  LogGrid2 L;
  L.mant = reinterpret_cast<const char*>(mt);
  L.rep16 = 16u * (threadIdx.x & (LG_REP - 1));
  L.n = (unsigned)n;
  L.K = &K;
  return L;
}
// Precondition: x >= 0 (or NaN).  The exponent is taken from the high word WITHOUT masking the sign bit (one integer
// instruction less in the three-point hot loop), so a negative x -- even -0.0 or a rounding-sized negative value -- would
// come out as a huge t' and land in the LAST cell, where reading A16 (max(s, 0): log 0 clamps to the first entry) wants the
// first.  Every caller guarantees it: set-up code clamps s at 0 before the call; the product-grid hot loop feeds
// x = (s_a + s_b + s_c)/3 with s_a, s_c >= 0 fixed per row and s_b = |q + p2|^2 at Gauss-Legendre nodes (|cos| < 1
// strictly), where the unclamped s_b >= (q - p2)^2 (1 - |cos|) stays far above rounding size relative to the sum.
__device__ __forceinline__ double lg2_coord(const LogGrid2& L, const double x) {
  const int hi = __double2hiint(x);
  unsigned off;                                   // 128 * (top 9 mantissa bits) + 16 * replica, as ONE three-input LOP3
  asm("lop3.b32 %0, %1, 0xff80, %2, 0xEA;" : "=r"(off) : "r"((unsigned)hi >> 4), "r"(L.rep16));
  const double2 T = *reinterpret_cast<const double2*>(L.mant + off);
  const int e = (int)((unsigned)hi >> 20) - 1023;
  const double inv = __hiloint2double(__double2hiint(T.x) - (e << 20), __double2loint(T.x));   // inv_j 2^-e
  const double r = fma(x, inv, -1.0);
  const double P = fma(r, fma(r, fma(r, L.K->a4, L.K->a3), L.K->a2), L.K->a1);
  return fma((double)e, L.K->ex1, fma(r, P, T.y));
}
// Guarded cells, one copy: cell F' in [0, n] as double4 (value, d1, d2, d3) in tau = t' - F'.  (n + 1) double4.
__device__ __forceinline__ void cells2_build(double4* cells, const double* __restrict__ v, const int n, const int interp) {
  for (int c = threadIdx.x; c <= n; c += blockDim.x) {
    const int F = c - 1;
    double4 k;
    if (F < 0) k = make_double4(v[0], 0.0, 0.0, 0.0);
    else if (F >= n - 1) k = make_double4(v[n - 1], 0.0, 0.0, 0.0);
    else if (interp == 3) {
      int i0 = F - 1;
      i0 = i0 < 0 ? 0 : i0;
      i0 = i0 > n - 4 ? n - 4 : i0;
      const int dl = F - i0;
      const double v0 = v[i0], v1 = v[i0 + 1], v2 = v[i0 + 2], v3 = v[i0 + 3];
      const double d3 = ((v3 - v0) + 3.0 * (v1 - v2)) * (1.0 / 6.0);
      if (dl == 0)
        k = make_double4(v0, (-11.0 * v0 + 18.0 * v1 - 9.0 * v2 + 2.0 * v3) * (1.0 / 6.0),
                         (2.0 * v0 - 5.0 * v1 + 4.0 * v2 - v3) * 0.5, d3);
      else if (dl == 1)
        k = make_double4(v1, (-2.0 * v0 - 3.0 * v1 + 6.0 * v2 - v3) * (1.0 / 6.0), (v0 - 2.0 * v1 + v2) * 0.5, d3);
      else
        k = make_double4(v2, (v0 - 6.0 * v1 + 3.0 * v2 + 2.0 * v3) * (1.0 / 6.0), (v1 - 2.0 * v2 + v3) * 0.5, d3);
    } else {
      k = make_double4(v[F], v[F + 1] - v[F], 0.0, 0.0);
    }
    cells[c] = k;
  }
}
__device__ __forceinline__ unsigned lg2_cell(const LogGrid2& L, const double tq) {
  const unsigned F = __double2uint_rd(tq);   // F2I.U32.F64.FLOOR: negative and NaN -> 0
  return min(F, L.n);
}
// stand-alone look-up (set-up code; the hot loop inlines the pieces around its cell cache)
__device__ __forceinline__ double lg2_lookup(const double4* __restrict__ cells, const LogGrid2& L, const double x) {
  const double tq = lg2_coord(L, x);
  const unsigned F = lg2_cell(L, tq);
  const double tau = tq - (double)F;
  const double4 k = cells[F];
  return fma(fma(fma(k.w, tau, k.z), tau, k.y), tau, k.x);
}

// k^2 e^-x from a table of k^2 2^(j/64), replicated 16 times (one copy per lane & 15: a 64-bit shared-memory load is
// served in half-warps, so the look-up is conflict free):  n = rint(-64 x / ln2), r = -x - n ln2/64, |r| <= ln2/128,
// e^r by its series to r^5/120.  Exactly 0 where libm underflows to 0 and where its result is a subnormal.
constexpr int FX_REP = 16;
constexpr int FX_DOUBLES = 64 * FX_REP;
__device__ __forceinline__ const double* fx_build(double* mem, const double k2) {
  for (int j = threadIdx.x; j < 64; j += blockDim.x) {
    const double v = k2 * kFmExp[j];
#pragma unroll
    for (int r = 0; r < FX_REP; ++r) mem[j * FX_REP + r] = v;
  }
  return mem + (threadIdx.x & (FX_REP - 1));
}
__device__ __forceinline__ double fx_exp_neg(const double* __restrict__ tab, const double* __restrict__ kc, double x) {
  x = clamp_hi(x, 746.0);
  const double MAGIC = kc[8];
  const double y = fma(x, kc[7], MAGIC);
  const int n = __double2loint(y);
  const double nd = y - MAGIC;
  double r = fma(nd, kc[9], -x);
  r = fma(nd, kc[10], r);
  double p = fma(r, kc[11], kc[12]);
  p = fma(r, p, kc[13]);
  p = fma(r, p, kc[14]);
  p = fma(r, p, kc[15]);
  p = fma(r, p, kc[15]);
  const double v = tab[(n & 63) * FX_REP] * p;
  return exp_scale_flush(v, n);
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
// Same, with a back-off between polls: for a producer that is far ahead and must not steal issue slots.
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* bar, uint32_t parity, unsigned ns) {
  for (;;) {
    uint32_t done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    if (done) break;
    __nanosleep(ns);
  }
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

__device__ __forceinline__ FastMath fm_stage(StageList& L, double* mem, const FastMathConsts& consts) {
  L.add(mem, kFmLog, 256);
  L.add(mem + 256, kFmExp, 64);
  FastMath fm;
  fm.logtab = reinterpret_cast<const double2*>(mem);
  fm.exptab = mem + 256;
  fm.k = consts.c;
  return fm;
}

// stage_issue + stage_wait = stage_to_smem; work placed between the two overlaps the copies' flight time.
// (The loops over the list are fully unrolled so that the list lives in registers: with run-time indices it sits in local
// memory and thread 0 spends ~3000 cycles walking it.  Copy a is issued by lane 0 of warp a mod n_warps: a bulk-copy
// instruction takes ~200 cycles to issue, five of them in one thread cost a microsecond at the head of a short kernel.  The
// barrier cannot complete before thread 0's arrive.expect_tx, whatever the order in which the copies' complete_tx land.)
__device__ __forceinline__ void stage_issue(const StageList& L, uint64_t* bar) {
  // bar must have been initialised (count 1) and fenced before the first call
  const int warp = threadIdx.x >> 5, n_warps = (blockDim.x + 31) >> 5;
  if ((threadIdx.x & 31) == 0) {
    if (threadIdx.x == 0) {
      uint32_t total = 0;
#pragma unroll
      for (int a = 0; a < 8; ++a)
        if (a < L.count && tma_ok(L.src[a], (size_t)L.n[a] * 8) && tma_ok(L.dst[a], 16)) total += (uint32_t)L.n[a] * 8u;
      mbar_expect_tx(bar, total);
    }
#pragma unroll
    for (int a = 0; a < 8; ++a)
      if (a < L.count && warp == a % n_warps && tma_ok(L.src[a], (size_t)L.n[a] * 8) && tma_ok(L.dst[a], 16))
        tma_bulk_g2s(L.dst[a], L.src[a], (uint32_t)L.n[a] * 8u, bar);
  }
#pragma unroll
  for (int a = 0; a < 8; ++a) {
    if (a < L.count && !(tma_ok(L.src[a], (size_t)L.n[a] * 8) && tma_ok(L.dst[a], 16)))
      for (int i = threadIdx.x; i < L.n[a]; i += blockDim.x) L.dst[a][i] = L.src[a][i];
  }
}
__device__ __forceinline__ void stage_wait(uint64_t* bar, uint32_t parity) {
  mbar_wait(bar, parity);
  __syncthreads();
}
__device__ __forceinline__ void stage_to_smem(const StageList& L, uint64_t* bar, uint32_t parity) {
  stage_issue(L, bar);
  stage_wait(bar, parity);
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
// Compensated sum of the per-CTA partial sums of an output (fix-up kernels).  north_star asks for Kahan-compensated partial
// sums "where ncu shows it is free": it is free here -- a fix-up kernel adds <= a handful of slots per output and waits on its
// loads -- and nowhere else: the hot loops are bound by the FP64 pipe ("Kahan"), where a compensated
// add costs three more FP64 instructions per term.  Neumaier's variant (the correction also covers |x| > |sum|); deterministic.
struct CompSum {
  double s, c;
  __device__ __forceinline__ explicit CompSum(double x) : s(x), c(0.0) {}
  __device__ __forceinline__ void add(double x) {
    const double t = s + x;
    c += (fabs(s) >= fabs(x)) ? (s - t) + x : (x - t) + s;
    s = t;
  }
  __device__ __forceinline__ double value() const { return s + c; }
};

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
