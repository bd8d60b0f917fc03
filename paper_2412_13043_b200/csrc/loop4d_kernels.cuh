// loop4d_kernels.cuh -- definitions shared by the translation units of dfrg_integrate_loop4d (one per integrand
// family, so that nvcc builds them side by side): parameter structs, the device helpers more than one family uses,
// and the host-side launchers each translation unit exports.  See loop4d.cu for the family descriptions.
#pragma once
#include "dfrg_device.cuh"
#include "dfrg_internal.h"

namespace dfrg {

// ---- two-point ----
constexpr int TP_FT = 128;      // field threads per consumer group
constexpr int TP_GROUPS = 4;
constexpr int TP_NCONS = TP_FT * TP_GROUPS;   // 512
constexpr int TP_NPROD = 128;                 // 4 producer warps
constexpr int TP_THREADS = TP_NCONS + TP_NPROD;
constexpr int TP_MAX_PAIRS = 12288;
constexpr double TP_JOINT_MASS_MAX = 1e150;   // (1e150 + |D0|)^2 stays finite for every |D0| < 1e153
constexpr int TP_CHUNK_NODES = 2048;          // most (radial x angular) nodes of a unit: 32 KB per stage

struct TwoPointParams {
  int nq, nc, n_field, n_ext;
  double prefactor;
  RegParams reg;
  GridParams grid;
  FastMathConsts fmc;
  const double *xq, *wq, *xc, *wc, *Z, *coef, *m2, *pext;
  double *out, *dmin, *dout;
  // scratch
  double* chunkmin;  // [n_ftiles][n_ext][NCH][TP_NPROD/32], then [1]: min over radial nodes of D0q
  double* part;      // [max_slots][dout ? 2 : 1][n_ext][n_field]
  int QC, NCH, tile, grid_main, max_slots;
};


// ---- three-point ----
struct ThreePointParams {
  int nq, n1, n2, nphi, n_ext;
  double prefactor;
  RegParams reg;
  GridParams grid;
  FastMathConsts fmc;
  const double *xq, *wq, *x1, *w1, *x2, *w2, *wphi, *ZA, *L3, *coef, *ext;
  double *out, *dmin;
  const int* skip_flag;  // nullable; the general kernel returns at once if *skip_flag == 0 (product-grid path did the work)
};

template <int REGK>  // 0 Litim, 1 EXP_POLY(1), 2 EXP_POLY(order)
__device__ __forceinline__ double t3_reg_R(const RegParams& rp, const double* __restrict__ fxtab,
                                           const double* __restrict__ kc, const double s) {
  if constexpr (REGK == 0) {
    return s < rp.k2 ? rp.zk * (rp.k2 - s) : 0.0;
  } else if constexpr (REGK == 1) {
    return fx_exp_neg(fxtab, kc, s * rp.inv_k2);
  } else {
    const double x = s * rp.inv_k2;
    double expo = x, xi = x;
    for (int i = 2; i <= rp.order; ++i) {
      xi *= x;
      expo += xi / (double)i;
    }
    return fx_exp_neg(fxtab, kc, expo);
  }
}

// ---- 3-D vertex dressing table (dfrg_table3d): device-side look-up, used by the product-grid kernels below and by
// t3d_kernel further down ----
struct Tab3DParams {
  int n[3];
  int is_log[3];
  double lo[3], inv_h[3];
};
struct ThreePoint3DParams {
  ThreePointParams B;   // L3 unused
  Tab3DParams T;
  const double* v3;
};
constexpr int T3D_MAX_TABLE = 12288;  // doubles (96 KB of shared memory)

__device__ __forceinline__ double tab3d_eval(const double* __restrict__ v, const Tab3DParams& T, const FastMath& fm,
                                             const double x0, const double x1, const double x2) {
  const double x[3] = {x0, x1, x2};
  int i[3];
  double tau[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double c = T.is_log[a] ? 0.5 * fm_log(fm, x[a]) : x[a];
    double t = (c - T.lo[a]) * T.inv_h[a];
    t = clamp_lo(t, 0.0);  // NaN -> 0
    t = clamp_hi(t, (double)(T.n[a] - 1));
    int ii = (int)t;
    ii = min(ii, T.n[a] - 2);
    i[a] = ii;
    tau[a] = t - (double)ii;
  }
  const int s1 = T.n[2], s0 = T.n[1] * T.n[2];
  const double* b = v + (i[0] * s0 + i[1] * s1 + i[2]);
  // lerp along axis 2, then 1, then 0
  const double v00 = fma(tau[2], b[1] - b[0], b[0]);
  const double v01 = fma(tau[2], b[s1 + 1] - b[s1], b[s1]);
  const double v10 = fma(tau[2], b[s0 + 1] - b[s0], b[s0]);
  const double v11 = fma(tau[2], b[s0 + s1 + 1] - b[s0 + s1], b[s0 + s1]);
  const double w0 = fma(tau[1], v01 - v00, v00);
  const double w1 = fma(tau[1], v11 - v10, v10);
  return fma(tau[0], w1 - w0, w0);
}

// The same look-up with the eight corners fetched as four 16-byte loads.  The corners come in pairs adjacent along the last
// axis, (i2, i2 + 1); vB is a second copy of the table shifted by one element (vB[j] = v[j + 1]), so that a pair starting at
// an odd offset is read, aligned, from vB at offset - 1.  The look-up is bound by the shared-memory pipe (eight scattered
// 8-byte loads per lane, each several wavefronts because of bank conflicts); four scattered 16-byte loads need fewer
// wavefronts.  Same arithmetic as tab3d_eval, bit for bit.  v and vB are 16-byte aligned.
__device__ __forceinline__ double tab3d_eval_paired(const double* __restrict__ v, const double* __restrict__ vB,
                                                    const Tab3DParams& T, const FastMath& fm, const double x0,
                                                    const double x1, const double x2) {
  const double x[3] = {x0, x1, x2};
  int i[3];
  double tau[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double c = T.is_log[a] ? 0.5 * fm_log(fm, x[a]) : x[a];
    double t = (c - T.lo[a]) * T.inv_h[a];
    t = clamp_lo(t, 0.0);  // NaN -> 0
    t = clamp_hi(t, (double)(T.n[a] - 1));
    int ii = (int)t;
    ii = min(ii, T.n[a] - 2);
    i[a] = ii;
    tau[a] = t - (double)ii;
  }
  const int s1 = T.n[2], s0 = T.n[1] * T.n[2];
  const int o = i[0] * s0 + i[1] * s1 + i[2];
  auto pair_at = [&](const int off) {
    return (off & 1) ? *reinterpret_cast<const double2*>(vB + off - 1) : *reinterpret_cast<const double2*>(v + off);
  };
  const double2 b00 = pair_at(o), b01 = pair_at(o + s1), b10 = pair_at(o + s0), b11 = pair_at(o + s0 + s1);
  const double v00 = fma(tau[2], b00.y - b00.x, b00.x);
  const double v01 = fma(tau[2], b01.y - b01.x, b01.x);
  const double v10 = fma(tau[2], b10.y - b10.x, b10.x);
  const double v11 = fma(tau[2], b11.y - b11.x, b11.x);
  const double w0 = fma(tau[1], v01 - v00, v00);
  const double w1 = fma(tau[1], v11 - v10, v10);
  return fma(tau[0], w1 - w0, w0);
}

// ... and with the eight corners of the current cell kept in registers: consecutive nodes of a cos2 row move the vertex
// coordinates slowly, so most look-ups fall into the cell of their predecessor and need no load at all (the reload is
// predicated on the flat cell offset; the arithmetic is that of tab3d_eval, bit for bit).
struct Tab3Cell {
  int o;                        // flat offset of the cached cell's first corner; -1 = empty
  double2 b00, b01, b10, b11;   // the corner pairs along the last axis
};
__device__ __forceinline__ double tab3d_eval_cached(const double* __restrict__ v, const double* __restrict__ vB,
                                                    const Tab3DParams& T, const FastMath& fm, Tab3Cell& cell,
                                                    const double x0, const double x1, const double x2) {
  const double x[3] = {x0, x1, x2};
  int i[3];
  double tau[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double c = T.is_log[a] ? 0.5 * fm_log(fm, x[a]) : x[a];
    double t = (c - T.lo[a]) * T.inv_h[a];
    t = clamp_lo(t, 0.0);  // NaN -> 0
    t = clamp_hi(t, (double)(T.n[a] - 1));
    int ii = (int)t;
    ii = min(ii, T.n[a] - 2);
    i[a] = ii;
    tau[a] = t - (double)ii;
  }
  const int s1 = T.n[2], s0 = T.n[1] * T.n[2];
  const int o = i[0] * s0 + i[1] * s1 + i[2];
  if (o != cell.o) {
    auto pair_at = [&](const int off) {
      return (off & 1) ? *reinterpret_cast<const double2*>(vB + off - 1) : *reinterpret_cast<const double2*>(v + off);
    };
    cell.b00 = pair_at(o); cell.b01 = pair_at(o + s1); cell.b10 = pair_at(o + s0); cell.b11 = pair_at(o + s0 + s1);
    cell.o = o;
  }
  const double v00 = fma(tau[2], cell.b00.y - cell.b00.x, cell.b00.x);
  const double v01 = fma(tau[2], cell.b01.y - cell.b01.x, cell.b01.x);
  const double v10 = fma(tau[2], cell.b10.y - cell.b10.x, cell.b10.x);
  const double v11 = fma(tau[2], cell.b11.y - cell.b11.x, cell.b11.x);
  const double w0 = fma(tau[1], v01 - v00, v00);
  const double w1 = fma(tau[1], v11 - v10, v10);
  return fma(tau[0], w1 - w0, w0);
}
__device__ __forceinline__ double tab3d_vertex_cached(const double* __restrict__ v, const double* __restrict__ vB,
                                                      const Tab3DParams& T, const FastMath& fm, Tab3Cell& cell,
                                                      const double k1, const double k2, const double k3) {
  const double six = k1 + k2 + k3;
  const double r = six > 0.0 ? fast_rcp(six) : 0.0;
  return tab3d_eval_cached(v, vB, T, fm, cell, six * (1.0 / 6.0), 1.7320508075688772 * (k2 - k1) * r, (k1 + k2 - 2.0 * k3) * r);
}

// lambda3 at the vertex with squared leg momenta (k1, k2, k3):  S0^2 = (k1+k2+k3)/6, a = sqrt3 (k2-k1)/(6 S0^2),
// s = (k1+k2-2 k3)/(6 S0^2);  S0 = 0: a = s = 0.
__device__ __forceinline__ double tab3d_vertex(const double* __restrict__ v, const Tab3DParams& T, const FastMath& fm,
                                               const double k1, const double k2, const double k3) {
  const double six = k1 + k2 + k3;
  const double r = six > 0.0 ? fast_rcp(six) : 0.0;
  return tab3d_eval(v, T, fm, six * (1.0 / 6.0), 1.7320508075688772 * (k2 - k1) * r, (k1 + k2 - 2.0 * k3) * r);
}

__device__ __forceinline__ double tab3d_vertex_paired(const double* __restrict__ v, const double* __restrict__ vB,
                                                      const Tab3DParams& T, const FastMath& fm, const double k1,
                                                      const double k2, const double k3) {
  const double six = k1 + k2 + k3;
  const double r = six > 0.0 ? fast_rcp(six) : 0.0;
  return tab3d_eval_paired(v, vB, T, fm, six * (1.0 / 6.0), 1.7320508075688772 * (k2 - k1) * r, (k1 + k2 - 2.0 * k3) * r);
}

// ---- three-point on a product grid ----
struct ThreeGridParams {
  ThreePointParams B;
  int G, S;        // n_ext = G S
  int KP, NCH;     // pairs per chunk, chunks per r
  int NODES;       // shared nodes per unit buffer of the main kernel
  int grid_main, max_slots;
  LogGrid2Consts lgc;   // series coefficients of lg2_coord (constant-bank operands of the hot loop)
  double m2k23;    // -2 k^2 / 3
  double* tabA;    // [npairs][G][8]: s_a/3 (TAB3D: s_a), the five quartic coefficients times w0, (unused), D_a
  double* tabR;    // [S][4]
  double* qmin;    // [1]   min over radial nodes of D(q^2)
  int* flag;       // [1]   != 0: the layout promise does not hold
  double* part;    // [max_slots][n_ext]
  double* partB;   // [max_slots][S]  min over the slot's nodes of D_b
  Tab3DParams T3;  // TAB3D instantiations: lambda3(S0^2, a, s) instead of the 1-D table
  const double* v3;
  int ntab3;
  int paired3;     // TAB3D main kernel: a second, shifted copy of the table sits behind the first (tab3d_eval_paired)
};

constexpr int T3G_THREADS = 256;
constexpr int T3G_NODES = 512;  // shared nodes per unit buffer
constexpr int T3G_MAXT = 512;   // threads of the main kernel (126 registers each)

// ---- four-point ----
struct FourPointParams {
  int nq, n1, n2, nphi, n_ext;
  double prefactor;
  RegParams reg;
  GridParams grid;
  FastMathConsts fmc;
  const double *xq, *wq, *x1, *w1, *x2, *w2, *xphi, *wphi, *ZA, *Zc, *L3, *coef, *ext;
  double *out, *dmin;
  int KP, NCH, grid_main, max_slots;
  double* part;    // [max_slots][n_ext]
  double* partD;   // [max_slots][n_ext]  min over the slot's nodes of D/1
};
constexpr int FP4_THREADS = 512;

inline void fill_common(const dfrg_regulator& r, const dfrg_table& t, RegParams* rp, GridParams* gp) {
  *rp = reg_params(r.kind, r.order, r.k, r.zk, r.eta);
  gp->lo = t.lnq_lo; gp->inv_h = (double)(t.n_q - 1) / (t.lnq_hi - t.lnq_lo); gp->n = t.n_q; gp->interp = t.interp;
}
inline int regulator_variant(const dfrg_regulator& r) {   // template argument REGK of the three- and four-point kernels
  return r.kind == DFRG_REG_LITIM ? 0 : (r.order == 1 ? 1 : 2);
}

// ---- launchers (validated arguments in, kernels enqueued on `stream`; DFRG_OK / DFRG_EUNSUPPORTED / DFRG_ECUDA / DFRG_ENOMEM;
//      nothing is enqueued unless DFRG_OK is certain up to the launch itself) ----
int twopoint_launch(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext, const double* ext, double* out,
                    double* dmin, int sm_count, cudaStream_t stream);                                   // loop4d_twopoint.cu
int fourpoint_launch(const dfrg_loop4d_desc* D, int n_ext, const double* ext, double* out, double* dmin, int sm_count,
                     cudaStream_t stream);                                                              // loop4d_fourpoint.cu
// general list of external configurations (loop4d_threepoint.cu); P.skip_flag as left by t3g_launch
size_t threepoint_general_smem(int nq, int n1, int n2, int nt);
int threepoint_general_launch(const ThreePointParams& P, int regk, int sm_count, cudaStream_t stream);
size_t threepoint3d_general_smem(int nq, int n1, int n2, int nt, int ntab3);
int threepoint3d_general_launch(const ThreePoint3DParams& Q3, int regk, int sm_count, cudaStream_t stream);
// product grid (loop4d_grid.cu): enqueues the product-grid kernels if the caller promised a product grid (G >= 2) and the
// shapes allow it; then P.skip_flag points at the device flag the general kernel must consult and *scratch_out at the
// scratch block to free after the general kernel.  T3 != nullptr: 3-D vertex table.
int t3g_launch(ThreePointParams& P, int G, int regk, const Tab3DParams* T3, const double* v3, int ntab3, int sm_count,
               cudaStream_t stream, void** scratch_out);

}  // namespace dfrg
