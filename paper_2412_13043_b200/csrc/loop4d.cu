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
#include "dfrg_device.cuh"
#include "dfrg_internal.h"

namespace dfrg {

// =====================================================================================================
// two-point
// =====================================================================================================
// One persistent, warp-specialised kernel (one CTA per SM) and a small fix-up kernel.
//  Work unit = (field tile, p, chunk of QC radial nodes); the units are dealt to the CTAs in contiguous ranges, so a
//  consumer keeps its accumulators while the CTA stays inside one (field tile, p).
//  Producer warps (S3, field independent), one unit ahead through a two-stage mbarrier ring (full[b] / empty[b]):
//        chunk[i][j] = (D0, W'),  D0 = Z(s_ij) s_ij + R(s_ij),  W' = wc_j sqrt(1-c_j^2) (coef0 + coef1 q_i p c_j/k^2)
//    and the chunk's minimum of D0 (for dmin).  outer[i] = (Z(q_i^2) q_i^2 + R(q_i^2), wq_i q_i^3 Rdot(q_i^2)) is built
//    once per CTA.  S2: nodes, weights and the Z table arrive by TMA bulk copy.
//  Consumers (S4 + S5): TP_GROUPS groups x TP_FT threads; a thread owns MF field points, a group every TP_GROUPS-th
//    radial node of the chunk.  Per node:  d_f = D0 + m2_f;  MF = 2: one seed + Newton reciprocal of d_0 d_1 serves both
//    field points (4.5 FP64 instructions per evaluation);  A_f += W'/d_f  (with mass derivatives also B_f += W'/d_f^2).
//    Per radial node:  acc_f += Wq G(q)^2 A_f.  Every table read is a shared-memory broadcast.
//    When (field tile, p) or the CTA's range ends, the groups are combined in fixed order and the partial sum goes to
//    part[slot]; slot = rank of the CTA among the owners of that (field tile, p).
//  tp_fixup_kernel (S5 + S6): out = prefactor sum_slots part in fixed order; dmin from the chunk minima
//    (fl(D0 + m2) is monotone in D0, so the minimum over nodes is (min D0) + m2).
constexpr int TP_FT = 128;      // field threads per consumer group
constexpr int TP_GROUPS = 4;
constexpr int TP_NCONS = TP_FT * TP_GROUPS;   // 512
constexpr int TP_NPROD = 128;                 // 4 producer warps
constexpr int TP_THREADS = TP_NCONS + TP_NPROD;
constexpr int TP_MAX_PAIRS = 12288;
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

// One batch of NB angular nodes for the MF field points of a thread.
template <int MF, bool WANT_D, int NB>
__device__ __forceinline__ void tp_batch(const double2* __restrict__ row, const double (&m2)[MF], double (&A)[MF],
                                         double (&B)[MF]) {
  double2 t[NB];
#pragma unroll
  for (int b = 0; b < NB; ++b) t[b] = row[b];
  if constexpr (MF == 2) {
    double d0[NB], d1[NB], R[NB], Rw[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) { d0[b] = t[b].x + m2[0]; d1[b] = t[b].x + m2[1]; }
#pragma unroll
    for (int b = 0; b < NB; ++b) R[b] = fast_rcp(d0[b] * d1[b]);
#pragma unroll
    for (int b = 0; b < NB; ++b) Rw[b] = R[b] * t[b].y;
#pragma unroll
    for (int b = 0; b < NB; ++b) { A[0] = fma(Rw[b], d1[b], A[0]); A[1] = fma(Rw[b], d0[b], A[1]); }
    if constexpr (WANT_D) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        B[0] = fma(Rw[b] * d1[b], R[b] * d1[b], B[0]);
        B[1] = fma(Rw[b] * d0[b], R[b] * d0[b], B[1]);
      }
    }
  } else {
#pragma unroll
    for (int k = 0; k < MF; ++k) {
      double r[NB];
#pragma unroll
      for (int b = 0; b < NB; ++b) r[b] = fast_rcp(t[b].x + m2[k]);
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        A[k] = fma(t[b].y, r[b], A[k]);
        if constexpr (WANT_D) B[k] = fma(t[b].y * r[b], r[b], B[k]);
      }
    }
  }
}

template <int MF, bool WANT_D>
__global__ void __launch_bounds__(TP_THREADS, 1) tp_main_kernel(const TwoPointParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar, full[2], empty[2];
  __shared__ double red[32];
  const int nq = P.nq, nc = P.nc, nt = P.grid.n, QC = P.QC, NCH = P.NCH;
  const int chunk_nodes = QC * nc;
  constexpr int ND = WANT_D ? 2 : 1;
  double2* buf = reinterpret_cast<double2*>(smem_raw);                // [2][chunk_nodes]
  double2* souter = buf + 2 * (size_t)chunk_nodes;                    // [nq]
  double4* cZ = reinterpret_cast<double4*>(souter + nq);              // [nt] per-cell cubics of Z
  double* sxq = reinterpret_cast<double*>(cZ + nt);
  double* swq = sxq + ((nq + 1) & ~1);
  double* sxc = swq + ((nq + 1) & ~1);
  double* swc = sxc + ((nc + 1) & ~1);                                // wc_j sqrt(1 - c_j^2) after the set-up
  double* sZ = swc + ((nc + 1) & ~1);
  double* fmmem = sZ + ((nt + 1) & ~1);
  double* comb = fmmem + FM_DOUBLES;                                  // [2][ND][TP_GROUPS][TP_FT * MF]

  const int tid = threadIdx.x;
  const int tile = TP_FT * MF;
  const int n_ftiles = (P.n_field + tile - 1) / tile;
  const long long upp = (long long)P.n_ext * NCH;                     // units per field tile
  const long long U = (long long)n_ftiles * upp;
  const long long u0 = (long long)blockIdx.x * U / gridDim.x, u1 = (long long)(blockIdx.x + 1) * U / gridDim.x;

  if (tid == 0) {
    mbar_init(&bar, 1);
    mbar_init(&full[0], TP_NPROD / 32);
    mbar_init(&full[1], TP_NPROD / 32);
    mbar_init(&empty[0], TP_NCONS / 32);
    mbar_init(&empty[1], TP_NCONS / 32);
    mbar_fence_init();
  }
  __syncthreads();
  StageList L;
  L.add(sxq, P.xq, nq); L.add(swq, P.wq, nq);
  L.add(sxc, P.xc, nc); L.add(swc, P.wc, nc);
  L.add(sZ, P.Z, nt);
  const FastMath fm = fm_build(fmmem, P.fmc);
  stage_to_smem(L, &bar, 0);
  cells_build(cZ, sZ, P.grid);
  __syncthreads();
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  {
    double dq = inf;
    for (int i = tid; i < nq; i += TP_THREADS) {
      const double q = sxq[i], s = q * q;
      double R, Rd;
      regulator(P.reg, fm, s, R, Rd);
      const double D0 = table_lookup(cZ, P.grid, fm, s) * s + R;
      souter[i] = make_double2(D0, swq[i] * q * q * q * Rd);
      dq = fmin(dq, D0);
    }
    for (int j = tid; j < nc; j += TP_THREADS) {
      const double c = sxc[j];
      swc[j] *= sqrt((1.0 - c) * (1.0 + c));
    }
    dq = block_min(dq, red);  // also publishes souter and swc
    if (blockIdx.x == 0 && tid == 0) P.chunkmin[(size_t)n_ftiles * P.n_ext * NCH * (TP_NPROD / 32)] = dq;
  }

  if (tid >= TP_NCONS) {
    // =========================== producers ===========================
    const int ptid = tid - TP_NCONS, lane = ptid & 31, pw = ptid >> 5;
    const double coef0 = P.coef[0], coef1 = P.coef[1];
    uint32_t g = 0;
    for (long long u = u0; u < u1; ++u, ++g) {
      const int b = g & 1;
      const long long rem = u % upp;
      const int e = (int)(rem / NCH), ch = (int)(rem - (long long)e * NCH);
      const int i0 = ch * QC;
      const int ni = min(QC, nq - i0);
      const double p = P.pext[e];
      mbar_wait(&empty[b], ((g >> 1) & 1) ^ 1);   // consumers drained this stage (passes at once for g < 2)
      double2* dst = buf + (size_t)b * chunk_nodes;
      double dmin0 = inf;
      for (int t = ptid; t < ni * nc; t += TP_NPROD) {
        const int il = t / nc, j = t - il * nc;
        const double q = sxq[i0 + il], c = sxc[j];
        double s = q * q + p * p + 2.0 * q * p * c;
        s = clamp_lo(s, 0.0);
        double R, Rd;
        regulator(P.reg, fm, s, R, Rd);
        const double D0 = table_lookup(cZ, P.grid, fm, s) * s + R;
        const double poly = coef0 + coef1 * (q * p * c * P.reg.inv_k2);
        dst[t] = make_double2(D0, swc[j] * poly);
        dmin0 = fmin(dmin0, D0);
      }
      dmin0 = warp_min(dmin0);
      if (lane == 0) {
        P.chunkmin[(size_t)(u * (TP_NPROD / 32)) + pw] = dmin0;
        mbar_arrive(&full[b]);  // release: the chunk is visible to whoever acquires full[b]
      }
    }
    return;
  }

  // =============================== consumers ===============================
  const int grp = tid / TP_FT, tf = tid - grp * TP_FT;
  const bool warp_leader = (tid & 31) == 0;
  double m2[MF], acc[MF], dacc[MF];
  int cur_ft = -1, seg_parity = 0;
  uint32_t g = 0;
  for (long long u = u0; u < u1; ++u, ++g) {
    const int ft = (int)(u / upp);
    const long long rem = u - (long long)ft * upp;
    const int e = (int)(rem / NCH), ch = (int)(rem - (long long)e * NCH);
    const int f0 = ft * tile + tf;
    const int b = g & 1;
    if (ft != cur_ft) {
      cur_ft = ft;
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        const int f = f0 + k * TP_FT;
        m2[k] = (f < P.n_field) ? P.m2[f] : 1.0;
      }
    }
    if (u == u0 || ch == 0) {
#pragma unroll
      for (int k = 0; k < MF; ++k) { acc[k] = 0.0; dacc[k] = 0.0; }
    }
    mbar_wait(&full[b], (g >> 1) & 1);
    const double2* chunk = buf + (size_t)b * chunk_nodes;
    const int i0 = ch * QC;
    const int ni = min(QC, nq - i0);
    for (int il = grp; il < ni; il += TP_GROUPS) {
      const double2* row = chunk + il * nc;
      double A[MF], B[MF];
#pragma unroll
      for (int k = 0; k < MF; ++k) { A[k] = 0.0; B[k] = 0.0; }
      int j = 0;
      for (; j + 4 <= nc; j += 4) tp_batch<MF, WANT_D, 4>(row + j, m2, A, B);
      for (; j < nc; ++j) tp_batch<MF, WANT_D, 1>(row + j, m2, A, B);
      const double2 o = souter[i0 + il];
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        const double gq = fast_rcp(o.x + m2[k]);
        const double wg2 = o.y * (gq * gq);
        acc[k] = fma(wg2, A[k], acc[k]);
        if constexpr (WANT_D) dacc[k] = fma(wg2, fma(2.0 * gq, A[k], B[k]), dacc[k]);
      }
    }
    __syncwarp();
    if (warp_leader) mbar_arrive(&empty[b]);
    if (ch == NCH - 1 || u == u1 - 1) {
      // combine the groups in fixed order; partial sum of this CTA for (field tile, p)
      double* cb = comb + (size_t)seg_parity * ND * TP_GROUPS * tile;
      seg_parity ^= 1;
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        cb[grp * tile + k * TP_FT + tf] = acc[k];
        if constexpr (WANT_D) cb[(TP_GROUPS + grp) * tile + k * TP_FT + tf] = dacc[k];
      }
      named_bar_sync(1, TP_NCONS);
      if (grp == 0) {
        const long long ufirst = (long long)ft * upp + (long long)e * NCH;
        const int c_first = (int)(((ufirst + 1) * gridDim.x - 1) / U);
        const int slot = (int)blockIdx.x - c_first;
        const size_t plane = (size_t)P.n_ext * P.n_field;
#pragma unroll
        for (int k = 0; k < MF; ++k) {
          const int f = f0 + k * TP_FT;
          if (f < P.n_field) {
            double r = cb[k * TP_FT + tf];
#pragma unroll
            for (int gg = 1; gg < TP_GROUPS; ++gg) r += cb[gg * tile + k * TP_FT + tf];
            P.part[((size_t)slot * ND) * plane + (size_t)e * P.n_field + f] = r;
            if constexpr (WANT_D) {
              double dr = cb[TP_GROUPS * tile + k * TP_FT + tf];
#pragma unroll
              for (int gg = 1; gg < TP_GROUPS; ++gg) dr += cb[(TP_GROUPS + gg) * tile + k * TP_FT + tf];
              P.part[((size_t)slot * 2 + 1) * plane + (size_t)e * P.n_field + f] = dr;
            }
          }
        }
      }
    }
  }
}
static size_t tp_main_smem(int nq, int nc, int nt, int chunk_nodes, int mf, bool want_d) {
  return 16 * (2 * (size_t)chunk_nodes + nq) + 32 * (size_t)nt +
         8 * (size_t)(2 * ((nq + 1) & ~1) + 2 * ((nc + 1) & ~1) + ((nt + 1) & ~1) + FM_DOUBLES +
                      2 * (want_d ? 2 : 1) * TP_GROUPS * TP_FT * mf);
}

__global__ void __launch_bounds__(256) tp_fixup_kernel(const TwoPointParams P) {
  const long long idx = (long long)blockIdx.x * 256 + threadIdx.x;
  const long long n_out = (long long)P.n_ext * P.n_field;
  if (idx >= n_out) return;
  const int f = (int)(idx % P.n_field), e = (int)(idx / P.n_field);
  const int n_ftiles = (P.n_field + P.tile - 1) / P.tile;
  const long long upp = (long long)P.n_ext * P.NCH, U = (long long)n_ftiles * upp;
  const long long ufirst = (long long)(f / P.tile) * upp + (long long)e * P.NCH, ulast = ufirst + P.NCH - 1;
  const int c_first = (int)(((ufirst + 1) * P.grid_main - 1) / U), c_last = (int)(((ulast + 1) * P.grid_main - 1) / U);
  const int nd = P.dout ? 2 : 1;
  const size_t plane = (size_t)n_out;
  double r = P.part[idx];
  for (int s = 1; s <= c_last - c_first; ++s) r += P.part[(size_t)s * nd * plane + idx];
  P.out[idx] = P.prefactor * r;
  if (P.dout) {
    double dr = P.part[plane + idx];
    for (int s = 1; s <= c_last - c_first; ++s) dr += P.part[((size_t)s * 2 + 1) * plane + idx];
    P.dout[idx] = -P.prefactor * dr;
  }
  if (P.dmin) {
    constexpr int NW = TP_NPROD / 32;
    double dm = P.chunkmin[(size_t)U * NW];
    for (long long t = ufirst * NW; t < (ulast + 1) * NW; ++t) dm = fmin(dm, P.chunkmin[t]);
    P.dmin[idx] = (dm + P.m2[f]) * P.reg.inv_k2;
  }
}

// =====================================================================================================
// three-point
// =====================================================================================================

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

// ---- three-point, general kernel (any list of external configurations) ----
// Persistent CTAs, thread = (q, c1) pairs, c2 loop inside.  The three table look-ups of a node go through lg_coord /
// lg_cell_eval (no separate logarithm, no FP64 clamps), e^-x through the replicated 64-entry table, every affine
// step is a single FMA, and the regulator kind is a template parameter.
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

// lambda3 at the vertex with squared leg momenta (k1, k2, k3):  S0^2 = (k1+k2+k3)/6, a = sqrt3 (k2-k1)/(6 S0^2),
// s = (k1+k2-2 k3)/(6 S0^2);  S0 = 0: a = s = 0.
__device__ __forceinline__ double tab3d_vertex(const double* __restrict__ v, const Tab3DParams& T, const FastMath& fm,
                                               const double k1, const double k2, const double k3) {
  const double six = k1 + k2 + k3;
  const double r = six > 0.0 ? fast_rcp(six) : 0.0;
  return tab3d_eval(v, T, fm, six * (1.0 / 6.0), 1.7320508075688772 * (k2 - k1) * r, (k1 + k2 - 2.0 * k3) * r);
}

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
//  (1) t3g_prepass_kernel: promise check; tabR[r] = (|p2|, cos alpha, sin alpha); tabA[pair][0..7][a] for every (q, c1) pair:
//        w0 = wq q^3 Rdot(q^2) G_A(q^2) w1 sqrt(1-c1^2) G_A(s_a) lambda3(.),  s_a/3,  the five quartic coefficients,  D_a.
//  (2) t3g_main_kernel: persistent, one CTA per SM.  Work unit = (r, chunk of KP pairs); the units are dealt to the
//      CTAs in contiguous ranges.  Phase 1 (all threads, one unit ahead, double buffered): the shared node data
//      (w2 G_A(s_b) lambda3(.), s_b/3, z) of the unit's KP x n2 nodes into shared memory.  Phase 2: thread = (a, pair
//      slot); per node one look-up, one Horner, two multiply-adds; the shared node data are warp-uniform broadcasts.
//      A thread keeps the running sum of its a while the CTA stays inside one r; the partial sums of an output are
//      written per CTA ("slot") and added in fixed order by
//  (3) t3g_fixup_kernel (deterministic: the ownership of units is a pure function of the grid size).
struct ThreeGridParams {
  ThreePointParams B;
  int G, S;        // n_ext = G S
  int KP, NCH;     // pairs per chunk, chunks per r
  int grid_main, max_slots;
  double* tabA;    // [npairs][8][G]
  double* tabR;    // [S][4]
  double* qmin;    // [1]   min over radial nodes of D(q^2)
  int* flag;       // [1]   != 0: the layout promise does not hold
  double* part;    // [max_slots][n_ext]
  double* partB;   // [max_slots][S]  min over the slot's nodes of D_b
  Tab3DParams T3;  // TAB3D instantiations: lambda3(S0^2, a, s) instead of the 1-D table
  const double* v3;
  int ntab3;
};

constexpr int T3G_THREADS = 256;
constexpr int T3G_NODES = 512;  // shared nodes per unit buffer
constexpr int T3G_MAXT = 512;   // threads of the main kernel (126 registers each)

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
    double* ta = Q.tabA + ((size_t)pair * 8) * G + a;
    ta[0] = wpair * (Ga * lam1);
    ta[(size_t)G] = TAB3D ? s_a : s_a * third;
#pragma unroll
    for (int c = 0; c < 5; ++c) ta[(size_t)(2 + c) * G] = gam[c];
    ta[(size_t)7 * G] = Da;
  }
}

template <int REGK, int NT, int UNR, bool TAB3D>
__global__ void __launch_bounds__(NT, 1) t3g_main_kernel(const ThreeGridParams Q) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ double red32[32];
  if (*Q.flag != 0) return;  // the layout promise does not hold: the general kernel does the work
  const ThreePointParams& P = Q.B;
  const int nq = P.nq, n1 = P.n1, n2 = P.n2, nt = P.grid.n, G = Q.G, S = Q.S, KP = Q.KP, NCH = Q.NCH;
  const int npairs = nq * n1;
  const T3GShared sm = t3g_carve(smem_raw, nq, n1, n2, nt);
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
    stage_to_smem(L, &bar, 0);
  }
  const FastMath fm = fm_build(sm.fmmem, P.fmc);   // the S0 axis of the 3-D table (TAB3D)
  const double* fxtab = fx_build(sm.fxmem, P.reg.zk * P.reg.k2);
  const LogGrid lg = lg_build(sm.lgmem, P.grid.lo, P.grid.inv_h, nt);
  const double* kc = P.fmc.c;
  const double2* cZA = cells_build_guarded(sm.cZA_all, sm.sZA, nt, P.grid.interp);
  const double2* cL3 = TAB3D ? nullptr : cells_build_guarded(sm.cL3_all, sm.sL3, nt, P.grid.interp);
  for (int j = tid; j < n2; j += NT) sm.xw2[j] = make_double2(sm.sx2[j], sm.sw2[j]);
  __syncthreads();

  const double ik2 = P.reg.inv_k2, third = 1.0 / 3.0, m2k2 = -2.0 * P.reg.k2;
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  const long long U = (long long)S * NCH;
  const long long u0 = (long long)blockIdx.x * U / gridDim.x, u1 = (long long)(blockIdx.x + 1) * U / gridDim.x;
  const int nw = NT / G;                 // pair slots
  const bool active = tid < nw * G;
  const int a = tid % G, w = tid / G;
  const double p1 = P.ext[3 * ((long long)a * S)];

  double dmB_cur = inf, dmB_nxt = inf;
  // Phase 1: shared node data of unit u into buffer b
  auto phase1 = [&](long long u, int b, double& dmB) {
    const int r = (int)(u / NCH), ch = (int)(u - (long long)r * NCH);
    const int pair0 = ch * KP;
    const int npl = min(KP, npairs - pair0);
    const double p2 = Q.tabR[4 * r], ca_ = Q.tabR[4 * r + 1], sa_ = Q.tabR[4 * r + 2];
    double2* nA = sm.nodeA + b * T3G_NODES;
    double* nZ = sm.nodeZ + b * T3G_NODES;
    for (int n = tid; n < npl * n2; n += NT) {
      const int pl = n / n2, j2 = n - pl * n2;
      const int pair = pair0 + pl;
      const int i = pair / n1, j1 = pair - i * n1;
      const double q = sm.sxq[i], c1 = sm.sx1[j1];
      const double sq = q * q;
      const double sin1 = sqrt((1.0 - c1) * (1.0 + c1));
      const double zc = q * p2 * ca_ * c1 * ik2;
      const double zs = q * p2 * sa_ * sin1 * ik2;
      const double sb0 = sq + p2 * p2;
      const double2 xw = sm.xw2[j2];
      const double z = fma(zs, xw.x, zc);
      double s_b = fma(m2k2, z, sb0);
      s_b = clamp_lo(s_b, 0.0);
      const double Db = fma(lg_lookup(cZA, lg, kc, s_b), s_b, t3_reg_R<REGK>(P.reg, fxtab, kc, s_b));
      dmB = fmin(dmB, Db);
      const double lam2 = TAB3D ? tab3d_vertex(sm.stab3, Q.T3, fm, p2 * p2, sq, s_b)
                                : lg_lookup(cL3, lg, kc, fma(s_b, third, sb0 * third));
      nA[n] = make_double2(xw.y * (fast_rcp(Db) * lam2), TAB3D ? s_b : s_b * third);
      nZ[n] = z;
    }
  };

  double acc = 0.0;
  if (u0 < u1) phase1(u0, 0, dmB_cur);
  __syncthreads();
  for (long long u = u0; u < u1; ++u) {
    const int b = (int)((u - u0) & 1);
    const int r = (int)(u / NCH), ch = (int)(u - (long long)r * NCH);
    const bool last_of_r = (u + 1 == u1) || ((u + 1) / NCH != r);
    if (u + 1 < u1) phase1(u + 1, b ^ 1, last_of_r ? dmB_nxt : dmB_cur);
    // ---- phase 2 ----
    const int pair0 = ch * KP;
    const int npl = min(KP, npairs - pair0);
    if (active) {
      const double p2 = Q.tabR[4 * r], ca_ = Q.tabR[4 * r + 1];
      double scc = p1 * p1 + p2 * p2 + 2.0 * p1 * p2 * ca_;
      scc = scc > 0.0 ? scc : 0.0;
      const double scc3 = scc * third;
      const double2* nA = sm.nodeA + b * T3G_NODES;
      const double* nZ = sm.nodeZ + b * T3G_NODES;
      double cur[7], nxt[7];
      if (w < npl) {
        const double* ta = Q.tabA + ((size_t)(pair0 + w) * 8) * G + a;
#pragma unroll
        for (int c = 0; c < 7; ++c) cur[c] = ta[(size_t)c * G];
      }
      for (int pl = w; pl < npl; pl += nw) {
        if (pl + nw < npl) {
          const double* ta = Q.tabA + ((size_t)(pair0 + pl + nw) * 8) * G + a;
#pragma unroll
          for (int c = 0; c < 7; ++c) nxt[c] = ta[(size_t)c * G];
        }
        const double l30 = cur[1] + scc3;
        const double2* na = nA + pl * n2;
        const double* nz = nZ + pl * n2;
        double acc2 = 0.0;
#pragma unroll UNR
        for (int j2 = 0; j2 < n2; ++j2) {
          const double2 bs = na[j2];
          const double z = nz[j2];
          const double lam3 = TAB3D ? tab3d_vertex(sm.stab3, Q.T3, fm, scc, cur[1], bs.y)
                                    : lg_lookup(cL3, lg, kc, bs.y + l30);
          const double poly = fma(fma(fma(fma(cur[6], z, cur[5]), z, cur[4]), z, cur[3]), z, cur[2]);
          acc2 = fma(bs.x * poly, lam3, acc2);
        }
        acc = fma(cur[0], acc2, acc);
#pragma unroll
        for (int c = 0; c < 7; ++c) cur[c] = nxt[c];
      }
    }
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
  double t = Q.part[e];
  for (int s = 1; s <= c_last - c_first; ++s) t += Q.part[(size_t)s * P.n_ext + e];
  double sum_wphi = 0.0;
  for (int jp = 0; jp < P.nphi; ++jp) sum_wphi += P.wphi[jp];
  P.out[e] = P.prefactor * sum_wphi * t;
  if (P.dmin) {
    double dm = *Q.qmin;
    for (int s = 0; s <= c_last - c_first; ++s) dm = fmin(dm, Q.partB[(size_t)s * S + r]);
    const int npairs = P.nq * P.n1;
    for (int pair = 0; pair < npairs; ++pair) dm = fmin(dm, Q.tabA[((size_t)pair * 8 + 7) * G + a]);
    P.dmin[e] = dm * P.reg.inv_k2;
  }
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
  double t = P.part[e];
  for (int s = 1; s <= c_last - c_first; ++s) t += P.part[(size_t)s * P.n_ext + e];
  P.out[e] = P.prefactor * t;
  if (P.dmin) {
    double dm = P.partD[e];
    for (int s = 1; s <= c_last - c_first; ++s) dm = fmin(dm, P.partD[(size_t)s * P.n_ext + e]);
    P.dmin[e] = dm * P.reg.inv_k2;
  }
}

// =====================================================================================================
// host side
// =====================================================================================================
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

static void fill_common(const dfrg_regulator& r, const dfrg_table& t, RegParams* rp, GridParams* gp) {
  *rp = reg_params(r.kind, r.order, r.k, r.zk, r.eta);
  gp->lo = t.lnq_lo; gp->inv_h = (double)(t.n_q - 1) / (t.lnq_hi - t.lnq_lo); gp->n = t.n_q; gp->interp = t.interp;
}

// Enqueues the product-grid kernels if the caller promised a product grid (G >= 2) and the shapes allow it; then
// P.skip_flag points at the device flag the general kernel must consult.  T3 != nullptr: 3-D vertex table.
static int t3g_launch(ThreePointParams& P, int G, int regk, const Tab3DParams* T3, const double* v3, int ntab3,
                      int sm_count, cudaStream_t stream, void** scratch_out) {
  const int n_ext = P.n_ext;
  if (!(G >= 2 && G <= 256 && n_ext % G == 0 && P.n2 <= T3G_NODES)) return DFRG_OK;
  const size_t smem_g = t3g_smem(P.nq, P.n1, P.n2, P.grid.n, T3 ? ntab3 : 0);
  if (smem_g > 227 * 1024) return DFRG_OK;   // (large 3-D tables: the general kernel)
  ThreeGridParams Q;
  Q.B = P;
  Q.G = G; Q.S = n_ext / G;
  Q.v3 = v3; Q.ntab3 = ntab3;
  if (T3) Q.T3 = *T3;
  const int npairs = P.nq * P.n1;
  Q.KP = T3G_NODES / P.n2 < npairs ? T3G_NODES / P.n2 : npairs;
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
#define DFRG_T3G_PICK(K)                                                                                  \
  if (regk == K) {                                                                                        \
    kpre = T3 ? t3g_prepass_kernel<K, true> : t3g_prepass_kernel<K, false>;                               \
    kmain = T3 ? t3g_main_kernel<K, T3G_MAXT, 8, true> : t3g_main_kernel<K, T3G_MAXT, 8, false>;          \
  }
  DFRG_T3G_PICK(0) DFRG_T3G_PICK(1) DFRG_T3G_PICK(2)
#undef DFRG_T3G_PICK
  if (e == cudaSuccess) e = cudaFuncSetAttribute(kpre, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_g);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(kmain, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_g);
  if (e != cudaSuccess) { scratch_free(scratch, stream); *scratch_out = nullptr; return check_cuda(e); }
  kpre<<<sm_count, T3G_THREADS, smem_g, stream>>>(Q);
  kmain<<<Q.grid_main, T3G_MAXT, smem_g, stream>>>(Q);
  t3g_fixup_kernel<<<(n_ext + 255) / 256, 256, 0, stream>>>(Q);
  rc = check_cuda(cudaGetLastError());
  if (rc != DFRG_OK) { scratch_free(scratch, stream); *scratch_out = nullptr; return rc; }
  P.skip_flag = Q.flag;
  return DFRG_OK;
}

static int loop4d_launch(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext, const double* ext,
                         double* out, double* dmin, int sm_count, cudaStream_t stream) {
  if (D->family == DFRG_LOOP_TWOPOINT) {
    TwoPointParams P;
    P.nq = D->q.n; P.nc = D->cos1.n; P.n_field = n_field; P.n_ext = n_ext;
    P.prefactor = D->prefactor;
    fill_common(D->reg, D->tab[0], &P.reg, &P.grid);
    P.fmc = fm_consts();
    P.xq = D->q.x; P.wq = D->q.w; P.xc = D->cos1.x; P.wc = D->cos1.w; P.Z = D->tab[0].v;
    P.coef = D->coef; P.m2 = m2; P.pext = ext; P.out = out; P.dmin = dmin; P.dout = D->dout_dm2;
    // ---- plan: chunk of QC radial nodes per unit, contiguous unit ranges per CTA ----
    const int mf = n_field > TP_FT ? 2 : 1;
    P.tile = TP_FT * mf;
    int qc = TP_CHUNK_NODES / P.nc;
    qc = qc > 8 ? 8 : qc;
    qc = qc > P.nq ? P.nq : qc;
    P.QC = qc;
    P.NCH = (P.nq + qc - 1) / qc;
    const int n_ftiles = (n_field + P.tile - 1) / P.tile;
    const long long upp = (long long)n_ext * P.NCH, U = (long long)n_ftiles * upp;
    P.grid_main = (int)(U < sm_count ? U : sm_count);
    P.max_slots = 1;
    for (long long seg = 0; seg < (long long)n_ftiles * n_ext; ++seg) {
      const long long ufirst = seg * P.NCH, ulast = ufirst + P.NCH - 1;
      const int c0 = (int)(((ufirst + 1) * P.grid_main - 1) / U), c1 = (int)(((ulast + 1) * P.grid_main - 1) / U);
      if (c1 - c0 + 1 > P.max_slots) P.max_slots = c1 - c0 + 1;
    }
    const bool want_d = D->dout_dm2 != nullptr;
    const size_t n_chunkmin = ((size_t)U * (TP_NPROD / 32) + 2) & ~(size_t)1,
                 n_part = (size_t)P.max_slots * (want_d ? 2 : 1) * n_ext * n_field;
    void* scratch = nullptr;
    int rc = scratch_alloc(&scratch, (n_chunkmin + n_part) * sizeof(double), stream);
    if (rc != DFRG_OK) return rc;
    P.chunkmin = (double*)scratch;
    P.part = P.chunkmin + n_chunkmin;
    const size_t smem_main = tp_main_smem(P.nq, P.nc, P.grid.n, P.QC * P.nc, mf, want_d);
    void (*kmain)(const TwoPointParams) =
        mf == 2 ? (want_d ? tp_main_kernel<2, true> : tp_main_kernel<2, false>)
                : (want_d ? tp_main_kernel<1, true> : tp_main_kernel<1, false>);
    cudaError_t e = cudaFuncSetAttribute(kmain, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_main);
    if (e != cudaSuccess) { scratch_free(scratch, stream); return check_cuda(e); }
    kmain<<<P.grid_main, TP_THREADS, smem_main, stream>>>(P);
    const long long n_out = (long long)n_ext * n_field;
    tp_fixup_kernel<<<(unsigned)((n_out + 255) / 256), 256, 0, stream>>>(P);
    rc = check_cuda(cudaGetLastError());
    scratch_free(scratch, stream);
    return rc;
  }
  if (D->family == DFRG_LOOP_FOURPOINT) {
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
    if (smem4 > 227 * 1024) { scratch_free(scratch4, stream); return DFRG_EUNSUPPORTED; }
    cudaError_t e4 = cudaFuncSetAttribute(k4, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem4);
    if (e4 != cudaSuccess) { scratch_free(scratch4, stream); return check_cuda(e4); }
    k4<<<P.grid_main, FP4_THREADS, smem4, stream>>>(P);
    fp4_fixup_kernel<<<(n_ext + 255) / 256, 256, 0, stream>>>(P);
    rc = check_cuda(cudaGetLastError());
    scratch_free(scratch4, stream);
    return rc;
  }
  ThreePointParams P;
  P.nq = D->q.n; P.n1 = D->cos1.n; P.n2 = D->cos2.n; P.nphi = D->phi.n; P.n_ext = n_ext;
  P.prefactor = D->prefactor;
  fill_common(D->reg, D->tab[0], &P.reg, &P.grid);
  P.fmc = fm_consts();
  P.xq = D->q.x; P.wq = D->q.w; P.x1 = D->cos1.x; P.w1 = D->cos1.w; P.x2 = D->cos2.x; P.w2 = D->cos2.w; P.wphi = D->phi.w;
  P.ZA = D->tab[0].v; P.L3 = D->tab[2].v; P.coef = D->coef; P.ext = ext; P.out = out; P.dmin = dmin;
  P.skip_flag = nullptr;
  if (D->family == DFRG_LOOP_THREEPOINT_TAB3D) {
    ThreePoint3DParams Q3;
    Q3.B = P;
    Q3.v3 = D->tab3d.v;
    int ntab3 = 1;
    for (int a = 0; a < 3; ++a) {
      Q3.T.n[a] = D->tab3d.n[a]; Q3.T.is_log[a] = D->tab3d.is_log[a]; Q3.T.lo[a] = D->tab3d.lo[a];
      Q3.T.inv_h[a] = (double)(D->tab3d.n[a] - 1) / (D->tab3d.hi[a] - D->tab3d.lo[a]);
      ntab3 *= D->tab3d.n[a];
    }
    const size_t smem3 = t3d_smem(P.nq, P.n1, P.n2, P.grid.n, ntab3);
    if (smem3 > 227 * 1024) return DFRG_EUNSUPPORTED;
    const int regk3 = D->reg.kind == DFRG_REG_LITIM ? 0 : (D->reg.order == 1 ? 1 : 2);
    void* scratch3 = nullptr;
    {  // product grid promised (ext_outer): share the |p1|-only and (|p2|, alpha)-only vertices as the 1-D family does
      const int rcg = t3g_launch(Q3.B, D->ext_outer, regk3, &Q3.T, Q3.v3, ntab3, sm_count, stream, &scratch3);
      if (rcg != DFRG_OK) return rcg;
    }
    void (*k3)(const ThreePoint3DParams) = nullptr;
#define DFRG_T3D_PICK(K) if (regk3 == K) k3 = dmin ? t3d_kernel<K, true> : t3d_kernel<K, false>;
    DFRG_T3D_PICK(0) DFRG_T3D_PICK(1) DFRG_T3D_PICK(2)
#undef DFRG_T3D_PICK
    cudaError_t e3 = cudaFuncSetAttribute(k3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem3);
    if (e3 != cudaSuccess) { scratch_free(scratch3, stream); return check_cuda(e3); }
    const int grid3 = n_ext < sm_count ? n_ext : sm_count;
    k3<<<grid3, 256, smem3, stream>>>(Q3);
    const int rc3 = check_cuda(cudaGetLastError());
    scratch_free(scratch3, stream);
    return rc3;
  }
  const int regk = D->reg.kind == DFRG_REG_LITIM ? 0 : (D->reg.order == 1 ? 1 : 2);
  void* scratch = nullptr;
  // ---- product-grid path (ext_outer = G promised by the caller, checked on the device) ----
  {
    const int rc = t3g_launch(P, D->ext_outer, regk, nullptr, nullptr, 0, sm_count, stream, &scratch);
    if (rc != DFRG_OK) return rc;   // P.skip_flag is set if the product-grid kernels were enqueued
  }
  const size_t smem = threepoint_v2_smem(P.nq, P.n1, P.n2, P.grid.n);
  void (*kern)(const ThreePointParams) = nullptr;
#define DFRG_T3_PICK(K) if (regk == K) kern = dmin ? threepoint_kernel_v2<K, true, 256, 8> : threepoint_kernel_v2<K, false, 256, 8>;
  DFRG_T3_PICK(0) DFRG_T3_PICK(1) DFRG_T3_PICK(2)
#undef DFRG_T3_PICK
  const int nthreads = 256;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) { scratch_free(scratch, stream); return check_cuda(e); }
  const int grid = n_ext < sm_count ? n_ext : sm_count;  // persistent: 1 CTA of 256 threads x 240 registers per SM (replicated tables: 140 KB)
  kern<<<grid, nthreads, smem, stream>>>(P);
  const int rc_last = check_cuda(cudaGetLastError());
  scratch_free(scratch, stream);
  return rc_last;
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
  size_t need = 2 * ((size_t)D->q.n + D->cos1.n + D->cos2.n + D->phi.n) + 3 * (size_t)D->tab[0].n_q + 128 + nf + next_d +
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
