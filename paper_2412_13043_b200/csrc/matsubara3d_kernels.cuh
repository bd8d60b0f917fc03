// matsubara3d_kernels.cuh -- kernels of dfrg_integrate_matsubara3d, shared by matsubara3d.cu (host API, pre-passes, the
// row-streaming kernel and the specialised moment kernel) and matsubara3d_anyshape.cu (the any-shape moment kernel).
#pragma once
#include <type_traits>
#include <stdlib.h>

#include "dfrg_device.cuh"
#include "dfrg_internal.h"

namespace dfrg {

constexpr int M3_MAX_PAIRS = 6144;
constexpr int M3_PRE_THREADS = 256;

struct Mats3dParams {
  int nq, nc, n_field, n_p, n_jext, n_max, n_rows, row_stride;
  double T, prefactor;
  RegParams reg;
  GridParams grid;
  FastMathConsts fmc;
  const double *xq, *wq, *xc, *wc, *Zpsi, *Zphi, *coef, *m2psi, *m2phi, *pext;
  double *d0phi;    // [n_p][n_rows][row_stride]
  double *rowmin;   // [n_p][n_rows]
  double2 *psi;     // [2 n_max + 1][psi_stride]
  double *psimin;   // [2 n_max + 1]
  int psi_stride;
  double *out, *dmin;
  // moment path (mats3d_moment_kernel): D0phi is laid out [p][i][m][c] in chunks of chunk_stride doubles
  int phi_layout;    // 0: [p][m][i*nc + c] (row_stride), 1: [p][i][m*nc + c] (chunk_stride)
  int chunk_stride;
  int tile_fields;   // field points per CTA tile of the moment kernel
  int max_slots;     // partial sums per (field tile, p) in part[]
  int grid_main;     // CTAs of the moment kernel (the fix-up kernel re-derives the unit ownership from it)
  double *part;      // [max_slots][n_p][n_jext][n_field]
  int sym_try;       // host: the cos rule is long enough for the symmetric-pair moment loop (nc % 8 == 0)
  int* symflag;      // device: 1 if the cos rule is exactly symmetric (x_c = -x_{nc-1-c}, equal weights), set by the pre-pass
  int reg_arg4d;     // 1: regulators at the 4-momentum squared; 0: spatial regulators
  int fermion_reg;   // 1: fermion line regulated with RF / RFdot on its Dirac structure (reading A25)
  double mu;         // chemical potential (complex fermion line when != 0)
  double *psi_im;    // [2 n_max + 1][psi_stride]  Im D0psi (mu != 0)
  double *psimin_f;  // [n_field]  min over (n, q) of |D0psi + m2psi_f| (mu != 0)
  double *out_im, *part_im;
  int mode;          // 0: value;  1: d/dm2_psi (G_psi^2 -> -2 G_psi^3);  2: d/dm2_phi (G_phi -> -G_phi^2, kernels with SQ)
};

// ---- (1) boson rows --------------------------------------------------------------------------------
static __global__ void __launch_bounds__(M3_PRE_THREADS) mats3d_phi_rows_kernel(const Mats3dParams P) {
  __shared__ __align__(32) double4 cells[1024];
  __shared__ __align__(16) double fmmem[FM_DOUBLES];
  __shared__ double red[32];
  const int m = blockIdx.x, e = blockIdx.y;
  const FastMath fm = fm_build(fmmem, P.fmc);
  cells_build(cells, P.Zphi + (size_t)m * P.grid.n, P.grid);
  __syncthreads();
  // Symmetric cos rule (Gauss-Legendre on [-1,1] is: x_c = -x_{nc-1-c}, equal weights)?  Then the moment path stores
  // each row as (node c, node nc-1-c) pairs, and the moment loop works on r+ + r-, r+ - r- (see mats3d_moment_kernel).
  int sym = 0;
  if (P.sym_try && P.phi_layout == 1) {
    int ok = 1;
    for (int c = threadIdx.x; c < P.nc / 2; c += M3_PRE_THREADS)
      if (P.xc[c] != -P.xc[P.nc - 1 - c] || P.wc[c] != P.wc[P.nc - 1 - c]) ok = 0;
    sym = __syncthreads_and(ok);
  }
  if (m == 0 && e == 0 && threadIdx.x == 0 && P.symflag) *P.symflag = sym;
  const double p = P.pext[e];
  const double om = 2.0 * 3.14159265358979323846 * (double)m * P.T;
  const int npairs = P.nq * P.nc;
  double* dst = P.d0phi + ((size_t)e * P.n_rows + m) * P.row_stride;
  double* dst1 = P.d0phi + (size_t)e * P.nq * P.chunk_stride + (size_t)m * P.nc;
  double dmin = __longlong_as_double(0x7ff0000000000000LL);
  for (int t = threadIdx.x; t < npairs; t += M3_PRE_THREADS) {
    const int i = t / P.nc, jc = t - i * P.nc;
    const double q = P.xq[i], c = P.xc[jc];
    double r2 = p * p + q * q - 2.0 * p * q * c;
    r2 = clamp_lo(r2, 0.0);
    const double sphi = om * om + r2;
    double R, Rd;
    regulator(P.reg, fm, P.reg_arg4d ? sphi : r2, R, Rd);
    const double D0 = table_lookup(cells, P.grid, fm, r2) * sphi + R;
    if (P.phi_layout == 0) dst[t] = D0;
    else dst1[(size_t)i * P.chunk_stride + (sym ? (2 * jc < P.nc ? 2 * jc : 2 * (P.nc - 1 - jc) + 1) : jc)] = D0;
    dmin = fmin(dmin, D0);
  }
  if (P.phi_layout == 0) {
    if (threadIdx.x == 0 && (npairs & 1)) dst[npairs] = 1.0;  // pad to the even row stride
  } else if (m == 0 && ((P.n_rows * P.nc) & 1)) {
    for (int i = threadIdx.x; i < P.nq; i += M3_PRE_THREADS)
      P.d0phi[((size_t)e * P.nq + i) * P.chunk_stride + P.n_rows * P.nc] = 1.0;  // pad to the even chunk stride
  }
  dmin = block_min(dmin, red);
  if (threadIdx.x == 0) P.rowmin[(size_t)e * P.n_rows + m] = dmin;
}

// ---- (2) fermion line --------------------------------------------------------------------------------
static __global__ void __launch_bounds__(128) mats3d_psi_kernel(const Mats3dParams P) {
  __shared__ __align__(32) double4 cells[1024];
  __shared__ __align__(16) double fmmem[FM_DOUBLES];
  __shared__ double red[32];
  const int it = blockIdx.x, n = it - P.n_max;
  const int nbar = n >= 0 ? n : -n - 1;
  const double nun = (2.0 * n + 1.0) * 3.14159265358979323846 * P.T;
  const FastMath fm = fm_build(fmmem, P.fmc);
  cells_build(cells, P.Zpsi + (size_t)nbar * P.grid.n, P.grid);
  __syncthreads();
  double dmin = __longlong_as_double(0x7ff0000000000000LL);
  for (int i = threadIdx.x; i < P.nq; i += 128) {
    const double q = P.xq[i];
    const double spsi = nun * nun - P.mu * P.mu + q * q;   // Re (nu + i mu)^2 + q^2
    const double Z = table_lookup(cells, P.grid, fm, q * q);
    double D0, Rd, Zt = Z;   // Zt: what multiplies the squared time component (nu + i mu)^2
    if (P.fermion_reg) {     // reading A25: D = Z^2 (s - sR) + (Z sqrt(sR) + RF(sR))^2 + m2, insertion 2 A RFdot
      const double sR = P.reg_arg4d ? spsi : q * q;   // (mu != 0 needs the spatial argument: spsi is real here)
      const double A = fermion_kinetic(P.reg, fm, Z, sR, Rd);
      Zt = Z * Z;
      D0 = fma(Zt, spsi - sR, A * A);
    } else {
      double R;
      regulator(P.reg, fm, P.reg_arg4d ? spsi : q * q, R, Rd);
      D0 = Z * spsi + R;
    }
    P.psi[(size_t)it * P.psi_stride + i] = make_double2(D0, P.wq[i] * q * q * Rd);
    if (P.psi_im) P.psi_im[(size_t)it * P.psi_stride + i] = Zt * (2.0 * nun * P.mu);
    dmin = fmin(dmin, D0);
  }
  dmin = block_min(dmin, red);
  if (threadIdx.x == 0) P.psimin[it] = dmin;
}

// ---- (3) main kernel -----------------------------------------------------------------------------------
// Persistent, warp-specialised.  One CTA per SM walks the work items (p, j, field tile) it owns
// (item = blockIdx.x + k gridDim.x) and, inside an item, the loop Matsubara index n.  One producer warp
// runs up to two (item, n) stages ahead of the consumers: it waits for a stage to drain (mbarrier
// empty[b]), issues the TMA bulk copies of row |j-n| of D0phi and row n of psi, builds the numerator row
// Nw in shared memory and arrives on full[b].  GROUPS x 256 consumer threads run the hot loop: thread =
// (MF field points, radial nodes i = group mod GROUPS); the groups' partial sums are combined in fixed
// order through shared memory once per item.
constexpr int M3_FT = 128;  // threads per consumer group; a group covers M3_FT x MF field points

// One quadrature node for the MF field points of a thread:  a_f += Nw / (D0 + m2_f).
// Batched inversion over the field points (same Nw): with d_f = D0 + m2_f,
//   MF = 2:  R = Nw/(d0 d1),               a0 += R d1,            a1 += R d0              (9 FP64 instr / 2 evals)
//   MF = 4:  R = Nw/((d0 d1)(d2 d3)),      a0 += (R p23) d1, ...                          (17 FP64 instr / 4 evals)
// i.e. 4 + 1/MF FP64-pipe instructions and 1/MF MUFU.RCP64H per evaluation instead of 5 and 1.  The products stay
// far inside the double range (|d| between ~1e-3 k^2 and ~1e5 k^2); each extra multiply costs half an ulp.
template <int MF, bool SQ>
__device__ __forceinline__ void accumulate_node(const double D0, const double Nw, const double (&m2)[MF],
                                                double (&a)[MF]) {
  if constexpr (SQ) {  // a_f -= Nw / (D0 + m2_f)^2   (mass derivative of the boson line)
#pragma unroll
    for (int m = 0; m < MF; ++m) {
      const double r = fast_rcp(D0 + m2[m]);
      a[m] = fma(-(Nw * r), r, a[m]);
    }
  } else if constexpr (MF == 1) {
    a[0] = fma(Nw, fast_rcp(D0 + m2[0]), a[0]);
  } else if constexpr (MF == 2) {
    const double d0 = D0 + m2[0], d1 = D0 + m2[1];
    const double R = fast_rcp(d0 * d1) * Nw;
    a[0] = fma(R, d1, a[0]);
    a[1] = fma(R, d0, a[1]);
  } else {
    static_assert(MF == 4, "MF must be 1, 2 or 4");
    const double d0 = D0 + m2[0], d1 = D0 + m2[1], d2 = D0 + m2[2], d3 = D0 + m2[3];
    const double p01 = d0 * d1, p23 = d2 * d3;
    const double R = fast_rcp(p01 * p23) * Nw;
    const double r01 = R * p23, r23 = R * p01;
    a[0] = fma(r01, d1, a[0]);
    a[1] = fma(r01, d0, a[1]);
    a[2] = fma(r23, d3, a[2]);
    a[3] = fma(r23, d2, a[3]);
  }
}

template <int GROUPS, int MF, bool SQ>
__global__ void __launch_bounds__(GROUPS * M3_FT + 32, 1) mats3d_main_kernel(const Mats3dParams P) {
  constexpr int NCONS = GROUPS * M3_FT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t full[2], empty[2];
  __shared__ double skap[20];

  const int nq = P.nq, nc = P.nc, npairs = nq * nc;
  const int rs = P.row_stride, ps = P.psi_stride;
  double* d0buf = reinterpret_cast<double*>(smem_raw);               // [2][rs]
  double2* psibuf = reinterpret_cast<double2*>(d0buf + 2 * rs);      // [2][ps]
  double* nwbuf = reinterpret_cast<double*>(psibuf + 2 * ps);        // [2][rs]
  double* beta = nwbuf + 2 * rs;                                     // [nq][4]   (producer only)
  double* sxq = beta + 4 * nq;
  double* sxc = sxq + ((nq + 1) & ~1);
  double* swc = sxc + ((nc + 1) & ~1);
  double* part = swc + ((nc + 1) & ~1);                              // [2][GROUPS][M3_FT * MF]

  const int n_terms = 2 * P.n_max + 1;
  const int n_ftiles = (P.n_field + M3_FT * MF - 1) / (M3_FT * MF);
  const int n_items = P.n_p * P.n_jext * n_ftiles;
  const uint32_t row_bytes = (uint32_t)rs * 8u, psi_bytes = (uint32_t)ps * 16u;
  const double pi = 3.14159265358979323846;
  const double ik2 = P.reg.inv_k2;

  if (threadIdx.x == 0) {
    mbar_init(&full[0], 1);
    mbar_init(&full[1], 1);
    mbar_init(&empty[0], NCONS / 32);
    mbar_init(&empty[1], NCONS / 32);
    mbar_fence_init();
  }
  if (threadIdx.x < 20) skap[threadIdx.x] = P.coef[threadIdx.x];
  for (int i = threadIdx.x; i < nq; i += blockDim.x) sxq[i] = P.xq[i];
  for (int i = threadIdx.x; i < nc; i += blockDim.x) { sxc[i] = P.xc[i]; swc[i] = P.wc[i]; }
  __syncthreads();

  if (threadIdx.x >= NCONS) {
    // =========================== producer warp ===========================
    const int lane = threadIdx.x - NCONS;
    uint32_t g = 0;  // global stage counter
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
      const int ej = item / n_ftiles;
      const int e = ej / P.n_jext, j = ej - e * P.n_jext;
      const double p = P.pext[e];
      const double nuj = (2.0 * j + 1.0) * pi * P.T;
      for (int it = 0; it < n_terms; ++it, ++g) {
        const int b = g & 1;
        const int n = it - P.n_max;
        const int mm = j - n, mabs = mm >= 0 ? mm : -mm;
        mbar_wait(&empty[b], ((g >> 1) & 1) ^ 1);  // consumers drained this stage (passes at once for g < 2)
        if (lane == 0) {
          mbar_expect_tx_only(&full[b], row_bytes + psi_bytes);
          tma_bulk_g2s(d0buf + (size_t)b * rs, P.d0phi + ((size_t)e * P.n_rows + mabs) * rs, row_bytes, &full[b]);
          tma_bulk_g2s(psibuf + (size_t)b * ps, P.psi + (size_t)it * ps, psi_bytes, &full[b]);
        }
        // P = sum_b y2^b beta_b,  beta_b = sum_{a+c<=3-b} kap_abc y1^a y3^c   (idx: a outermost, then b, then c)
        const double nun = (2.0 * n + 1.0) * pi * P.T;
        const double y1 = nun * nuj * ik2;
        for (int i = lane; i < nq; i += 32) {
          const double q = sxq[i];
          const double y3 = fma(nun, nun, __dmul_rn(q, q)) * ik2;   // (explicit: the same bits in every instantiation)
          double be[4] = {0.0, 0.0, 0.0, 0.0};
          int idx = 0;
          double y1a = 1.0;
#pragma unroll
          for (int a = 0; a <= 3; ++a) {
#pragma unroll
            for (int bb = 0; bb <= 3 - a; ++bb) {
              double y3c = y1a;
#pragma unroll
              for (int c = 0; c <= 3 - a - bb; ++c) {
                be[bb] = fma(skap[idx++], y3c, be[bb]);
                y3c *= y3;
              }
            }
            y1a *= y1;
          }
          beta[4 * i + 0] = be[0]; beta[4 * i + 1] = be[1]; beta[4 * i + 2] = be[2]; beta[4 * i + 3] = be[3];
        }
        __syncwarp();
        double* nw = nwbuf + (size_t)b * rs;
        for (int i = 0; i < nq; ++i) {
          const double pq = p * sxq[i] * ik2;
          const double b0 = beta[4 * i], b1 = beta[4 * i + 1], b2 = beta[4 * i + 2], b3 = beta[4 * i + 3];
          for (int jc = lane; jc < nc; jc += 32) {
            const double y2 = pq * sxc[jc];
            nw[i * nc + jc] = swc[jc] * fma(fma(fma(b3, y2, b2), y2, b1), y2, b0);
          }
        }
        if (lane == 0 && (npairs & 1)) nw[npairs] = 0.0;
        __syncwarp();
        if (lane == 0) mbar_arrive(&full[b]);  // release: the Nw row is visible to whoever acquires full[b]
      }
    }
    return;
  }

  // =============================== consumers ===============================
  const int grp = threadIdx.x / M3_FT, tf = threadIdx.x - grp * M3_FT;
  const bool warp_leader = (threadIdx.x & 31) == 0;
  uint32_t g = 0;
  int item_parity = 0;
  for (int item = blockIdx.x; item < n_items; item += gridDim.x, item_parity ^= 1) {
    const int ej = item / n_ftiles, ftile = item - ej * n_ftiles;
    const int e = ej / P.n_jext, j = ej - e * P.n_jext;
    const int f0 = ftile * (M3_FT * MF) + tf;
    double m2psi[MF], m2phi[MF], acc[MF];
#pragma unroll
    for (int m = 0; m < MF; ++m) {
      const int f = f0 + m * M3_FT;
      m2psi[m] = (f < P.n_field) ? P.m2psi[f] : 1.0;
      m2phi[m] = (f < P.n_field) ? P.m2phi[f] : 1.0;
      acc[m] = 0.0;
    }
    for (int it = 0; it < n_terms; ++it, ++g) {
      const int b = g & 1;
      mbar_wait(&full[b], (g >> 1) & 1);
      const double* d0 = d0buf + (size_t)b * rs;
      const double* nw = nwbuf + (size_t)b * rs;
      const double2* psi = psibuf + (size_t)b * ps;
      for (int i = grp; i < nq; i += GROUPS) {
        // fermion line first: its reciprocal chain overlaps with the angular loop below
        const double2 o = psi[i];
        double h[MF], a[MF];
#pragma unroll
        for (int m = 0; m < MF; ++m) {
          const double gpsi = fast_rcp(o.x + m2psi[m]);
          const double g2 = gpsi * gpsi;
          h[m] = o.y * (P.mode == 1 ? -2.0 * g2 * gpsi : g2);
          a[m] = 0.0;
        }
        if ((nc & 1) == 0) {
          const double2* drow = reinterpret_cast<const double2*>(d0 + i * nc);
          const double2* nrow = reinterpret_cast<const double2*>(nw + i * nc);
#pragma unroll 2
          for (int jc = 0; jc < nc / 2; ++jc) {
            const double2 dd = drow[jc], nn = nrow[jc];
            accumulate_node<MF, SQ>(dd.x, nn.x, m2phi, a);
            accumulate_node<MF, SQ>(dd.y, nn.y, m2phi, a);
          }
        } else {
          for (int jc = 0; jc < nc; ++jc) accumulate_node<MF, SQ>(d0[i * nc + jc], nw[i * nc + jc], m2phi, a);
        }
#pragma unroll
        for (int m = 0; m < MF; ++m) acc[m] = fma(h[m], a[m], acc[m]);
      }
      __syncwarp();
      if (warp_leader) mbar_arrive(&empty[b]);
    }
    // ---- S5/S6: combine the radial-node groups in fixed order, write the item's outputs ----
    double* mypart = part + (size_t)item_parity * GROUPS * (M3_FT * MF);
#pragma unroll
    for (int m = 0; m < MF; ++m) mypart[grp * (M3_FT * MF) + m * M3_FT + tf] = acc[m];
    named_bar_sync(1, NCONS);
    if (grp == 0) {
      const double scale = P.prefactor * P.T;
      double dpsi = 0.0, dphi = 0.0;
      if (P.dmin) {
        const double inf = __longlong_as_double(0x7ff0000000000000LL);
        dpsi = inf;
        dphi = inf;
        for (int it = 0; it < n_terms; ++it) {
          const int mm = j - (it - P.n_max), mabs = mm >= 0 ? mm : -mm;
          dpsi = fmin(dpsi, P.psimin[it]);
          dphi = fmin(dphi, P.rowmin[(size_t)e * P.n_rows + mabs]);
        }
      }
#pragma unroll
      for (int m = 0; m < MF; ++m) {
        const int f = f0 + m * M3_FT;
        if (f < P.n_field) {
          double r = mypart[m * M3_FT + tf];
#pragma unroll
          for (int gg = 1; gg < GROUPS; ++gg) r += mypart[gg * (M3_FT * MF) + m * M3_FT + tf];
          const size_t o = (size_t)ej * P.n_field + f;
          P.out[o] = scale * r;
          if (P.dmin) P.dmin[o] = fmin(dpsi + m2psi[m], dphi + m2phi[m]) * ik2;
        }
      }
    }
  }
}

static size_t mats3d_main_smem(int nq, int nc, int rs, int ps, int groups, int mf) {
  return 8 * (size_t)(2 * rs + 4 * ps + 2 * rs + 4 * nq + ((nq + 1) & ~1) + 2 * ((nc + 1) & ~1) +
                      2 * groups * M3_FT * mf);
}

// ---- (3b) moment kernel ---------------------------------------------------------------------------------
// The numerator polynomial is a cubic in y2 = p q c / k^2 whose coefficients depend on (j, n, i) only, and the
// boson denominator depends on (j, n) only through m = |j - n|.  Hence
//     sum_c wc_c P G_phi  =  sum_{b=0..3} beta_b(j,n,i) (p q_i/k^2)^b  M_b(m, i; f),
//     M_b(m, i; f) = sum_c wc_c c^b / (D0phi[p][m][i][c] + m2phi_f)              (angular moments of the boson line)
// and the moments are shared by every (j, n) with |j - n| = m: n_jext + n_max rows of moments serve
// n_jext (2 n_max + 1) (j, n) pairs (27 for 368 in config 4).  Likewise G_psi depends on n only through
// nbar (nu_{-n-1} = -nu_n): n_max + 1 fermion reciprocals serve 2 n_max + 1 terms.  Per (p, i, f):
//     (n_jext + n_max) nc  x (DADD + reciprocal (3 DFMA) + 4 DFMA)        moments
//   + (n_max + 1)          x (DADD + reciprocal + DMUL)                    H_nbar = G_psi^2
//   + n_jext (2 n_max + 1) x (DMUL + 3 DFMA + DFMA)                        acc_j += H_nbar (beta' . M)
// = 7084 FP64 instructions for config 4 instead of 16 x 23 x (24 x 4.25 + 8) = 40 480.
//
// Mapping.  Work unit = (field tile, p, radial node i); the units are dealt to the CTAs (one per SM, persistent)
// in contiguous ranges, so a CTA keeps its NJ accumulators per field point in registers while it walks the radial
// nodes of one p, and writes them as a partial sum when p (or its range) ends; mats3d_fixup_kernel adds the
// <= max_slots partial sums of an output in fixed order (deterministic: the ownership of units is a pure
// function of the grid size).  A producer warp runs one unit ahead: TMA bulk copy of the unit's D0phi chunk
// [m][c] (5 KB), the fermion denominators, and beta'[j][n] = Wpsi (p q/k^2)^b beta_b (12 KB, field independent).
// NTC consumer threads x MF field points: everything they read in the hot loop is a shared-memory broadcast.
// The loops over m and j are unrolled at compile time (NMAX, NJ are template parameters) so that the
// accumulators, the moments and H stay in registers.
// Reciprocals 1/(D0[t] + m2[k]) of M3_NBAT consecutive nodes for the MF field points of a thread, stage by stage.
// MF = 2: one hardware seed per node serves both field points, 1/(d0 d1) then r0 = R d1, r1 = R d0 -- the same
// FP64 instruction count as two separate Newton reciprocals (8 per node) and half the MUFU.RCP64H.
constexpr int M3_NBAT = 4;
template <int MF, bool SQ>
__device__ __forceinline__ void mats3d_recip_batch(const double* __restrict__ dptr, const double (&m2)[MF],
                                                   double (&r)[M3_NBAT][MF]) {
  double d[M3_NBAT][MF];
  static_assert(M3_NBAT % 2 == 0, "vector loads of D0");
#pragma unroll
  for (int t = 0; t < M3_NBAT; t += 2) {
    const double2 D0 = *reinterpret_cast<const double2*>(dptr + t);   // dptr is 16-byte aligned (even node index)
#pragma unroll
    for (int k = 0; k < MF; ++k) { d[t][k] = D0.x + m2[k]; d[t + 1][k] = D0.y + m2[k]; }
  }
  if constexpr (MF == 2) {
    // one hardware seed per TWO nodes x two field points: R = 1/((d00 d01)(d10 d11)), 1/(d00 d01) = R (d10 d11), ...
    // 16 FP64 instructions per 4 reciprocals (as four separate Newton reciprocals) and a quarter of the MUFU.RCP64H
    double pr[M3_NBAT], R[M3_NBAT / 2], q[M3_NBAT / 2];
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t) pr[t] = d[t][0] * d[t][1];
#pragma unroll
    for (int h = 0; h < M3_NBAT / 2; ++h) q[h] = pr[2 * h] * pr[2 * h + 1];
#pragma unroll
    for (int h = 0; h < M3_NBAT / 2; ++h) R[h] = rcp_seed(q[h]);
#pragma unroll
    for (int h = 0; h < M3_NBAT / 2; ++h) q[h] = fma(-q[h], R[h], 1.0);
#pragma unroll
    for (int h = 0; h < M3_NBAT / 2; ++h) q[h] = fma(q[h], q[h], q[h]);
#pragma unroll
    for (int h = 0; h < M3_NBAT / 2; ++h) R[h] = fma(R[h], q[h], R[h]);
#pragma unroll
    for (int h = 0; h < M3_NBAT / 2; ++h) {
      const double ra_ = R[h] * pr[2 * h + 1], rb_ = R[h] * pr[2 * h];   // 1/(d d) of node 2h, of node 2h+1
      r[2 * h][0] = ra_ * d[2 * h][1]; r[2 * h][1] = ra_ * d[2 * h][0];
      r[2 * h + 1][0] = rb_ * d[2 * h + 1][1]; r[2 * h + 1][1] = rb_ * d[2 * h + 1][0];
    }
  } else {
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t)
#pragma unroll
      for (int k = 0; k < MF; ++k) r[t][k] = rcp_seed(d[t][k]);
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t)
#pragma unroll
      for (int k = 0; k < MF; ++k) d[t][k] = fma(-d[t][k], r[t][k], 1.0);
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t)
#pragma unroll
      for (int k = 0; k < MF; ++k) d[t][k] = fma(d[t][k], d[t][k], d[t][k]);
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t)
#pragma unroll
      for (int k = 0; k < MF; ++k) r[t][k] = fma(r[t][k], d[t][k], r[t][k]);
  }
  if constexpr (SQ) {  // mass derivative of the boson line: the moments are taken of -G_phi^2
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t)
#pragma unroll
      for (int k = 0; k < MF; ++k) r[t][k] = -(r[t][k] * r[t][k]);
  }
}

// Field points are independent outputs (reading A4: whatever IEEE arithmetic gives, PER OUTPUT), but mats3d_recip_batch
// inverts the denominators of a thread's two field points at two neighbouring nodes through ONE product.  A field point
// whose mass term has blown up (NaN, infinite, or so large that the product of four denominators overflows) would spoil
// the reciprocals of its partner as well.  The masses are fixed per thread and field tile, so this is known before the
// unit starts: `solo` is set where either mass is not below M3_JOINT_MASS_MAX in magnitude, and such a thread redoes every
// row with one Newton reciprocal per denominator, as the one-field-point kernels do (a branch on a flag that has long
// been known: measured cost nil.  Flags derived from the data inside the loop -- the hardware seeds of the products, or
// the finished moments -- cost 4.2 % and 2.3 % of the bench kernel's time: integer work and a branch at the end of the
// dependent chain are not free at two warps per scheduler).  The blown-up field point gets what IEEE arithmetic gives
// for it, its partner its own regular value.  Not covered: a denominator D0 + m2 that is EXACTLY zero at a node (D0 and
// -m2 equal bit for bit) still costs the partner's output too; include/dfrg.h says so.
constexpr double M3_JOINT_MASS_MAX = 1e70;   // (1e70 + |D0|)^4 stays finite for every |D0| < 1e76
template <int MF, bool SQ, bool SYM>
__device__ __forceinline__ void mats3d_row_decouple(const double* __restrict__ drow, const double4* __restrict__ num4,
                                                    const int nc, const double (&m2phi)[MF], double (&M)[4][MF],
                                                    const bool solo) {
  if constexpr (MF == 2) {
    if (solo) {
#pragma unroll
      for (int k = 0; k < MF; ++k) { M[0][k] = 0.0; M[1][k] = 0.0; M[2][k] = 0.0; M[3][k] = 0.0; }
#pragma unroll 1
      for (int c = 0; c < nc; ++c) {
        const double D0 = drow[c];
        double4 w;
        if constexpr (SYM) {   // pair-ordered chunk (x-, x+), one weight vector (w, w x+, w x+^2, w x+^3) per pair
          w = num4[c >> 1];
          if (!(c & 1)) { w.y = -w.y; w.w = -w.w; }
        } else {
          w = num4[c];
        }
#pragma unroll
        for (int k = 0; k < MF; ++k) {
          double r = fast_rcp(D0 + m2phi[k]);
          if constexpr (SQ) r = -(r * r);
          M[0][k] = fma(w.x, r, M[0][k]);
          M[1][k] = fma(w.y, r, M[1][k]);
          M[2][k] = fma(w.z, r, M[2][k]);
          M[3][k] = fma(w.w, r, M[3][k]);
        }
      }
    }
  }
}

// M_b += sum_t w[t].b r[t]  for a batch of M3_NBAT nodes (w = wc c^b, broadcast from shared memory).
template <int MF>
__device__ __forceinline__ void mats3d_moment_accumulate(const double4* __restrict__ w4, const double (&r)[M3_NBAT][MF],
                                                         double (&M)[4][MF]) {
  double4 w[M3_NBAT];
#pragma unroll
  for (int t = 0; t < M3_NBAT; ++t) w[t] = w4[t];
#pragma unroll
  for (int t = 0; t < M3_NBAT; ++t)
#pragma unroll
    for (int k = 0; k < MF; ++k) {
      M[0][k] = fma(w[t].x, r[t][k], M[0][k]);
      M[1][k] = fma(w[t].y, r[t][k], M[1][k]);
      M[2][k] = fma(w[t].z, r[t][k], M[2][k]);
      M[3][k] = fma(w[t].w, r[t][k], M[3][k]);
    }
}

// Symmetric cos rule: the batch holds two (x-, x+) pairs, x- = -x+, equal weights, so with s = r+ + r-, d = r+ - r-
//   M_0 += w s,  M_1 += w x+ d,  M_2 += w x+^2 s,  M_3 += w x+^3 d :  6 FP64 instructions per pair and field point instead
// of 8, and one weight vector per pair instead of per node.  w4[p] = (w, w x+, w x+^2, w x+^3) of the pair's positive node.
template <int MF>
__device__ __forceinline__ void mats3d_moment_accumulate_sym(const double4* __restrict__ w4,
                                                             const double (&r)[M3_NBAT][MF], double (&M)[4][MF]) {
  double4 w[M3_NBAT / 2];
#pragma unroll
  for (int p = 0; p < M3_NBAT / 2; ++p) w[p] = w4[p];
  double sm[M3_NBAT / 2][MF], df[M3_NBAT / 2][MF];
#pragma unroll
  for (int p = 0; p < M3_NBAT / 2; ++p)
#pragma unroll
    for (int k = 0; k < MF; ++k) { sm[p][k] = r[2 * p + 1][k] + r[2 * p][k]; df[p][k] = r[2 * p + 1][k] - r[2 * p][k]; }
#pragma unroll
  for (int p = 0; p < M3_NBAT / 2; ++p)
#pragma unroll
    for (int k = 0; k < MF; ++k) {
      M[0][k] = fma(w[p].x, sm[p][k], M[0][k]);
      M[1][k] = fma(w[p].y, df[p][k], M[1][k]);
      M[2][k] = fma(w[p].z, sm[p][k], M[2][k]);
      M[3][k] = fma(w[p].w, df[p][k], M[3][k]);
    }
}

// The (j, n) pairs with |j - n| = m of the moment kernel:  acc[j] += H[nbar(n)] (beta'[j][n] . M),  in groups of
// four (two j x two signs), written stage by stage so that each stage is a set of independent instructions.
template <int m, int NMAX, int NJ, int MF>
__device__ __forceinline__ void mats3d_pairs(const double4* __restrict__ bet4, const double (&M)[4][MF],
                                             const double (&H)[NMAX + 1][MF], double (&acc)[NJ][MF]) {
  constexpr int NT = 2 * NMAX + 1;
#pragma unroll
  for (int j0 = 0; j0 < NJ; j0 += 2) {
    double4 B[4];
    double t[4][MF];
#pragma unroll
    for (int qd = 0; qd < 4; ++qd) {
      const int j = j0 + (qd >> 1), n = (qd & 1) ? j + m : j - m;
      const bool valid = j < NJ && ((qd & 1) ? (m > 0 && n <= NMAX) : (n >= -NMAX && n <= NMAX));
      if (valid) B[qd] = bet4[j * NT + n + NMAX];
    }
#pragma unroll
    for (int qd = 0; qd < 4; ++qd) {
      const int j = j0 + (qd >> 1), n = (qd & 1) ? j + m : j - m;
      const bool valid = j < NJ && ((qd & 1) ? (m > 0 && n <= NMAX) : (n >= -NMAX && n <= NMAX));
      if (valid)
#pragma unroll
        for (int k = 0; k < MF; ++k) t[qd][k] = B[qd].x * M[0][k];
    }
#pragma unroll
    for (int qd = 0; qd < 4; ++qd) {
      const int j = j0 + (qd >> 1), n = (qd & 1) ? j + m : j - m;
      const bool valid = j < NJ && ((qd & 1) ? (m > 0 && n <= NMAX) : (n >= -NMAX && n <= NMAX));
      if (valid)
#pragma unroll
        for (int k = 0; k < MF; ++k) t[qd][k] = fma(B[qd].y, M[1][k], t[qd][k]);
    }
#pragma unroll
    for (int qd = 0; qd < 4; ++qd) {
      const int j = j0 + (qd >> 1), n = (qd & 1) ? j + m : j - m;
      const bool valid = j < NJ && ((qd & 1) ? (m > 0 && n <= NMAX) : (n >= -NMAX && n <= NMAX));
      if (valid)
#pragma unroll
        for (int k = 0; k < MF; ++k) t[qd][k] = fma(B[qd].z, M[2][k], t[qd][k]);
    }
#pragma unroll
    for (int qd = 0; qd < 4; ++qd) {
      const int j = j0 + (qd >> 1), n = (qd & 1) ? j + m : j - m;
      const bool valid = j < NJ && ((qd & 1) ? (m > 0 && n <= NMAX) : (n >= -NMAX && n <= NMAX));
      if (valid)
#pragma unroll
        for (int k = 0; k < MF; ++k) t[qd][k] = fma(B[qd].w, M[3][k], t[qd][k]);
    }
#pragma unroll
    for (int qd = 0; qd < 4; ++qd) {
      const int j = j0 + (qd >> 1), n = (qd & 1) ? j + m : j - m;
      const bool valid = j < NJ && ((qd & 1) ? (m > 0 && n <= NMAX) : (n >= -NMAX && n <= NMAX));
      if (valid) {
        const int nbar = n >= 0 ? n : -n - 1;
#pragma unroll
        for (int k = 0; k < MF; ++k) acc[j][k] = fma(H[nbar][k], t[qd][k], acc[j][k]);
      }
    }
  }
}

template <int NMAX, int NJ, int MF, int NTC, bool SQ, bool SYM>
__global__ void __launch_bounds__(NTC, 1) mats3d_moment_kernel(const Mats3dParams P) {
  // two instantiations are enqueued when the symmetric-pair loop is possible; the pre-pass decided which one works
  if (P.sym_try && (*P.symflag != 0) != SYM) return;
  constexpr int NT = 2 * NMAX + 1, NROWS = NJ + NMAX, NB = NJ * NT * 4, NPS = NMAX + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t full[2];
  __shared__ double skap[20];

  const int nq = P.nq, nc = P.nc, cs = P.chunk_stride, ps = P.psi_stride;
  double* d0buf = reinterpret_cast<double*>(smem_raw);           // [2][cs]
  double* betabuf = d0buf + 2 * cs;                              // [2][NB]
  double2* psibuf = reinterpret_cast<double2*>(betabuf + 2 * NB);  // [2][NPS] (D0psi, Wpsi)
  double* numbuf = reinterpret_cast<double*>(psibuf + 2 * NPS);  // [nc][4]  wc c^b
  double* sxq = numbuf + 4 * nc;                                 // [nq]

  const int tid = threadIdx.x;
  const int tile = NTC * MF;
  const int n_ftiles = (P.n_field + tile - 1) / tile;
  const long long upp = (long long)P.n_p * nq;                   // units per field tile
  const long long U = (long long)n_ftiles * upp;
  const long long u0 = (long long)blockIdx.x * U / gridDim.x, u1 = (long long)(blockIdx.x + 1) * U / gridDim.x;
  const double pi = 3.14159265358979323846;
  const double ik2 = P.reg.inv_k2;

  if (tid == 0) {
    mbar_init(&full[0], 1);
    mbar_init(&full[1], 1);
    mbar_fence_init();
  }
  if (tid < 20) skap[tid] = P.coef[tid];
  for (int i = tid; i < nq; i += NTC) sxq[i] = P.xq[i];
  for (int c = tid; c < (SYM ? nc / 2 : nc); c += NTC) {
    const int cn = SYM ? nc - 1 - c : c;   // SYM: pair c = (node c, node nc-1-c), weights of the positive node
    const double x = P.xc[cn], w = P.wc[cn];
    numbuf[4 * c] = w; numbuf[4 * c + 1] = w * x; numbuf[4 * c + 2] = w * x * x; numbuf[4 * c + 3] = w * x * x * x;
  }
  __syncthreads();

  // Stage of unit u into buffer b (S2 + the field-independent S3 remainder), by all threads of the CTA: the TMA
  // bulk copy of the unit's D0phi chunk, the fermion denominators, and beta'[j][n].  Called one unit ahead.
  auto produce = [&](const int e, const int i, int b) {   // unit (., e, i); the caller advances (ft, e, i) without divisions
    if (tid == 0) {
      mbar_expect_tx(&full[b], (uint32_t)cs * 8u);
      tma_bulk_g2s(d0buf + (size_t)b * cs, P.d0phi + ((size_t)e * nq + i) * cs, (uint32_t)cs * 8u, &full[b]);
    }
    if (tid < NPS) psibuf[b * NPS + tid] = P.psi[(size_t)(tid + P.n_max) * ps + i];   // rows n >= 0: nbar = n
    const double q = sxq[i];
    const double pq = P.pext[e] * q * ik2;
    double* bet = betabuf + (size_t)b * NB;
    for (int t = tid; t < NJ * NT; t += NTC) {
      const int j = t / NT, n = t - j * NT - NMAX;
      const int nbar = n >= 0 ? n : -n - 1;
      const double nun = (2.0 * n + 1.0) * pi * P.T, nuj = (2.0 * j + 1.0) * pi * P.T;
      const double y1 = nun * nuj * ik2;
      const double y3 = fma(nun, nun, __dmul_rn(q, q)) * ik2;   // (explicit: the same bits in every instantiation)
      // P = sum_b y2^b beta_b,  beta_b = sum_{a+c<=3-b} kap_abc y1^a y3^c   (idx: a outermost, then b, then c)
      double be[4] = {0.0, 0.0, 0.0, 0.0};
      int idx = 0;
      double y1a = 1.0;
#pragma unroll
      for (int a = 0; a <= 3; ++a) {
#pragma unroll
        for (int bb = 0; bb <= 3 - a; ++bb) {
          double y3c = y1a;
#pragma unroll
          for (int c = 0; c <= 3 - a - bb; ++c) {
            be[bb] = fma(skap[idx++], y3c, be[bb]);
            y3c *= y3;
          }
        }
        y1a *= y1;
      }
      const double W = P.psi[(size_t)(nbar + P.n_max) * ps + i].y;
      const double s1 = W * pq, s2 = s1 * pq, s3 = s2 * pq;
      bet[4 * t] = be[0] * W; bet[4 * t + 1] = be[1] * s1; bet[4 * t + 2] = be[2] * s2; bet[4 * t + 3] = be[3] * s3;
    }
  };

  const double4* num4 = reinterpret_cast<const double4*>(numbuf);
  double m2psi[MF], m2phi[MF], acc[NJ][MF];
  int cur_ft = -1;
  bool solo = false;   // this thread inverts every denominator on its own (mats3d_row_decouple)
  uint32_t g = 0;
  // unit u = (ft, e, i), decoded once (64-bit divisions cost ~100 instructions each) and advanced incrementally
  int ft_u = (int)(u0 / upp);
  int e_u = (int)((u0 - (long long)ft_u * upp) / nq);
  int i_u = (int)(u0 - (long long)ft_u * upp - (long long)e_u * nq);
  if (u0 < u1) produce(e_u, i_u, 0);
  __syncthreads();
  for (long long u = u0; u < u1; ++u, ++g) {
    const int ft = ft_u, e = e_u, i = i_u;
    if (++i_u == nq) { i_u = 0; if (++e_u == P.n_p) { e_u = 0; ++ft_u; } }   // (ft_u, e_u, i_u): unit u + 1
    const int f0 = ft * tile + tid;
    const int b = g & 1;
    if (u + 1 < u1) produce(e_u, i_u, b ^ 1);   // buffer b^1 was drained before the barrier that ended unit u-1
    if (ft != cur_ft) {
      cur_ft = ft;
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        const int f = f0 + k * NTC;
        m2psi[k] = (f < P.n_field) ? P.m2psi[f] : 1.0;
        m2phi[k] = (f < P.n_field) ? P.m2phi[f] : 1.0;
      }
      if constexpr (MF == 2)   // a padding lane beside a real field point: the real one's masses (its joint products are then its own)
        if (f0 + NTC >= P.n_field && f0 < P.n_field) { m2psi[1] = m2psi[0]; m2phi[1] = m2phi[0]; }
      if constexpr (MF == 2) solo = !(fabs(m2phi[0]) < M3_JOINT_MASS_MAX) || !(fabs(m2phi[1]) < M3_JOINT_MASS_MAX);
    }
    if (u == u0 || i == 0) {
#pragma unroll
      for (int j = 0; j < NJ; ++j)
#pragma unroll
        for (int k = 0; k < MF; ++k) acc[j][k] = 0.0;
    }
    mbar_wait(&full[b], (g >> 1) & 1);
    const double* d0 = d0buf + (size_t)b * cs;
    const double4* bet4 = reinterpret_cast<const double4*>(betabuf + (size_t)b * NB);
    const double2* psb = psibuf + b * NPS;

    double H[NPS][MF];
#pragma unroll
    for (int nb = 0; nb < NPS; ++nb) {
      const double D0 = psb[nb].x;
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        const double gp = fast_rcp(D0 + m2psi[k]);
        const double g2 = gp * gp;
        H[nb][k] = P.mode == 1 ? -2.0 * g2 * gp : g2;
      }
    }
    const bool pipelined = (nc % (2 * M3_NBAT)) == 0;
    const int l_last = NROWS * nc - M3_NBAT;
    double ra[M3_NBAT][MF], rb[M3_NBAT][MF];
    if (pipelined) mats3d_recip_batch<MF, SQ>(d0, m2phi, ra);
#pragma unroll 1
    for (int m = 0; m < NROWS; ++m) {
      // ---- angular moments of row m.  Written stage by stage over a batch of M3_NBAT nodes x MF field points so
      // that every stage holds independent instructions, and software-pipelined: the reciprocals of the next batch
      // (which may belong to the next row: the chunk is contiguous in [m][c]) are computed while the current batch
      // is accumulated.  With two warps per scheduler the FP64 pipe is fed by instruction-level parallelism. ----
      double M[4][MF];
#pragma unroll
      for (int k = 0; k < MF; ++k) { M[0][k] = 0.0; M[1][k] = 0.0; M[2][k] = 0.0; M[3][k] = 0.0; }
      // angular rules of 16, 24 (BASELINE config 4) and 32 nodes: the trips of the loop below unrolled at compile time (no
      // loop control per row, and the scheduler sees across the trips: cfg4 1.64 -> 1.60 ms)
      auto unrolled_row = [&](auto ncc) {
        constexpr int NCC = decltype(ncc)::value;
#pragma unroll
        for (int c = 0; c < NCC; c += 2 * M3_NBAT) {
          const int L = m * NCC + c;
          mats3d_recip_batch<MF, SQ>(d0 + L + M3_NBAT, m2phi, rb);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + c / 2, ra, M);
          else mats3d_moment_accumulate<MF>(num4 + c, ra, M);
          int Ln = L + 2 * M3_NBAT;
          Ln = Ln < l_last ? Ln : l_last;
          mats3d_recip_batch<MF, SQ>(d0 + Ln, m2phi, ra);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + (c + M3_NBAT) / 2, rb, M);
          else mats3d_moment_accumulate<MF>(num4 + c + M3_NBAT, rb, M);
        }
      };
      if (nc == 24) {
        unrolled_row(std::integral_constant<int, 24>{});
      } else if (nc == 16) {
        unrolled_row(std::integral_constant<int, 16>{});
      } else if (nc == 32) {
        unrolled_row(std::integral_constant<int, 32>{});
      } else if (pipelined) {
        // two batches per trip, the reciprocals ping-ponging between ra and rb (no register moves):
        //   ra = batch at c (ready), rb <- batch at c+4 while ra is accumulated, ra <- batch at c+8 while rb is ...
        for (int c = 0; c < nc; c += 2 * M3_NBAT) {
          const int L = m * nc + c;
          mats3d_recip_batch<MF, SQ>(d0 + L + M3_NBAT, m2phi, rb);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + c / 2, ra, M);
          else mats3d_moment_accumulate<MF>(num4 + c, ra, M);
          int Ln = L + 2 * M3_NBAT;
          Ln = Ln < l_last ? Ln : l_last;   // past the end of the chunk: recompute the last batch (result unused)
          mats3d_recip_batch<MF, SQ>(d0 + Ln, m2phi, ra);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + (c + M3_NBAT) / 2, rb, M);
          else mats3d_moment_accumulate<MF>(num4 + c + M3_NBAT, rb, M);
        }
      } else {
        const double* drow = d0 + m * nc;
#pragma unroll 1
        for (int c = 0; c < nc; ++c) {
          const double D0 = drow[c];
          const double4 w = num4[c];
#pragma unroll
          for (int k = 0; k < MF; ++k) {
            double r = fast_rcp(D0 + m2phi[k]);
            if constexpr (SQ) r = -(r * r);
            M[0][k] = fma(w.x, r, M[0][k]);
            M[1][k] = fma(w.y, r, M[1][k]);
            M[2][k] = fma(w.z, r, M[2][k]);
            M[3][k] = fma(w.w, r, M[3][k]);
          }
        }
      }
      if (pipelined) mats3d_row_decouple<MF, SQ, SYM>(d0 + m * nc, num4, nc, m2phi, M, solo);
      // ---- the (j, n) pairs with |j - n| = m: compile-time code per m (static register indices), reached through
      // a jump table so that the moment loop above exists once in the instruction stream ----
      switch (m) {
#define DFRG_M3_CASE(k) case k: if constexpr (k < NROWS) mats3d_pairs<(k < NROWS ? k : 0), NMAX, NJ, MF>(bet4, M, H, acc); break;
        DFRG_M3_CASE(0) DFRG_M3_CASE(1) DFRG_M3_CASE(2) DFRG_M3_CASE(3) DFRG_M3_CASE(4) DFRG_M3_CASE(5) DFRG_M3_CASE(6)
        DFRG_M3_CASE(7) DFRG_M3_CASE(8) DFRG_M3_CASE(9) DFRG_M3_CASE(10) DFRG_M3_CASE(11) DFRG_M3_CASE(12) DFRG_M3_CASE(13)
        DFRG_M3_CASE(14) DFRG_M3_CASE(15) DFRG_M3_CASE(16) DFRG_M3_CASE(17) DFRG_M3_CASE(18) DFRG_M3_CASE(19)
        DFRG_M3_CASE(20) DFRG_M3_CASE(21) DFRG_M3_CASE(22) DFRG_M3_CASE(23) DFRG_M3_CASE(24) DFRG_M3_CASE(25)
        DFRG_M3_CASE(26) DFRG_M3_CASE(27) DFRG_M3_CASE(28) DFRG_M3_CASE(29) DFRG_M3_CASE(30) DFRG_M3_CASE(31)
#undef DFRG_M3_CASE
        default: break;
      }
    }
    if (i == nq - 1 || u == u1 - 1) {
      // partial sum of this CTA for (field tile, p): slot = rank of this CTA among the owners of the p's units
      const long long ufirst = (long long)ft * upp + (long long)e * nq;
      const int c_first = (int)(((ufirst + 1) * gridDim.x - 1) / U);
      const int slot = (int)blockIdx.x - c_first;
#pragma unroll
      for (int j = 0; j < NJ; ++j)
#pragma unroll
        for (int k = 0; k < MF; ++k) {
          const int f = f0 + k * NTC;
          if (f < P.n_field)
            P.part[(((size_t)slot * P.n_p + e) * NJ + j) * P.n_field + f] = acc[j][k];
        }
    }
    __syncthreads();   // unit u is drained: its buffers may be refilled, and the stage of unit u+1 is complete
  }
}

// JB consecutive values of j of one side of row m:  acc[j0 + t] += H[nbar(n0 + t)] (beta'[j0 + t][n0 + t] . M),  written
// stage by stage (loads, then JB x MF independent chains).  b: first beta' entry, bstride between consecutive j; H: this
// thread's column, hstride between consecutive nbar.  j0 is a compile-time value at every call site (unrolled loops).
template <int JB, int MF, int NJ>
__device__ __forceinline__ void gm_pair_block(const double4* __restrict__ b, const int bstride,
                                              const double* __restrict__ H, const int hstride, const int n0,
                                              const double (&M)[4][MF], double (&acc)[NJ][MF], const int j0) {
  double4 B[JB];
  double h[JB][MF], t[JB][MF];
#pragma unroll
  for (int q = 0; q < JB; ++q) {
    B[q] = b[q * bstride];
    const int n = n0 + q, nbar = n >= 0 ? n : -n - 1;
#pragma unroll
    for (int k = 0; k < MF; ++k) h[q][k] = H[(size_t)nbar * hstride + k];
  }
#pragma unroll
  for (int q = 0; q < JB; ++q)
#pragma unroll
    for (int k = 0; k < MF; ++k) t[q][k] = B[q].x * M[0][k];
#pragma unroll
  for (int q = 0; q < JB; ++q)
#pragma unroll
    for (int k = 0; k < MF; ++k) t[q][k] = fma(B[q].y, M[1][k], t[q][k]);
#pragma unroll
  for (int q = 0; q < JB; ++q)
#pragma unroll
    for (int k = 0; k < MF; ++k) t[q][k] = fma(B[q].z, M[2][k], t[q][k]);
#pragma unroll
  for (int q = 0; q < JB; ++q)
#pragma unroll
    for (int k = 0; k < MF; ++k) t[q][k] = fma(B[q].w, M[3][k], t[q][k]);
#pragma unroll
  for (int q = 0; q < JB; ++q)
#pragma unroll
    for (int k = 0; k < MF; ++k) acc[j0 + q][k] = fma(h[q][k], t[q][k], acc[j0 + q][k]);
}

// ---- (3c) moment kernel for any (n_max, n_jext) ---------------------------------------------------------------
// The same factorisation, unit walk, staging and moment loop as mats3d_moment_kernel, with n_max a run-time value and
// n_jext <= NJ (NJ = 2, 4, 8, 16, 32 compiled).  The accumulators acc[j] stay in registers (the j loop is unrolled over
// NJ); what the specialised kernel indexes at compile time through its per-row jump table -- H[nbar] and beta'[j][n] --
// is read from shared memory here: H sits in a thread-private column Hs[nbar][tid] (no synchronisation needed), and the
// (j, n) pairs of row m are enumerated by two warp-uniform range tests per j
//     n = j - m:  max(0, m - n_max) <= j <= min(n_jext - 1, n_max + m);     n = j + m (m > 0):  j <= min(n_jext - 1, n_max - m).
// Cost against the specialised kernel: one LDS per pair and two uniform range tests per block of eight j.
template <int NJ, int MF, int NTC, bool SQ, bool SYM>
__global__ void __launch_bounds__(NTC, 1) mats3d_gmoment_kernel(const Mats3dParams P) {
  if (P.sym_try && (*P.symflag != 0) != SYM) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t full[2];
  __shared__ double skap[20];

  const int nq = P.nq, nc = P.nc, cs = P.chunk_stride, ps = P.psi_stride;
  const int n_max = P.n_max, n_jext = P.n_jext;
  const int NT = 2 * n_max + 1, NROWS = n_jext + n_max, NB = n_jext * NT * 4, NPS = n_max + 1;
  double* d0buf = reinterpret_cast<double*>(smem_raw);             // [2][cs]
  double* betabuf = d0buf + 2 * cs;                                // [2][NB]
  double2* psibuf = reinterpret_cast<double2*>(betabuf + 2 * NB);  // [2][NPS] (D0psi, Wpsi)
  double* numbuf = reinterpret_cast<double*>(psibuf + 2 * NPS);    // [nc][4]  wc c^b
  double* sxq = numbuf + 4 * nc;                                   // [nq]
  double* Hs = sxq + ((nq + 1) & ~1);                              // [NPS][NTC][MF]

  const int tid = threadIdx.x;
  const int tile = NTC * MF;
  const int n_ftiles = (P.n_field + tile - 1) / tile;
  const long long upp = (long long)P.n_p * nq;
  const long long U = (long long)n_ftiles * upp;
  const long long u0 = (long long)blockIdx.x * U / gridDim.x, u1 = (long long)(blockIdx.x + 1) * U / gridDim.x;
  const double pi = 3.14159265358979323846;
  const double ik2 = P.reg.inv_k2;

  if (tid == 0) {
    mbar_init(&full[0], 1);
    mbar_init(&full[1], 1);
    mbar_fence_init();
  }
  if (tid < 20) skap[tid] = P.coef[tid];
  for (int i = tid; i < nq; i += NTC) sxq[i] = P.xq[i];
  for (int c = tid; c < (SYM ? nc / 2 : nc); c += NTC) {
    const int cn = SYM ? nc - 1 - c : c;
    const double x = P.xc[cn], w = P.wc[cn];
    numbuf[4 * c] = w; numbuf[4 * c + 1] = w * x; numbuf[4 * c + 2] = w * x * x; numbuf[4 * c + 3] = w * x * x * x;
  }
  __syncthreads();

  auto produce = [&](const int e, const int i, int b) {   // unit (., e, i); the caller advances (ft, e, i) without divisions
    if (tid == 0) {
      mbar_expect_tx(&full[b], (uint32_t)cs * 8u);
      tma_bulk_g2s(d0buf + (size_t)b * cs, P.d0phi + ((size_t)e * nq + i) * cs, (uint32_t)cs * 8u, &full[b]);
    }
    for (int t = tid; t < NPS; t += NTC) psibuf[b * NPS + t] = P.psi[(size_t)(t + n_max) * ps + i];
    const double q = sxq[i];
    const double pq = P.pext[e] * q * ik2;
    double* bet = betabuf + (size_t)b * NB;
    for (int t = tid; t < n_jext * NT; t += NTC) {
      const int j = t / NT, n = t - j * NT - n_max;
      const int nbar = n >= 0 ? n : -n - 1;
      const double nun = (2.0 * n + 1.0) * pi * P.T, nuj = (2.0 * j + 1.0) * pi * P.T;
      const double y1 = nun * nuj * ik2;
      const double y3 = fma(nun, nun, __dmul_rn(q, q)) * ik2;   // (explicit: the same bits in every instantiation)
      double be[4] = {0.0, 0.0, 0.0, 0.0};
      int idx = 0;
      double y1a = 1.0;
#pragma unroll
      for (int a = 0; a <= 3; ++a) {
#pragma unroll
        for (int bb = 0; bb <= 3 - a; ++bb) {
          double y3c = y1a;
#pragma unroll
          for (int c = 0; c <= 3 - a - bb; ++c) {
            be[bb] = fma(skap[idx++], y3c, be[bb]);
            y3c *= y3;
          }
        }
        y1a *= y1;
      }
      const double W = P.psi[(size_t)(nbar + n_max) * ps + i].y;
      const double s1 = W * pq, s2 = s1 * pq, s3 = s2 * pq;
      bet[4 * t] = be[0] * W; bet[4 * t + 1] = be[1] * s1; bet[4 * t + 2] = be[2] * s2; bet[4 * t + 3] = be[3] * s3;
    }
  };

  const double4* num4 = reinterpret_cast<const double4*>(numbuf);
  double* myH = Hs + (size_t)tid * MF;
  double m2psi[MF], m2phi[MF], acc[NJ][MF];
  int cur_ft = -1;
  bool solo = false;   // this thread inverts every denominator on its own (mats3d_row_decouple)
  uint32_t g = 0;
  // unit u = (ft, e, i), decoded once (64-bit divisions cost ~100 instructions each) and advanced incrementally
  int ft_u = (int)(u0 / upp);
  int e_u = (int)((u0 - (long long)ft_u * upp) / nq);
  int i_u = (int)(u0 - (long long)ft_u * upp - (long long)e_u * nq);
  if (u0 < u1) produce(e_u, i_u, 0);
  __syncthreads();
  for (long long u = u0; u < u1; ++u, ++g) {
    const int ft = ft_u, e = e_u, i = i_u;
    if (++i_u == nq) { i_u = 0; if (++e_u == P.n_p) { e_u = 0; ++ft_u; } }   // (ft_u, e_u, i_u): unit u + 1
    const int f0 = ft * tile + tid;
    const int b = g & 1;
    if (u + 1 < u1) produce(e_u, i_u, b ^ 1);
    if (ft != cur_ft) {
      cur_ft = ft;
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        const int f = f0 + k * NTC;
        m2psi[k] = (f < P.n_field) ? P.m2psi[f] : 1.0;
        m2phi[k] = (f < P.n_field) ? P.m2phi[f] : 1.0;
      }
      if constexpr (MF == 2)   // a padding lane beside a real field point: the real one's masses (its joint products are then its own)
        if (f0 + NTC >= P.n_field && f0 < P.n_field) { m2psi[1] = m2psi[0]; m2phi[1] = m2phi[0]; }
      if constexpr (MF == 2) solo = !(fabs(m2phi[0]) < M3_JOINT_MASS_MAX) || !(fabs(m2phi[1]) < M3_JOINT_MASS_MAX);
    }
    if (u == u0 || i == 0) {
#pragma unroll
      for (int j = 0; j < NJ; ++j)
#pragma unroll
        for (int k = 0; k < MF; ++k) acc[j][k] = 0.0;
    }
    mbar_wait(&full[b], (g >> 1) & 1);
    const double* d0 = d0buf + (size_t)b * cs;
    const double4* bet4 = reinterpret_cast<const double4*>(betabuf + (size_t)b * NB);
    const double2* psb = psibuf + b * NPS;

    for (int nb = 0; nb < NPS; ++nb) {   // fermion line into this thread's column of Hs
      const double D0 = psb[nb].x;
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        const double gp = fast_rcp(D0 + m2psi[k]);
        const double g2 = gp * gp;
        myH[(size_t)nb * NTC * MF + k] = P.mode == 1 ? -2.0 * g2 * gp : g2;
      }
    }
    const bool pipelined = (nc % (2 * M3_NBAT)) == 0;
    const int l_last = NROWS * nc - M3_NBAT;
    double ra[M3_NBAT][MF], rb[M3_NBAT][MF];
    if (pipelined) mats3d_recip_batch<MF, SQ>(d0, m2phi, ra);
#pragma unroll 1
    for (int m = 0; m < NROWS; ++m) {
      double M[4][MF];
#pragma unroll
      for (int k = 0; k < MF; ++k) { M[0][k] = 0.0; M[1][k] = 0.0; M[2][k] = 0.0; M[3][k] = 0.0; }
      auto unrolled_row = [&](auto ncc) {   // as in mats3d_moment_kernel: 16, 24 and 32 angular nodes unrolled
        constexpr int NCC = decltype(ncc)::value;
#pragma unroll
        for (int c = 0; c < NCC; c += 2 * M3_NBAT) {
          const int L = m * NCC + c;
          mats3d_recip_batch<MF, SQ>(d0 + L + M3_NBAT, m2phi, rb);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + c / 2, ra, M);
          else mats3d_moment_accumulate<MF>(num4 + c, ra, M);
          int Ln = L + 2 * M3_NBAT;
          Ln = Ln < l_last ? Ln : l_last;
          mats3d_recip_batch<MF, SQ>(d0 + Ln, m2phi, ra);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + (c + M3_NBAT) / 2, rb, M);
          else mats3d_moment_accumulate<MF>(num4 + c + M3_NBAT, rb, M);
        }
      };
      if (nc == 24) {
        unrolled_row(std::integral_constant<int, 24>{});
      } else if (nc == 16) {
        unrolled_row(std::integral_constant<int, 16>{});
      } else if (nc == 32) {
        unrolled_row(std::integral_constant<int, 32>{});
      } else if (pipelined) {
        for (int c = 0; c < nc; c += 2 * M3_NBAT) {
          const int L = m * nc + c;
          mats3d_recip_batch<MF, SQ>(d0 + L + M3_NBAT, m2phi, rb);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + c / 2, ra, M);
          else mats3d_moment_accumulate<MF>(num4 + c, ra, M);
          int Ln = L + 2 * M3_NBAT;
          Ln = Ln < l_last ? Ln : l_last;
          mats3d_recip_batch<MF, SQ>(d0 + Ln, m2phi, ra);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + (c + M3_NBAT) / 2, rb, M);
          else mats3d_moment_accumulate<MF>(num4 + c + M3_NBAT, rb, M);
        }
      } else {
        const double* drow = d0 + m * nc;
#pragma unroll 1
        for (int c = 0; c < nc; ++c) {
          const double D0 = drow[c];
          const double4 w = num4[c];
#pragma unroll
          for (int k = 0; k < MF; ++k) {
            double r = fast_rcp(D0 + m2phi[k]);
            if constexpr (SQ) r = -(r * r);
            M[0][k] = fma(w.x, r, M[0][k]);
            M[1][k] = fma(w.y, r, M[1][k]);
            M[2][k] = fma(w.z, r, M[2][k]);
            M[3][k] = fma(w.w, r, M[3][k]);
          }
        }
      }
      if (pipelined) mats3d_row_decouple<MF, SQ, SYM>(d0 + m * nc, num4, nc, m2phi, M, solo);
      // ---- the (j, n) pairs with |j - n| = m ----
      const int jlo1 = max(0, m - n_max), jhi1 = min(n_jext - 1, n_max + m);
      const int jhi2 = m > 0 ? min(n_jext - 1, n_max - m) : -1;
      const double4* brow1 = bet4 + (n_max - m);   // entry (j, n = j - m) at brow1[j (NT + 1)]
      const double4* brow2 = bet4 + (n_max + m);   // entry (j, n = j + m) at brow2[j (NT + 1)]
      constexpr int JB = NJ < 8 ? NJ : 8;          // blocks of JB values of j: one range test per block when it is
#pragma unroll                                     // entirely inside the valid range (stage-wise code: JB x MF chains)
      for (int j0 = 0; j0 < NJ; j0 += JB) {
        if (j0 >= jlo1 && j0 + JB - 1 <= jhi1) {
          gm_pair_block<JB, MF, NJ>(brow1 + j0 * (NT + 1), NT + 1, myH, NTC * MF, j0 - m, M, acc, j0);
        } else if (j0 <= jhi1 && j0 + JB - 1 >= jlo1) {
#pragma unroll
          for (int jj = 0; jj < JB; ++jj)
            if (j0 + jj >= jlo1 && j0 + jj <= jhi1)
              gm_pair_block<1, MF, NJ>(brow1 + (j0 + jj) * (NT + 1), NT + 1, myH, NTC * MF, j0 + jj - m, M, acc, j0 + jj);
        }
        if (j0 + JB - 1 <= jhi2) {
          gm_pair_block<JB, MF, NJ>(brow2 + j0 * (NT + 1), NT + 1, myH, NTC * MF, j0 + m, M, acc, j0);
        } else if (j0 <= jhi2) {
#pragma unroll
          for (int jj = 0; jj < JB; ++jj)
            if (j0 + jj <= jhi2)
              gm_pair_block<1, MF, NJ>(brow2 + (j0 + jj) * (NT + 1), NT + 1, myH, NTC * MF, j0 + jj + m, M, acc, j0 + jj);
        }
      }
    }
    if (i == nq - 1 || u == u1 - 1) {
      const long long ufirst = (long long)ft * upp + (long long)e * nq;
      const int c_first = (int)(((ufirst + 1) * gridDim.x - 1) / U);
      const int slot = (int)blockIdx.x - c_first;
#pragma unroll
      for (int j = 0; j < NJ; ++j)
        if (j < n_jext) {
#pragma unroll
          for (int k = 0; k < MF; ++k) {
            const int f = f0 + k * NTC;
            if (f < P.n_field)
              P.part[(((size_t)slot * P.n_p + e) * n_jext + j) * P.n_field + f] = acc[j][k];
          }
        }
    }
    __syncthreads();
  }
}

// ---- (3d) moment kernel at finite chemical potential (complex fermion line) ------------------------------------
// mu != 0 (include/dfrg.h, dfrg_mats3d_desc::mu; reading A24): the boson line and hence the angular moments
// M_b stay real; the fermion line H = G_psi^2 and the polynomial coefficients beta'_b(j, n) are complex, and so are the
// accumulators.  Same unit walk, staging and moment loop as mats3d_gmoment_kernel (one field point per thread):
//   H[nbar] = 1/(D0re + m2 + i D0im)^2 per field point (thread-private shared-memory column; H(n < 0) = conj H(nbar)),
//   beta' = (re[4], im[4]) per (j, n) in shared memory,  t = beta' . M (8 FP64),  acc[j] += H t (4 FP64).
struct cplx_t { double re, im; };
// (explicit roundings: left to the compiler, the contraction of a*b + c*d differs between the instantiations of the kernel,
//  and the compile-time and run-time pair enumerations must agree bit for bit)
__device__ __forceinline__ cplx_t cmul(const cplx_t a, const cplx_t b) {
  cplx_t r;
  r.re = fma(a.re, b.re, -__dmul_rn(a.im, b.im));
  r.im = fma(a.re, b.im, __dmul_rn(a.im, b.re));
  return r;
}
// JB consecutive j of one side of row m, complex:  acc[j0+t] += H(n0+t) (beta'[j0+t][n0+t] . M), H(n < 0) = conj H(nbar);
// stage-wise (loads, then 2 JB independent chains).  b: first beta' entry (re, then im), bstride in double4 per j.
template <int JB, int NJ>
__device__ __forceinline__ void gm_cpair_block(const double4* __restrict__ b, const int bstride,
                                               const double* __restrict__ H, const int hstride, const int n0,
                                               const double (&M)[4][1], double (&accr)[NJ], double (&acci)[NJ],
                                               const int j0) {
  double4 Br[JB], Bi[JB];
  double hr[JB], hi[JB], tr[JB], ti[JB];
#pragma unroll
  for (int q = 0; q < JB; ++q) {
    Br[q] = b[q * bstride];
    Bi[q] = b[q * bstride + 1];
    const int n = n0 + q, nbar = n >= 0 ? n : -n - 1;
    hr[q] = H[(size_t)nbar * hstride];
    const double him = H[(size_t)nbar * hstride + 1];
    hi[q] = n >= 0 ? him : -him;
  }
#pragma unroll
  for (int q = 0; q < JB; ++q) { tr[q] = Br[q].x * M[0][0]; ti[q] = Bi[q].x * M[0][0]; }
#pragma unroll
  for (int q = 0; q < JB; ++q) { tr[q] = fma(Br[q].y, M[1][0], tr[q]); ti[q] = fma(Bi[q].y, M[1][0], ti[q]); }
#pragma unroll
  for (int q = 0; q < JB; ++q) { tr[q] = fma(Br[q].z, M[2][0], tr[q]); ti[q] = fma(Bi[q].z, M[2][0], ti[q]); }
#pragma unroll
  for (int q = 0; q < JB; ++q) { tr[q] = fma(Br[q].w, M[3][0], tr[q]); ti[q] = fma(Bi[q].w, M[3][0], ti[q]); }
#pragma unroll
  for (int q = 0; q < JB; ++q) {
    accr[j0 + q] = fma(hr[q], tr[q], fma(-hi[q], ti[q], accr[j0 + q]));
    acci[j0 + q] = fma(hr[q], ti[q], fma(hi[q], tr[q], acci[j0 + q]));
  }
}

// Row m of the complex pair section with (n_max, n_jext) = (NMAX, NJ) known at compile time: the valid (j, n) pairs are
// enumerated by the compiler (no range tests), as the jump-table pair code of the specialised real kernel.
template <int m, int NMAX, int NJ>
__device__ __forceinline__ void gm_cpairs_static(const double4* __restrict__ bet4, const double* __restrict__ H,
                                                 const int hstride, const double (&M)[4][1], double (&accr)[NJ],
                                                 double (&acci)[NJ]) {
  constexpr int NT = 2 * NMAX + 1;
#pragma unroll
  for (int j = 0; j < NJ; ++j) {
    const int n1 = j - m, n2 = j + m;
    if (n1 >= -NMAX && n1 <= NMAX) gm_cpair_block<1, NJ>(bet4 + 2 * (j * NT + n1 + NMAX), 0, H, hstride, n1, M, accr, acci, j);
    if (m > 0 && n2 <= NMAX) gm_cpair_block<1, NJ>(bet4 + 2 * (j * NT + n2 + NMAX), 0, H, hstride, n2, M, accr, acci, j);
  }
}

// NMAX_T >= 0: (n_max, n_jext) = (NMAX_T, NJ) exactly, pair code per row behind a jump table; NMAX_T < 0: any n_max, n_jext <= NJ.
template <int NJ, bool SYM, bool SQ, int NMAX_T = -1>
__global__ void __launch_bounds__(256, 1) mats3d_cmoment_kernel(const Mats3dParams P) {
  constexpr int NTC = 256, MF = 1;
  if (P.sym_try && (*P.symflag != 0) != SYM) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t full[2];
  __shared__ double skap[20];

  const int nq = P.nq, nc = P.nc, cs = P.chunk_stride, ps = P.psi_stride;
  const int n_max = P.n_max, n_jext = P.n_jext;
  const int NT = 2 * n_max + 1, NROWS = n_jext + n_max, NB = n_jext * NT * 8, NPS = n_max + 1;
  double* d0buf = reinterpret_cast<double*>(smem_raw);             // [2][cs]
  double* betabuf = d0buf + 2 * cs;                                // [2][NB]  (re[4], im[4]) per (j, n)
  double* psibuf = betabuf + 2 * NB;                               // [2][NPS][2] (Re D0psi, Im D0psi)
  double* numbuf = psibuf + 4 * NPS;                               // [nc][4]  wc c^b
  double* sxq = numbuf + 4 * nc;                                   // [nq]
  double* Hs = sxq + ((nq + 1) & ~1);                              // [NPS][NTC][2]

  const int tid = threadIdx.x;
  const int n_ftiles = (P.n_field + NTC - 1) / NTC;
  const long long upp = (long long)P.n_p * nq;
  const long long U = (long long)n_ftiles * upp;
  const long long u0 = (long long)blockIdx.x * U / gridDim.x, u1 = (long long)(blockIdx.x + 1) * U / gridDim.x;
  const double pi = 3.14159265358979323846;
  const double ik2 = P.reg.inv_k2;

  if (tid == 0) {
    mbar_init(&full[0], 1);
    mbar_init(&full[1], 1);
    mbar_fence_init();
  }
  if (tid < 20) skap[tid] = P.coef[tid];
  for (int i = tid; i < nq; i += NTC) sxq[i] = P.xq[i];
  for (int c = tid; c < (SYM ? nc / 2 : nc); c += NTC) {
    const int cn = SYM ? nc - 1 - c : c;
    const double x = P.xc[cn], w = P.wc[cn];
    numbuf[4 * c] = w; numbuf[4 * c + 1] = w * x; numbuf[4 * c + 2] = w * x * x; numbuf[4 * c + 3] = w * x * x * x;
  }
  __syncthreads();

  auto produce = [&](const int e, const int i, int b) {   // unit (., e, i); the caller advances (ft, e, i) without divisions
    if (tid == 0) {
      mbar_expect_tx(&full[b], (uint32_t)cs * 8u);
      tma_bulk_g2s(d0buf + (size_t)b * cs, P.d0phi + ((size_t)e * nq + i) * cs, (uint32_t)cs * 8u, &full[b]);
    }
    for (int t = tid; t < NPS; t += NTC) {
      const size_t at = (size_t)(t + n_max) * ps + i;
      psibuf[(b * NPS + t) * 2] = P.psi[at].x;
      psibuf[(b * NPS + t) * 2 + 1] = P.psi_im[at];
    }
    const double q = sxq[i];
    const double pq = P.pext[e] * q * ik2;
    double* bet = betabuf + (size_t)b * NB;
    for (int t = tid; t < n_jext * NT; t += NTC) {
      const int j = t / NT, n = t - j * NT - n_max;
      const int nbar = n >= 0 ? n : -n - 1;
      const double nun = (2.0 * n + 1.0) * pi * P.T, nuj = (2.0 * j + 1.0) * pi * P.T;
      cplx_t p0n, p0j, y1, y3;
      p0n.re = nun; p0n.im = P.mu; p0j.re = nuj; p0j.im = P.mu;
      y1 = cmul(p0n, p0j); y1.re *= ik2; y1.im *= ik2;
      y3 = cmul(p0n, p0n); y3.re = fma(q, q, y3.re) * ik2; y3.im *= ik2;
      // P = sum_b y2^b beta_b,  beta_b = sum_{a+c<=3-b} kap_abc y1^a y3^c   (idx: a outermost, then b, then c)
      cplx_t be[4];
#pragma unroll
      for (int bb = 0; bb < 4; ++bb) { be[bb].re = 0.0; be[bb].im = 0.0; }
      int idx = 0;
      cplx_t y1a; y1a.re = 1.0; y1a.im = 0.0;
#pragma unroll
      for (int a = 0; a <= 3; ++a) {
#pragma unroll
        for (int bb = 0; bb <= 3 - a; ++bb) {
          cplx_t y3c = y1a;
#pragma unroll
          for (int c = 0; c <= 3 - a - bb; ++c) {
            const double kap = skap[idx++];
            be[bb].re = fma(kap, y3c.re, be[bb].re);
            be[bb].im = fma(kap, y3c.im, be[bb].im);
            y3c = cmul(y3c, y3);
          }
        }
        y1a = cmul(y1a, y1);
      }
      const double W = P.psi[(size_t)(nbar + n_max) * ps + i].y;
      double sc = W;
#pragma unroll
      for (int bb = 0; bb < 4; ++bb) {
        bet[8 * t + bb] = be[bb].re * sc;
        bet[8 * t + 4 + bb] = be[bb].im * sc;
        sc *= pq;
      }
    }
  };

  const double4* num4 = reinterpret_cast<const double4*>(numbuf);
  double* myH = Hs + (size_t)tid * 2;
  double m2psi[MF], m2phi[MF], accr[NJ], acci[NJ];
  int cur_ft = -1;
  uint32_t g = 0;
  // unit u = (ft, e, i), decoded once (64-bit divisions cost ~100 instructions each) and advanced incrementally
  int ft_u = (int)(u0 / upp);
  int e_u = (int)((u0 - (long long)ft_u * upp) / nq);
  int i_u = (int)(u0 - (long long)ft_u * upp - (long long)e_u * nq);
  if (u0 < u1) produce(e_u, i_u, 0);
  __syncthreads();
  for (long long u = u0; u < u1; ++u, ++g) {
    const int ft = ft_u, e = e_u, i = i_u;
    if (++i_u == nq) { i_u = 0; if (++e_u == P.n_p) { e_u = 0; ++ft_u; } }   // (ft_u, e_u, i_u): unit u + 1
    const int f = ft * NTC + tid;
    const int b = g & 1;
    if (u + 1 < u1) produce(e_u, i_u, b ^ 1);
    if (ft != cur_ft) {
      cur_ft = ft;
      m2psi[0] = (f < P.n_field) ? P.m2psi[f] : 1.0;
      m2phi[0] = (f < P.n_field) ? P.m2phi[f] : 1.0;
    }
    if (u == u0 || i == 0) {
#pragma unroll
      for (int j = 0; j < NJ; ++j) { accr[j] = 0.0; acci[j] = 0.0; }
    }
    mbar_wait(&full[b], (g >> 1) & 1);
    const double* d0 = d0buf + (size_t)b * cs;
    const double4* bet4 = reinterpret_cast<const double4*>(betabuf + (size_t)b * NB);
    const double* psb = psibuf + (size_t)b * NPS * 2;

    for (int nb = 0; nb < NPS; ++nb) {   // H = G_psi^2, G_psi = conj(D)/|D|^2, D = a + i bb
      const double a = psb[2 * nb] + m2psi[0], bb = psb[2 * nb + 1];
      const double r = fast_rcp(fma(a, a, __dmul_rn(bb, bb)));
      const double gr = a * r, gi = -(bb * r);
      const double g2r = fma(gr, gr, -__dmul_rn(gi, gi)), g2i = 2.0 * gr * gi;
      if (P.mode == 1) {   // d/dm2_psi: G^2 -> -2 G^3
        myH[(size_t)nb * NTC * 2] = -2.0 * fma(g2r, gr, -__dmul_rn(g2i, gi));
        myH[(size_t)nb * NTC * 2 + 1] = -2.0 * fma(g2r, gi, __dmul_rn(g2i, gr));
      } else {
        myH[(size_t)nb * NTC * 2] = g2r;
        myH[(size_t)nb * NTC * 2 + 1] = g2i;
      }
    }
    const bool pipelined = (nc % (2 * M3_NBAT)) == 0;
    const int l_last = NROWS * nc - M3_NBAT;
    double ra[M3_NBAT][MF], rb[M3_NBAT][MF];
    if (pipelined) mats3d_recip_batch<MF, SQ>(d0, m2phi, ra);
#pragma unroll 1
    for (int m = 0; m < NROWS; ++m) {
      double M[4][MF];
      M[0][0] = 0.0; M[1][0] = 0.0; M[2][0] = 0.0; M[3][0] = 0.0;
      auto unrolled_row = [&](auto ncc) {   // as in mats3d_moment_kernel: 16, 24 and 32 angular nodes unrolled
        constexpr int NCC = decltype(ncc)::value;
#pragma unroll
        for (int c = 0; c < NCC; c += 2 * M3_NBAT) {
          const int L = m * NCC + c;
          mats3d_recip_batch<MF, SQ>(d0 + L + M3_NBAT, m2phi, rb);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + c / 2, ra, M);
          else mats3d_moment_accumulate<MF>(num4 + c, ra, M);
          int Ln = L + 2 * M3_NBAT;
          Ln = Ln < l_last ? Ln : l_last;
          mats3d_recip_batch<MF, SQ>(d0 + Ln, m2phi, ra);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + (c + M3_NBAT) / 2, rb, M);
          else mats3d_moment_accumulate<MF>(num4 + c + M3_NBAT, rb, M);
        }
      };
      if (nc == 24) {
        unrolled_row(std::integral_constant<int, 24>{});
      } else if (nc == 16) {
        unrolled_row(std::integral_constant<int, 16>{});
      } else if (nc == 32) {
        unrolled_row(std::integral_constant<int, 32>{});
      } else if (pipelined) {
        for (int c = 0; c < nc; c += 2 * M3_NBAT) {
          const int L = m * nc + c;
          mats3d_recip_batch<MF, SQ>(d0 + L + M3_NBAT, m2phi, rb);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + c / 2, ra, M);
          else mats3d_moment_accumulate<MF>(num4 + c, ra, M);
          int Ln = L + 2 * M3_NBAT;
          Ln = Ln < l_last ? Ln : l_last;
          mats3d_recip_batch<MF, SQ>(d0 + Ln, m2phi, ra);
          if constexpr (SYM) mats3d_moment_accumulate_sym<MF>(num4 + (c + M3_NBAT) / 2, rb, M);
          else mats3d_moment_accumulate<MF>(num4 + c + M3_NBAT, rb, M);
        }
      } else {
        const double* drow = d0 + m * nc;
#pragma unroll 1
        for (int c = 0; c < nc; ++c) {
          double r = fast_rcp(drow[c] + m2phi[0]);
          if constexpr (SQ) r = -(r * r);
          const double4 w = num4[c];
          M[0][0] = fma(w.x, r, M[0][0]);
          M[1][0] = fma(w.y, r, M[1][0]);
          M[2][0] = fma(w.z, r, M[2][0]);
          M[3][0] = fma(w.w, r, M[3][0]);
        }
      }
      // ---- the (j, n) pairs with |j - n| = m ----
      if constexpr (NMAX_T >= 0) {
        switch (m) {
#define DFRG_M3C_CASE(k) case k: if constexpr (k < NJ + NMAX_T) gm_cpairs_static<(k < NJ + NMAX_T ? k : 0), NMAX_T, NJ>(bet4, myH, NTC * 2, M, accr, acci); break;
          DFRG_M3C_CASE(0) DFRG_M3C_CASE(1) DFRG_M3C_CASE(2) DFRG_M3C_CASE(3) DFRG_M3C_CASE(4) DFRG_M3C_CASE(5) DFRG_M3C_CASE(6)
          DFRG_M3C_CASE(7) DFRG_M3C_CASE(8) DFRG_M3C_CASE(9) DFRG_M3C_CASE(10) DFRG_M3C_CASE(11) DFRG_M3C_CASE(12)
          DFRG_M3C_CASE(13) DFRG_M3C_CASE(14) DFRG_M3C_CASE(15) DFRG_M3C_CASE(16) DFRG_M3C_CASE(17) DFRG_M3C_CASE(18)
          DFRG_M3C_CASE(19) DFRG_M3C_CASE(20) DFRG_M3C_CASE(21) DFRG_M3C_CASE(22) DFRG_M3C_CASE(23) DFRG_M3C_CASE(24)
          DFRG_M3C_CASE(25) DFRG_M3C_CASE(26) DFRG_M3C_CASE(27) DFRG_M3C_CASE(28) DFRG_M3C_CASE(29) DFRG_M3C_CASE(30)
          DFRG_M3C_CASE(31)
#undef DFRG_M3C_CASE
          default: break;
        }
      } else {
      const int jlo1 = max(0, m - n_max), jhi1 = min(n_jext - 1, n_max + m);
      const int jhi2 = m > 0 ? min(n_jext - 1, n_max - m) : -1;
      const double4* brow1 = bet4 + 2 * (n_max - m);   // entry (j, n = j - m) at brow1[2 j (NT + 1)] (re), +1 (im)
      const double4* brow2 = bet4 + 2 * (n_max + m);
      constexpr int JB = NJ < 8 ? NJ : 8;
#pragma unroll
      for (int j0 = 0; j0 < NJ; j0 += JB) {
        if (j0 >= jlo1 && j0 + JB - 1 <= jhi1) {
          gm_cpair_block<JB, NJ>(brow1 + 2 * j0 * (NT + 1), 2 * (NT + 1), myH, NTC * 2, j0 - m, M, accr, acci, j0);
        } else if (j0 <= jhi1 && j0 + JB - 1 >= jlo1) {
#pragma unroll
          for (int jj = 0; jj < JB; ++jj)
            if (j0 + jj >= jlo1 && j0 + jj <= jhi1)
              gm_cpair_block<1, NJ>(brow1 + 2 * (j0 + jj) * (NT + 1), 2 * (NT + 1), myH, NTC * 2, j0 + jj - m, M, accr, acci,
                                    j0 + jj);
        }
        if (j0 + JB - 1 <= jhi2) {
          gm_cpair_block<JB, NJ>(brow2 + 2 * j0 * (NT + 1), 2 * (NT + 1), myH, NTC * 2, j0 + m, M, accr, acci, j0);
        } else if (j0 <= jhi2) {
#pragma unroll
          for (int jj = 0; jj < JB; ++jj)
            if (j0 + jj <= jhi2)
              gm_cpair_block<1, NJ>(brow2 + 2 * (j0 + jj) * (NT + 1), 2 * (NT + 1), myH, NTC * 2, j0 + jj + m, M, accr, acci,
                                    j0 + jj);
        }
      }
          }
    }
    if (i == nq - 1 || u == u1 - 1) {
      const long long ufirst = (long long)ft * upp + (long long)e * nq;
      const int c_first = (int)(((ufirst + 1) * gridDim.x - 1) / U);
      const int slot = (int)blockIdx.x - c_first;
      if (f < P.n_field) {
#pragma unroll
        for (int j = 0; j < NJ; ++j)
          if (j < n_jext) {
            const size_t at = (((size_t)slot * P.n_p + e) * n_jext + j) * P.n_field + f;
            P.part[at] = accr[j];
            P.part_im[at] = acci[j];
          }
      }
    }
    __syncthreads();
  }
}

// mu != 0: min over (n >= 0, q) of |D0psi + m2psi_f| per field point (the rows n < 0 are the complex conjugates).
static __global__ void __launch_bounds__(128) mats3d_psimin_cplx_kernel(const Mats3dParams P) {
  const int f = blockIdx.x * 128 + threadIdx.x;
  if (f >= P.n_field) return;
  const double m2 = P.m2psi[f];
  double best = __longlong_as_double(0x7ff0000000000000LL);
  for (int nb = 0; nb <= P.n_max; ++nb)
    for (int i = 0; i < P.nq; ++i) {
      const size_t at = (size_t)(nb + P.n_max) * P.psi_stride + i;
      const double a = P.psi[at].x + m2, b = P.psi_im[at];
      best = fmin(best, fma(a, a, b * b));
    }
  P.psimin_f[f] = sqrt(best);
}

// S5/S6 of the moment path: out = prefactor T sum_slots part, dmin from the row minima.
static __global__ void __launch_bounds__(256) mats3d_fixup_kernel(const Mats3dParams P) {
  const long long idx = (long long)blockIdx.x * 256 + threadIdx.x;
  const long long n_out = (long long)P.n_p * P.n_jext * P.n_field;
  if (idx >= n_out) return;
  const int f = (int)(idx % P.n_field);
  const long long ej = idx / P.n_field;
  const int e = (int)(ej / P.n_jext), j = (int)(ej - (long long)e * P.n_jext);
  const int n_ftiles = (P.n_field + P.tile_fields - 1) / P.tile_fields;
  const long long upp = (long long)P.n_p * P.nq, U = (long long)n_ftiles * upp;
  const long long ufirst = (long long)(f / P.tile_fields) * upp + (long long)e * P.nq, ulast = ufirst + P.nq - 1;
  const int c_first = (int)(((ufirst + 1) * P.grid_main - 1) / U), c_last = (int)(((ulast + 1) * P.grid_main - 1) / U);
  const size_t stride = (size_t)P.n_p * P.n_jext * P.n_field;
  CompSum r(P.part[idx]);
  for (int s = 1; s <= c_last - c_first; ++s) r.add(P.part[(size_t)s * stride + idx]);
  P.out[idx] = P.prefactor * P.T * r.value();
  if (P.out_im) {
    double ri = 0.0;
    if (P.part_im) {
      CompSum ci(P.part_im[idx]);
      for (int s = 1; s <= c_last - c_first; ++s) ci.add(P.part_im[(size_t)s * stride + idx]);
      ri = ci.value();
    }
    P.out_im[idx] = P.prefactor * P.T * ri;
  }
  if (P.dmin && P.psimin_f) {   // complex fermion line: |D_psi| does not split into (min D0) + m2
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    double dphi = inf;
    for (int it = 0; it < 2 * P.n_max + 1; ++it) {
      const int mm = j - (it - P.n_max), mabs = mm >= 0 ? mm : -mm;
      dphi = fmin(dphi, P.rowmin[(size_t)e * P.n_rows + mabs]);
    }
    P.dmin[idx] = fmin(P.psimin_f[f], dphi + P.m2phi[f]) * P.reg.inv_k2;
  } else if (P.dmin) {
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    double dpsi = inf, dphi = inf;
    for (int it = 0; it < 2 * P.n_max + 1; ++it) {
      const int mm = j - (it - P.n_max), mabs = mm >= 0 ? mm : -mm;
      dpsi = fmin(dpsi, P.psimin[it]);
      dphi = fmin(dphi, P.rowmin[(size_t)e * P.n_rows + mabs]);
    }
    P.dmin[idx] = fmin(dpsi + P.m2psi[f], dphi + P.m2phi[f]) * P.reg.inv_k2;
  }
}



// X(NMAX, NJ) for every specialised instantiation of mats3d_moment_kernel: BASELINE.json config 4 and one small shape
// that keeps the specialised kernel under the test-suite's small cases.
#define DFRG_M3_SHAPES(X) X(11, 16) X(3, 3)

struct MomentPlan {
  int variant;     // 0: MF 2 x 256 threads, 2: MF 1 x 256 threads
  int tile, grid, max_slots;
  size_t smem;
  bool generic;    // mats3d_gmoment_kernel (any n_max, n_jext <= 32) instead of a specialised instantiation
  bool any_shape_forced;   // dfrg_mats3d_desc::path & DFRG_M3_ANY_SHAPE: no compile-time-enumerated instantiation
};

}  // namespace dfrg
