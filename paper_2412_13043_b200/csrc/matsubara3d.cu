// matsubara3d.cu -- dfrg_integrate_matsubara3d: 3-D spatial loop + Matsubara sum (BASELINE.json config 4).
//
// Three launches per call, all on the caller's stream:
//
//  (1) mats3d_phi_rows_kernel  (S3, field independent, once per call)
//        D0phi[p][m][i][c] = Z_phi(r^2; row m) s_phi + R(s_phi),  m = 0 .. n_jext-1+n_max
//      The boson denominator depends on the external and loop Matsubara indices only through
//      |j - n|, so the 16 x 23 (j, n) combinations of config 4 share 27 rows per momentum p.
//      Rows go to a stream-ordered scratch buffer (31 MB for config 4: L2 resident) together with
//      their minima (for dmin).
//  (2) mats3d_psi_kernel       (S3, once per call)
//        psi[n][i] = (D0psi, Wpsi) = (Z_psi(q_i^2; row nbar) s_psi + R(s_psi),  wq_i q_i^2 Rdot(s_psi))
//  (3) mats3d_main_kernel      (S2 + S3 remainder + S4 + S5 + S6): persistent, one CTA per SM, warp-specialised
//      (see the comment at the kernel).  Row |j-n| of D0phi and row n of psi arrive by TMA bulk copy into a
//      double-buffered shared-memory stage; a producer warp builds the numerator row Nw[i][c] = wc_c P(y1, y2, y3)
//      (P as a cubic in y2 = p q c/k^2 by Horner, its four coefficients depending on (n, i) only).  Hot loop:
//      thread = MF field points; per node  d_f = D0 + m2phi_f;  two-way batched inversion
//      r = 1/(d_a d_b), 1/d_a = r d_b, 1/d_b = r d_a  (one MUFU.RCP64H seed + cubic Newton step per two
//      evaluations: 10 FP64 instructions per two evaluations, the same as two separate reciprocals, but
//      half the load on the XU pipe);  a_f += Nw / d_f  on two accumulators per field point.
//      Every lane of a warp reads the same table entries (shared-memory broadcast).
//      Then acc_f += Wpsi G_psi(f)^2 a_f.
// dmin: fl(D0 + m2) is monotone in D0, so the minimum over nodes is (min D0) + m2: no hot-loop work.
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
  int mode;          // 0: value;  1: d/dm2_psi (G_psi^2 -> -2 G_psi^3);  2: d/dm2_phi (G_phi -> -G_phi^2, kernels with SQ)
};

// ---- (1) boson rows --------------------------------------------------------------------------------
__global__ void __launch_bounds__(M3_PRE_THREADS) mats3d_phi_rows_kernel(const Mats3dParams P) {
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
    regulator(P.reg, fm, sphi, R, Rd);
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
__global__ void __launch_bounds__(128) mats3d_psi_kernel(const Mats3dParams P) {
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
    const double spsi = nun * nun + q * q;
    double R, Rd;
    regulator(P.reg, fm, spsi, R, Rd);
    const double D0 = table_lookup(cells, P.grid, fm, q * q) * spsi + R;
    P.psi[(size_t)it * P.psi_stride + i] = make_double2(D0, P.wq[i] * q * q * Rd);
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
          const double y3 = (nun * nun + q * q) * ik2;
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
    double pr[M3_NBAT], R[M3_NBAT];
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t) pr[t] = d[t][0] * d[t][1];
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t) R[t] = rcp_seed(pr[t]);
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t) pr[t] = fma(-pr[t], R[t], 1.0);
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t) pr[t] = fma(pr[t], pr[t], pr[t]);
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t) R[t] = fma(R[t], pr[t], R[t]);
#pragma unroll
    for (int t = 0; t < M3_NBAT; ++t) { r[t][0] = R[t] * d[t][1]; r[t][1] = R[t] * d[t][0]; }
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
  auto produce = [&](long long u, int b) {
    const long long rem = u % upp;
    const int e = (int)(rem / nq), i = (int)(rem - (long long)e * nq);
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
      const double y3 = (nun * nun + q * q) * ik2;
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
  uint32_t g = 0;
  if (u0 < u1) produce(u0, 0);
  __syncthreads();
  for (long long u = u0; u < u1; ++u, ++g) {
    const int ft = (int)(u / upp);
    const long long rem = u - (long long)ft * upp;
    const int e = (int)(rem / nq), i = (int)(rem - (long long)e * nq);
    const int f0 = ft * tile + tid;
    const int b = g & 1;
    if (u + 1 < u1) produce(u + 1, b ^ 1);   // buffer b^1 was drained before the barrier that ended unit u-1
    if (ft != cur_ft) {
      cur_ft = ft;
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        const int f = f0 + k * NTC;
        m2psi[k] = (f < P.n_field) ? P.m2psi[f] : 1.0;
        m2phi[k] = (f < P.n_field) ? P.m2phi[f] : 1.0;
      }
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
      if (pipelined) {
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

// S5/S6 of the moment path: out = prefactor T sum_slots part, dmin from the row minima.
__global__ void __launch_bounds__(256) mats3d_fixup_kernel(const Mats3dParams P) {
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
  double r = P.part[idx];
  for (int s = 1; s <= c_last - c_first; ++s) r += P.part[(size_t)s * stride + idx];
  P.out[idx] = P.prefactor * P.T * r;
  if (P.dmin) {
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
  return DFRG_OK;
}

template <int GROUPS, int MF>
static int mats3d_launch_main(const Mats3dParams& P, int sm_count, cudaStream_t stream) {
  const size_t smem = mats3d_main_smem(P.nq, P.nc, P.row_stride, P.psi_stride, GROUPS, MF);
  if (smem > 227 * 1024) return DFRG_EUNSUPPORTED;
  auto kern = P.mode == 2 ? mats3d_main_kernel<GROUPS, MF, true> : mats3d_main_kernel<GROUPS, MF, false>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return check_cuda(e);
  const long long n_ftiles = (P.n_field + M3_FT * MF - 1) / (M3_FT * MF);
  const long long n_items = (long long)P.n_p * P.n_jext * n_ftiles;
  const int grid = (int)(n_items < sm_count ? n_items : sm_count);
  kern<<<grid, GROUPS * M3_FT + 32, smem, stream>>>(P);
  return check_cuda(cudaGetLastError());
}

// ---- moment-path dispatch: (n_max, n_jext) pairs with a compiled instantiation ---------------------------
struct MomentPlan {
  int variant;     // 0: MF 2 x 256 threads, 1: MF 1 x 512 threads, 2: MF 1 x 256 threads
  int tile, grid, max_slots;
  size_t smem;
};

template <int NMAX, int NJ, bool SYM>
static int mats3d_moment_go(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream) {
  cudaError_t e;
#define DFRG_M3_GO(MF, NTC)                                                                                          \
  {                                                                                                                  \
    auto kern = P.mode == 2 ? mats3d_moment_kernel<NMAX, NJ, MF, NTC, true, SYM>                                     \
                            : mats3d_moment_kernel<NMAX, NJ, MF, NTC, false, SYM>;                                   \
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);                       \
    if (e != cudaSuccess) return check_cuda(e);                                                                      \
    kern<<<pl.grid, NTC, pl.smem, stream>>>(P);                                                                      \
  }
  if (pl.variant == 0) { DFRG_M3_GO(2, 256) }
  else if (pl.variant == 1) { DFRG_M3_GO(1, 512) }
  else { DFRG_M3_GO(1, 256) }
#undef DFRG_M3_GO
  return check_cuda(cudaGetLastError());
}

// X(NMAX, NJ) for every compiled instantiation: BASELINE.json config 4 and the small shapes of the test-suite.
#ifdef DFRG_M3_ONLY_CFG4  // faster builds while tuning
#define DFRG_M3_SHAPES(X) X(11, 16)
#else
#define DFRG_M3_SHAPES(X) X(11, 16) X(11, 2) X(3, 3) X(2, 2)
#endif

static bool mats3d_moment_shape(int n_max, int n_jext) {
#define X(a, b) if (n_max == a && n_jext == b) return true;
  DFRG_M3_SHAPES(X)
#undef X
  return false;
}
static int mats3d_moment_dispatch(Mats3dParams& P, const MomentPlan& pl, cudaStream_t stream) {
  // symmetric-pair instantiation first (runs iff the pre-pass found the cos rule symmetric), then the plain one
#define X(a, b)                                                                    \
  if (P.n_max == a && P.n_jext == b) {                                             \
    if (P.sym_try) {                                                               \
      const int rc = mats3d_moment_go<a, b, true>(P, pl, stream);                  \
      if (rc != DFRG_OK) return rc;                                                \
    }                                                                              \
    return mats3d_moment_go<a, b, false>(P, pl, stream);                           \
  }
  DFRG_M3_SHAPES(X)
#undef X
  return DFRG_EUNSUPPORTED;
}

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

  // ---- path: moment factorisation where an instantiation exists (DFRG_M3_PATH=generic forces the other one) ----
  const char* vpath = getenv("DFRG_M3_PATH");
  bool moment = mats3d_moment_shape(D->n_max, n_jext) && !(vpath && vpath[0] == 'g');
  MomentPlan pl = {};
  if (moment) {
    const char* vm = getenv("DFRG_M3_MF");
    pl.variant = n_field <= 256 ? 2 : ((vm && atoi(vm) == 1) ? 1 : 0);
    pl.tile = pl.variant == 0 ? 512 : (pl.variant == 1 ? 512 : 256);
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
    if (pl.smem > 220 * 1024) moment = false;
  }
  P.phi_layout = moment ? 1 : 0;
  {
    const char* vs = getenv("DFRG_M3_SYM");
    P.sym_try = (moment && (P.nc % (2 * M3_NBAT)) == 0 && !(vs && vs[0] == '0')) ? 1 : 0;
  }
  P.tile_fields = pl.tile; P.max_slots = pl.max_slots; P.grid_main = pl.grid;

  const int n_terms = 2 * D->n_max + 1;
  const size_t n_d0 = moment ? (size_t)n_p * P.nq * P.chunk_stride : (size_t)n_p * P.n_rows * P.row_stride;
  const size_t n_rowmin = ((size_t)n_p * P.n_rows + 1) & ~(size_t)1;
  const size_t n_psi = (size_t)n_terms * P.psi_stride * 2;
  const size_t n_psimin = ((size_t)n_terms + 1) & ~(size_t)1;
  const size_t n_part = moment ? (size_t)pl.max_slots * n_p * n_jext * n_field : 0;
  void* scratch = nullptr;
  int rc = scratch_alloc(&scratch, (n_d0 + n_rowmin + n_psi + n_psimin + n_part + 2) * sizeof(double), stream);
  if (rc != DFRG_OK) return rc;
  P.d0phi = (double*)scratch;
  P.psi = (double2*)(P.d0phi + n_d0);
  P.rowmin = (double*)(P.psi) + n_psi;
  P.psimin = P.rowmin + n_rowmin;
  P.part = P.psimin + n_psimin;
  P.symflag = (int*)(P.part + n_part);

  mats3d_phi_rows_kernel<<<dim3(P.n_rows, n_p), M3_PRE_THREADS, 0, stream>>>(P);
  rc = check_cuda(cudaGetLastError());
  if (rc == DFRG_OK) {
    mats3d_psi_kernel<<<n_terms, 128, 0, stream>>>(P);
    rc = check_cuda(cudaGetLastError());
  }
  // one pass for the values, one more for each requested mass derivative (same kernels, mode 1 / 2)
  double* const pass_out[3] = {out, D->dout_dm2_psi, D->dout_dm2_phi};
  for (int mode = 0; mode < 3 && rc == DFRG_OK; ++mode) {
    if (!pass_out[mode]) continue;
    P.mode = mode;
    P.out = pass_out[mode];
    P.dmin = mode == 0 ? dmin : nullptr;
    if (moment) {
      rc = mats3d_moment_dispatch(P, pl, stream);
      if (rc == DFRG_OK) {
        const long long n_out = (long long)n_p * n_jext * n_field;
        mats3d_fixup_kernel<<<(unsigned)((n_out + 255) / 256), 256, 0, stream>>>(P);
        rc = check_cuda(cudaGetLastError());
      }
    } else {
      // generic path: consumer groups per CTA (radial nodes are dealt round-robin to the groups) and field points per
      // thread; DFRG_M3_GROUPS / DFRG_M3_MF override the defaults (tuning knobs)
      const char* vg = getenv("DFRG_M3_GROUPS");
      const char* vm = getenv("DFRG_M3_MF");
      int mf = n_field > 2 * M3_FT ? 4 : (n_field > M3_FT ? 2 : 1);
      if (vm && atoi(vm) >= 1 && atoi(vm) < mf) mf = atoi(vm) == 3 ? 2 : atoi(vm);
      const int groups = vg ? atoi(vg) : 6;
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
  const size_t need = 2 * ((size_t)D->q.n + D->cos1.n) + (rows_psi + rows_phi) * nt + 20 + 2 * nf + n_p + 4 * n_out;
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
  if (A.status() != DFRG_OK) return A.status();
  rc = mats3d_launch(&Dd, n_field, d_mpsi, d_mphi, n_p, d_p, n_jext, d_out, d_dmin, sms, A.stream());
  if (rc != DFRG_OK) return rc;
  A.fetch(out, d_out, n_out);
  if (dmin) A.fetch(dmin, d_dmin, n_out);
  if (D->dout_dm2_psi) A.fetch(D->dout_dm2_psi, Dd.dout_dm2_psi, n_out);
  if (D->dout_dm2_phi) A.fetch(D->dout_dm2_phi, Dd.dout_dm2_phi, n_out);
  return A.finish();
}
