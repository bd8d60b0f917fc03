// loop4d_twopoint.cu -- two-point family of dfrg_integrate_loop4d (BASELINE.json config 2).
#include <mutex>
#include <type_traits>

#include "loop4d_kernels.cuh"

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
  long long u0, u1;
  if ((long long)gridDim.x * U < (1ll << 32)) {   // (32-bit divisions where they suffice: ~300 cycles each otherwise)
    u0 = (unsigned)(blockIdx.x * (unsigned)U) / gridDim.x;
    u1 = (unsigned)((blockIdx.x + 1) * (unsigned)U) / gridDim.x;
  } else {
    u0 = (long long)blockIdx.x * U / gridDim.x;
    u1 = (long long)(blockIdx.x + 1) * U / gridDim.x;
  }

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
  const FastMath fm = fm_stage(L, fmmem, P.fmc);   // the constant log/exp tables travel with the inputs
  const double coef0 = P.coef[0], coef1 = P.coef[1];   // (producers; loaded here so that the latency hides behind the staging)
  stage_issue(L, &bar);
  stage_wait(&bar, 0);
  cells_build(cZ, sZ, P.grid);
  for (int j = tid; j < nc; j += TP_THREADS) {
    const double c = sxc[j];
    swc[j] *= sqrt((1.0 - c) * (1.0 + c));
  }
  __syncthreads();   // the producers start on their first chunk from here; the consumers build souter meanwhile
  const double inf = __longlong_as_double(0x7ff0000000000000LL);
  // unit u = (ft, e, ch); advanced without divisions
  int ft_u, e_u, ch_u;
  if (U < (1ll << 31)) {   // (32-bit divisions: the 64-bit ones cost ~1000 cycles at the head of every CTA)
    const unsigned v = (unsigned)u0, uppu = (unsigned)upp;
    ft_u = (int)(v / uppu);
    const unsigned rem = v - (unsigned)ft_u * uppu;
    e_u = (int)(rem / (unsigned)NCH);
    ch_u = (int)(rem - (unsigned)e_u * (unsigned)NCH);
  } else {
    ft_u = (int)(u0 / upp);
    e_u = (int)((u0 - (long long)ft_u * upp) / NCH);
    ch_u = (int)(u0 - (long long)ft_u * upp - (long long)e_u * NCH);
  }
  auto next_unit = [&]() {
    if (++ch_u == NCH) { ch_u = 0; if (++e_u == P.n_ext) { e_u = 0; ++ft_u; } }
  };

  if (tid >= TP_NCONS) {
    // =========================== producers ===========================
    const int ptid = tid - TP_NCONS, lane = ptid & 31, pw = ptid >> 5;
    uint32_t g = 0;
    for (long long u = u0; u < u1; ++u, ++g, next_unit()) {
      const int b = g & 1;
      const int e = e_u, ch = ch_u;
      const int i0 = ch * QC;
      const int ni = min(QC, nq - i0);
      const double p = P.pext[e];
      mbar_wait(&empty[b], ((g >> 1) & 1) ^ 1);   // consumers drained this stage (passes at once for g < 2)
      double2* dst = buf + (size_t)b * chunk_nodes;
      double dmin0 = inf;
      for (int t = ptid; t < ni * nc; t += TP_NPROD) {
        const int il = t / nc, j = t - il * nc;
        const double q = sxq[i0 + il], c = sxc[j];
        // (explicit FMAs: left to the compiler, the contraction of a*b + c may differ between the template instantiations
        //  of this kernel, and the values must not depend on whether derivatives were asked for)
        const double qpc = q * p * c;
        double s = fma(2.0, qpc, fma(q, q, p * p));
        s = clamp_lo(s, 0.0);
        double R, Rd;
        regulator(P.reg, fm, s, R, Rd);
        const double D0 = fma(table_lookup(cZ, P.grid, fm, s), s, R);
        const double poly = fma(coef1, qpc * P.reg.inv_k2, coef0);
        dst[t] = make_double2(D0, swc[j] * poly);
        dmin0 = fmin(dmin0, D0);
      }
      dmin0 = warp_min(dmin0);
      __syncwarp();           // every lane's stores to the chunk precede lane 0's release-arrive below
      if (lane == 0) {
        P.chunkmin[(size_t)(u * (TP_NPROD / 32)) + pw] = dmin0;
        mbar_arrive(&full[b]);  // release: the chunk is visible to whoever acquires full[b]
      }
    }
    return;
  }

  // =============================== consumers ===============================
  {
    // outer[i] = (Z(q^2) q^2 + R(q^2), wq q^3 Rdot(q^2)) and its minimum (for dmin), by the consumers while the
    // producers are on the first chunk; published among the consumers by a named barrier
    double dq = inf;
    for (int i = tid; i < nq; i += TP_NCONS) {
      const double q = sxq[i], s = q * q;
      double R, Rd;
      regulator(P.reg, fm, s, R, Rd);
      const double D0 = fma(table_lookup(cZ, P.grid, fm, s), s, R);
      souter[i] = make_double2(D0, swq[i] * q * q * q * Rd);
      dq = fmin(dq, D0);
    }
    dq = warp_min(dq);
    if ((tid & 31) == 0) red[tid >> 5] = dq;
    named_bar_sync(1, TP_NCONS);
    if (blockIdx.x == 0 && tid == 0) {
      for (int w = 1; w < TP_NCONS / 32; ++w) dq = fmin(dq, red[w]);
      P.chunkmin[(size_t)n_ftiles * P.n_ext * NCH * (TP_NPROD / 32)] = dq;
    }
  }
  const int grp = tid / TP_FT, tf = tid - grp * TP_FT;
  const bool warp_leader = (tid & 31) == 0;
  double m2[MF], acc[MF], dacc[MF];
  int cur_ft = -1, seg_parity = 0;
  bool solo = false;   // this thread inverts every denominator on its own (close_row)
  uint32_t g = 0;
  for (long long u = u0; u < u1; ++u, ++g, next_unit()) {
    const int ft = ft_u, e = e_u, ch = ch_u;
    const int f0 = ft * tile + tf;
    const int b = g & 1;
    if (ft != cur_ft) {
      cur_ft = ft;
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        const int f = f0 + k * TP_FT;
        m2[k] = (f < P.n_field) ? P.m2[f] : 1.0;
      }
      if constexpr (MF == 2)   // a padding lane beside a real field point: the real one's mass (its joint products are then its own)
        if (f0 + TP_FT >= P.n_field && f0 < P.n_field) m2[1] = m2[0];
      if constexpr (MF == 2) solo = !(fabs(m2[0]) < TP_JOINT_MASS_MAX) || !(fabs(m2[1]) < TP_JOINT_MASS_MAX);
    }
    if (u == u0 || ch == 0) {
#pragma unroll
      for (int k = 0; k < MF; ++k) { acc[k] = 0.0; dacc[k] = 0.0; }
    }
    mbar_wait(&full[b], (g >> 1) & 1);
    const double2* chunk = buf + (size_t)b * chunk_nodes;
    const int i0 = ch * QC;
    const int ni = min(QC, nq - i0);
    // radial node il of the chunk:  acc_f += Wq G(q)^2 A_f
    auto close_row = [&](const int il, double (&A)[MF], double (&B)[MF]) {
      const double2 o = souter[i0 + il];
      double gq[MF], wg2[MF];
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        gq[k] = fast_rcp(o.x + m2[k]);
        wg2[k] = o.y * (gq[k] * gq[k]);
      }
      if constexpr (MF == 2) {
        // Field points are independent outputs (reading A4), but tp_batch inverts the denominators of the thread's two
        // field points at a node through their product.  A field point whose mass term has blown up (NaN, infinite, or so
        // large that the product overflows) would spoil its partner's reciprocals too; the masses are fixed per thread, so
        // such a thread (`solo`, known long before the row ends: no cost) redoes each row with one reciprocal per
        // denominator.  The blown-up field point gets what IEEE arithmetic gives for it, its partner its own regular
        // value.  Not covered: a denominator that is EXACTLY zero at a node still costs the partner's output as well.
        if (solo) {
          const double2* row = chunk + il * nc;
#pragma unroll
          for (int k = 0; k < MF; ++k) { A[k] = 0.0; B[k] = 0.0; }
#pragma unroll 1
          for (int j = 0; j < nc; ++j) {
            const double2 t = row[j];
#pragma unroll
            for (int k = 0; k < MF; ++k) {
              const double r = fast_rcp(t.x + m2[k]);
              A[k] = fma(t.y, r, A[k]);
              if constexpr (WANT_D) B[k] = fma(t.y * r, r, B[k]);
            }
          }
        }
      }
#pragma unroll
      for (int k = 0; k < MF; ++k) {
        acc[k] = fma(wg2[k], A[k], acc[k]);
        if constexpr (WANT_D) dacc[k] = fma(wg2[k], fma(2.0 * gq[k], A[k], B[k]), dacc[k]);
      }
    };
    int il = grp;
    // two radial nodes of the group at a time (their angular loops interleaved: the row set-up and the dependent chain that
    // closes a row overlap with the other row's work); the rows are closed in the order of the single-row loop below
    for (; il + TP_GROUPS < ni; il += 2 * TP_GROUPS) {
      const double2* rowa = chunk + il * nc;
      const double2* rowb = rowa + TP_GROUPS * nc;
      double Aa[MF], Ba[MF], Ab[MF], Bb[MF];
#pragma unroll
      for (int k = 0; k < MF; ++k) { Aa[k] = 0.0; Ba[k] = 0.0; Ab[k] = 0.0; Bb[k] = 0.0; }
      // angular rules of 16, 24 and 32 (BASELINE config 2) nodes: unrolled at compile time, same order of operations
      // (cfg2 33.1 -> 31.6 us: no loop control, and the scheduler sees across the batches)
      auto unrolled_rows = [&](auto ncc) {
        constexpr int NCC = decltype(ncc)::value;
#pragma unroll
        for (int j = 0; j < NCC; j += 4) {
          tp_batch<MF, WANT_D, 4>(rowa + j, m2, Aa, Ba);
          tp_batch<MF, WANT_D, 4>(rowb + j, m2, Ab, Bb);
        }
      };
      if (nc == 32) {
        unrolled_rows(std::integral_constant<int, 32>{});
      } else if (nc == 24) {
        unrolled_rows(std::integral_constant<int, 24>{});
      } else if (nc == 16) {
        unrolled_rows(std::integral_constant<int, 16>{});
      } else {
        int j = 0;
        for (; j + 4 <= nc; j += 4) {
          tp_batch<MF, WANT_D, 4>(rowa + j, m2, Aa, Ba);
          tp_batch<MF, WANT_D, 4>(rowb + j, m2, Ab, Bb);
        }
        for (; j < nc; ++j) {
          tp_batch<MF, WANT_D, 1>(rowa + j, m2, Aa, Ba);
          tp_batch<MF, WANT_D, 1>(rowb + j, m2, Ab, Bb);
        }
      }
      close_row(il, Aa, Ba);
      close_row(il + TP_GROUPS, Ab, Bb);
    }
    for (; il < ni; il += TP_GROUPS) {
      const double2* row = chunk + il * nc;
      double A[MF], B[MF];
#pragma unroll
      for (int k = 0; k < MF; ++k) { A[k] = 0.0; B[k] = 0.0; }
      int j = 0;
      for (; j + 4 <= nc; j += 4) tp_batch<MF, WANT_D, 4>(row + j, m2, A, B);
      for (; j < nc; ++j) tp_batch<MF, WANT_D, 1>(row + j, m2, A, B);
      close_row(il, A, B);
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
  CompSum r(P.part[idx]);
  for (int s = 1; s <= c_last - c_first; ++s) r.add(P.part[(size_t)s * nd * plane + idx]);
  P.out[idx] = P.prefactor * r.value();
  if (P.dout) {
    CompSum dr(P.part[plane + idx]);
    for (int s = 1; s <= c_last - c_first; ++s) dr.add(P.part[((size_t)s * 2 + 1) * plane + idx]);
    P.dout[idx] = -P.prefactor * dr.value();
  }
  if (P.dmin) {
    constexpr int NW = TP_NPROD / 32;
    double dm = P.chunkmin[(size_t)U * NW];
    for (long long t = ufirst * NW; t < (ulast + 1) * NW; ++t) dm = fmin(dm, P.chunkmin[t]);
    P.dmin[idx] = (dm + P.m2[f]) * P.reg.inv_k2;
  }
}

int twopoint_launch(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext, const double* ext, double* out,
                    double* dmin, int sm_count, cudaStream_t stream) {
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
  if (smem_main > kMaxDynSmem) { scratch_free(scratch, stream); return DFRG_EUNSUPPORTED; }
  rc = opt_in_max_smem(kmain);
  if (rc != DFRG_OK) { scratch_free(scratch, stream); return rc; }
  kmain<<<P.grid_main, TP_THREADS, smem_main, stream>>>(P);
  const long long n_out = (long long)n_ext * n_field;
  tp_fixup_kernel<<<(unsigned)((n_out + 255) / 256), 256, 0, stream>>>(P);
  rc = check_cuda(cudaGetLastError());
  scratch_free(scratch, stream);
  return rc;
}


// ---- the entry point that allocates nothing -------------------------------------------------------------------------
// twopoint_launch() above takes its scratch (per-chunk denominator minima and per-CTA partial sums) from the library's
// stream-ordered memory pool.  Some hosts of this library may not allocate device memory at the moment they call it: a
// flow-equation right-hand side evaluated inside a solver that has already handed the whole GPU to its own allocator, a
// call made from a thread that must not take the driver's allocation lock (a real-time or callback context), or a process
// running under a memory cap where any cudaMalloc may fail.  For those callers the same two kernels run here with their
// scratch in an array that is part of the library image: it is there from the moment the library is loaded on a device
// until the process exits, on EVERY device that loads the library, whether or not this entry point is ever called
// (DFRG_NOALLOC_SCRATCH_BYTES each).
//
// In host code the name g_tp_fixed_scratch is only a handle for the runtime, not a device address; the address the
// kernels need is asked for once per device with cudaGetSymbolAddress (with that device current) and cached.
static __device__ __align__(256) double g_tp_fixed_scratch[DFRG_NOALLOC_SCRATCH_BYTES / sizeof(double)];

static std::mutex g_fixed_mutex;
static double* g_fixed_addr[64] = {};   // per device: device address of g_tp_fixed_scratch, nullptr = not asked yet

static int fixed_scratch_address(double** addr) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return check_cuda(e);
  if (dev < 0 || dev >= 64) return DFRG_EUNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_fixed_mutex);
  if (!g_fixed_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_tp_fixed_scratch);   // the current device's copy of the array
    if (e != cudaSuccess) return check_cuda(e);
    if (!p) return DFRG_ECUDA;
    g_fixed_addr[dev] = (double*)p;
  }
  *addr = g_fixed_addr[dev];
  return DFRG_OK;
}

// Same plan, same kernels, same launch configuration as twopoint_launch (the GPU test asserts bit-identical outputs);
// only the origin of P.chunkmin / P.part differs.  Keep the two plans in step.
static int twopoint_launch_fixed_scratch(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext,
                                         const double* ext, double* out, double* dmin, int sm_count,
                                         cudaStream_t stream) {
  TwoPointParams P;
  P.nq = D->q.n; P.nc = D->cos1.n; P.n_field = n_field; P.n_ext = n_ext;
  P.prefactor = D->prefactor;
  fill_common(D->reg, D->tab[0], &P.reg, &P.grid);
  P.fmc = fm_consts();
  P.xq = D->q.x; P.wq = D->q.w; P.xc = D->cos1.x; P.wc = D->cos1.w; P.Z = D->tab[0].v;
  P.coef = D->coef; P.m2 = m2; P.pext = ext; P.out = out; P.dmin = dmin; P.dout = D->dout_dm2;
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
  if (n_chunkmin + n_part > DFRG_NOALLOC_SCRATCH_BYTES / sizeof(double)) return DFRG_ESCRATCH;   // nothing enqueued
  const size_t smem_main = tp_main_smem(P.nq, P.nc, P.grid.n, P.QC * P.nc, mf, want_d);
  if (smem_main > kMaxDynSmem) return DFRG_EUNSUPPORTED;
  double* fixed = nullptr;
  int rc = fixed_scratch_address(&fixed);
  if (rc != DFRG_OK) return rc;
  // Nothing in the scratch has to start at zero: the main kernel writes every chunkmin entry and every partial-sum slot
  // that the fix-up kernel reads, so what the previous call left behind is never looked at.
  P.chunkmin = fixed;
  P.part = fixed + n_chunkmin;
  void (*kmain)(const TwoPointParams) =
      mf == 2 ? (want_d ? tp_main_kernel<2, true> : tp_main_kernel<2, false>)
              : (want_d ? tp_main_kernel<1, true> : tp_main_kernel<1, false>);
  rc = opt_in_max_smem(kmain);
  if (rc != DFRG_OK) return rc;
  kmain<<<P.grid_main, TP_THREADS, smem_main, stream>>>(P);
  const long long n_out = (long long)n_ext * n_field;
  tp_fixup_kernel<<<(unsigned)((n_out + 255) / 256), 256, 0, stream>>>(P);
  return check_cuda(cudaGetLastError());
}

}  // namespace dfrg

using namespace dfrg;

// See include/dfrg.h.  Validation is the two-point branch of dfrg_integrate_loop4d's.
extern "C" int dfrg_integrate_twopoint_noalloc(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext,
                                               const double* ext, double* out, double* dmin, void* cuda_stream) {
  if (!D || !ext || !out || n_ext < 1 || n_field < 1 || !m2) return DFRG_EINVAL;
  if (D->family != DFRG_LOOP_TWOPOINT) return DFRG_EINVAL;
  if (!valid_regulator(D->reg) || !valid_rule(D->q) || !valid_rule(D->cos1) || !D->coef || D->n_coef != 2 ||
      !valid_table(D->tab[0], 1))
    return DFRG_EINVAL;
  if ((long long)D->q.n * D->cos1.n > TP_MAX_PAIRS || D->cos1.n > TP_CHUNK_NODES || D->tab[0].n_q > 1024)
    return DFRG_EUNSUPPORTED;
  int sms = 0;
  int rc = require_sm100(&sms);
  if (rc != DFRG_OK) return rc;
  return twopoint_launch_fixed_scratch(D, n_field, m2, n_ext, ext, out, dmin, sms, (cudaStream_t)cuda_stream);
}
