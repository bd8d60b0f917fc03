// dfrg_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, double-precision CPU implementation of the momentum-loop
// integrals on the right-hand side of fRG flow equations (the hot path of
// arxiv 2412.13043, "DiFfRG"), written from the paper text and the workload
// definitions of BASELINE.json / SURVEY.md section 8(c).  It exists to check
// the CUDA library; only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call it.  It shares
// no code, header, table or constant with paper_2412_13043_b200/csrc.
//
// What it follows (PAPER.md line : passage):
//   * fixed tensor-product quadrature "of arbitrary order", radial x angles in
//     the vacuum, Matsubara sum in the time direction at finite T
//     (sec. 5.3.2, integrator types Quadrature / Quadraturex0);
//   * angle variables cos1, cos2, phi (App. F.1);
//   * polynomial exponential regulator s_N(x) = k^2 exp(-sum_{i<=N} x^i/i)
//     (eq. 14) and its RG-time derivative through
//     k d/dk = -2x d/dx on the shape (Fig. 2 caption);
//   * flat (Litim) regulator, shape (1/x - 1) Theta(1 - x);
//   * propagator G = 1/(p^2 + m^2 + R_k) (eq. G.1);
//   * dressing functions as tables on a logarithmic momentum grid
//      and stacks of such tables indexed by an integer
//     Matsubara index with no interpolation across it.
// Everything concrete (integrands, measures, prefactors, loop order) is the
// reading listed in DESIGN.md section "Readings".
//
// Every integrator also returns, per output, dmin (signed minimum over nodes and propagators of
// denominator/k^2, reading A4) and sens: the sum over nodes of |term| -- with |P| replaced by the sum of
// |monomials| -- times (1 + sum over propagators of (|D - m2| + |m2|)/|D| per power), i.e. the first-order
// bound on the output's change under relative perturbations of every input of a term.  The parity tests
// use eps*sens as the condition-aware tolerance for outputs whose denominators vanish or change sign.
//
// Style: one full integrand evaluation per quadrature node, nothing shared
// between field points or external momenta, libm exp/log/sqrt, accumulation in
// long double in exactly the loop order written, OpenMP only across outputs.
//
// Pins (tests/test_oracle_pins.py): Gauss-Legendre closed forms and
// polynomial exactness; Litim threshold functions d=3,4; finite-T Litim
// truncated Matsubara sum vs coth/digamma closed form; exponential-regulator
// weight integrals; regulator derivative vs mpmath differentiation; cubic
// interpolator exactness on cubics; p=0 identity; coefficient linearity;
// dimensional scaling; brute-force convergence; an independent mpmath
// restatement on tiny inputs.
// Mass derivatives (orc_*_dm2, at the end of the file): pinned by the derivatives of the Litim closed forms
// (T = 0 and truncated Matsubara sum), the m2 -> inf weight integrals, and five-point finite differences of
// the pinned value functions.
// Further families: dressed regulator (tests/test_oracle_pins_dressed.py), four-point box (..._fourpoint.py),
// fermionic loop at chemical potential (..._fermion.py), 3-D tables and vertex coordinates (..._tab3d.py).
// Every function here has a pin from outside this file.  What no pin can fix is the choice of READING where the
// words of BASELINE.json / the paper leave an integrand open (configs 3, 4 and the 8(f) families): those readings
// are stated in DESIGN.md section 2; the arithmetic of each reading is pinned by scipy/mpmath adaptive quadrature of
// the continuum integrand it states, unit-monomial runs, Cartesian restatements and closed forms.

#include <cmath>
#include <complex>
#include <cstddef>
#include <cstdint>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef long double acc_t;

const double kInf = std::numeric_limits<double>::infinity();

// ---- regulators: PAPER.md:192 (eq. 14), PAPER.md:178 ---------------------------------
// kind 0: Litim      R = (k^2 - s) Theta(k^2 - s),  Rdot = 2 k^2 Theta(k^2 - s), Theta(0)=0
// kind 1: EXP_POLY(N) R = k^2 exp(-sum_{i=1..N} x^i / i), Rdot = 2 R (1 + sum_{i=1..N} x^i)
// s is the squared momentum, x = s/k^2, Rdot = k dR/dk.
// Dressed regulator (wave-function renormalisation Z_k with anomalous dimension eta = -k dZ_k/dk / Z_k,
// PAPER.md:367 "only the eta_i = -d_t Z_i/Z_i enter the flow equations"):
//   R = zk R_shape,  Rdot = k d(Z_k R_shape)/dk = zk (Rdot_shape - eta R_shape);  zk = 1, eta = 0: the plain shapes.
void regulator_shape(int kind, int order, double k, double s, double* R, double* Rdot);
void regulator(int kind, int order, double k, double zk, double eta, double s, double* R, double* Rdot) {
  double Rs, Rds;
  regulator_shape(kind, order, k, s, &Rs, &Rds);
  *R = zk * Rs;
  *Rdot = zk * (Rds - eta * Rs);
}
void regulator_shape(int kind, int order, double k, double s, double* R, double* Rdot) {
  const double k2 = k * k;
  if (kind == 0) {
    if (s < k2) { *R = k2 - s; *Rdot = 2.0 * k2; }
    else        { *R = 0.0;    *Rdot = 0.0; }
    return;
  }
  const double x = s / k2;
  double expo = 0.0, geo = 0.0, xi = 1.0;
  for (int i = 1; i <= order; ++i) {
    xi *= x;
    expo += xi / (double)i;
    geo += xi;
  }
  const double r = k2 * std::exp(-expo);
  *R = r;
  *Rdot = 2.0 * r * (1.0 + geo);
}

// ---- fermionic regulator RF / RFdot ------------------------------------------------------------------
// The paper makes four functions available in every integration kernel, RB, RF, RBdot, RFdot, and
// its finite-temperature / finite-density examples are fermionic; it prints no fermionic
// shape.  Reading A25: the regulator of a Dirac operator, i pslash (1 + r_F), with the standard relation
// (1 + r_F)^2 = 1 + r_B to the bosonic shape, i.e. with R_F = |p| r_F of momentum dimension one
//   (sqrt(s) + R_F(s))^2 = s + R_B(s)   =>   R_F = sqrt(s + R_B) - sqrt(s),   k dR_F/dk = RBdot / (2 sqrt(s + R_B))
// (flat shape: R_F = (k - sqrt(s)) Theta(k^2 - s), the flat fermionic regulator).  Dressed as the bosonic one:
//   RF = zk R_F,   RFdot = k d(Z_k R_F)/dk = zk (k dR_F/dk - eta R_F).
// A fermion line regulated this way has the scalar denominator of  Z (pslash + ...) + RF-slash + i m:
//   D = Z^2 (s - sR) + (Z sqrt(sR) + RF(sR))^2 + m^2,   insertion  k dD/dk at fixed Z, m  =  2 (Z sqrt(sR) + RF) RFdot
// where sR is the argument of the regulator (the 4-momentum squared, or the spatial part for "3D" regulators, in which
// case s - sR is the squared time component) and m^2 the squared fermion mass.
void regulator_fermion(int kind, int order, double k, double zk, double eta, double s, double* RF, double* RFdot) {
  double Rb, Rbd;
  regulator_shape(kind, order, k, s, &Rb, &Rbd);
  const double root = std::sqrt(s + Rb);
  const double rf = Rb / (root + std::sqrt(s));   // = root - sqrt(s), written without the cancellation at s >> R_B
  const double rfd = Rbd / (2.0 * root);
  *RF = zk * rf;
  *RFdot = zk * (rfd - eta * rf);
}

// ---- log-grid table look-up: PAPER.md:1854-1880; stacks PAPER.md:1898-1905 -----------
// v[0..n-1] sits on ln q_i = lo + i h, h = (hi - lo)/(n - 1).  The argument is the
// SQUARED momentum s; l = log(s)/2; t = clamp((l - lo)/h, 0, n-1).
//   interp 3: i0 = clamp(floor(t) - 1, 0, n - 4), sg = t - i0, 4-point Lagrange on 0,1,2,3
//   interp 1: i = min(floor(t), n - 2), linear
// Outside the grid the end value is returned (clamp-to-edge).
double table_lookup(const double* v, int n, double lo, double hi, int interp, double s) {
  const double h = (hi - lo) / (double)(n - 1);
  const double l = 0.5 * std::log(s);  // s == 0 -> -inf -> clamps low
  double t = (l - lo) / h;
  if (!(t > 0.0)) t = 0.0;             // also catches NaN
  if (t > (double)(n - 1)) t = (double)(n - 1);
  if (interp == 3) {
    int i0 = (int)std::floor(t) - 1;
    if (i0 < 0) i0 = 0;
    if (i0 > n - 4) i0 = n - 4;
    const double sg = t - (double)i0;
    const double L0 = -(sg - 1.0) * (sg - 2.0) * (sg - 3.0) / 6.0;
    const double L1 = sg * (sg - 2.0) * (sg - 3.0) / 2.0;
    const double L2 = -sg * (sg - 1.0) * (sg - 3.0) / 2.0;
    const double L3 = sg * (sg - 1.0) * (sg - 2.0) / 6.0;
    return v[i0] * L0 + v[i0 + 1] * L1 + v[i0 + 2] * L2 + v[i0 + 3] * L3;
  }
  int i = (int)std::floor(t);
  if (i > n - 2) i = n - 2;
  const double tau = t - (double)i;
  return v[i] * (1.0 - tau) + v[i + 1] * tau;
}

// ---- 3-D dressing tables, trilinear: PAPER.md:1860-1896 (LinearInterpolator3D with Log x Log x Lin or
// Log x Lin x Lin coordinates) -------------------------------------------------------------------------
// v is row-major [n0][n1][n2].  Axis a has n_a >= 2 points on a uniform grid in its coordinate c_a between lo_a and
// hi_a; c_a = log(x_a)/2 for a logarithmic axis (x_a = SQUARED momentum, as for the 1-D tables) and c_a = x_a for a
// linear one.  t_a = clamp((c_a - lo_a)/h_a, 0, n_a - 1), cell i_a = min(floor(t_a), n_a - 2), tau_a = t_a - i_a, and
// the value is the trilinear combination of the 8 corners.  Outside the grid the edge value is returned.
struct Table3D {
  const double* v;
  int n[3];
  double lo[3], hi[3];
  int is_log[3];
};
double table3d_lookup(const Table3D& tb, double x0, double x1, double x2) {
  const double x[3] = {x0, x1, x2};
  int i[3];
  double tau[3];
  for (int a = 0; a < 3; ++a) {
    const double h = (tb.hi[a] - tb.lo[a]) / (double)(tb.n[a] - 1);
    const double c = tb.is_log[a] ? 0.5 * std::log(x[a]) : x[a];
    double t = (c - tb.lo[a]) / h;
    if (!(t > 0.0)) t = 0.0;
    if (t > (double)(tb.n[a] - 1)) t = (double)(tb.n[a] - 1);
    i[a] = (int)std::floor(t);
    if (i[a] > tb.n[a] - 2) i[a] = tb.n[a] - 2;
    tau[a] = t - (double)i[a];
  }
  double val = 0.0;
  for (int d0 = 0; d0 < 2; ++d0)
    for (int d1 = 0; d1 < 2; ++d1)
      for (int d2 = 0; d2 < 2; ++d2) {
        const double w = (d0 ? tau[0] : 1.0 - tau[0]) * (d1 ? tau[1] : 1.0 - tau[1]) * (d2 ? tau[2] : 1.0 - tau[2]);
        val += w * tb.v[((size_t)(i[0] + d0) * tb.n[1] + (i[1] + d1)) * tb.n[2] + (i[2] + d2)];
      }
  return val;
}

// Vertex coordinates of a three-point function with squared leg momenta (k1, k2, k3) = (k1^2, k2^2, k3^2): the
// permutation-group variables used for the paper's 96 x 8 x 7 vertex grids ("average momentum S0 and two angles a, s,
// in a parametrisation as introduced in [34]"; reading A23):
//   S0^2 = (k1 + k2 + k3)/6,   a = sqrt(3) (k2 - k1)/(6 S0^2),   s = (k1 + k2 - 2 k3)/(6 S0^2);   S0 = 0: a = s = 0.
// Momentum conservation confines (a, s) to the unit disc.
void vertex_coords(double k1, double k2, double k3, double* S0sq, double* a, double* s) {
  const double six_s0 = k1 + k2 + k3;
  *S0sq = six_s0 / 6.0;
  if (six_s0 > 0.0) {
    *a = std::sqrt(3.0) * (k2 - k1) / six_s0;
    *s = (k1 + k2 - 2.0 * k3) / six_s0;
  } else {
    *a = 0.0;
    *s = 0.0;
  }
}

inline double ipow(double x, int e) {
  double r = 1.0;
  for (int i = 0; i < e; ++i) r *= x;
  return r;
}

inline double clamp0(double s) { return s > 0.0 ? s : 0.0; }  // reading A16

}  // namespace

extern "C" {

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

// Gauss-Legendre rule GL(n;[a,b]): x_i = (b-a)/2 xi_i + (a+b)/2, w_i = (b-a)/2 om_i with
// xi_i the roots of P_n ascending and om_i = 2/((1 - xi_i^2) P_n'(xi_i)^2).
// Newton on the three-term recurrence (j+1)P_{j+1} = (2j+1) x P_j - j P_{j-1}, every root
// on its own from the guess cos(pi (i - 1/4)/(n + 1/2)), all in long double.
int orc_gl_rule(int n, double a, double b, double* x, double* w) {
  if (n < 1 || !x || !w) return -1;
  const long double pi = 3.141592653589793238462643383279502884L;
  const long double half = 0.5L * ((long double)b - (long double)a);
  const long double mid = 0.5L * ((long double)b + (long double)a);
  for (int i = 1; i <= n; ++i) {
    long double z = cosl(pi * ((long double)i - 0.25L) / ((long double)n + 0.5L));
    long double dp = 1.0L;
    for (int it = 0; it < 100; ++it) {
      long double p0 = 1.0L, p1 = z;  // P_0, P_1
      for (int j = 1; j < n; ++j) {
        const long double p2 = ((2.0L * j + 1.0L) * z * p1 - (long double)j * p0) / ((long double)j + 1.0L);
        p0 = p1;
        p1 = p2;
      }
      // n == 1: p1 = z = P_1, p0 = 1 = P_0
      dp = (long double)n * (z * p1 - p0) / (z * z - 1.0L);  // P_n'(z)
      const long double dz = p1 / dp;
      z -= dz;
      if (fabsl(dz) < 2e-19L) break;
    }
    {  // derivative at the converged root
      long double p0 = 1.0L, p1 = z;
      for (int j = 1; j < n; ++j) {
        const long double p2 = ((2.0L * j + 1.0L) * z * p1 - (long double)j * p0) / ((long double)j + 1.0L);
        p0 = p1;
        p1 = p2;
      }
      dp = (long double)n * (z * p1 - p0) / (z * z - 1.0L);
    }
    if (2 * i == n + 1) z = 0.0L;  // middle root of odd n is exactly 0
    const long double om = 2.0L / ((1.0L - z * z) * dp * dp);
    // the guess enumerates roots descending; store ascending
    x[n - i] = (double)(mid + half * z);
    w[n - i] = (double)(half * om);
  }
  return 0;
}

void orc_regulator(int kind, int order, double k, double zk, double eta, double s, double* R, double* Rdot) {
  regulator(kind, order, k, zk, eta, s, R, Rdot);
}

void orc_regulator_fermion(int kind, int order, double k, double zk, double eta, double s, double* RF, double* RFdot) {
  regulator_fermion(kind, order, k, zk, eta, s, RF, RFdot);
}
double orc_table_lookup(const double* v, int n_q, double lnq_lo, double lnq_hi, int interp, double s) {
  return table_lookup(v, n_q, lnq_lo, lnq_hi, interp, s);
}

// ---- LPA O(N) flow right-hand side (configs 0 and 1) ---------------------------------
// T == 0:  I(m2) = C sum_i w_i q_i^(d-1) Rdot(q_i^2) / (q_i^2 + R(q_i^2) + m2)
// T  > 0:  I(m2) = C T sum_{n=-n_max..n_max} sum_i w_i q_i^(d-1) Rdot(sR) / (s + R(sR) + m2),
//          s = w_n^2 + q_i^2, w_n = 2 pi n T, sR = s if reg_arg4d else q_i^2
// flow[f] = (N-1) I(u[f]) + I(u[f] + 2 rho[f] du[f]);  chan = [I_pi | I_sigma] (nullable);
// dmin[f] = signed min over nodes and both channels of (denominator / k^2) (nullable).
int orc_lpa(int d, double T, int n_max, int reg_arg4d, double N, double prefactor,
            int reg_kind, int reg_order, double k, double zk, double eta,
            int nq, const double* xq, const double* wq,
            int n_field, const double* rho, const double* u, const double* du,
            double* flow, double* chan, double* dmin, double* sens) {
  if (d < 1 || nq < 1 || n_field < 0 || T < 0 || n_max < 0 || k <= 0) return -1;
  const double pi = 3.14159265358979323846;
  const double k2 = k * k;
#pragma omp parallel for schedule(static)
  for (int f = 0; f < n_field; ++f) {
    const double m2c[2] = {u[f], u[f] + 2.0 * rho[f] * du[f]};
    double I[2];
    double dm = kInf;
    acc_t sn[2] = {0.0L, 0.0L};
    for (int ch = 0; ch < 2; ++ch) {
      const double m2 = m2c[ch];
      acc_t acc = 0.0L;
      if (T == 0.0) {
        for (int i = 0; i < nq; ++i) {
          const double q = xq[i];
          const double s = q * q;
          double R, Rd;
          regulator(reg_kind, reg_order, k, zk, eta, s, &R, &Rd);
          const double D = s + R + m2;
          if (D / k2 < dm) dm = D / k2;
          const double term = wq[i] * ipow(q, d - 1) * Rd / D;
          acc += (acc_t)term;
          sn[ch] += (acc_t)(std::fabs(term) * (1.0 + (std::fabs(s + R) + std::fabs(m2)) / std::fabs(D)));
        }
        I[ch] = (double)((acc_t)prefactor * acc);
      } else {
        for (int n = -n_max; n <= n_max; ++n) {
          const double wn = 2.0 * pi * (double)n * T;
          for (int i = 0; i < nq; ++i) {
            const double q = xq[i];
            const double s = wn * wn + q * q;
            const double sR = reg_arg4d ? s : q * q;
            double R, Rd;
            regulator(reg_kind, reg_order, k, zk, eta, sR, &R, &Rd);
            const double D = s + R + m2;
            if (D / k2 < dm) dm = D / k2;
            const double term = wq[i] * ipow(q, d - 1) * Rd / D;
            acc += (acc_t)term;
            sn[ch] += (acc_t)(std::fabs(term) * (1.0 + (std::fabs(s + R) + std::fabs(m2)) / std::fabs(D)));
          }
        }
        I[ch] = (double)((acc_t)prefactor * (acc_t)T * acc);
      }
    }
    flow[f] = (N - 1.0) * I[0] + I[1];
    if (chan) { chan[f] = I[0]; chan[n_field + f] = I[1]; }
    if (dmin) dmin[f] = dm;
    if (sens) {
      const acc_t sc = (acc_t)std::fabs(prefactor) * (T == 0.0 ? (acc_t)1.0 : (acc_t)T);
      sens[f] = (double)(sc * sn[0]);
      sens[n_field + f] = (double)(sc * sn[1]);
    }
  }
  return 0;
}

// ---- fermionic LPA loop at finite temperature and chemical potential -------------
// Fermionic Matsubara frequencies nu_n = (2n+1) pi T shifted by the chemical potential, p0 -> nu_n + i mu
// (external fermion legs carry p0f - i mu_q; "T" and "muq"), spatial ("3D")
// regulator R(q^2) as in the paper's finite-density example.  Reading A22:
//   I_F(m2) = C T sum_{n=-n_max-1..n_max} sum_i w_i q_i^(d-1) Rdot(q_i^2) Re[ 1 / ((nu_n + i mu)^2 + q_i^2 + R(q_i^2) + m2) ]
// (the sum over n = -n_max-1 .. n_max is symmetric under nu -> -nu, which makes it real; the real part is written out:
//  D = a + i b, a = nu^2 - mu^2 + q^2 + R + m2, b = 2 nu mu, Re 1/D = a/(a^2+b^2)).
//   dI[j] = d I_F / d m2 = -C T sum sum w q^(d-1) Rdot Re[1/D^2],  Re 1/D^2 = (a^2 - b^2)/(a^2+b^2)^2
//   dmin[j] = min over nodes of |D| / k^2;   sens, sens_d: sum |term| (1 + (|D - m2| + |m2|)/|D| per power of 1/D)
// freg != 0 (reading A25): the loop is regulated with RF / RFdot on the Dirac structure (Z = 1, spatial argument):
//   D = (nu_n + i mu)^2 + (q + RF(q^2))^2 + m2,   Rdot(q^2) -> 2 (q + RF(q^2)) RFdot(q^2);
// with zk = 1, eta = 0 this is the same function as freg = 0 ((q + R_F)^2 = q^2 + R_B, 2 (q + R_F) k dR_F/dk = RBdot).
int orc_lpa_fermion(int d, double T, int n_max, double mu, double prefactor,
                    int reg_kind, int reg_order, double k, double zk, double eta, int freg,
                    int nq, const double* xq, const double* wq,
                    int n_m2, const double* m2v,
                    double* I, double* dI, double* dmin, double* sens, double* sens_d) {
  if (d < 1 || nq < 1 || n_m2 < 0 || !(T > 0) || n_max < 0 || k <= 0) return -1;
  const double pi = 3.14159265358979323846;
  const double k2 = k * k;
#pragma omp parallel for schedule(static)
  for (int j = 0; j < n_m2; ++j) {
    const double m2 = m2v[j];
    acc_t acc = 0.0L, accd = 0.0L, sn = 0.0L, snd = 0.0L;
    double dm = kInf;
    for (int n = -n_max - 1; n <= n_max; ++n) {
      const double nu = (2.0 * (double)n + 1.0) * pi * T;
      for (int i = 0; i < nq; ++i) {
        const double q = xq[i];
        double R, Rd;      // freg: R = (q + RF)^2 - q^2 is not formed; a0 is written with the kinetic term A = q + RF
        double a0;                                             // Re(D - m2)
        if (freg) {
          double RF, RFd;
          regulator_fermion(reg_kind, reg_order, k, zk, eta, q * q, &RF, &RFd);
          const double A = q + RF;
          a0 = nu * nu - mu * mu + A * A;
          Rd = 2.0 * A * RFd;
        } else {
          regulator(reg_kind, reg_order, k, zk, eta, q * q, &R, &Rd);
          a0 = nu * nu - mu * mu + q * q + R;
        }
        const double a = a0 + m2, b = 2.0 * nu * mu;
        const double den = a * a + b * b;                      // |D|^2
        const double absD = std::sqrt(den);
        if (absD / k2 < dm) dm = absD / k2;
        const double w = wq[i] * ipow(q, d - 1) * Rd;
        const double term = w * (a / den);
        const double termd = w * ((a * a - b * b) / (den * den));
        const double cond = (std::sqrt(a0 * a0 + b * b) + std::fabs(m2)) / absD;
        acc += (acc_t)term;
        accd += (acc_t)termd;
        sn += (acc_t)(std::fabs(w) / absD * (1.0 + cond));
        snd += (acc_t)(std::fabs(w) / den * (1.0 + 2.0 * cond));
      }
    }
    const acc_t sc = (acc_t)prefactor * (acc_t)T;
    I[j] = (double)(sc * acc);
    if (dI) dI[j] = (double)(-sc * accd);
    if (dmin) dmin[j] = dm;
    if (sens) sens[j] = (double)(fabsl(sc) * sn);
    if (sens_d) sens_d[j] = (double)(fabsl(sc) * snd);
  }
  return 0;
}

// ---- 4-D vacuum two-point loop (config 2) --------------------------------------------
// out[e][f] = C sum_i wq_i q_i^3 Rdot(q_i^2) G(q_i^2;f)^2
//               sum_j wc_j sqrt(1-c_j^2) (coef0 + coef1 q_i p_e c_j / k^2) G(s_ij;f),
// s_ij = q_i^2 + p_e^2 + 2 q_i p_e c_j,  G(s;f) = 1/(Z(sqrt s) s + R(s) + m2_f).
// sel (nullable): flat output indices e*n_field+f to compute; out/dmin then have n_sel entries.
int orc_loop4d_twopoint(double prefactor, int reg_kind, int reg_order, double k, double zk, double eta,
                        int nq, const double* xq, const double* wq,
                        int nc, const double* xc, const double* wc,
                        const double* Zv, int Z_nq, double Z_lo, double Z_hi, int Z_interp,
                        const double* coef, int n_coef,
                        int n_field, const double* m2, int n_ext, const double* pext,
                        long long n_sel, const long long* sel,
                        double* out, double* dmin, double* sens) {
  if (n_coef != 2 || nq < 1 || nc < 1 || n_field < 1 || n_ext < 1 || k <= 0) return -1;
  const double k2 = k * k;
  const long long n_out = sel ? n_sel : (long long)n_ext * n_field;
#pragma omp parallel for schedule(static)
  for (long long o = 0; o < n_out; ++o) {
    const long long flat = sel ? sel[o] : o;
    const int e = (int)(flat / n_field), f = (int)(flat % n_field);
    const double p = pext[e], mm = m2[f];
    double dm = kInf;
    acc_t acc_q = 0.0L, sn = 0.0L;
    for (int i = 0; i < nq; ++i) {
      const double q = xq[i];
      const double sq = q * q;
      double Rq, Rdq;
      regulator(reg_kind, reg_order, k, zk, eta, sq, &Rq, &Rdq);
      const double Dq = table_lookup(Zv, Z_nq, Z_lo, Z_hi, Z_interp, sq) * sq + Rq + mm;
      if (Dq / k2 < dm) dm = Dq / k2;
      const double Gq = 1.0 / Dq;
      const double condq = 2.0 * (std::fabs(Dq - mm) + std::fabs(mm)) / std::fabs(Dq);
      acc_t acc_c = 0.0L, sn_c = 0.0L;
      for (int j = 0; j < nc; ++j) {
        const double c = xc[j];
        const double s = clamp0(sq + p * p + 2.0 * q * p * c);
        double R, Rd;
        regulator(reg_kind, reg_order, k, zk, eta, s, &R, &Rd);
        const double D = table_lookup(Zv, Z_nq, Z_lo, Z_hi, Z_interp, s) * s + R + mm;
        if (D / k2 < dm) dm = D / k2;
        const double poly = coef[0] + coef[1] * (q * p * c / k2);
        acc_c += (acc_t)(wc[j] * std::sqrt((1.0 - c) * (1.0 + c)) * poly / D);
        const double apoly = std::fabs(coef[0]) + std::fabs(coef[1] * (q * p * c / k2));
        sn_c += (acc_t)(std::fabs(wc[j] * std::sqrt((1.0 - c) * (1.0 + c)) * apoly / D) *
                        (1.0 + condq + (std::fabs(D - mm) + std::fabs(mm)) / std::fabs(D)));
      }
      acc_q += (acc_t)(wq[i] * q * q * q * Rdq * Gq * Gq) * acc_c;
      sn += (acc_t)std::fabs(wq[i] * q * q * q * Rdq * Gq * Gq) * sn_c;
    }
    out[o] = (double)((acc_t)prefactor * acc_q);
    if (dmin) dmin[o] = dm;
    if (sens) sens[o] = (double)((acc_t)std::fabs(prefactor) * sn);
  }
  return 0;
}

// ---- 4-D vacuum three-point vertex loop (config 3) -----------------------------------
// ext = (|p1|, |p2|, alpha)[e];  p1 = |p1|(1,0,0,0), p2 = |p2|(cos a, sin a, 0, 0).
// q.p1 = q|p1|c1,  q.p2 = q|p2|(cos a c1 + sin a sqrt(1-c1^2) c2),
// s_a = |q+p1|^2, s_b = |q-p2|^2, s_c = |p1+p2|^2,  G_A(s) = 1/(Z_A(sqrt s) s + R(s)),
// Lam = l3((p1^2+q^2+s_a)/3) l3((p2^2+q^2+s_b)/3) l3((s_c+s_a+s_b)/3)   (table argument = squared momentum),
// P = sum_{a+b+c<=4} kap_abc (q^2/k^2)^a (q.p1/k^2)^b (q.p2/k^2)^c, a outermost, then b, then c.
// out[e] = C sum_q w q^3 Rdot(q^2) G_A(q^2) sum_c1 w sqrt(1-c1^2) sum_c2 w sum_phi w G_A(s_a) G_A(s_b) Lam P
// The integrand does not depend on phi; literal_phi != 0 evaluates it inside the phi loop
// anyway (tiny inputs only), literal_phi == 0 evaluates it once and multiplies by sum_phi w.
int orc_loop4d_threepoint(double prefactor, int reg_kind, int reg_order, double k, double zk, double eta,
                          int nq, const double* xq, const double* wq,
                          int n1, const double* x1, const double* w1,
                          int n2, const double* x2, const double* w2,
                          int nphi, const double* xphi, const double* wphi,
                          const double* ZA, const double* Zc, const double* L3,
                          int t_nq, double t_lo, double t_hi, int t_interp,
                          const double* coef, int n_coef,
                          int n_ext, const double* ext,
                          long long n_sel, const long long* sel, int literal_phi,
                          double* out, double* dmin, double* sens) {
  (void)Zc;    // accepted, not used by this integrand (reading A14)
  (void)xphi;  // the integrand has no phi dependence
  if (n_coef != 35 || nq < 1 || n1 < 1 || n2 < 1 || nphi < 1 || n_ext < 1 || k <= 0) return -1;
  const double k2 = k * k;
  const long long n_out = sel ? n_sel : (long long)n_ext;
#pragma omp parallel for schedule(dynamic, 1)
  for (long long o = 0; o < n_out; ++o) {
    const long long e = sel ? sel[o] : o;
    const double p1 = ext[3 * e], p2 = ext[3 * e + 1], al = ext[3 * e + 2];
    const double ca = std::cos(al), sa = std::sin(al);
    const double sc = clamp0(p1 * p1 + p2 * p2 + 2.0 * p1 * p2 * ca);
    double dm = kInf;
    acc_t acc_q = 0.0L, sn_q = 0.0L;
    for (int i = 0; i < nq; ++i) {
      const double q = xq[i];
      const double sq = q * q;
      double Rq, Rdq;
      regulator(reg_kind, reg_order, k, zk, eta, sq, &Rq, &Rdq);
      const double Dq = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, sq) * sq + Rq;
      if (Dq / k2 < dm) dm = Dq / k2;
      acc_t acc_1 = 0.0L, sn_1 = 0.0L;
      for (int j1 = 0; j1 < n1; ++j1) {
        const double c1 = x1[j1];
        const double sin1 = std::sqrt((1.0 - c1) * (1.0 + c1));
        acc_t acc_2 = 0.0L, sn_2 = 0.0L;
        for (int j2 = 0; j2 < n2; ++j2) {
          const double c2 = x2[j2];
          const double qp1 = q * p1 * c1;
          const double qp2 = q * p2 * (ca * c1 + sa * sin1 * c2);
          const double s_a = clamp0(sq + p1 * p1 + 2.0 * qp1);
          const double s_b = clamp0(sq + p2 * p2 - 2.0 * qp2);
          acc_t acc_phi = 0.0L;
          const int nphi_eval = literal_phi ? nphi : 1;
          double F = 0.0, Fabs = 0.0;
          for (int jp = 0; jp < nphi_eval; ++jp) {
            double Ra, Rda, Rb, Rdb;
            regulator(reg_kind, reg_order, k, zk, eta, s_a, &Ra, &Rda);
            regulator(reg_kind, reg_order, k, zk, eta, s_b, &Rb, &Rdb);
            const double Da = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, s_a) * s_a + Ra;
            const double Db = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, s_b) * s_b + Rb;
            if (Da / k2 < dm) dm = Da / k2;
            if (Db / k2 < dm) dm = Db / k2;
            const double lam =
                table_lookup(L3, t_nq, t_lo, t_hi, t_interp, (p1 * p1 + sq + s_a) / 3.0) *
                table_lookup(L3, t_nq, t_lo, t_hi, t_interp, (p2 * p2 + sq + s_b) / 3.0) *
                table_lookup(L3, t_nq, t_lo, t_hi, t_interp, (sc + s_a + s_b) / 3.0);
            double P = 0.0, Pabs = 0.0;
            int idx = 0;
            for (int a = 0; a <= 4; ++a)
              for (int b = 0; a + b <= 4; ++b)
                for (int c = 0; a + b + c <= 4; ++c) {
                  const double mono = coef[idx++] * ipow(sq / k2, a) * ipow(qp1 / k2, b) * ipow(qp2 / k2, c);
                  P += mono;
                  Pabs += std::fabs(mono);
                }
            F = (1.0 / Da) * (1.0 / Db) * lam * P;
            Fabs = std::fabs((1.0 / Da) * (1.0 / Db) * lam) * Pabs;
            if (literal_phi) acc_phi += (acc_t)(wphi[jp] * F);
          }
          if (!literal_phi) {
            acc_t sw = 0.0L;
            for (int jp = 0; jp < nphi; ++jp) sw += (acc_t)wphi[jp];
            acc_phi = sw * (acc_t)F;
          }
          acc_2 += (acc_t)w2[j2] * acc_phi;
          sn_2 += (acc_t)(w2[j2] * Fabs);
        }
        acc_1 += (acc_t)(w1[j1] * sin1) * acc_2;
        sn_1 += (acc_t)(w1[j1] * sin1) * sn_2;
      }
      acc_q += (acc_t)(wq[i] * q * q * q * Rdq / Dq) * acc_1;
      sn_q += (acc_t)std::fabs(wq[i] * q * q * q * Rdq / Dq) * sn_1;
    }
    out[o] = (double)((acc_t)prefactor * acc_q);
    if (dmin) dmin[o] = dm;
    if (sens) {  // sum of |terms| with |P| replaced by the sum of |monomials|, times sum_phi w
      acc_t sw = 0.0L;
      for (int jp = 0; jp < nphi; ++jp) sw += (acc_t)wphi[jp];
      sens[o] = (double)((acc_t)std::fabs(prefactor) * sw * sn_q);
    }
  }
  return 0;
}

// ---- three-point vertex loop with a 3-D vertex dressing table ---------------------
// As orc_loop4d_threepoint (same kinematics, propagators, polynomial, measure), but every three-gluon vertex is
// dressed by lambda3(S0, a, s) from a 3-D table at the vertex coordinates of its legs (vertex_coords above):
//   Lam = l3d(p1^2, q^2, s_a) l3d(p2^2, q^2, s_b) l3d(s_c, s_a, s_b)      (leg order as written)
// Table axes: 0 = S0^2 (logarithmic or linear), 1 = a, 2 = s.
int orc_loop4d_threepoint_tab3d(double prefactor, int reg_kind, int reg_order, double k, double zk, double eta,
                                int nq, const double* xq, const double* wq,
                                int n1, const double* x1, const double* w1,
                                int n2, const double* x2, const double* w2,
                                int nphi, const double* wphi,
                                const double* ZA, int t_nq, double t_lo, double t_hi, int t_interp,
                                const double* v3, const int* n3, const double* lo3, const double* hi3, const int* log3,
                                const double* coef, int n_coef,
                                int n_ext, const double* ext,
                                long long n_sel, const long long* sel,
                                double* out, double* dmin, double* sens) {
  if (n_coef != 35 || nq < 1 || n1 < 1 || n2 < 1 || nphi < 1 || n_ext < 1 || k <= 0) return -1;
  Table3D tb;
  tb.v = v3;
  for (int a = 0; a < 3; ++a) {
    tb.n[a] = n3[a]; tb.lo[a] = lo3[a]; tb.hi[a] = hi3[a]; tb.is_log[a] = log3[a];
    if (n3[a] < 2 || !(hi3[a] > lo3[a])) return -1;
  }
  const double k2 = k * k;
  acc_t sw = 0.0L;
  for (int jp = 0; jp < nphi; ++jp) sw += (acc_t)wphi[jp];
  const long long n_out = sel ? n_sel : (long long)n_ext;
#pragma omp parallel for schedule(dynamic, 1)
  for (long long o = 0; o < n_out; ++o) {
    const long long e = sel ? sel[o] : o;
    const double p1 = ext[3 * e], p2 = ext[3 * e + 1], al = ext[3 * e + 2];
    const double ca = std::cos(al), sa = std::sin(al);
    const double sc = clamp0(p1 * p1 + p2 * p2 + 2.0 * p1 * p2 * ca);
    double dm = kInf;
    acc_t acc_q = 0.0L, sn_q = 0.0L;
    for (int i = 0; i < nq; ++i) {
      const double q = xq[i];
      const double sq = q * q;
      double Rq, Rdq;
      regulator(reg_kind, reg_order, k, zk, eta, sq, &Rq, &Rdq);
      const double Dq = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, sq) * sq + Rq;
      if (Dq / k2 < dm) dm = Dq / k2;
      acc_t acc_1 = 0.0L, sn_1 = 0.0L;
      for (int j1 = 0; j1 < n1; ++j1) {
        const double c1 = x1[j1];
        const double sin1 = std::sqrt((1.0 - c1) * (1.0 + c1));
        acc_t acc_2 = 0.0L, sn_2 = 0.0L;
        for (int j2 = 0; j2 < n2; ++j2) {
          const double c2 = x2[j2];
          const double qp1 = q * p1 * c1;
          const double qp2 = q * p2 * (ca * c1 + sa * sin1 * c2);
          const double s_a = clamp0(sq + p1 * p1 + 2.0 * qp1);
          const double s_b = clamp0(sq + p2 * p2 - 2.0 * qp2);
          double Ra, Rb, dummy;
          regulator(reg_kind, reg_order, k, zk, eta, s_a, &Ra, &dummy);
          regulator(reg_kind, reg_order, k, zk, eta, s_b, &Rb, &dummy);
          const double Da = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, s_a) * s_a + Ra;
          const double Db = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, s_b) * s_b + Rb;
          if (Da / k2 < dm) dm = Da / k2;
          if (Db / k2 < dm) dm = Db / k2;
          double lam = 1.0;
          const double legs[3][3] = {{p1 * p1, sq, s_a}, {p2 * p2, sq, s_b}, {sc, s_a, s_b}};
          for (int v = 0; v < 3; ++v) {
            double S0sq, a_, s_;
            vertex_coords(legs[v][0], legs[v][1], legs[v][2], &S0sq, &a_, &s_);
            lam *= table3d_lookup(tb, S0sq, a_, s_);
          }
          double P = 0.0, Pabs = 0.0;
          int idx = 0;
          for (int a = 0; a <= 4; ++a)
            for (int b = 0; a + b <= 4; ++b)
              for (int c = 0; a + b + c <= 4; ++c) {
                const double mono = coef[idx++] * ipow(sq / k2, a) * ipow(qp1 / k2, b) * ipow(qp2 / k2, c);
                P += mono;
                Pabs += std::fabs(mono);
              }
          const double F = (1.0 / Da) * (1.0 / Db) * lam * P;
          const double Fabs = std::fabs((1.0 / Da) * (1.0 / Db) * lam) * Pabs;
          acc_2 += (acc_t)w2[j2] * (sw * (acc_t)F);
          sn_2 += (acc_t)(w2[j2] * Fabs);
        }
        acc_1 += (acc_t)(w1[j1] * sin1) * acc_2;
        sn_1 += (acc_t)(w1[j1] * sin1) * sn_2;
      }
      acc_q += (acc_t)(wq[i] * q * q * q * Rdq / Dq) * acc_1;
      sn_q += (acc_t)std::fabs(wq[i] * q * q * q * Rdq / Dq) * sn_1;
    }
    out[o] = (double)((acc_t)prefactor * acc_q);
    if (dmin) dmin[o] = dm;
    if (sens) sens[o] = (double)((acc_t)std::fabs(prefactor) * sw * sn_q);
  }
  return 0;
}

double orc_table3d_lookup(const double* v3, const int* n3, const double* lo3, const double* hi3, const int* log3,
                          double x0, double x1, double x2) {
  Table3D tb;
  tb.v = v3;
  for (int a = 0; a < 3; ++a) { tb.n[a] = n3[a]; tb.lo[a] = lo3[a]; tb.hi[a] = hi3[a]; tb.is_log[a] = log3[a]; }
  return table3d_lookup(tb, x0, x1, x2);
}

void orc_vertex_coords(double k1, double k2, double k3, double* S0sq, double* a, double* s) {
  vertex_coords(k1, k2, k3, S0sq, a, s);
}

// ---- 4-D vacuum four-point box loop: genuine three-angle kinematics + ghost loop ----
// "Angles -> 3": cos1, cos2, phi; four-gluon vertex configurations.  Reading A21.
// ext = (|p1|, |p2|, |p3|, alpha, beta, gamma)[e]:
//   p1 = |p1| (1, 0, 0, 0),  p2 = |p2| (cos al, sin al, 0, 0),  p3 = |p3| (cos be, sin be cos ga, sin be sin ga, 0),
//   q  = q (c1, s1 c2, s1 s2 cos phi, s1 s2 sin phi),  s1 = sqrt(1-c1^2), s2 = sqrt(1-c2^2)
//   u1 = q.p1 = q|p1| c1,  u2 = q.p2 = q|p2| (cos al c1 + sin al s1 c2),
//   u3 = q.p3 = q|p3| (cos be c1 + sin be cos ga s1 c2 + sin be sin ga s1 s2 cos phi)
// Box routing: internal lines q, q+p1, q+p1+p2, q+p1+p2+p3:
//   s12 = |p1+p2|^2,  s123 = |p1+p2+p3|^2 (= p4^2),
//   s_a = q^2 + p1^2 + 2 u1,  s_b = q^2 + s12 + 2 (u1 + u2),  s_d = q^2 + s123 + 2 (u1 + u2 + u3)
// Gluon box: four three-gluon vertices, each dressed at the mean squared momentum of its legs,
//   l1 = (q^2 + p1^2 + s_a)/3, l2 = (s_a + p2^2 + s_b)/3, l3 = (s_b + p3^2 + s_d)/3, l4 = (s_d + s123 + q^2)/3
//   T_A = G_A(q^2) G_A(s_a) G_A(s_b) G_A(s_d) l3(l1) l3(l2) l3(l3) l3(l4) P_A,   G_A(s) = 1/(Z_A(s) s + R(s))
// Ghost box (undressed ghost-gluon vertices):
//   T_c = G_c(q^2) G_c(s_a) G_c(s_b) G_c(s_d) P_c,                                 G_c(s) = 1/(Z_c(s) s + R(s))
// P_X = sum_{a+b+c+d<=3} kap^X_abcd (q^2/k^2)^a (u1/k^2)^b (u2/k^2)^c (u3/k^2)^d, a outermost, then b, c, d, ascending
//   (35 coefficients each; coef = [kap^A | kap^c], n_coef = 70).
// out[e] = C sum_q w q^3 Rdot(q^2) sum_c1 w sqrt(1-c1^2) sum_c2 w sum_phi w (T_A + T_c)
int orc_loop4d_fourpoint(double prefactor, int reg_kind, int reg_order, double k, double zk, double eta,
                         int nq, const double* xq, const double* wq,
                         int n1, const double* x1, const double* w1,
                         int n2, const double* x2, const double* w2,
                         int nphi, const double* xphi, const double* wphi,
                         const double* ZA, const double* Zc, const double* L3,
                         int t_nq, double t_lo, double t_hi, int t_interp,
                         const double* coef, int n_coef,
                         int n_ext, const double* ext,
                         long long n_sel, const long long* sel,
                         double* out, double* dmin, double* sens) {
  if (n_coef != 70 || nq < 1 || n1 < 1 || n2 < 1 || nphi < 1 || n_ext < 1 || k <= 0) return -1;
  const double k2 = k * k;
  const long long n_out = sel ? n_sel : (long long)n_ext;
#pragma omp parallel for schedule(dynamic, 1)
  for (long long o = 0; o < n_out; ++o) {
    const long long e = sel ? sel[o] : o;
    const double p1 = ext[6 * e], p2 = ext[6 * e + 1], p3 = ext[6 * e + 2];
    const double al = ext[6 * e + 3], be = ext[6 * e + 4], ga = ext[6 * e + 5];
    const double ca = std::cos(al), sa = std::sin(al), cb = std::cos(be), sb = std::sin(be);
    const double cg = std::cos(ga), sg = std::sin(ga);
    const double p1p2 = p1 * p2 * ca, p1p3 = p1 * p3 * cb, p2p3 = p2 * p3 * (ca * cb + sa * sb * cg);
    const double s12 = clamp0(p1 * p1 + p2 * p2 + 2.0 * p1p2);
    const double s123 = clamp0(p1 * p1 + p2 * p2 + p3 * p3 + 2.0 * (p1p2 + p1p3 + p2p3));
    double dm = kInf;
    acc_t acc_q = 0.0L, sn_q = 0.0L;
    for (int i = 0; i < nq; ++i) {
      const double q = xq[i];
      const double sq = q * q;
      double Rq, Rdq;
      regulator(reg_kind, reg_order, k, zk, eta, sq, &Rq, &Rdq);
      const double DqA = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, sq) * sq + Rq;
      const double Dqc = table_lookup(Zc, t_nq, t_lo, t_hi, t_interp, sq) * sq + Rq;
      if (DqA / k2 < dm) dm = DqA / k2;
      if (Dqc / k2 < dm) dm = Dqc / k2;
      acc_t acc_1 = 0.0L, sn_1 = 0.0L;
      for (int j1 = 0; j1 < n1; ++j1) {
        const double c1 = x1[j1];
        const double sin1 = std::sqrt((1.0 - c1) * (1.0 + c1));
        acc_t acc_2 = 0.0L, sn_2 = 0.0L;
        for (int j2 = 0; j2 < n2; ++j2) {
          const double c2 = x2[j2];
          const double sin2 = std::sqrt((1.0 - c2) * (1.0 + c2));
          acc_t acc_phi = 0.0L, sn_phi = 0.0L;
          for (int jp = 0; jp < nphi; ++jp) {
            const double cphi = std::cos(xphi[jp]);
            const double u1 = q * p1 * c1;
            const double u2 = q * p2 * (ca * c1 + sa * sin1 * c2);
            const double u3 = q * p3 * (cb * c1 + sb * cg * sin1 * c2 + sb * sg * sin1 * sin2 * cphi);
            const double s_a = clamp0(sq + p1 * p1 + 2.0 * u1);
            const double s_b = clamp0(sq + s12 + 2.0 * (u1 + u2));
            const double s_d = clamp0(sq + s123 + 2.0 * (u1 + u2 + u3));
            double Ra, Rb, Rd, dummy;
            regulator(reg_kind, reg_order, k, zk, eta, s_a, &Ra, &dummy);
            regulator(reg_kind, reg_order, k, zk, eta, s_b, &Rb, &dummy);
            regulator(reg_kind, reg_order, k, zk, eta, s_d, &Rd, &dummy);
            const double DaA = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, s_a) * s_a + Ra;
            const double DbA = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, s_b) * s_b + Rb;
            const double DdA = table_lookup(ZA, t_nq, t_lo, t_hi, t_interp, s_d) * s_d + Rd;
            const double Dac = table_lookup(Zc, t_nq, t_lo, t_hi, t_interp, s_a) * s_a + Ra;
            const double Dbc = table_lookup(Zc, t_nq, t_lo, t_hi, t_interp, s_b) * s_b + Rb;
            const double Ddc = table_lookup(Zc, t_nq, t_lo, t_hi, t_interp, s_d) * s_d + Rd;
            const double Dall[6] = {DaA, DbA, DdA, Dac, Dbc, Ddc};
            for (int t = 0; t < 6; ++t)
              if (Dall[t] / k2 < dm) dm = Dall[t] / k2;
            const double lam =
                table_lookup(L3, t_nq, t_lo, t_hi, t_interp, (sq + p1 * p1 + s_a) / 3.0) *
                table_lookup(L3, t_nq, t_lo, t_hi, t_interp, (s_a + p2 * p2 + s_b) / 3.0) *
                table_lookup(L3, t_nq, t_lo, t_hi, t_interp, (s_b + p3 * p3 + s_d) / 3.0) *
                table_lookup(L3, t_nq, t_lo, t_hi, t_interp, (s_d + s123 + sq) / 3.0);
            double PA = 0.0, PAabs = 0.0, Pc = 0.0, Pcabs = 0.0;
            int idx = 0;
            for (int a = 0; a <= 3; ++a)
              for (int b = 0; a + b <= 3; ++b)
                for (int c = 0; a + b + c <= 3; ++c)
                  for (int d = 0; a + b + c + d <= 3; ++d) {
                    const double mono = ipow(sq / k2, a) * ipow(u1 / k2, b) * ipow(u2 / k2, c) * ipow(u3 / k2, d);
                    PA += coef[idx] * mono;
                    PAabs += std::fabs(coef[idx] * mono);
                    Pc += coef[35 + idx] * mono;
                    Pcabs += std::fabs(coef[35 + idx] * mono);
                    ++idx;
                  }
            const double gA = (1.0 / DqA) * (1.0 / DaA) * (1.0 / DbA) * (1.0 / DdA) * lam;
            const double gc = (1.0 / Dqc) * (1.0 / Dac) * (1.0 / Dbc) * (1.0 / Ddc);
            acc_phi += (acc_t)(wphi[jp] * (gA * PA + gc * Pc));
            sn_phi += (acc_t)(wphi[jp] * (std::fabs(gA) * PAabs + std::fabs(gc) * Pcabs));
          }
          acc_2 += (acc_t)w2[j2] * acc_phi;
          sn_2 += (acc_t)w2[j2] * sn_phi;
        }
        acc_1 += (acc_t)(w1[j1] * sin1) * acc_2;
        sn_1 += (acc_t)(w1[j1] * sin1) * sn_2;
      }
      acc_q += (acc_t)(wq[i] * q * q * q * Rdq) * acc_1;
      sn_q += (acc_t)std::fabs(wq[i] * q * q * q * Rdq) * sn_1;
    }
    out[o] = (double)((acc_t)prefactor * acc_q);
    if (dmin) dmin[o] = dm;
    if (sens) sens[o] = (double)((acc_t)std::fabs(prefactor) * sn_q);
  }
  return 0;
}

// ---- 3-D spatial + Matsubara loop (config 4) -----------------------------------------
// nu_n = (2n+1) pi T (fermionic, loop n = -n_max..n_max, external j = 0..n_jext-1),
// boson line (nu_j - nu_n, p - q): m = j - n, om_m = 2 pi m T, r^2 = p^2 + q^2 - 2 p q c.
// s_psi = nu_n^2 + q^2,  s_phi = om_m^2 + r^2
// G_psi = 1/(Z_psi(q, nbar) s_psi + R(s_psi) + m2_psi),  nbar = n >= 0 ? n : -n-1
// G_phi = 1/(Z_phi(r, |m|) s_phi + R(s_phi) + m2_phi)
// P = sum_{a+b+c<=3} kap_abc y1^a y2^b y3^c, y1 = nu_n nu_j/k^2, y2 = p q c/k^2, y3 = s_psi/k^2
// out[p][j][f] = C T sum_n sum_q w q^2 Rdot(s_psi) G_psi^2 sum_c w P G_phi
// Tables are row-major [n_freq][n_q]; the momentum argument is the spatial one (q^2, r^2).
// freg != 0 (reading A25): the fermion line carries the fermionic regulator on its Dirac structure (4-D argument):
//   A = Z_psi sqrt(s_psi) + RF(s_psi),  G_psi = 1/(A^2 + m2_psi),  Rdot(s_psi) -> 2 A RFdot(s_psi);  boson line unchanged.
int orc_matsubara3d(double T, int n_max, double prefactor, int reg_kind, int reg_order, double k, double zk, double eta,
                    int freg,
                    int nq, const double* xq, const double* wq,
                    int nc, const double* xc, const double* wc,
                    const double* Zpsi, const double* Zphi, int t_nq, int t_nfreq,
                    double t_lo, double t_hi, int t_interp,
                    const double* coef, int n_coef,
                    int n_field, const double* m2psi, const double* m2phi,
                    int n_p, const double* pext, int n_jext,
                    long long n_sel, const long long* sel,
                    double* out, double* dmin, double* sens) {
  if (n_coef != 20 || nq < 1 || nc < 1 || n_field < 1 || n_p < 1 || n_jext < 1 || k <= 0 || T <= 0) return -1;
  if (n_max + 1 > t_nfreq || n_jext - 1 + n_max + 1 > t_nfreq) return -1;
  const double pi = 3.14159265358979323846;
  const double k2 = k * k;
  const long long n_out = sel ? n_sel : (long long)n_p * n_jext * n_field;
#pragma omp parallel for schedule(static)
  for (long long o = 0; o < n_out; ++o) {
    const long long flat = sel ? sel[o] : o;
    const int f = (int)(flat % n_field);
    const int j = (int)((flat / n_field) % n_jext);
    const int e = (int)(flat / ((long long)n_field * n_jext));
    const double p = pext[e];
    const double nuj = (2.0 * j + 1.0) * pi * T;
    double dm = kInf;
    acc_t acc_n = 0.0L, sn_n = 0.0L;
    for (int n = -n_max; n <= n_max; ++n) {
      const double nun = (2.0 * n + 1.0) * pi * T;
      const int nbar = n >= 0 ? n : -n - 1;
      const int m = j - n;
      const int mabs = m >= 0 ? m : -m;
      const double om = 2.0 * pi * (double)m * T;
      for (int i = 0; i < nq; ++i) {
        const double q = xq[i];
        const double spsi = nun * nun + q * q;
        double Rp, Rdp, Dpsi;
        const double Zq = table_lookup(Zpsi + (size_t)nbar * t_nq, t_nq, t_lo, t_hi, t_interp, q * q);
        if (freg) {
          double RF, RFd;
          regulator_fermion(reg_kind, reg_order, k, zk, eta, spsi, &RF, &RFd);
          const double A = Zq * std::sqrt(spsi) + RF;
          Dpsi = A * A + m2psi[f];
          Rdp = 2.0 * A * RFd;
        } else {
          regulator(reg_kind, reg_order, k, zk, eta, spsi, &Rp, &Rdp);
          Dpsi = Zq * spsi + Rp + m2psi[f];
        }
        if (Dpsi / k2 < dm) dm = Dpsi / k2;
        const double Gpsi = 1.0 / Dpsi;
        const double condpsi = 2.0 * (std::fabs(Dpsi - m2psi[f]) + std::fabs(m2psi[f])) / std::fabs(Dpsi);
        acc_t acc_c = 0.0L, sn_c = 0.0L;
        for (int jc = 0; jc < nc; ++jc) {
          const double c = xc[jc];
          const double r2 = clamp0(p * p + q * q - 2.0 * p * q * c);
          const double sphi = om * om + r2;
          double Rb, Rdb;
          regulator(reg_kind, reg_order, k, zk, eta, sphi, &Rb, &Rdb);
          const double Dphi =
              table_lookup(Zphi + (size_t)mabs * t_nq, t_nq, t_lo, t_hi, t_interp, r2) * sphi + Rb + m2phi[f];
          if (Dphi / k2 < dm) dm = Dphi / k2;
          const double y1 = nun * nuj / k2, y2 = p * q * c / k2, y3 = spsi / k2;
          double P = 0.0, Pabs = 0.0;
          int idx = 0;
          for (int a = 0; a <= 3; ++a)
            for (int b = 0; a + b <= 3; ++b)
              for (int cc = 0; a + b + cc <= 3; ++cc) {
                const double mono = coef[idx++] * ipow(y1, a) * ipow(y2, b) * ipow(y3, cc);
                P += mono;
                Pabs += std::fabs(mono);
              }
          acc_c += (acc_t)(wc[jc] * P / Dphi);
          sn_c += (acc_t)(std::fabs(wc[jc] * Pabs / Dphi) *
                          (1.0 + condpsi + (std::fabs(Dphi - m2phi[f]) + std::fabs(m2phi[f])) / std::fabs(Dphi)));
        }
        acc_n += (acc_t)(wq[i] * q * q * Rdp * Gpsi * Gpsi) * acc_c;
        sn_n += (acc_t)std::fabs(wq[i] * q * q * Rdp * Gpsi * Gpsi) * sn_c;
      }
    }
    out[o] = (double)((acc_t)prefactor * (acc_t)T * acc_n);
    if (dmin) dmin[o] = dm;
    if (sens) sens[o] = (double)((acc_t)std::fabs(prefactor) * (acc_t)T * sn_n);
  }
  return 0;
}

// ---- 3-D spatial + Matsubara loop at finite chemical potential, spatial regulators ----
// As orc_matsubara3d, with (reading A24):
//   * spatial ("3D") regulators, as the paper's finite-density example: R(q^2), Rdot(q^2) on the fermion
//     line, R(r^2) on the boson line;
//   * every fermion leg carries the time component nu + i mu (PAPER.md:1947-1952 writes p0f - i mu_q: the complex
//     conjugate convention; out(-mu) = conj(out(mu))): loop fermion nu_n + i mu, external fermion nu_j + i mu; the boson
//     line carries their difference nu_j - nu_n, so mu drops out of it;
//   s_psi = (nu_n + i mu)^2 + q^2 (complex),  G_psi = 1/(Z_psi(q^2; nbar) s_psi + R(q^2) + m2_psi)
//   s_phi = om_m^2 + r^2,                      G_phi = 1/(Z_phi(r^2; |m|) s_phi + R(r^2) + m2_phi)
//   y1 = (nu_n + i mu)(nu_j + i mu)/k^2,  y2 = p q c/k^2,  y3 = s_psi/k^2
//   out[p][j][f] = C T sum_n sum_q w q^2 Rdot(q^2) G_psi^2 sum_c w P(y1, y2, y3) G_phi        (complex: out_re, out_im)
// mu = 0 gives the real spatial-regulator variant of the family (out_im = 0 exactly).
// dmin = min over nodes of min(|D_psi|, D_phi)/k^2;  sens as orc_matsubara3d with moduli.
// freg != 0 (reading A25): fermion line with the fermionic regulator on the Dirac structure, spatial argument:
//   A = Z_psi q + RF(q^2),  G_psi = 1/(Z_psi^2 (nu_n + i mu)^2 + A^2 + m2_psi),  Rdot(q^2) -> 2 A RFdot(q^2).
int orc_matsubara3d_mu(double T, int n_max, double mu, double prefactor, int reg_kind, int reg_order, double k,
                       double zk, double eta, int freg,
                       int nq, const double* xq, const double* wq,
                       int nc, const double* xc, const double* wc,
                       const double* Zpsi, const double* Zphi, int t_nq, int t_nfreq,
                       double t_lo, double t_hi, int t_interp,
                       const double* coef, int n_coef,
                       int n_field, const double* m2psi, const double* m2phi,
                       int n_p, const double* pext, int n_jext,
                       long long n_sel, const long long* sel,
                       double* out_re, double* out_im, double* dmin, double* sens) {
  typedef std::complex<double> cd;
  typedef std::complex<long double> cld;
  if (n_coef != 20 || nq < 1 || nc < 1 || n_field < 1 || n_p < 1 || n_jext < 1 || k <= 0 || T <= 0) return -1;
  if (n_max + 1 > t_nfreq || n_jext - 1 + n_max + 1 > t_nfreq) return -1;
  const double pi = 3.14159265358979323846;
  const double k2 = k * k;
  const long long n_out = sel ? n_sel : (long long)n_p * n_jext * n_field;
#pragma omp parallel for schedule(static)
  for (long long o = 0; o < n_out; ++o) {
    const long long flat = sel ? sel[o] : o;
    const int f = (int)(flat % n_field);
    const int j = (int)((flat / n_field) % n_jext);
    const int e = (int)(flat / ((long long)n_field * n_jext));
    const double p = pext[e];
    const cd p0j((2.0 * j + 1.0) * pi * T, mu);
    double dm = kInf;
    cld acc_n(0.0L, 0.0L);
    acc_t sn_n = 0.0L;
    for (int n = -n_max; n <= n_max; ++n) {
      const cd p0n((2.0 * n + 1.0) * pi * T, mu);
      const int nbar = n >= 0 ? n : -n - 1;
      const int m = j - n;
      const int mabs = m >= 0 ? m : -m;
      const double om = 2.0 * pi * (double)m * T;
      for (int i = 0; i < nq; ++i) {
        const double q = xq[i];
        const cd spsi = p0n * p0n + q * q;
        double Rp, Rdp;
        cd Dpsi;
        const double Zq = table_lookup(Zpsi + (size_t)nbar * t_nq, t_nq, t_lo, t_hi, t_interp, q * q);
        if (freg) {
          double RF, RFd;
          regulator_fermion(reg_kind, reg_order, k, zk, eta, q * q, &RF, &RFd);
          const double A = Zq * q + RF;
          Dpsi = (Zq * Zq) * (p0n * p0n) + A * A + m2psi[f];
          Rdp = 2.0 * A * RFd;
        } else {
          regulator(reg_kind, reg_order, k, zk, eta, q * q, &Rp, &Rdp);
          Dpsi = Zq * spsi + Rp + m2psi[f];
        }
        if (std::abs(Dpsi) / k2 < dm) dm = std::abs(Dpsi) / k2;
        const cd Gpsi = 1.0 / Dpsi;
        const double condpsi = 2.0 * (std::abs(Dpsi - m2psi[f]) + std::fabs(m2psi[f])) / std::abs(Dpsi);
        cld acc_c(0.0L, 0.0L);
        acc_t sn_c = 0.0L;
        for (int jc = 0; jc < nc; ++jc) {
          const double c = xc[jc];
          const double r2 = clamp0(p * p + q * q - 2.0 * p * q * c);
          const double sphi = om * om + r2;
          double Rb, Rdb;
          regulator(reg_kind, reg_order, k, zk, eta, r2, &Rb, &Rdb);
          const double Dphi =
              table_lookup(Zphi + (size_t)mabs * t_nq, t_nq, t_lo, t_hi, t_interp, r2) * sphi + Rb + m2phi[f];
          if (Dphi / k2 < dm) dm = Dphi / k2;
          const cd y1 = p0n * p0j / k2, y3 = spsi / k2;
          const double y2 = p * q * c / k2;
          cd P(0.0, 0.0);
          double Pabs = 0.0;
          int idx = 0;
          for (int a = 0; a <= 3; ++a)
            for (int b = 0; a + b <= 3; ++b)
              for (int cc = 0; a + b + cc <= 3; ++cc) {
                cd mono(coef[idx++], 0.0);
                for (int t = 0; t < a; ++t) mono *= y1;
                for (int t = 0; t < b; ++t) mono *= y2;
                for (int t = 0; t < cc; ++t) mono *= y3;
                P += mono;
                Pabs += std::abs(mono);
              }
          const cd term = wc[jc] * P / Dphi;
          acc_c += cld(term.real(), term.imag());
          sn_c += (acc_t)(std::fabs(wc[jc] * Pabs / Dphi) *
                          (1.0 + condpsi + (std::fabs(Dphi - m2phi[f]) + std::fabs(m2phi[f])) / std::fabs(Dphi)));
        }
        const cd wgt = wq[i] * q * q * Rdp * Gpsi * Gpsi;
        acc_n += cld(wgt.real(), wgt.imag()) * acc_c;
        sn_n += (acc_t)std::abs(wgt) * sn_c;
      }
    }
    out_re[o] = (double)((acc_t)prefactor * (acc_t)T * acc_n.real());
    out_im[o] = (double)((acc_t)prefactor * (acc_t)T * acc_n.imag());
    if (dmin) dmin[o] = dm;
    if (sens) sens[o] = (double)((acc_t)std::fabs(prefactor) * (acc_t)T * sn_n);
  }
  return 0;
}

// Mass derivatives of orc_matsubara3d_mu (spatial regulators, any mu), term by term on the same nodes:
//   dpsi = d out / d m2_psi = C T sum_n sum_q w q^2 Rdot(q^2) (-2 G_psi^3) sum_c w P G_phi
//   dphi = d out / d m2_phi = C T sum_n sum_q w q^2 Rdot(q^2) G_psi^2 sum_c w P (-G_phi^2)
// (complex for mu != 0: *_re, *_im).  sens_* as orc_matsubara3d_dm2 with moduli.
// freg != 0 (reading A25): fermion line with the fermionic regulator on the Dirac structure, spatial argument:
//   A = Z_psi q + RF(q^2),  G_psi = 1/(Z_psi^2 (nu_n + i mu)^2 + A^2 + m2_psi),  Rdot(q^2) -> 2 A RFdot(q^2).
int orc_matsubara3d_mu_dm2(double T, int n_max, double mu, double prefactor, int reg_kind, int reg_order, double k,
                           double zk, double eta, int freg,
                           int nq, const double* xq, const double* wq,
                           int nc, const double* xc, const double* wc,
                           const double* Zpsi, const double* Zphi, int t_nq, int t_nfreq,
                           double t_lo, double t_hi, int t_interp,
                           const double* coef, int n_coef,
                           int n_field, const double* m2psi, const double* m2phi,
                           int n_p, const double* pext, int n_jext,
                           long long n_sel, const long long* sel,
                           double* dpsi_re, double* dpsi_im, double* dphi_re, double* dphi_im,
                           double* sens_psi, double* sens_phi) {
  typedef std::complex<double> cd;
  typedef std::complex<long double> cld;
  if (n_coef != 20 || nq < 1 || nc < 1 || n_field < 1 || n_p < 1 || n_jext < 1 || k <= 0 || T <= 0) return -1;
  if (n_max + 1 > t_nfreq || n_jext - 1 + n_max + 1 > t_nfreq) return -1;
  const double pi = 3.14159265358979323846;
  const double k2 = k * k;
  const long long n_out = sel ? n_sel : (long long)n_p * n_jext * n_field;
#pragma omp parallel for schedule(static)
  for (long long o = 0; o < n_out; ++o) {
    const long long flat = sel ? sel[o] : o;
    const int f = (int)(flat % n_field);
    const int j = (int)((flat / n_field) % n_jext);
    const int e = (int)(flat / ((long long)n_field * n_jext));
    const double p = pext[e];
    const cd p0j((2.0 * j + 1.0) * pi * T, mu);
    cld a_psi(0.0L, 0.0L), a_phi(0.0L, 0.0L);
    acc_t s_psi = 0.0L, s_phi = 0.0L;
    for (int n = -n_max; n <= n_max; ++n) {
      const cd p0n((2.0 * n + 1.0) * pi * T, mu);
      const int nbar = n >= 0 ? n : -n - 1;
      const int m = j - n;
      const int mabs = m >= 0 ? m : -m;
      const double om = 2.0 * pi * (double)m * T;
      for (int i = 0; i < nq; ++i) {
        const double q = xq[i];
        const cd spsi = p0n * p0n + q * q;
        double Rp, Rdp;
        cd Dpsi;
        const double Zq = table_lookup(Zpsi + (size_t)nbar * t_nq, t_nq, t_lo, t_hi, t_interp, q * q);
        if (freg) {
          double RF, RFd;
          regulator_fermion(reg_kind, reg_order, k, zk, eta, q * q, &RF, &RFd);
          const double A = Zq * q + RF;
          Dpsi = (Zq * Zq) * (p0n * p0n) + A * A + m2psi[f];
          Rdp = 2.0 * A * RFd;
        } else {
          regulator(reg_kind, reg_order, k, zk, eta, q * q, &Rp, &Rdp);
          Dpsi = Zq * spsi + Rp + m2psi[f];
        }
        const cd Gpsi = 1.0 / Dpsi;
        const double condpsi = (std::abs(Dpsi - m2psi[f]) + std::fabs(m2psi[f])) / std::abs(Dpsi);
        cld c_psi(0.0L, 0.0L), c_phi(0.0L, 0.0L);
        acc_t sc_psi = 0.0L, sc_phi = 0.0L;
        for (int jc = 0; jc < nc; ++jc) {
          const double c = xc[jc];
          const double r2 = clamp0(p * p + q * q - 2.0 * p * q * c);
          const double sphi = om * om + r2;
          double Rb, Rdb;
          regulator(reg_kind, reg_order, k, zk, eta, r2, &Rb, &Rdb);
          const double Dphi =
              table_lookup(Zphi + (size_t)mabs * t_nq, t_nq, t_lo, t_hi, t_interp, r2) * sphi + Rb + m2phi[f];
          const double Gphi = 1.0 / Dphi;
          const double condphi = (std::fabs(Dphi - m2phi[f]) + std::fabs(m2phi[f])) / std::fabs(Dphi);
          const cd y1 = p0n * p0j / k2, y3 = spsi / k2;
          const double y2 = p * q * c / k2;
          cd P(0.0, 0.0);
          double Pabs = 0.0;
          int idx = 0;
          for (int a = 0; a <= 3; ++a)
            for (int b = 0; a + b <= 3; ++b)
              for (int cc = 0; a + b + cc <= 3; ++cc) {
                cd mono(coef[idx++], 0.0);
                for (int t = 0; t < a; ++t) mono *= y1;
                for (int t = 0; t < b; ++t) mono *= y2;
                for (int t = 0; t < cc; ++t) mono *= y3;
                P += mono;
                Pabs += std::abs(mono);
              }
          const cd t_psi = wc[jc] * P * Gphi, t_phi = -wc[jc] * P * Gphi * Gphi;
          c_psi += cld(t_psi.real(), t_psi.imag());
          c_phi += cld(t_phi.real(), t_phi.imag());
          sc_psi += (acc_t)(std::fabs(wc[jc] * Pabs * Gphi) * (1.0 + 3.0 * condpsi + condphi));
          sc_phi += (acc_t)(std::fabs(wc[jc] * Pabs * Gphi * Gphi) * (1.0 + 2.0 * condpsi + 2.0 * condphi));
        }
        const double W = wq[i] * q * q * Rdp;
        const cd w_psi = -2.0 * W * Gpsi * Gpsi * Gpsi, w_phi = W * Gpsi * Gpsi;
        a_psi += cld(w_psi.real(), w_psi.imag()) * c_psi;
        a_phi += cld(w_phi.real(), w_phi.imag()) * c_phi;
        s_psi += (acc_t)std::abs(w_psi) * sc_psi;
        s_phi += (acc_t)std::abs(w_phi) * sc_phi;
      }
    }
    const acc_t sc = (acc_t)prefactor * (acc_t)T;
    dpsi_re[o] = (double)(sc * a_psi.real()); dpsi_im[o] = (double)(sc * a_psi.imag());
    dphi_re[o] = (double)(sc * a_phi.real()); dphi_im[o] = (double)(sc * a_phi.imag());
    if (sens_psi) sens_psi[o] = (double)(fabsl(sc) * s_psi);
    if (sens_phi) sens_phi[o] = (double)(fabsl(sc) * s_phi);
  }
  return 0;
}

// =====================================================================================================
// Mass derivatives (Jacobian support).  Implicit time-steppers need dR_i/du_j (eq. 27;
// kernel option "AD"): for the loop integrals that is the derivative of the quadrature
// sum with respect to the mass term of its propagators.  Each function below is the term-by-term
// derivative of the sum its value twin above computes, d/dm2 (1/D^p) = -p/D^(p+1), written out plainly.
// sens_* = sum |term| (1 + sum over propagators of power (|D - m2| + |m2|)/|D|), as for the values.
// =====================================================================================================

// dchan[ch][f] = dI/dm2 at m2 = m2_channel:  -C [T] sum w q^(d-1) Rdot / D^2
int orc_lpa_dm2(int d, double T, int n_max, int reg_arg4d, double prefactor,
                int reg_kind, int reg_order, double k, double zk, double eta,
                int nq, const double* xq, const double* wq,
                int n_field, const double* rho, const double* u, const double* du,
                double* dchan, double* sens) {
  if (d < 1 || nq < 1 || n_field < 0 || T < 0 || n_max < 0 || k <= 0 || !dchan) return -1;
  const double pi = 3.14159265358979323846;
#pragma omp parallel for schedule(static)
  for (int f = 0; f < n_field; ++f) {
    const double m2c[2] = {u[f], u[f] + 2.0 * rho[f] * du[f]};
    for (int ch = 0; ch < 2; ++ch) {
      const double m2 = m2c[ch];
      acc_t acc = 0.0L, sn = 0.0L;
      const int n_lo = (T == 0.0) ? 0 : -n_max, n_hi = (T == 0.0) ? 0 : n_max;
      for (int n = n_lo; n <= n_hi; ++n) {
        const double wn = 2.0 * pi * (double)n * T;
        for (int i = 0; i < nq; ++i) {
          const double q = xq[i];
          const double s = wn * wn + q * q;
          const double sR = (T == 0.0 || reg_arg4d) ? s : q * q;
          double R, Rd;
          regulator(reg_kind, reg_order, k, zk, eta, sR, &R, &Rd);
          const double D = s + R + m2;
          const double term = -wq[i] * ipow(q, d - 1) * Rd / (D * D);
          acc += (acc_t)term;
          sn += (acc_t)(std::fabs(term) * (1.0 + 2.0 * (std::fabs(s + R) + std::fabs(m2)) / std::fabs(D)));
        }
      }
      const acc_t sc = (acc_t)prefactor * (T == 0.0 ? (acc_t)1.0 : (acc_t)T);
      dchan[(size_t)ch * n_field + f] = (double)(sc * acc);
      if (sens) sens[(size_t)ch * n_field + f] = (double)(fabsl(sc) * sn);
    }
  }
  return 0;
}

// dout[e][f] = d out / d m2_f with the same m2 in all three propagators:
//   C sum_i wq q^3 Rdot [ -2 G(q)^3 sum_j W'_ij G(s_ij) - G(q)^2 sum_j W'_ij G(s_ij)^2 ]
int orc_loop4d_twopoint_dm2(double prefactor, int reg_kind, int reg_order, double k, double zk, double eta,
                            int nq, const double* xq, const double* wq,
                            int nc, const double* xc, const double* wc,
                            const double* Zv, int Z_nq, double Z_lo, double Z_hi, int Z_interp,
                            const double* coef, int n_coef,
                            int n_field, const double* m2, int n_ext, const double* pext,
                            long long n_sel, const long long* sel,
                            double* dout, double* sens) {
  if (n_coef != 2 || nq < 1 || nc < 1 || n_field < 1 || n_ext < 1 || k <= 0 || !dout) return -1;
  const double k2 = k * k;
  const long long n_out = sel ? n_sel : (long long)n_ext * n_field;
#pragma omp parallel for schedule(static)
  for (long long o = 0; o < n_out; ++o) {
    const long long flat = sel ? sel[o] : o;
    const int e = (int)(flat / n_field), f = (int)(flat % n_field);
    const double p = pext[e], mm = m2[f];
    acc_t acc_q = 0.0L, sn = 0.0L;
    for (int i = 0; i < nq; ++i) {
      const double q = xq[i];
      const double sq = q * q;
      double Rq, Rdq;
      regulator(reg_kind, reg_order, k, zk, eta, sq, &Rq, &Rdq);
      const double Dq = table_lookup(Zv, Z_nq, Z_lo, Z_hi, Z_interp, sq) * sq + Rq + mm;
      const double Gq = 1.0 / Dq;
      const double condq = (std::fabs(Dq - mm) + std::fabs(mm)) / std::fabs(Dq);
      acc_t acc_c = 0.0L, sn_c = 0.0L;
      for (int j = 0; j < nc; ++j) {
        const double c = xc[j];
        const double s = clamp0(sq + p * p + 2.0 * q * p * c);
        double R, Rd;
        regulator(reg_kind, reg_order, k, zk, eta, s, &R, &Rd);
        const double D = table_lookup(Zv, Z_nq, Z_lo, Z_hi, Z_interp, s) * s + R + mm;
        const double G = 1.0 / D;
        const double poly = coef[0] + coef[1] * (q * p * c / k2);
        const double Wp = wc[j] * std::sqrt((1.0 - c) * (1.0 + c));
        const double t1 = -2.0 * Gq * Gq * Gq * G, t2 = -Gq * Gq * G * G;
        acc_c += (acc_t)(Wp * poly * (t1 + t2));
        const double apoly = std::fabs(coef[0]) + std::fabs(coef[1] * (q * p * c / k2));
        const double condc = (std::fabs(D - mm) + std::fabs(mm)) / std::fabs(D);
        sn_c += (acc_t)(std::fabs(Wp * apoly) * (std::fabs(t1) * (1.0 + 3.0 * condq + condc) +
                                                 std::fabs(t2) * (1.0 + 2.0 * condq + 2.0 * condc)));
      }
      acc_q += (acc_t)(wq[i] * q * q * q * Rdq) * acc_c;
      sn += (acc_t)std::fabs(wq[i] * q * q * q * Rdq) * sn_c;
    }
    dout[o] = (double)((acc_t)prefactor * acc_q);
    if (sens) sens[o] = (double)((acc_t)std::fabs(prefactor) * sn);
  }
  return 0;
}

// dpsi[p][j][f] = d out / d m2_psi_f = C T sum_n sum_q w q^2 Rdot (-2 G_psi^3) sum_c w P G_phi
// dphi[p][j][f] = d out / d m2_phi_f = C T sum_n sum_q w q^2 Rdot G_psi^2 sum_c w P (-G_phi^2)
// freg: as orc_matsubara3d.
int orc_matsubara3d_dm2(double T, int n_max, double prefactor, int reg_kind, int reg_order, double k, double zk, double eta,
                        int freg,
                        int nq, const double* xq, const double* wq,
                        int nc, const double* xc, const double* wc,
                        const double* Zpsi, const double* Zphi, int t_nq, int t_nfreq,
                        double t_lo, double t_hi, int t_interp,
                        const double* coef, int n_coef,
                        int n_field, const double* m2psi, const double* m2phi,
                        int n_p, const double* pext, int n_jext,
                        long long n_sel, const long long* sel,
                        double* dpsi, double* dphi, double* sens_psi, double* sens_phi) {
  if (n_coef != 20 || nq < 1 || nc < 1 || n_field < 1 || n_p < 1 || n_jext < 1 || k <= 0 || T <= 0) return -1;
  if (n_max + 1 > t_nfreq || n_jext - 1 + n_max + 1 > t_nfreq || !dpsi || !dphi) return -1;
  const double pi = 3.14159265358979323846;
  const double k2 = k * k;
  const long long n_out = sel ? n_sel : (long long)n_p * n_jext * n_field;
#pragma omp parallel for schedule(static)
  for (long long o = 0; o < n_out; ++o) {
    const long long flat = sel ? sel[o] : o;
    const int f = (int)(flat % n_field);
    const int j = (int)((flat / n_field) % n_jext);
    const int e = (int)(flat / ((long long)n_field * n_jext));
    const double p = pext[e];
    const double nuj = (2.0 * j + 1.0) * pi * T;
    acc_t a_psi = 0.0L, a_phi = 0.0L, s_psi = 0.0L, s_phi = 0.0L;
    for (int n = -n_max; n <= n_max; ++n) {
      const double nun = (2.0 * n + 1.0) * pi * T;
      const int nbar = n >= 0 ? n : -n - 1;
      const int m = j - n;
      const int mabs = m >= 0 ? m : -m;
      const double om = 2.0 * pi * (double)m * T;
      for (int i = 0; i < nq; ++i) {
        const double q = xq[i];
        const double spsi = nun * nun + q * q;
        double Rp, Rdp, Dpsi;
        const double Zq = table_lookup(Zpsi + (size_t)nbar * t_nq, t_nq, t_lo, t_hi, t_interp, q * q);
        if (freg) {
          double RF, RFd;
          regulator_fermion(reg_kind, reg_order, k, zk, eta, spsi, &RF, &RFd);
          const double A = Zq * std::sqrt(spsi) + RF;
          Dpsi = A * A + m2psi[f];
          Rdp = 2.0 * A * RFd;
        } else {
          regulator(reg_kind, reg_order, k, zk, eta, spsi, &Rp, &Rdp);
          Dpsi = Zq * spsi + Rp + m2psi[f];
        }
        const double Gpsi = 1.0 / Dpsi;
        const double condpsi = (std::fabs(Dpsi - m2psi[f]) + std::fabs(m2psi[f])) / std::fabs(Dpsi);
        acc_t c_psi = 0.0L, c_phi = 0.0L, sc_psi = 0.0L, sc_phi = 0.0L;
        for (int jc = 0; jc < nc; ++jc) {
          const double c = xc[jc];
          const double r2 = clamp0(p * p + q * q - 2.0 * p * q * c);
          const double sphi = om * om + r2;
          double Rb, Rdb;
          regulator(reg_kind, reg_order, k, zk, eta, sphi, &Rb, &Rdb);
          const double Dphi =
              table_lookup(Zphi + (size_t)mabs * t_nq, t_nq, t_lo, t_hi, t_interp, r2) * sphi + Rb + m2phi[f];
          const double Gphi = 1.0 / Dphi;
          const double condphi = (std::fabs(Dphi - m2phi[f]) + std::fabs(m2phi[f])) / std::fabs(Dphi);
          const double y1 = nun * nuj / k2, y2 = p * q * c / k2, y3 = spsi / k2;
          double P = 0.0, Pabs = 0.0;
          int idx = 0;
          for (int a = 0; a <= 3; ++a)
            for (int b = 0; a + b <= 3; ++b)
              for (int cc = 0; a + b + cc <= 3; ++cc) {
                const double mono = coef[idx++] * ipow(y1, a) * ipow(y2, b) * ipow(y3, cc);
                P += mono;
                Pabs += std::fabs(mono);
              }
          c_psi += (acc_t)(wc[jc] * P * Gphi);
          c_phi += (acc_t)(-wc[jc] * P * Gphi * Gphi);
          sc_psi += (acc_t)(std::fabs(wc[jc] * Pabs * Gphi) * (1.0 + 3.0 * condpsi + condphi));
          sc_phi += (acc_t)(std::fabs(wc[jc] * Pabs * Gphi * Gphi) * (1.0 + 2.0 * condpsi + 2.0 * condphi));
        }
        const double W = wq[i] * q * q * Rdp;
        a_psi += (acc_t)(-2.0 * W * Gpsi * Gpsi * Gpsi) * c_psi;
        a_phi += (acc_t)(W * Gpsi * Gpsi) * c_phi;
        s_psi += (acc_t)std::fabs(2.0 * W * Gpsi * Gpsi * Gpsi) * sc_psi;
        s_phi += (acc_t)std::fabs(W * Gpsi * Gpsi) * sc_phi;
      }
    }
    const acc_t sc = (acc_t)prefactor * (acc_t)T;
    dpsi[o] = (double)(sc * a_psi);
    dphi[o] = (double)(sc * a_phi);
    if (sens_psi) sens_psi[o] = (double)(fabsl(sc) * s_psi);
    if (sens_phi) sens_phi[o] = (double)(fabsl(sc) * s_phi);
  }
  return 0;
}

}  // extern "C"
