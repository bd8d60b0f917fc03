/* dfrg.h -- C ABI of the B200-native loop-integral library (FP64 only).
 *
 * What it computes: the momentum-loop integrals on the right-hand side of functional
 * renormalisation group flow equations, the "momentum integration of flow kernels"
 * of arxiv 2412.13043 (DiFfRG), sec. 5.3.2: fixed tensor-product
 * Gauss-Legendre quadrature over a radial loop momentum and 1-3 angles in the vacuum
 * (integrator type "Quadrature"), or over a spatial radial momentum, one angle and a
 * truncated Matsubara sum at finite temperature (type "Quadraturex0"), of
 *     d_t R_k  x  products of propagators G = 1/(Z s + R_k(s) + m^2)  x  dressings,
 * with the regulator shapes of PAPER.md:190-194 (eq. 14) and PAPER.md:178 (flat),
 * the propagator of PAPER.md:1915-1918 (eq. G.1) and dressing functions tabulated on
 * a logarithmic momentum grid.  Where the paper's interface
 * returns ONE integral per call (integrator.get<double>(k, args...))
 * this library evaluates a whole batch -- every field-grid point times every external
 * momentum -- per call.  The integrand families, measures, prefactors and loop
 * conventions are the readings listed in DESIGN.md ("Readings").
 *
 * Conventions common to all entry points
 *  - Arrays are FP64, contiguous.  In the `dfrg_integrate_*` functions every pointer inside
 *    the descriptors and in the argument list is a CUDA DEVICE pointer on the current device,
 *    owned by the caller; the library never allocates, frees or retains them.  In the
 *    `dfrg_integrate_*_host` functions the same pointers are HOST pointers (pinned memory
 *    gives asynchronous copies); the library stages them through a per-thread device arena.
 *  - Device entry points are asynchronous: they validate on the host, enqueue on `cuda_stream`
 *    (a cudaStream_t passed as void*, NULL = default stream) and return.  No hidden
 *    synchronisation.  Host entry points return after the outputs have landed in host memory.
 *  - Return value: a dfrg_status.  Nothing is written to any output on DFRG_EINVAL /
 *    DFRG_EUNSUPPORTED.  The library never throws across the ABI and has no CPU fallback.
 *  - Device pointers must be 8-byte aligned.  Tables and node arrays that are 16-byte aligned
 *    with a size that is a multiple of 16 bytes are staged into shared memory with TMA bulk
 *    copies; others with plain loads (same results).
 *  - Numerical special cases are not errors: a vanishing or negative propagator denominator
 *    gives whatever IEEE arithmetic gives; `dmin` reports it (signed minimum over all quadrature
 *    nodes and all propagators of an output of denominator / k^2; reading A4 in DESIGN.md).
 *    An exactly zero denominator yields NaN (the reciprocal is a Newton iteration on a hardware seed).
 *    NaN inputs: a NaN momentum or mass reaches the output through the Z s + m^2 terms of its denominators; the regulator
 *    term alone does not carry it (the device e^-x maps a NaN argument to 0, so R(NaN) = 0), which matters only where a
 *    caller inspects intermediate quantities -- the outputs that depend on the NaN input are NaN either way.
 *    Field points are independent outputs, also where the kernels batch: the two-point and Matsubara kernels invert the
 *    denominators of the TWO field points a thread owns (f and f + 128, resp. f + 256 of a field tile) through one product,
 *    1/(d_1 d_2 [d_3 d_4]) from one hardware seed.  A field point whose mass term has blown up -- NaN, infinite, or beyond
 *    1e150 (two-point) / 1e70 (Matsubara) in magnitude, where the product would overflow -- is detected from the masses
 *    before the loop starts and its thread inverts every denominator on its own: that field point gets what IEEE arithmetic
 *    gives for it, its partner its own regular value, as in the oracle
 *    (tests/test_gpu_parity.py::test_field_points_are_independent_outputs_also_where_reciprocals_are_batched).
 *    What remains coupled: a denominator D0 + m2 that is EXACTLY zero at a quadrature node (D0 and -m2 equal bit for bit;
 *    a mere sign change between nodes is not this case) yields NaN for the partner field point as well, and the partner's
 *    own dmin does not show it (data-dependent tests inside the hot loop were measured at 2-4 % of the kernel time and left
 *    out).  The field-independent part D0 of every denominator must stay below ~1e75 in magnitude (physical values lie
 *    between ~1e-3 k^2 and ~1e6 k^2).  dfrg_mats3d_desc::path = DFRG_M3_ONE_FIELD never batches across field points.
 *  - Mass derivatives (Jacobian support; the paper's "AD" kernels for implicit time-steppers, PAPER.md:713-723
 *    eq. 27 and PAPER.md:1842): every descriptor of a family with a field axis carries nullable output pointers
 *    for the derivative of each integral with respect to the mass term of its propagators,
 *    d/dm2 (1/D^p) = -p/D^(p+1) term by term on the same nodes.  NULL = not computed, no cost.
 *  - Deterministic: fixed thread -> node mapping, fixed reduction trees, no atomics.
 *  - Re-entrant; concurrent calls on different streams are allowed.
 */
#ifndef DFRG_H_
#define DFRG_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  DFRG_OK = 0,
  DFRG_EINVAL = -1,       /* null required pointer, non-positive size, T < 0, k <= 0, bad interp, wrong n_coef ... */
  DFRG_EUNSUPPORTED = -2, /* sizes beyond the shared-memory budget, unsupported dimension, not an sm_100 device */
  DFRG_ECUDA = -3,        /* CUDA runtime / launch error; see dfrg_last_cuda_error() */
  DFRG_ENOMEM = -4,       /* device arena allocation failed (host entry points only) */
  DFRG_ESCRATCH = -5      /* dfrg_integrate_twopoint_noalloc only: the call needs more scratch than the fixed array holds */
} dfrg_status;

const char* dfrg_strerror(int status);  /* static string */
int dfrg_last_cuda_error(void);         /* cudaError_t of the last DFRG_ECUDA on the calling thread */
int dfrg_version(void);                 /* 100*major + minor */
void dfrg_shutdown(void);               /* frees the calling thread's device arena (host entry points) */

/* Regulator R_k(s), s = squared momentum, x = s/k^2; Rdot = k dR/dk (k d/dk = -2x d/dx).
 *   DFRG_REG_LITIM:    R = (k^2 - s) Theta(k^2 - s),            Rdot = 2 k^2 Theta(k^2 - s), Theta(0) = 0
 *   DFRG_REG_EXP_POLY: R = k^2 exp(-sum_{i=1..order} x^i / i),  Rdot = 2 R (1 + sum_{i=1..order} x^i)       (eq. 14)
 * order in [1, 16] for EXP_POLY; ignored for LITIM.
 * Dressed regulator (the paper's RB / RBdot with a wave-function renormalisation; "only the
 * eta_i = -d_t Z_i/Z_i enter the flow equations"):  with Z_k = zk and eta = -k dZ_k/dk / Z_k
 *   R = zk R_shape,   Rdot = k d(Z_k R_shape)/dk = zk (Rdot_shape - eta R_shape)
 * in every propagator and in the insertion.  zk > 0 is required (DFRG_EINVAL otherwise: a zero-initialised struct is
 * rejected); zk = 1, eta = 0 gives the plain shapes.  Z_k dresses the regulator only, not the s term (reading A12/A20). */
/* Fermionic regulator (the paper's RF / RFdot; its finite-temperature and finite-density examples are
 * fermionic; the paper prints no fermionic shape -- DESIGN.md reading A25).  A fermion line of a
 * descriptor with fermion_reg = 1 is regulated on its Dirac structure, i pslash (1 + r_F), with (1 + r_F)^2 = 1 + r_B:
 *   R_F(s) = sqrt(s + R_shape(s)) - sqrt(s)      (momentum dimension one; flat shape: (k - sqrt(s)) Theta(k^2 - s))
 *   k dR_F/dk = Rdot_shape(s) / (2 sqrt(s + R_shape(s)))
 *   RF = zk R_F,  RFdot = zk (k dR_F/dk - eta R_F)
 * and has the denominator  D = Z^2 (s - sR) + (Z sqrt(sR) + RF(sR))^2 + m2  with the insertion  2 (Z sqrt(sR) + RF(sR)) RFdot(sR)
 * in place of  Z s + R(sR) + m2  and  Rdot(sR)   (sR = argument of the regulator: s, or its spatial part for "3D" regulators,
 * s - sR then being the squared time component; Z = the line's dressing table; m2 = the squared fermion mass).
 * With zk = 1, eta = 0 and Z = 1 the two switches describe the same function. */
typedef enum { DFRG_REG_LITIM = 0, DFRG_REG_EXP_POLY = 1 } dfrg_reg_kind;
typedef struct {
  int kind;
  int order;
  double k;
  double zk;
  double eta;
} dfrg_regulator;

/* S1 (host): Gauss-Legendre rule of order n mapped to [a, b]: x ascending, w > 0, sum w = b - a
 * ("quadrature rules of arbitrary order").  x_host, w_host: caller-owned HOST arrays of n doubles.
 * 1 <= n <= 4096.  Nodes are correct to 1 ulp; weights to 1 ulp for n <= 512 (the outermost weights of longer rules lose
 * digits to the factor 1 - x^2: ~3e-14 relative at n = 4096).  The rule is exactly symmetric about (a + b)/2 when a = -b. */
typedef enum { DFRG_RULE_GAUSS_LEGENDRE = 0 } dfrg_rule_kind;
int dfrg_quad_nodes(int rule_kind, int n, double a, double b, double* x_host, double* w_host);

typedef struct {
  const double* x; /* nodes   [n] */
  const double* w; /* weights [n] */
  int n;           /* 0 = axis unused */
} dfrg_rule;

/* Dressing function tabulated on a uniform grid in ln q:
 *   ln q_i = lnq_lo + i (lnq_hi - lnq_lo)/(n_q - 1),  v row-major [n_freq][n_q]; n_freq = 1 for 1-D tables.
 * Evaluated at a squared momentum s through l = log(s)/2, t = clamp((l - lnq_lo)/h, 0, n_q - 1):
 *   interp 3: 4-point Lagrange on the stencil i0..i0+3, i0 = clamp(floor(t) - 1, 0, n_q - 4)
 *   interp 1: linear between floor(t) and floor(t)+1 (the paper's interpolators)
 * Outside the grid the end value is returned.  The frequency index of a stacked table selects a row
 * exactly; there is no interpolation across it. */
typedef struct {
  const double* v;
  int n_q;
  int n_freq;
  double lnq_lo, lnq_hi;
  int interp;
} dfrg_table;

/* ---- LPA O(N) flow right-hand side (BASELINE.json configs 0 and 1) -------------------------------------
 *   flow[f] = (N - 1) I(u[f]) + I(u[f] + 2 rho[f] du[f])
 *   T == 0: I(m2) = prefactor sum_i w_i q_i^(d-1) Rdot(q_i^2) / (q_i^2 + R(q_i^2) + m2)
 *   T  > 0: I(m2) = prefactor T sum_{n=-n_max..n_max} sum_i w_i q_i^(d-1) Rdot(sR) / (s + R(sR) + m2),
 *           s = (2 pi n T)^2 + q_i^2,  sR = s if reg_arg4d else q_i^2      (Matsubara sum)
 * d = dimension of the radial integral (1..8): 4 in the vacuum config, 3 at finite T.
 * flow [n_field]; chan nullable [2][n_field] = I_pi, I_sigma; dmin nullable [n_field].
 * dchan (in the descriptor, nullable) [2][n_field] = dI/dm2 at m2 = u and at m2 = u + 2 rho du, from which
 *   dflow/du = (N-1) dchan[0] + dchan[1],  dflow/d(du) = 2 rho dchan[1].
 * Limits: (n_max + 1) * q.n <= 12288.
 * Fermionic statistics at chemical potential mu (statistics = DFRG_STAT_FERMION; requires T > 0 and reg_arg4d = 0,
 * the spatial "3D" regulators of the paper's finite-density example; the time component of a fermion
 * momentum is nu_n + i mu, PAPER.md:1947-1952 -- the paper writes p0f - i mu_q, the real part below is even in mu;
 * DESIGN.md reading A22):  nu_n = (2n+1) pi T,
 *   I(m2) = prefactor T sum_{n=-n_max-1..n_max} sum_i w_i q_i^(d-1) Rdot(q_i^2) Re[ 1/((nu_n + i mu)^2 + q_i^2 + R(q_i^2) + m2) ]
 * in the same combination flow = (N-1) I(u) + I(u + 2 rho du) (a single quark loop: N = 1, du = 0; signs and
 * degeneracies go into prefactor); dchan = dI/dm2 = -prefactor T sum sum w q^(d-1) Rdot Re[1/(...)^2];
 * dmin = min over nodes and both channels of |denominator| / k^2.  Limit: (n_max + 1) * q.n <= 6144. */
typedef enum { DFRG_STAT_BOSON = 0, DFRG_STAT_FERMION = 1 } dfrg_statistics;
/* Number of Matsubara terms on either side for a cut-off in the time direction:
 *   DFRG_DOMAIN_X0 ("Quadraturex0": the domain scales with k):   n_max = ceil(extent * k / (2 pi T)),  extent in units of k
 *   DFRG_DOMAIN_Q0 ("Quadratureq0": fixed, bounded domain):       n_max = ceil(extent / (2 pi T)),      extent in units of T's
 * Host function.  Returns n_max >= 0, or DFRG_EINVAL (T <= 0, k <= 0, extent < 0, unknown domain, n_max beyond 2^30). */
typedef enum { DFRG_DOMAIN_X0 = 0, DFRG_DOMAIN_Q0 = 1 } dfrg_time_domain;
int dfrg_matsubara_n_max(int domain, double T, double k, double extent);

typedef struct {
  int d;
  double T;
  int n_max;
  int reg_arg4d;
  double N;
  double prefactor;
  dfrg_regulator reg;
  dfrg_rule q;
  double* dchan; /* nullable output [2][n_field] */
  int statistics; /* DFRG_STAT_BOSON (0): the sums above.  DFRG_STAT_FERMION (1): see below */
  double mu;      /* chemical potential (fermionic statistics only; must be 0 otherwise) */
  int fermion_reg; /* fermionic statistics only (must be 0 otherwise).  0: the loop is regulated with R / Rdot as written above.
                      1: with RF / RFdot (see dfrg_regulator):  D = (nu_n + i mu)^2 + (q_i + RF(q_i^2))^2 + m2,
                      Rdot(q_i^2) -> 2 (q_i + RF(q_i^2)) RFdot(q_i^2) */
} dfrg_lpa_desc;

int dfrg_integrate_lpa(const dfrg_lpa_desc* D, int n_field, const double* rho, const double* u, const double* du,
                       double* flow, double* chan, double* dmin, void* cuda_stream);
int dfrg_integrate_lpa_host(const dfrg_lpa_desc* D, int n_field, const double* rho, const double* u,
                            const double* du, double* flow, double* chan, double* dmin);
/* Several temperatures in ONE launch (BASELINE.json config 1 runs T in {0.05, 0.1, 0.2, 0.5} k on the same field grid):
 * the integrals of dfrg_integrate_lpa with D->T, D->n_max replaced by T_host[t], n_max_host[t] for t < n_T (HOST arrays,
 * read before the call returns; 1 <= n_T <= 16, else DFRG_EUNSUPPORTED; every entry must satisfy the limits above).
 * Outputs gain a leading axis: flow [n_T][n_field]; chan, D->dchan (nullable) [n_T][2][n_field]; dmin (nullable)
 * [n_T][n_field].  Entry t is bit-identical to a single call at (T_host[t], n_max_host[t]).  Device pointers, asynchronous. */
int dfrg_integrate_lpa_batch(const dfrg_lpa_desc* D, int n_T, const double* T_host, const int* n_max_host, int n_field,
                             const double* rho, const double* u, const double* du, double* flow, double* chan,
                             double* dmin, void* cuda_stream);
int dfrg_integrate_lpa_batch_host(const dfrg_lpa_desc* D, int n_T, const double* T_host, const int* n_max_host, int n_field,
                                  const double* rho, const double* u, const double* du, double* flow, double* chan,
                                  double* dmin);   /* host pointers throughout; returns when the outputs have landed */

/* ---- 4-D vacuum loops (BASELINE.json configs 2 and 3; angles cos1, cos2, phi of PAPER.md:1837-1840) ------
 * DFRG_LOOP_TWOPOINT (tab[0] = Z, n_coef = 2, axes q, cos1; cos2/phi unused, their measure is in prefactor):
 *   out[e][f] = prefactor sum_i wq_i q_i^3 Rdot(q_i^2) G(q_i^2; f)^2
 *                 sum_j wc_j sqrt(1 - c_j^2) (coef[0] + coef[1] q_i p_e c_j / k^2) G(s_ij; f)
 *   s_ij = max(q_i^2 + p_e^2 + 2 q_i p_e c_j, 0),   G(s; f) = 1/(Z(s) s + R(s) + m2[f]);  ext = |p|[n_ext]
 * DFRG_LOOP_THREEPOINT (tab = Z_A, Z_c, lambda3 sharing one grid, n_coef = 35, axes q, cos1, cos2, phi; n_field = 0):
 *   ext = (|p1|, |p2|, alpha)[n_ext];  q.p1 = q |p1| c1,  q.p2 = q |p2| (cos(alpha) c1 + sin(alpha) sqrt(1-c1^2) c2)
 *   s_a = |q + p1|^2, s_b = |q - p2|^2, s_c = |p1 + p2|^2,  G_A(s) = 1/(Z_A(s) s + R(s))
 *   Lam = l3((p1^2+q^2+s_a)/3) l3((p2^2+q^2+s_b)/3) l3((s_c+s_a+s_b)/3)
 *   P = sum_{a+b+c<=4} coef[idx(a,b,c)] (q^2/k^2)^a (q.p1/k^2)^b (q.p2/k^2)^c,  idx: a outermost, then b, then c, ascending
 *   out[e] = prefactor sum_q w q^3 Rdot(q^2) G_A(q^2) sum_c1 w sqrt(1-c1^2) sum_c2 w sum_phi w  G_A(s_a) G_A(s_b) Lam P
 *   (the integrand is phi-independent: the phi axis contributes sum_phi w; Z_c is accepted and not used.)
 * DFRG_LOOP_FOURPOINT (tab = Z_A, Z_c, lambda3 sharing one grid, n_coef = 70, axes q, cos1, cos2, phi; n_field = 0): a box
 *   with genuine three-angle kinematics ("Angles" -> 3: cos1, cos2, phi; four-gluon vertex configurations,
 *   PAPER.md:334) plus a ghost box; every node of the (q, c1, c2, phi) grid is a distinct evaluation.  DESIGN.md reading A21.
 *   ext = (|p1|, |p2|, |p3|, alpha, beta, gamma)[n_ext]:
 *     p1 = |p1| (1,0,0,0), p2 = |p2| (cos al, sin al, 0, 0), p3 = |p3| (cos be, sin be cos ga, sin be sin ga, 0)
 *     q = q (c1, s1 c2, s1 s2 cos phi, s1 s2 sin phi), s_i = sqrt(1 - c_i^2);  u_i = q.p_i
 *   internal lines q, q+p1, q+p1+p2, q+p1+p2+p3:  s_a = q^2 + p1^2 + 2 u1,  s_b = q^2 + |p1+p2|^2 + 2 (u1+u2),
 *     s_d = q^2 + |p1+p2+p3|^2 + 2 (u1+u2+u3)   (each clamped at 0)
 *   T_A = G_A(q^2) G_A(s_a) G_A(s_b) G_A(s_d) l3((q^2+p1^2+s_a)/3) l3((s_a+p2^2+s_b)/3) l3((s_b+p3^2+s_d)/3)
 *         l3((s_d+|p1+p2+p3|^2+q^2)/3) P_A,        G_X(s) = 1/(Z_X(s) s + R(s))
 *   T_c = G_c(q^2) G_c(s_a) G_c(s_b) G_c(s_d) P_c
 *   P_X = sum_{a+b+c+d<=3} coef_X[idx(a,b,c,d)] (q^2/k^2)^a (u1/k^2)^b (u2/k^2)^c (u3/k^2)^d, idx: a outermost, then b, c, d,
 *         ascending; coef = [coef_A (35) | coef_c (35)]
 *   out[e] = prefactor sum_q w q^3 Rdot(q^2) sum_c1 w sqrt(1-c1^2) sum_c2 w sum_phi w (T_A + T_c)
 * DFRG_LOOP_THREEPOINT_TAB3D (tab[0] = Z_A, tab3d = lambda3(S0^2, a, s); n_coef = 35; n_field = 0): the three-point family
 *   above with every vertex factor looked up in the 3-D table at the vertex coordinates of its squared leg momenta
 *   (k1, k2, k3) (the paper's vertex grids "for the average momentum S0 and two angles a, s"; reading A23):
 *     S0^2 = (k1 + k2 + k3)/6,  a = sqrt(3) (k2 - k1)/(6 S0^2),  s = (k1 + k2 - 2 k3)/(6 S0^2)   (S0 = 0: a = s = 0)
 *     Lam = l3(p1^2, q^2, s_a) l3(p2^2, q^2, s_b) l3(s_c, s_a, s_b)      table axes: 0 = S0^2, 1 = a, 2 = s
 *   tab[1], tab[2] and ext_outer are ignored.
 * out, dmin (nullable): [n_ext][max(n_field, 1)].
 * Limits: four-point cos2.n <= 512, phi.n <= 4096, q.n * cos1.n <= 65536; two-point q.n * cos1.n <= 12288; three-point q.n * cos1.n <= 65536, every tab[i].n_q <= 1024. */
typedef enum {
  DFRG_LOOP_TWOPOINT = 0,
  DFRG_LOOP_THREEPOINT = 1,
  DFRG_LOOP_FOURPOINT = 2,
  DFRG_LOOP_THREEPOINT_TAB3D = 3
} dfrg_loop_family;
/* Dressing function on a 3-D grid, trilinear (the paper's LinearInterpolator3D with Log x Lin x Lin or Log x Log x Lin
 * coordinates): v row-major [n[0]][n[1]][n[2]], axis a uniform in its coordinate c_a between lo[a]
 * and hi[a] with n[a] >= 2 points; c_a = log(x_a)/2 for a logarithmic axis (x_a = SQUARED momentum, as dfrg_table) and
 * c_a = x_a for a linear one.  t_a = clamp((c_a - lo_a)/h_a, 0, n_a - 1), cell min(floor(t_a), n_a - 2); the value is the
 * trilinear combination of the 8 corners; outside the grid the edge value.  n[0] n[1] n[2] <= 12288. */
typedef struct {
  const double* v;
  int n[3];
  double lo[3], hi[3];
  int is_log[3];
} dfrg_table3d;
typedef struct {
  int family;
  double prefactor;
  dfrg_regulator reg;
  dfrg_rule q, cos1, cos2, phi;
  dfrg_table tab[3];
  const double* coef;
  int n_coef;
  int ext_outer; /* three-point only; 0 or 1: no layout promised.  G >= 2: the caller promises a product grid,
                    n_ext = G S and ext[a S + r] = (|p1|_a, |p2|_r, alpha_r) for a < G, r < S (the paper's vertex
                    grids), which lets the library share everything that depends on |p1| alone or on
                    (|p2|, alpha) alone.  The promise is checked on the device; if it does not hold the general
                    path runs and the results are the same.  Ignored (general path) if G > 256 or cos2.n > 512. */
  double* dout_dm2; /* two-point only, nullable output [n_ext][n_field]: d out[e][f] / d m2[f] (the same m2 sits in all
                       three propagators):  prefactor sum_i wq q^3 Rdot [-2 G(q)^3 A_i - G(q)^2 B_i],
                       A_i = sum_j W'_ij G(s_ij), B_i = sum_j W'_ij G(s_ij)^2.  Must be NULL for the three- and four-point families. */
  dfrg_table3d tab3d; /* DFRG_LOOP_THREEPOINT_TAB3D only */
} dfrg_loop4d_desc;

int dfrg_integrate_loop4d(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext, const double* ext,
                          double* out, double* dmin, void* cuda_stream);
int dfrg_integrate_loop4d_host(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext,
                               const double* ext, double* out, double* dmin);

/* ---- Two-point loop for callers that cannot allocate device memory ------------------------------------------
 * Every other device entry point of this library takes the scratch of its kernels (partial sums of the fixed-order
 * reduction, denominator minima) from a library-owned CUDA memory pool, which now and then has to grow, i.e. allocate.
 * That is not acceptable to every caller: a solver that has given all device memory to its own allocator and wants no
 * second one beside it, a thread that must never block on the driver's allocation lock (callbacks, latency-bound
 * loops), a job under a device-memory cap where an allocation in the middle of a flow may fail.  This entry point is
 * the two-point family (DFRG_LOOP_TWOPOINT; same descriptor, same arguments, same integrand, PAPER.md:1007-1030 and the
 * "Two-point" block above) with NO allocation of any kind on the device: it calls neither cudaMalloc / cudaFree nor
 * their stream-ordered or pooled relatives, nor any library routine that does.  The kernels and the launch plan are the
 * ones dfrg_integrate_loop4d uses, so out / dmin / D->dout_dm2 are bit-identical to that call's.
 *
 * Where the scratch lives: in a fixed array of DFRG_NOALLOC_SCRATCH_BYTES that is part of the library image.  Every GPU
 * on which the library is loaded carries it from load to process exit, used or not; that is the price of the guarantee.
 * The limit: the call needs
 *     8 * ( 4 U + 2  +  slots * (dout_dm2 ? 2 : 1) * n_ext * n_field )  bytes,
 *     U = ceil(n_field / tile) * n_ext * ceil(q.n / QC),  tile = 256 (128 if n_field <= 128),
 *     QC = min(8, q.n, floor(2048 / cos1.n)),  slots <= 2 + ceil(q.n / QC) * (number of SMs) / U  (CTAs sharing one output),
 * about 0.6 MB for BASELINE.json config 2 with derivatives (64 momenta x 256 field points, 128 x 32 nodes).  A call
 * that needs more returns DFRG_ESCRATCH before anything is enqueued and writes nothing; use dfrg_integrate_loop4d then.
 *
 * First call on a device: looks up the device address of the array and raises the kernels' shared-memory limit (two
 * CUDA runtime queries, a few host-side table entries).  Make this first call outside any stream capture; later calls
 * only enqueue the two kernels.
 *
 * Sharing: there is ONE array per device, and every call on that device uses it from its start.  Two calls whose kernels
 * can overlap on the GPU (different streams without an ordering between them, or two host threads) race on it and both
 * results are garbage: order such calls on one stream or with events.  The array keeps whatever the last call left in
 * it; no call depends on its contents (every entry that is read has been written by the same call before), so there is
 * nothing to clear between calls.
 *
 * Other return values as dfrg_integrate_loop4d; D->family must be DFRG_LOOP_TWOPOINT (DFRG_EINVAL otherwise). */
#define DFRG_NOALLOC_SCRATCH_BYTES (8u * 1024u * 1024u)
int dfrg_integrate_twopoint_noalloc(const dfrg_loop4d_desc* D, int n_field, const double* m2, int n_ext,
                                    const double* ext, double* out, double* dmin, void* cuda_stream);

/* ---- 3-D spatial momentum + Matsubara sum (BASELINE.json config 4; "Quadraturex0") -------
 *   nu_n = (2n+1) pi T (loop fermion, n = -n_max..n_max; external fermion index j = 0..n_jext-1)
 *   boson line (nu_j - nu_n, p - q): m = j - n, om_m = 2 pi m T, r^2 = max(p^2 + q^2 - 2 p q c, 0)
 *   s_psi = nu_n^2 + q^2,  s_phi = om_m^2 + r^2
 *   G_psi = 1/(Z_psi(q^2; row nbar) s_psi + R(s_psi) + m2_psi[f]),  nbar = n >= 0 ? n : -n-1
 *   G_phi = 1/(Z_phi(r^2; row |m|) s_phi + R(s_phi) + m2_phi[f])
 *   P = sum_{a+b+c<=3} coef[idx(a,b,c)] y1^a y2^b y3^c,  y1 = nu_n nu_j/k^2, y2 = p q c/k^2, y3 = s_psi/k^2   (n_coef = 20)
 *   out[p][j][f] = prefactor T sum_n sum_q w q^2 Rdot(s_psi) G_psi^2 sum_c w P G_phi
 * Performance note: a cos1 rule of 8 k nodes that is EXACTLY symmetric (x_c = -x_{n-1-c}, equal weights: what dfrg_quad_nodes
 * returns for [-1, 1]) takes a faster moment loop (checked on the device; any other rule gives the same sums at ~10 % more time).
 * tab_psi and tab_phi share n_q, lnq_lo, lnq_hi, interp; rows needed: tab_psi.n_freq > n_max,
 * tab_phi.n_freq > n_jext - 1 + n_max.  out, dmin (nullable): [n_p][n_jext][n_field].
 * Limits: q.n * cos1.n <= 6144, table n_q <= 1024. */
typedef struct {
  double T;
  int n_max;
  double prefactor;
  dfrg_regulator reg;
  dfrg_rule q, cos1;
  dfrg_table tab_psi, tab_phi;
  const double* coef;
  int n_coef;
  double* dout_dm2_psi; /* nullable output [n_p][n_jext][n_field]: d out / d m2_psi[f]  (G_psi^2 -> -2 G_psi^3) */
  double* dout_dm2_phi; /* nullable output [n_p][n_jext][n_field]: d out / d m2_phi[f]  (G_phi   -> -G_phi^2)   */
  int reg_arg4d;        /* 1: R, Rdot at the 4-momentum squared (s_psi, s_phi) as written above (BASELINE.json config 4);
                           0: spatial ("3D") regulators R(q^2), Rdot(q^2) on the fermion line and R(r^2) on the boson line */
  double mu;            /* chemical potential (reading A24).  mu != 0 needs reg_arg4d = 0 and out_im:
                           every fermion leg carries nu + i mu (loop nu_n + i mu, external nu_j + i mu; the boson line carries
                           their difference and is unchanged), so s_psi = (nu_n + i mu)^2 + q^2, y1 = (nu_n + i mu)(nu_j + i mu)/k^2
                           and y3 = s_psi/k^2 are complex and so is the result: out = real part, out_im = imaginary part
                           (out(-mu) = conj out(mu): the paper writes p0f - i mu_q).  dmin = min(|D_psi|, D_phi)/k^2.
                           The mass derivatives are complex too: dout_dm2_psi / dout_dm2_phi receive the real parts and need
                           their partners dout_dm2_psi_im / dout_dm2_phi_im (DFRG_EINVAL otherwise).  n_jext <= 32 and
                           128 n_jext (2 n_max + 1) + 4096 (n_max + 1) bytes of shared memory must fit (else DFRG_EUNSUPPORTED). */
  double* out_im;       /* nullable unless mu != 0; output [n_p][n_jext][n_field] (zero-filled when mu == 0) */
  double* dout_dm2_psi_im; /* imaginary parts of the mass derivatives: nullable unless mu != 0 and the real part is requested; */
  double* dout_dm2_phi_im; /* zero-filled when mu == 0 */
  int path;             /* kernel-path selection, an OR of dfrg_mats3d_path bits; 0 = the library's own choice.  Every path
                           computes the same sums (the tests run them all on the same inputs); the field exists for testing
                           and tuning and is part of the descriptor so that the call stays free of global state. */
  int fermion_reg;      /* 0: the fermion line is regulated with R / Rdot as written above (BASELINE.json config 4).
                           1: with RF / RFdot on its Dirac structure (see dfrg_regulator; reading A25):
                              A = Z_psi sqrt(sR) + RF(sR),  sR = s_psi (reg_arg4d = 1) or q^2 (reg_arg4d = 0)
                              G_psi = 1/(Z_psi^2 (s_psi - sR) + A^2 + m2_psi[f]),   Rdot(sR) -> 2 A RFdot(sR)
                              (s_psi - sR = (nu_n + i mu)^2 for spatial regulators, 0 otherwise); the boson line is unchanged. */
} dfrg_mats3d_desc;
typedef enum {
  DFRG_M3_AUTO = 0,
  DFRG_M3_ROW_STREAMING = 1,      /* the kernel without the moment factorisation (the library's choice for n_jext > 32) */
  DFRG_M3_ANY_SHAPE = 2,          /* the any-shape moment kernel even where a compile-time-specialised one exists */
  DFRG_M3_PLAIN_MOMENTS = 4,      /* plain moment loop even if the cos rule is exactly symmetric */
  DFRG_M3_ONE_FIELD = 8,          /* one field point per thread (512-thread CTAs) where the default is two */
  DFRG_M3_GROUPS_4 = 16,          /* row-streaming kernel: 4 consumer groups per CTA (default 6) */
  DFRG_M3_GROUPS_7 = 32           /* row-streaming kernel: 7 consumer groups per CTA */
} dfrg_mats3d_path;

int dfrg_integrate_matsubara3d(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi, const double* m2_phi,
                               int n_p, const double* p, int n_jext, double* out, double* dmin, void* cuda_stream);
int dfrg_integrate_matsubara3d_host(const dfrg_mats3d_desc* D, int n_field, const double* m2_psi,
                                    const double* m2_phi, int n_p, const double* p, int n_jext, double* out,
                                    double* dmin);

#ifdef __cplusplus
}
#endif
#endif /* DFRG_H_ */
