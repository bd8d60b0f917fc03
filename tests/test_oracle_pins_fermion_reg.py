"""Pins for the fermionic regulator RF / RFdot (PAPER.md:968-975 names the four functions RB, RF, RBdot, RFdot;
DESIGN.md reading A25: (sqrt(s) + R_F)^2 = s + R_B on the Dirac structure) and for the fermion lines regulated with it
(`freg = 1` of orc_lpa_fermion, orc_matsubara3d, orc_matsubara3d_mu and their mass-derivative twins), against things
other than the oracle:
  * the shape: the defining relation to the pinned bosonic shape; the flat fermionic regulator (k - |p|) Theta; RFdot
    against mpmath differentiation in k of Z(k) R_F(k, s) with a running Z(k) = zk (k/k0)^-eta;
  * flat regulator on [0,k]: the textbook fermionic threshold function (2 k^(d+2)/d) (1 - eta/(d+1)) / ... -- the factor
    differs from the bosonic 1 - eta/(d+2) -- times the pinned truncated fermionic Matsubara sum; its m2 derivative;
  * zk != 1 (where (q + zk R_F)^2 is NOT q^2 + zk R_B), exponential shape: mpmath quadrature of the continuum radial
    integral with mpmath's own k-derivative;
  * zk = 1, eta = 0, Z = 1: the fermionic and the bosonic regularisation of a line are the same function;
  * Matsubara family: heavy-mass weight integrals with Z_psi != 1 (mpmath), the full integrand against scipy adaptive
    quadrature (4-D argument and spatial + chemical potential), mass derivatives against five-point finite differences.
CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_2412_13043_b200 import inputs
from test_oracle_pins_fermion import truncated_fermi_sum

PI = math.pi


# ---- the shape ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind,order", [(oracle.REG_LITIM, 1), (oracle.REG_EXP_POLY, 1), (oracle.REG_EXP_POLY, 2),
                                        (oracle.REG_EXP_POLY, 8)])
def test_rf_squares_to_the_bosonic_shape(kind, order):
    """(sqrt(s) + R_F)^2 - s = R_B  (the relation (1 + r_F)^2 = 1 + r_B), with R_B from the pinned bosonic regulator (P5),
    and 2 (sqrt(s) + R_F) k dR_F/dk = RBdot."""
    k = 1.3
    for s in (0.0, 1e-8, 0.02, 0.5, 1.0, 1.69 - 1e-9, 1.7, 3.0, 9.0):
        RB, RBd = oracle.regulator(kind, order, k, s)
        RF, RFd = oracle.regulator_fermion(kind, order, k, s)
        assert abs((math.sqrt(s) + RF) ** 2 - s - RB) <= 4e-16 * (s + RB)
        assert abs(2 * (math.sqrt(s) + RF) * RFd - RBd) <= 4e-16 * max(RBd, 1e-300) + 1e-300


def test_rf_flat_is_the_flat_fermionic_regulator():
    k = 0.8
    for q in (0.0, 0.1, 0.5, 0.79):
        RF, RFd = oracle.regulator_fermion(oracle.REG_LITIM, 1, k, q * q)
        assert abs(RF - (k - q)) < 1e-15 and abs(RFd - k) < 1e-15        # r_F = (1/sqrt(x) - 1) Theta(1 - x)
    assert oracle.regulator_fermion(oracle.REG_LITIM, 1, k, k * k) == (0.0, 0.0)
    assert oracle.regulator_fermion(oracle.REG_LITIM, 1, k, 2.0) == (0.0, 0.0)


@pytest.mark.parametrize("order", [1, 2, 8])
def test_rfdot_vs_mpmath_total_derivative(order):
    """RFdot = k d/dk [Z(k) R_F(k, s)] with Z(k) = zk (k/k0)^-eta, i.e. eta = -k dZ/dk / Z, at k = k0."""
    mp.mp.dps = 40
    k0, zk, eta = 1.1, 1.3, 0.27

    def dressed(kk, s):
        x = s / kk ** 2
        RB = kk ** 2 * mp.exp(-sum(x ** i / i for i in range(1, order + 1)))
        return zk * (kk / k0) ** (-eta) * (mp.sqrt(s + RB) - mp.sqrt(s))
    for s in (0.0, 0.3, 1.21, 2.5, 6.0):
        ref = k0 * mp.diff(lambda kk: dressed(kk, mp.mpf(s)), mp.mpf(k0))
        RF, RFd = oracle.regulator_fermion(oracle.REG_EXP_POLY, order, k0, s, zk=zk, eta=eta)
        assert abs(RF - float(dressed(mp.mpf(k0), mp.mpf(s)))) <= 1e-15 * (1 + RF)
        assert abs(RFd - float(ref)) <= 1e-14 * abs(float(ref)) + 1e-18


# ---- fermionic LPA loop ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("d", [3, 4])
@pytest.mark.parametrize("T,mu,n_max", [(0.1, 0.3, 10), (0.3, 0.0, 4)])
def test_fermionic_threshold_function_flat(d, T, mu, n_max):
    """Flat fermionic regulator, zk = 1: q + R_F = k on [0,k], D = (nu + i mu)^2 + k^2 + m2, insertion 2 k (k - eta (k - q)):
    int_0^k q^(d-1) 2k (k(1 - eta) + eta q) dq = (2 k^(d+2)/d) (1 - eta/(d+1))  -- the fermionic threshold-function factor."""
    mp.mp.dps = 30
    k, C, eta = 1.1, 0.37, 0.4
    xq, wq = oracle.gl_rule(32, 0.0, k)
    m2 = np.array([-0.4, 0.0, 0.3, 2.5, 40.0])
    I, dI, dmin, sens, sens_d = oracle.lpa_fermion(d, T, n_max, mu, C, oracle.REG_LITIM, 1, k, xq, wq, m2, eta=eta, freg=1)
    Ib = oracle.lpa_fermion(d, T, n_max, mu, C, oracle.REG_LITIM, 1, k, xq, wq, m2, eta=eta, freg=0)[0]
    for j, m in enumerate(m2):
        E2 = k * k + m
        rad = (2 * k ** (d + 2) / d) * (1 - eta / (d + 1))
        ref = C * rad * truncated_fermi_sum(E2, T, mu, n_max)
        assert abs(I[j] - float(ref)) <= 1e-13 * sens[j], (j, I[j], float(ref))
        dref = C * rad * mp.diff(lambda e2: truncated_fermi_sum(e2, T, mu, n_max), mp.mpf(E2))
        assert abs(dI[j] - float(dref)) <= 1e-12 * sens_d[j]
        nu0 = PI * T
        assert abs(dmin[j] - abs(complex(nu0 * nu0 - mu * mu + E2, 2 * nu0 * mu)) / (k * k)) < 1e-13 * (1 + dmin[j])
        # the bosonic regularisation of the same line has the factor 1 - eta/(d+2): the two switches are told apart
        assert abs(Ib[j] / I[j] - (1 - eta / (d + 2)) / (1 - eta / (d + 1))) < 1e-12


def test_fermionic_loop_dressed_exp_vs_mpmath_quadrature():
    """zk != 1: (q + zk R_F)^2 differs from q^2 + zk R_B.  Continuum radial integral by mpmath, the k-derivative by mpmath."""
    mp.mp.dps = 25
    k, T, mu, n_max, d, C, zk, eta = 1.0, 0.15, 0.5, 8, 3, 1.0, 1.25, 0.15
    xq, wq = oracle.gl_rule(128, 0.0, 8.0 * k)
    m2 = np.array([0.2, 1.5])
    I, dI, _, sens, _ = oracle.lpa_fermion(d, T, n_max, mu, C, oracle.REG_EXP_POLY, 1, k, xq, wq, m2, zk=zk, eta=eta, freg=1)

    def RFd(kk, q):      # Z(k) R_F(k, q^2), Z(k) = zk (k/k0)^-eta with k0 = k
        return zk * (kk / k) ** (-eta) * (mp.sqrt(q * q + kk * kk * mp.exp(-q * q / (kk * kk))) - q)
    for j, m in enumerate(m2):
        def integrand(q):
            A = q + RFd(mp.mpf(k), q)
            ins = 2 * A * k * mp.diff(lambda kk: RFd(kk, q), mp.mpf(k))
            return q ** (d - 1) * ins * truncated_fermi_sum(A * A + m, T, mu, n_max)
        ref = C * mp.quad(integrand, [0, 0.5, 1, 2, 4, 8])
        assert abs(I[j] / float(ref) - 1) < 1e-11
    # and it is not the bosonic dressing of the same line
    Ib = oracle.lpa_fermion(d, T, n_max, mu, C, oracle.REG_EXP_POLY, 1, k, xq, wq, m2, zk=zk, eta=eta, freg=0)[0]
    assert np.all(np.abs(Ib / I - 1) > 1e-3)


@pytest.mark.parametrize("kind,order", [(oracle.REG_LITIM, 1), (oracle.REG_EXP_POLY, 1), (oracle.REG_EXP_POLY, 8)])
def test_fermionic_equals_bosonic_regularisation_when_undressed(kind, order):
    """zk = 1, eta = 0 (and Z = 1): (q + R_F)^2 = q^2 + R_B and 2 (q + R_F) k dR_F/dk = RBdot, so freg = 1 is freg = 0."""
    k, T, mu = 0.9, 0.12, 0.4
    xq, wq = oracle.gl_rule(40, 0.0, 6.0 * k)
    m2 = np.array([-0.2, 0.1, 3.0])
    a = oracle.lpa_fermion(3, T, 6, mu, 0.7, kind, order, k, xq, wq, m2, freg=1)
    b = oracle.lpa_fermion(3, T, 6, mu, 0.7, kind, order, k, xq, wq, m2, freg=0)
    assert np.all(np.abs(a[0] - b[0]) <= 1e-14 * b[3]) and np.all(np.abs(a[1] - b[1]) <= 1e-14 * b[4])
    assert np.all(np.abs(a[2] - b[2]) <= 1e-14 * (1 + b[2]))


# ---- Matsubara family -----------------------------------------------------------------------------------------------
def monomial_order(deg=3):
    return [(a, b, c) for a in range(deg + 1) for b in range(deg + 1 - a) for c in range(deg + 1 - a - b)]


def run4d(c, rq, rc, **over):
    a = dict(c)
    a.update(over)
    return oracle.matsubara3d(a["T"], a["n_max"], a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], *rq, *rc,
                              a["Zpsi"], a["Zphi"], a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"], a["m2psi"], a["m2phi"],
                              a["pext"], a["n_jext"], want_sens=True, zk=a.get("zk", 1.0), eta=a.get("eta", 0.0),
                              freg=a.get("freg", 0))


def run3d(c, rq, rc, mu, **over):
    a = dict(c)
    a.update(over)
    return oracle.matsubara3d_mu(a["T"], a["n_max"], mu, a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], *rq, *rc,
                                 a["Zpsi"], a["Zphi"], a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"], a["m2psi"],
                                 a["m2phi"], a["pext"], a["n_jext"], want_sens=True, zk=a.get("zk", 1.0),
                                 eta=a.get("eta", 0.0), freg=a.get("freg", 0))


@pytest.mark.parametrize("kind", [oracle.REG_LITIM, oracle.REG_EXP_POLY])
def test_matsubara_fermionic_equals_bosonic_when_undressed_and_Zpsi_is_one(kind):
    c = inputs.config4(n_field=3, n_p=2, n_jext=2, T_over_k=0.2)
    ones = np.ones_like(c["Zpsi"])
    rq, rc = oracle.gl_rule(12, 0, 5), oracle.gl_rule(6, -1, 1)
    kw = dict(n_max=3, reg_kind=kind, Zpsi=ones, m2psi=np.array([0.1, 0.5, 2.0]), m2phi=np.array([0.3, 0.2, 1.0]))
    a, da, sa = run4d(c, rq, rc, freg=1, **kw)
    b, db, sb = run4d(c, rq, rc, freg=0, **kw)
    assert np.all(np.abs(a - b) <= 1e-14 * sb) and np.all(np.abs(da - db) <= 1e-14 * (1 + db))
    a, da, sa = run3d(c, rq, rc, 0.3, freg=1, **kw)
    b, db, sb = run3d(c, rq, rc, 0.3, freg=0, **kw)
    assert np.all(np.abs(a - b) <= 1e-14 * sb) and np.all(np.abs(da - db) <= 1e-14 * (1 + db))
    # with the tabulated Z_psi != 1 the two regularisations are different functions
    a, _, _ = run4d(c, rq, rc, freg=1, **dict(kw, Zpsi=c["Zpsi"]))
    b, _, _ = run4d(c, rq, rc, freg=0, **dict(kw, Zpsi=c["Zpsi"]))
    assert np.all(np.abs(a / b - 1) > 1e-4)


def test_matsubara_fermionic_heavy_mass_weights():
    """m2 -> inf, kappa_000 = 1, constant Z_psi = z0 != 1, dressed regulator: out m_psi^4 m_phi^2 / (C T) is
    2 sum_n int q^2 2 (z0 sqrt(s) + RF(s)) RFdot(s) dq  with s = nu_n^2 + q^2 (4-D argument) or s -> q^2 (spatial)."""
    mp.mp.dps = 30
    k, T, n_max, M, z0, zk, eta = 1.0, 0.3, 2, 1e15, 1.4, 0.8, 0.2
    c = inputs.config4(n_field=1, n_p=1, n_jext=1, T_over_k=T)
    rq, rc = oracle.gl_rule(96, 0, 9), oracle.gl_rule(4, -1, 1)
    coef = np.zeros(20)
    coef[0] = 1.0
    kw = dict(n_max=n_max, coef=coef, Zpsi=z0 * np.ones_like(c["Zpsi"]), m2psi=np.array([M]), m2phi=np.array([M]),
              pext=np.array([0.7]), n_jext=1, zk=zk, eta=eta, freg=1)

    def ins(s, sq):     # s: regulator argument, sq = sqrt(s)
        RB = mp.exp(-s)
        RBd = 2 * RB * (1 + s)
        rf = mp.sqrt(s + RB) - sq
        rfd = RBd / (2 * mp.sqrt(s + RB))
        return 2 * (z0 * sq + zk * rf) * zk * (rfd - eta * rf)
    out, _, _ = run4d(c, rq, rc, **kw)
    ref = 2 * sum(mp.quad(lambda q: q * q * ins(((2 * n + 1) * mp.pi * T) ** 2 + q * q,
                                               mp.sqrt(((2 * n + 1) * mp.pi * T) ** 2 + q * q)), [0, 1, 3, 9])
                  for n in range(-n_max, n_max + 1))
    assert abs(out[0, 0, 0] * M ** 3 / (c["prefactor"] * T) / float(ref) - 1) < 1e-11
    out, _, _ = run3d(c, rq, rc, 0.0, **kw)
    ref = 2 * (2 * n_max + 1) * mp.quad(lambda q: q * q * ins(q * q, q), [0, 1, 3, 9])
    assert abs(out[0, 0, 0].real * M ** 3 / (c["prefactor"] * T) / float(ref) - 1) < 1e-11


def _analytic_dressings():
    U = inputs.splitmix64_uniform(4, 4)
    return 0.1 + 0.4 * U[0], 0.5 + 1.5 * U[1], 0.1 + 0.4 * U[2], 0.5 + 1.5 * U[3]


@pytest.mark.parametrize("mu,arg4d", [(0.0, True), (0.35, False)])
def test_matsubara_fermionic_vs_scipy_dblquad(mu, arg4d):
    """The whole integrand of reading A25 with analytic dressings, restated in Python, under scipy's adaptive 2-D quadrature."""
    k, T, n_max, p, j, zk, eta = 1.0, 0.15, 3, 0.9, 2, 1.2, 0.1
    c = inputs.config4(n_field=1, n_p=1, n_jext=4, n_tab=4096, T_over_k=T)
    A_psi, B_psi, A_phi, B_phi = _analytic_dressings()
    kap, order = c["coef"], monomial_order()
    mpsi, mphi = 0.3, 0.5
    p0j = complex((2 * j + 1) * PI * T, mu)
    ref = 0.0
    for n in range(-n_max, n_max + 1):
        p0n = complex((2 * n + 1) * PI * T, mu)
        nbar = n if n >= 0 else -n - 1
        m = j - n
        om = 2 * PI * m * T
        nu_row, om_row = (2 * nbar + 1) * PI * T, 2 * PI * abs(m) * T

        def g(cth, q):
            spsi = p0n * p0n + q * q
            r2 = p * p + q * q - 2 * p * q * cth
            sphi = om * om + r2
            Zp = 1 + A_psi / (1 + B_psi * (q * q + nu_row ** 2))
            Zb = 1 + A_phi / (1 + B_phi * (r2 + om_row ** 2))
            sR = spsi.real if arg4d else q * q                      # regulator argument of the fermion line
            RB = math.exp(-sR)
            root = math.sqrt(sR + RB)
            rf, rfd = root - math.sqrt(sR), 2 * RB * (1 + sR) / (2 * root)
            A = Zp * math.sqrt(sR) + zk * rf
            Dpsi = Zp * Zp * (spsi - sR) + A * A + mpsi
            insert = 2 * A * zk * (rfd - eta * rf)
            sRb = sphi if arg4d else r2
            Gphi = 1 / (Zb * sphi + zk * math.exp(-sRb) + mphi)
            y1, y2, y3 = p0n * p0j, p * q * cth, spsi
            P = sum(kap[i] * y1 ** a * y2 ** b * y3 ** cc for i, (a, b, cc) in enumerate(order))
            return q * q * insert / Dpsi ** 2 * P * Gphi
        re, _ = integrate.dblquad(lambda cth, q: g(cth, q).real, 0, 10, -1, 1, epsabs=1e-13, epsrel=1e-10)
        im = 0.0
        if mu != 0.0:
            im, _ = integrate.dblquad(lambda cth, q: g(cth, q).imag, 0, 10, -1, 1, epsabs=1e-13, epsrel=1e-10)
        ref += complex(re, im)
    ref *= c["prefactor"] * T
    kw = dict(n_max=n_max, m2psi=np.array([mpsi]), m2phi=np.array([mphi]), pext=np.array([p]), n_jext=4, zk=zk, eta=eta,
              freg=1)
    rq, rc = oracle.gl_rule(128, 0, 10), oracle.gl_rule(48, -1, 1)
    if arg4d:
        out, _, _ = run4d(c, rq, rc, **kw)
        assert abs(out[0, j, 0] / ref.real - 1) < 1e-8
    else:
        out, _, _ = run3d(c, rq, rc, mu, **kw)
        assert abs(out[0, j, 0] / ref - 1) < 1e-8


def test_matsubara_fermionic_mass_derivatives_five_point():
    c = inputs.config4(n_field=1, n_p=1, n_jext=2, T_over_k=0.2)
    rq, rc = oracle.gl_rule(16, 0, 6), oracle.gl_rule(6, -1, 1)
    mpsi, mphi, h = 0.4, 0.6, 1e-3
    kw = dict(n_max=2, pext=np.array([0.8]), n_jext=2, zk=1.1, eta=0.05, freg=1)

    def val4(a, b):
        return run4d(c, rq, rc, m2psi=np.array([a]), m2phi=np.array([b]), **kw)[0][0, 1, 0]

    def val3(a, b):
        return run3d(c, rq, rc, 0.3, m2psi=np.array([a]), m2phi=np.array([b]), **kw)[0][0, 1, 0]

    def fd(f, x):
        return (f(x - 2 * h) - 8 * f(x - h) + 8 * f(x + h) - f(x + 2 * h)) / (12 * h)
    d = oracle.matsubara3d_dm2(c["T"], 2, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *rq, *rc, c["Zpsi"], c["Zphi"],
                               c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], np.array([mpsi]), np.array([mphi]),
                               np.array([0.8]), 2, zk=1.1, eta=0.05, freg=1)
    assert abs(d[0][0, 1, 0] / fd(lambda x: val4(x, mphi), mpsi) - 1) < 1e-8
    assert abs(d[1][0, 1, 0] / fd(lambda x: val4(mpsi, x), mphi) - 1) < 1e-8
    d = oracle.matsubara3d_mu_dm2(c["T"], 2, 0.3, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *rq, *rc, c["Zpsi"],
                                  c["Zphi"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], np.array([mpsi]),
                                  np.array([mphi]), np.array([0.8]), 2, zk=1.1, eta=0.05, freg=1)
    assert abs(d[0][0, 1, 0] / fd(lambda x: val3(x, mphi), mpsi) - 1) < 1e-8
    assert abs(d[1][0, 1, 0] / fd(lambda x: val3(mpsi, x), mphi) - 1) < 1e-8


def test_matsubara_fermionic_sens_is_the_positive_term_identity():
    """m2 = 0 on both lines, positive coefficients, n >= 0 and j >= 0 frequencies: every term is positive and
    (|D - m2| + |m2|)/|D| = 1, so sens = out (1 + 2 + 1) exactly (G_psi^2 G_phi), with the fermionic regulator too."""
    c = inputs.config4(n_field=1, n_p=1, n_jext=1, T_over_k=0.2)
    rq, rc = oracle.gl_rule(10, 0, 4), oracle.gl_rule(4, -1, 1)
    coef = np.zeros(20)
    coef[0], coef[monomial_order().index((0, 0, 1))] = 1.0, 0.5     # 1 + y3/2 > 0
    out, _, sens = run4d(c, rq, rc, n_max=0, coef=coef, m2psi=np.zeros(1), m2phi=np.zeros(1), pext=np.array([0.3]),
                         n_jext=1, zk=1.3, eta=0.1, freg=1)
    assert abs(sens[0, 0, 0] / out[0, 0, 0] - 4.0) < 1e-13
