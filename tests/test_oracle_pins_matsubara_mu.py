"""Pins for the Matsubara family at finite chemical potential (orc_matsubara3d_mu, DESIGN.md
reading A24) against things other than the oracle:
  * the full integrand (complex fermion line, spatial regulators, analytic dressings) against scipy adaptive 2-D
    quadrature of its real and imaginary parts, term by term in n;
  * unit monomials in the heavy-mass limit with complex y1, y3 (mpmath radial integrals);
  * flat spatial regulator, Z = 1, p = 0, kappa_000 = 1: every (n, q, c) integral is elementary, the result is a finite
    sum of closed-form complex terms (the sign of i mu, the square of G_psi, the mu-free boson line);
  * mu -> -mu conjugates the result; mu = 0 is real.
CPU only."""
import math

import mpmath as mp
import numpy as np
from scipy import integrate

import oracle
from paper_2412_13043_b200 import inputs

PI = math.pi


def monomial_order(deg=3):
    return [(a, b, c) for a in range(deg + 1) for b in range(deg + 1 - a) for c in range(deg + 1 - a - b)]


def run(c, rq, rc, mu, **over):
    a = dict(c)
    a.update(over)
    return oracle.matsubara3d_mu(a["T"], a["n_max"], mu, a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], *rq, *rc,
                                 a["Zpsi"], a["Zphi"], a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"],
                                 a["m2psi"], a["m2phi"], a["pext"], a["n_jext"], sel=a.get("sel"),
                                 want_sens=True)


def test_matsubara_mu_vs_scipy_dblquad():
    k, T, n_max, p, j, mu = 1.0, 0.15, 3, 0.9, 2, 0.35
    c = inputs.config4(n_field=1, n_p=1, n_jext=4, n_tab=4096, T_over_k=T)
    U = inputs.splitmix64_uniform(4, 4)
    A_psi, B_psi, A_phi, B_phi = 0.1 + 0.4 * U[0], 0.5 + 1.5 * U[1], 0.1 + 0.4 * U[2], 0.5 + 1.5 * U[3]
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
            Gpsi = 1 / (Zp * spsi + math.exp(-q * q) + mpsi)                  # spatial regulator
            Gphi = 1 / (Zb * sphi + math.exp(-r2) + mphi)
            y1, y2, y3 = p0n * p0j, p * q * cth, spsi
            P = sum(kap[i] * y1 ** a * y2 ** b * y3 ** cc for i, (a, b, cc) in enumerate(order))
            return q * q * 2 * math.exp(-q * q) * (1 + q * q) * Gpsi ** 2 * P * Gphi
        re, _ = integrate.dblquad(lambda cth, q: g(cth, q).real, 0, 10, -1, 1, epsabs=1e-13, epsrel=1e-10)
        im, _ = integrate.dblquad(lambda cth, q: g(cth, q).imag, 0, 10, -1, 1, epsabs=1e-13, epsrel=1e-10)
        ref += complex(re, im)
    ref *= c["prefactor"] * T
    out, _, _ = run(c, oracle.gl_rule(128, 0, 10), oracle.gl_rule(48, -1, 1), mu, n_max=n_max,
                    m2psi=np.array([mpsi]), m2phi=np.array([mphi]), pext=np.array([p]), n_jext=4)
    assert abs(out[0, j, 0] / ref - 1) < 1e-8


def test_matsubara_mu_monomials_heavy_mass_limit():
    mp.mp.dps = 30
    k, T, n_max, p, j, M, mu = 1.0, 0.3, 2, 0.7, 1, 1e15, 0.45
    c = inputs.config4(n_field=1, n_p=1, n_jext=2, T_over_k=T)
    rq, rc = oracle.gl_rule(64, 0, 9), oracle.gl_rule(6, -1, 1)
    p0j = mp.mpc((2 * j + 1) * mp.pi * T, mu)
    for idx, (a, b, cc) in enumerate(monomial_order()):
        coef = np.zeros(20)
        coef[idx] = 1.0
        out, _, _ = run(c, rq, rc, mu, n_max=n_max, coef=coef, m2psi=np.array([M]), m2phi=np.array([M]),
                        pext=np.array([p]), n_jext=2)
        got = complex(out[0, j, 0]) * M ** 3 / (c["prefactor"] * T)
        ref, scale = mp.mpc(0), mp.mpf(0)
        for n in range(-n_max, n_max + 1):
            p0n = mp.mpc((2 * n + 1) * mp.pi * T, mu)
            rad = mp.quad(lambda q: q * q * 2 * mp.exp(-q * q) * (1 + q * q) * (p * q) ** b * (p0n ** 2 + q * q) ** cc,
                          [0, 1, 3, 9])
            term = (p0n * p0j) ** a * rad * (mp.mpf(2) / (b + 1) if b % 2 == 0 else 0)
            ref += term
            scale += abs((p0n * p0j) ** a * rad) * 2 / (b + 1)           # int |c|^b dc: the size of what cancels for odd b
        if b % 2:
            assert abs(got) < 1e-13 * float(scale), (idx, a, b, cc)
        else:
            assert abs(got - complex(ref)) < 2e-11 * float(scale), (idx, a, b, cc)


def test_matsubara_mu_flat_regulator_closed_form():
    """Flat spatial regulator, Z = 1, radial [0,k], p = 0, kappa_000 = 1:  q^2 + R = k^2 on both lines, so
    out[j] = C T (2 k^5/3) 2 sum_n 1/(((nu_n + i mu)^2 + k^2 + m_psi^2)^2 ((nu_j - nu_n)^2 + k^2 + m_phi^2))."""
    k, T, n_max, mu = 1.2, 0.2, 4, 0.5
    c = inputs.config4(n_field=3, n_p=1, n_jext=3, T_over_k=T / k, k=k)
    ones = np.ones_like(c["Zpsi"])
    coef = np.zeros(20)
    coef[0] = 1.0
    rq, rc = oracle.gl_rule(16, 0, k), oracle.gl_rule(4, -1, 1)
    mpsi, mphi = np.array([0.1, 0.7, 2.0]), np.array([0.4, -0.3, 1.5])
    out, dmin, _ = run(c, rq, rc, mu, n_max=n_max, reg_kind=oracle.REG_LITIM, Zpsi=ones, Zphi=ones, coef=coef,
                       m2psi=mpsi, m2phi=mphi, pext=np.zeros(1), n_jext=3)
    for j in range(3):
        for f in range(3):
            tot = 0.0
            for n in range(-n_max, n_max + 1):
                p0n = complex((2 * n + 1) * PI * c["T"], mu)
                om = 2 * PI * (j - n) * c["T"]
                tot += 1.0 / ((p0n * p0n + k * k + mpsi[f]) ** 2 * (om * om + k * k + mphi[f]))
            ref = c["prefactor"] * c["T"] * (2 * k ** 5 / 3) * 2 * tot
            assert abs(out[0, j, f] / ref - 1) < 1e-12
    # |D_psi| is smallest at n = 0 / n = -1
    d0 = abs(complex((PI * c["T"]) ** 2 - mu * mu + k * k + mpsi[0], 2 * PI * c["T"] * mu))
    assert abs(dmin[0, 0, 0] - min(d0, k * k + mphi[0]) / (k * k)) < 1e-13


def test_matsubara_mu_conjugation_and_mu0_is_real():
    c = inputs.config4(n_field=3, n_p=2, n_jext=3)
    rq, rc = oracle.gl_rule(8, 0, 10), oracle.gl_rule(4, -1, 1)
    a, _, _ = run(c, rq, rc, 0.3, n_max=2)
    b, _, _ = run(c, rq, rc, -0.3, n_max=2)
    assert np.array_equal(a, np.conj(b)) and np.any(a.imag != 0)
    z, _, _ = run(c, rq, rc, 0.0, n_max=2)
    assert np.all(z.imag == 0)
    sel = np.array([0, 5, 17, 9])
    s, _, _ = run(c, rq, rc, 0.3, n_max=2, sel=sel)
    assert np.array_equal(s, a.ravel()[sel])


# ---- mass derivatives at chemical potential (orc_matsubara3d_mu_dm2) -------------------------------------------
def _dm2(c, rq, rc, mu, **over):
    a = dict(c)
    a.update(over)
    return oracle.matsubara3d_mu_dm2(a["T"], a["n_max"], mu, a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], *rq, *rc,
                                     a["Zpsi"], a["Zphi"], a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"],
                                     a["m2psi"], a["m2phi"], a["pext"], a["n_jext"], sel=a.get("sel"))


def test_matsubara_mu_dm2_vs_finite_differences_of_the_pinned_value_function():
    """Five-point central differences of orc_matsubara3d_mu (pinned above) in m2_psi and in m2_phi, mu != 0 and mu = 0."""
    c = inputs.config4(n_field=4, n_p=2, n_jext=3)
    rq, rc = oracle.gl_rule(10, 0, 10), oracle.gl_rule(6, -1, 1)
    mpsi, mphi = np.array([0.2, 0.6, 1.1, 2.0]), np.array([0.3, 0.8, 1.5, 3.0])
    h = 1e-3
    fd5 = lambda fun: (fun(-2 * h) - 8 * fun(-h) + 8 * fun(h) - fun(2 * h)) / (12 * h)
    for mu in (0.4, 0.0):
        dpsi, dphi, spsi, sphi = _dm2(c, rq, rc, mu, n_max=2, m2psi=mpsi, m2phi=mphi)
        val = lambda dpsi_, dphi_: run(c, rq, rc, mu, n_max=2, m2psi=mpsi + dpsi_, m2phi=mphi + dphi_)[0]
        fpsi = fd5(lambda t: val(t, 0.0))
        fphi = fd5(lambda t: val(0.0, t))
        scale = np.abs(run(c, rq, rc, mu, n_max=2, m2psi=mpsi, m2phi=mphi)[0])
        assert np.all(np.abs(dpsi - fpsi) <= 1e-8 * (np.abs(dpsi) + scale))
        assert np.all(np.abs(dphi - fphi) <= 1e-8 * (np.abs(dphi) + scale))
        assert np.all(spsi >= np.abs(dpsi)) and np.all(sphi >= np.abs(dphi))
        if mu == 0.0:
            assert np.all(dpsi.imag == 0) and np.all(dphi.imag == 0)


def test_matsubara_mu_dm2_flat_regulator_closed_form():
    """As test_matsubara_mu_flat_regulator_closed_form: d/dm2_psi (A + m)^-2 = -2 (A + m)^-3, d/dm2_phi (B + m)^-1 = -(B + m)^-2."""
    k, T, n_max, mu = 1.2, 0.2, 4, 0.5
    c = inputs.config4(n_field=3, n_p=1, n_jext=3, T_over_k=T / k, k=k)
    ones = np.ones_like(c["Zpsi"])
    coef = np.zeros(20)
    coef[0] = 1.0
    rq, rc = oracle.gl_rule(16, 0, k), oracle.gl_rule(4, -1, 1)
    mpsi, mphi = np.array([0.1, 0.7, 2.0]), np.array([0.4, -0.3, 1.5])
    dpsi, dphi, _, _ = _dm2(c, rq, rc, mu, n_max=n_max, reg_kind=oracle.REG_LITIM, Zpsi=ones, Zphi=ones, coef=coef,
                            m2psi=mpsi, m2phi=mphi, pext=np.zeros(1), n_jext=3)
    for j in range(3):
        for f in range(3):
            tpsi = tphi = 0.0
            for n in range(-n_max, n_max + 1):
                p0n = complex((2 * n + 1) * PI * c["T"], mu)
                A = p0n * p0n + k * k + mpsi[f]
                Bq = (2 * PI * (j - n) * c["T"]) ** 2 + k * k + mphi[f]
                tpsi += -2.0 / (A ** 3 * Bq)
                tphi += -1.0 / (A ** 2 * Bq ** 2)
            pref = c["prefactor"] * c["T"] * (2 * k ** 5 / 3) * 2
            assert abs(dpsi[0, j, f] / (pref * tpsi) - 1) < 1e-12
            assert abs(dphi[0, j, f] / (pref * tphi) - 1) < 1e-12
