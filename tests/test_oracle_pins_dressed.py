"""Pins for the dressed regulator of the CPU oracle (reading A20):
    R = Z_k R_shape,   Rdot = k d(Z_k R_shape)/dk = Z_k (Rdot_shape - eta R_shape),   eta = -k dZ_k/dk / Z_k
("only the eta_i = -d_t Z_i/Z_i enter the flow equations"; RB / RBdot).
Fixed by things other than the oracle: mpmath differentiation of Z_k R_k with a running Z_k, the textbook
(1 - eta/(d+2)) threshold functions of the flat regulator, and mpmath adaptive quadrature.  CPU only.
"""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2412_13043_b200 import inputs

PI = math.pi


@pytest.mark.parametrize("kind,order", [(oracle.REG_EXP_POLY, 1), (oracle.REG_EXP_POLY, 2), (oracle.REG_EXP_POLY, 8),
                                        (oracle.REG_LITIM, 0)])
def test_dressed_regulator_vs_mpmath_total_derivative(kind, order):
    """k d/dk of Z(k) R_k(s) with Z(k) = zk (k/k0)^(-eta), evaluated at k = k0."""
    mp.mp.dps = 40
    zk, eta = 1.3, 0.27
    for k0 in (1.0, 1.7):
        for s in (0.0, 1e-3, 0.3, 0.9, 2.5):
            if kind == oracle.REG_LITIM and s >= k0 * k0:
                continue

            def ZR(kk):
                x = mp.mpf(s) / kk ** 2
                shape = (kk ** 2 - mp.mpf(s)) if kind == oracle.REG_LITIM else \
                    kk ** 2 * mp.exp(-sum(x ** i / i for i in range(1, order + 1)))
                return mp.mpf(zk) * (kk / mp.mpf(k0)) ** (-mp.mpf(eta)) * shape
            R_ref = ZR(mp.mpf(k0))
            Rd_ref = mp.mpf(k0) * mp.diff(ZR, mp.mpf(k0))
            R, Rd = oracle.regulator(kind, order, k0, s, zk=zk, eta=eta)
            assert abs(R - float(R_ref)) <= 1e-13 * abs(float(R_ref))
            assert abs(Rd - float(Rd_ref)) <= 1e-13 * abs(float(Rd_ref))
    # zk = 1, eta = 0 is bit-identical to the plain shapes
    assert oracle.regulator(kind, order, 1.3, 0.4, zk=1.0, eta=0.0) == oracle.regulator(kind, order, 1.3, 0.4)


@pytest.mark.parametrize("d,k,eta", [(4, 1.0, 0.3), (3, 1.0, -0.2), (4, 1.7, 1.1)])
def test_litim_threshold_function_with_eta(d, k, eta):
    """Flat regulator, zk = 1, radial [0,k]:  I = C (2 k^(d+2)/d) (1 - eta/(d+2)) / (k^2 + m^2)."""
    c = inputs.config0(n_field=65, k=k, litim=True, d=d)
    xq, wq = oracle.gl_rule(*c["rule_q"])
    flow, chan, dmin = oracle.lpa(d, 0.0, 0, 1, c["N"], c["prefactor"], oracle.REG_LITIM, 1, k, xq, wq,
                                  c["rho"], c["u"], c["du"], eta=eta)
    m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
    E2 = k * k + m2
    ok = np.abs(E2) > 1e-9
    ref = c["prefactor"] * 2 * k ** (d + 2) / d * (1 - eta / (d + 2)) / E2
    np.testing.assert_allclose(chan[ok], ref[ok], rtol=1e-13)
    # derivative twin
    dchan, _ = oracle.lpa_dm2(d, 0.0, 0, 1, c["prefactor"], oracle.REG_LITIM, 1, k, xq, wq, c["rho"], c["u"], c["du"],
                              eta=eta)
    np.testing.assert_allclose(dchan[ok], -ref[ok] / E2[ok], rtol=1e-13)


@pytest.mark.parametrize("d", [3, 4])
def test_litim_dressed_zk_vs_mpmath_quadrature(d):
    """zk != 1: the denominator is q^2 + zk (k^2 - q^2) + m^2 (Z_k dresses the regulator only, reading A12)."""
    mp.mp.dps = 30
    k, zk, eta = 1.2, 1.6, 0.35
    c = inputs.config0(n_field=9, k=k, litim=True, d=d)
    xq, wq = oracle.gl_rule(64, 0.0, k)
    flow, chan, dmin = oracle.lpa(d, 0.0, 0, 1, c["N"], c["prefactor"], oracle.REG_LITIM, 1, k, xq, wq,
                                  c["rho"], c["u"], c["du"], zk=zk, eta=eta)
    for f in range(9):
        m2 = float(c["u"][f])
        if zk * k * k + m2 < 0.05:
            continue
        ref = c["prefactor"] * mp.quad(
            lambda q: q ** (d - 1) * zk * (2 * k * k - eta * (k * k - q * q)) / (q * q + zk * (k * k - q * q) + m2),
            [0, k])
        assert abs(chan[0, f] / float(ref) - 1) < 1e-12


@pytest.mark.parametrize("T_over_k", [0.1, 0.5])
def test_finite_T_litim_with_eta(T_over_k):
    """Spatial flat regulator at T > 0, zk = 1: the eta term multiplies every Matsubara term by (1 - eta/5)."""
    k, eta = 1.0, 0.4
    c = inputs.config1(T_over_k, n_field=33, k=k, litim=True)
    xq, wq = oracle.gl_rule(*c["rule_q"])
    T, N = c["T"], c["n_max"]
    _, chan0, _ = oracle.lpa(3, T, N, 0, 4.0, c["prefactor"], oracle.REG_LITIM, 1, k, xq, wq, c["rho"], c["u"], c["du"])
    _, chan1, _ = oracle.lpa(3, T, N, 0, 4.0, c["prefactor"], oracle.REG_LITIM, 1, k, xq, wq, c["rho"], c["u"], c["du"],
                             eta=eta)
    m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
    ok = k * k + m2 > 1e-3
    np.testing.assert_allclose(chan1[ok], chan0[ok] * (1 - eta / 5), rtol=1e-13)


def test_exp_regulator_dressed_vs_mpmath_quadrature():
    """EXP_POLY(1), d = 4, zk and eta: the whole lpa integrand against adaptive quadrature of the continuum integral."""
    mp.mp.dps = 30
    k, zk, eta = 1.0, 0.8, 0.25
    c = inputs.config0(n_field=5, k=k)
    xq, wq = oracle.gl_rule(96, 0.0, 8.0 * k)
    _, chan, _ = oracle.lpa(4, 0.0, 0, 1, c["N"], c["prefactor"], oracle.REG_EXP_POLY, 1, k, xq, wq,
                            c["rho"], c["u"], c["du"], zk=zk, eta=eta)
    for f in range(5):
        m2 = float(c["u"][f] + 2 * c["rho"][f] * c["du"][f])
        if m2 < -0.5:
            continue

        def integrand(q):
            x = q * q / (k * k)
            R = zk * k * k * mp.exp(-x)
            Rd = zk * (2 * k * k * mp.exp(-x) * (1 + x) - eta * k * k * mp.exp(-x))
            return q ** 3 * Rd / (q * q + R + m2)
        ref = c["prefactor"] * mp.quad(integrand, [0, 1, 2, 4, 8])
        assert abs(chan[1, f] / float(ref) - 1) < 1e-11


def test_dressing_reaches_every_family():
    """The dressing in the two-point, Matsubara and three-point families.  m2 -> infinity: out m2^p / C is the weight
    sum of Rdot, linear in zk, and the eta part is -eta times the same sum with R in place of Rdot (numpy sums over the
    same nodes); three-point: flat regulator below k^2 everywhere, against a numpy restatement of the whole sum."""
    k, zk = 1.0, 1.4
    big = 1e15
    # two-point at p = 0: out = C Sc coef0 sum_i w q^3 Rdot / m2^3
    c = inputs.config2(n_field=1, n_ext=1, k=k)
    xq, wq = oracle.gl_rule(48, 0, 8 * k)
    xc, wc = oracle.gl_rule(8, -1, 1)
    args = (c["prefactor"], oracle.REG_EXP_POLY, 1, k, xq, wq, xc, wc, np.ones(8), c["lnq_lo"], c["lnq_hi"], 1,
            np.array([1.0, 0.0]), np.array([big]), np.zeros(1))
    o = {eta: oracle.loop4d_twopoint(*args, zk=zk, eta=eta)[0][0, 0] * big ** 3 / c["prefactor"] for eta in (0.0, 1.0)}
    Sc = np.sum(wc * np.sqrt(1 - xc ** 2))
    x = xq ** 2
    sumRd = np.sum(wq * xq ** 3 * 2 * np.exp(-x) * (1 + x))
    sumR = np.sum(wq * xq ** 3 * np.exp(-x))
    assert abs(o[0.0] / (zk * Sc * sumRd) - 1) < 1e-12
    assert abs((o[0.0] - o[1.0]) / (zk * Sc * sumR) - 1) < 1e-11
    # Matsubara: out = C T sum_n sum_q w q^2 Rdot(s_psi) / (m2psi^2 m2phi) sum_c w  (kappa_000 = 1)
    c4 = inputs.config4(n_field=1, n_p=1, n_jext=1, n_q=32, n_c=4)
    xq, wq = oracle.gl_rule(*c4["rule_q"])
    xc, wc = oracle.gl_rule(*c4["rule_c"])
    coef = np.zeros(20)
    coef[0] = 1.0
    T, nm = c4["T"], c4["n_max"]
    a4 = (T, nm, c4["prefactor"], oracle.REG_EXP_POLY, 1, k, xq, wq, xc, wc, c4["Zpsi"], c4["Zphi"], c4["lnq_lo"],
          c4["lnq_hi"], c4["interp"], coef, np.array([big]), np.array([big]), c4["pext"], 1)
    o4 = {eta: oracle.matsubara3d(*a4, zk=zk, eta=eta)[0][0, 0, 0] * big ** 3 / (c4["prefactor"] * T)
          for eta in (0.0, 1.0)}
    nu = (2 * np.arange(-nm, nm + 1) + 1) * PI * T
    s = nu[:, None] ** 2 + xq[None, :] ** 2
    sumRd = np.sum(wq[None, :] * xq[None, :] ** 2 * 2 * np.exp(-s) * (1 + s)) * np.sum(wc)
    sumR = np.sum(wq[None, :] * xq[None, :] ** 2 * np.exp(-s)) * np.sum(wc)
    assert abs(o4[0.0] / (zk * sumRd) - 1) < 1e-12
    assert abs((o4[0.0] - o4[1.0]) / (zk * sumR) - 1) < 1e-11
    # three-point: Litim, small momenta, Z_A = lambda3 = 1, kappa_000 = 1, radial [0, k/2]: every argument stays below
    # k^2, so G_A(s) = 1/(s + zk (k^2 - s)); reference = an independent numpy sum over the same grid
    c3 = inputs.config3(n_p=1, n_alpha=1, n_q=8, n_c1=6, n_c2=4)
    xq, wq = oracle.gl_rule(8, 0, 0.5 * k)
    x1, w1 = oracle.gl_rule(6, -1, 1)
    x2, w2 = oracle.gl_rule(4, -1, 1)
    xp, wp = oracle.gl_rule(4, 0, 2 * PI)
    coef3 = np.zeros(35)
    coef3[0] = 1.0
    ones = np.ones(8)
    p1, p2, al = 0.1, 0.2, 0.7
    ext = np.array([[p1, p2, al]])
    eta = 0.3
    o3 = oracle.loop4d_threepoint(c3["prefactor"], oracle.REG_LITIM, 1, k, xq, wq, x1, w1, x2, w2, xp, wp, ones, ones,
                                  ones, c3["lnq_lo"], c3["lnq_hi"], 1, coef3, ext, zk=zk, eta=eta)[0][0]
    Q, C1, C2 = np.meshgrid(xq, x1, x2, indexing="ij")
    W = (wq * xq ** 3)[:, None, None] * (w1 * np.sqrt(1 - x1 ** 2))[None, :, None] * w2[None, None, :]
    S1 = np.sqrt(1 - C1 ** 2)
    sa = Q ** 2 + p1 ** 2 + 2 * Q * p1 * C1
    sb = Q ** 2 + p2 ** 2 - 2 * Q * p2 * (math.cos(al) * C1 + math.sin(al) * S1 * C2)
    assert sa.max() < k * k and sb.max() < k * k
    G = lambda s_: 1.0 / (s_ + zk * (k * k - s_))
    Rd = zk * (2 * k * k - eta * (k * k - Q ** 2))
    ref = c3["prefactor"] * np.sum(wp) * np.sum(W * Rd * G(Q ** 2) * G(sa) * G(sb))
    assert abs(o3 / ref - 1) < 1e-12
