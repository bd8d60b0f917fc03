"""Pins for the CPU oracle (oracle/dfrg_oracle.cpp) against things other than itself.

Closed forms, library routines (mpmath / scipy adaptive quadrature of the CONTINUUM
integrals the quadrature sums approximate), invariants and brute force on tiny inputs.
Numbering P1..P12 follows SURVEY.md section 8(c) / DESIGN.md "Pins".  CPU only.
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_2412_13043_b200 import inputs

PI = math.pi


def rule(r):
    return oracle.gl_rule(*r)


# ----------------------------------------------------------------------------------------
# P1  Gauss-Legendre nodes and weights (textbook values, exactness, independent library)
# ----------------------------------------------------------------------------------------
def test_p1_gl_closed_forms():
    x, w = oracle.gl_rule(1, -1, 1)
    assert x[0] == 0.0 and w[0] == 2.0
    x, w = oracle.gl_rule(2, -1, 1)
    np.testing.assert_allclose(x, [-1 / math.sqrt(3), 1 / math.sqrt(3)], rtol=2e-16)
    np.testing.assert_allclose(w, [1.0, 1.0], rtol=2e-16)
    x, w = oracle.gl_rule(3, -1, 1)
    np.testing.assert_allclose(x, [-math.sqrt(0.6), 0.0, math.sqrt(0.6)], rtol=2e-16, atol=0)
    np.testing.assert_allclose(w, [5 / 9, 8 / 9, 5 / 9], rtol=2e-16)
    # golden file: 5-point rule, Abramowitz & Stegun table 25.4 closed forms
    g = np.loadtxt("tests/golden/gl5_abramowitz_stegun.txt")
    x, w = oracle.gl_rule(5, -1, 1)
    np.testing.assert_allclose(x, g[:, 0], rtol=0, atol=1e-15)
    np.testing.assert_allclose(w, g[:, 1], rtol=0, atol=1e-15)


@pytest.mark.parametrize("n", [16, 24, 32, 64, 96, 128])
def test_p1_gl_vs_mpmath_and_numpy(n):
    x, w = oracle.gl_rule(n, -1, 1)
    assert np.all(np.diff(x) > 0)
    np.testing.assert_allclose(x, -x[::-1], rtol=0, atol=1e-16)
    np.testing.assert_allclose(w, w[::-1], rtol=4e-16)
    mp.mp.dps = 40
    for i in (0, 1, n // 3, n // 2, n - 1):
        r = mp.mpf(float(x[i]))
        for _ in range(4):                                # Newton on mpmath's own (hypergeometric) P_n
            r -= mp.legendre(n, r) / mp.diff(lambda z: mp.legendre(n, z), r)
        d = mp.diff(lambda z: mp.legendre(n, z), r)
        wi = 2 / ((1 - r * r) * d * d)
        assert abs(x[i] - float(r)) <= 2.3e-16 * max(abs(float(r)), 0.05)
        assert abs(w[i] / float(wi) - 1) <= 4.5e-16
    xn, wn = np.polynomial.legendre.leggauss(n)          # independent library, less accurate weights
    np.testing.assert_allclose(x, xn, rtol=0, atol=4.5e-16)
    np.testing.assert_allclose(w, wn, rtol=1e-10)   # numpy documents its weights as less accurate at high n


def test_p1_gl_exactness_and_mapping():
    n, a, b = 12, 0.5, 6.0
    x, w = oracle.gl_rule(n, a, b)
    assert abs(w.sum() - (b - a)) < 1e-14
    for m in range(0, 2 * n):
        exact = (b ** (m + 1) - a ** (m + 1)) / (m + 1)
        assert abs(np.dot(w, x ** m) / exact - 1) < 5e-14
    # degree 2n is NOT integrated exactly
    x, w = oracle.gl_rule(4, -1, 1)
    assert abs(np.dot(w, x ** 6) - 2 / 7) < 1e-15 and abs(np.dot(w, x ** 8) - 2 / 9) > 1e-3


# ----------------------------------------------------------------------------------------
# P5  regulators: eq. (14) and k d/dk
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("order", [1, 2, 8])
def test_p5_regulator_exp_poly_vs_mpmath(order):
    mp.mp.dps = 40
    for k in (1.0, 1.7):
        for s in (0.0, 1e-3, 0.3, 1.0, 2.5, 7.0):
            def Rk(kk):
                x = mp.mpf(s) / kk ** 2
                return kk ** 2 * mp.exp(-sum(x ** i / i for i in range(1, order + 1)))
            R_ref = Rk(mp.mpf(k))
            Rd_ref = mp.mpf(k) * mp.diff(Rk, mp.mpf(k))
            R, Rd = oracle.regulator(oracle.REG_EXP_POLY, order, k, s)
            # exp() amplifies the rounding of its argument by |argument| (<= ~3000 here for order 8)
            assert abs(R - float(R_ref)) <= 1e-13 * abs(float(R_ref)) + 1e-300
            assert abs(Rd - float(Rd_ref)) <= 1e-13 * abs(float(Rd_ref)) + 1e-300


def test_p5_regulator_order1_is_baseline_form():
    # BASELINE.json configs[0]: R = k^2 e^{-q^2/k^2}, dtR = 2 k^2 e^{-q^2/k^2} (1 + q^2/k^2)
    for s in (0.0, 0.25, 1.0, 9.0, 36.0):
        R, Rd = oracle.regulator(oracle.REG_EXP_POLY, 1, 1.0, s)
        assert abs(R - math.exp(-s)) <= 2e-16 * math.exp(-s)
        assert abs(Rd - 2 * math.exp(-s) * (1 + s)) <= 4e-16 * 2 * math.exp(-s) * (1 + s)


def test_p5_regulator_litim():
    k = 1.3
    assert oracle.regulator(oracle.REG_LITIM, 0, k, 0.5) == (k * k - 0.5, 2 * k * k)
    assert oracle.regulator(oracle.REG_LITIM, 0, k, k * k) == (0.0, 0.0)      # Theta(0) = 0
    assert oracle.regulator(oracle.REG_LITIM, 0, k, 2.0) == (0.0, 0.0)


# ----------------------------------------------------------------------------------------
# P6  log-grid interpolator
# ----------------------------------------------------------------------------------------
def test_p6_cubic_exact_on_cubics_linear_on_lines():
    n, lo, hi = 37, math.log(1e-4), math.log(2e2)
    lnq = lo + (hi - lo) * np.arange(n) / (n - 1)
    cub = lambda l: 0.3 - 0.2 * l + 0.05 * l ** 2 + 0.01 * l ** 3
    lin = lambda l: 1.5 - 0.25 * l
    rng = np.random.default_rng(0)
    for l in np.concatenate([rng.uniform(lo, hi, 200), lnq[[0, 1, 2, n - 3, n - 2, n - 1]]]):
        s = math.exp(2 * l)                      # the argument is the SQUARED momentum
        assert abs(oracle.table_lookup(cub(lnq), lo, hi, 3, s) - cub(l)) < 2e-13
        assert abs(oracle.table_lookup(lin(lnq), lo, hi, 1, s) - lin(l)) < 2e-14
    # linear mode is not exact on a cubic, cubic mode is not exact on a quartic
    l = lo + 10.4 * (hi - lo) / (n - 1)
    assert abs(oracle.table_lookup(cub(lnq), lo, hi, 1, math.exp(2 * l)) - cub(l)) > 1e-4
    assert abs(oracle.table_lookup(lnq ** 4, lo, hi, 3, math.exp(2 * l)) - l ** 4) > 1e-6


def test_p6_clamp_nodes_and_continuity():
    n, lo, hi = 16, -2.0, 3.0
    h = (hi - lo) / (n - 1)
    v = np.random.default_rng(1).uniform(0.5, 1.5, n)
    for interp in (1, 3):
        assert oracle.table_lookup(v, lo, hi, interp, 0.0) == v[0]            # log(0) = -inf clamps low
        assert oracle.table_lookup(v, lo, hi, interp, math.exp(2 * (lo - 5))) == v[0]
        assert oracle.table_lookup(v, lo, hi, interp, math.exp(2 * (hi + 5))) == v[-1]
        for i in range(n):                                                     # reproduces node values
            assert abs(oracle.table_lookup(v, lo, hi, interp, math.exp(2 * (lo + i * h))) - v[i]) < 1e-13
        for i in range(1, n - 1):                                              # continuous across cell edges
            a = oracle.table_lookup(v, lo, hi, interp, math.exp(2 * (lo + (i - 1e-9) * h)))
            b = oracle.table_lookup(v, lo, hi, interp, math.exp(2 * (lo + (i + 1e-9) * h)))
            assert abs(a - b) < 1e-7


def test_p6_cubic_stencil_is_centred_and_edge_shifted():
    # 4-point Lagrange through nodes i0..i0+3 with i0 = clamp(floor(t)-1, 0, n-4): a table that
    # is a delta at node j contributes the Lagrange basis polynomial of the centred stencil.
    n, lo, hi = 10, 0.0, 9.0      # h = 1, ln q_i = i
    def L(nodes, j, t):
        return np.prod([(t - m) / (j - m) for m in nodes if m != j])
    for t, nodes in ((4.3, (3, 4, 5, 6)), (0.6, (0, 1, 2, 3)), (8.7, (6, 7, 8, 9)), (1.5, (0, 1, 2, 3))):
        for j in range(n):
            v = np.zeros(n)
            v[j] = 1.0
            ref = L(nodes, j, t) if j in nodes else 0.0
            assert abs(oracle.table_lookup(v, lo, hi, 3, math.exp(2 * t)) - ref) < 1e-13


# ----------------------------------------------------------------------------------------
# P2  Litim threshold functions at T = 0 (closed form)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("d,k", [(4, 1.0), (3, 1.0), (4, 1.7), (3, 0.6)])
def test_p2_litim_threshold_closed_form(d, k):
    c = inputs.config0(n_field=257, k=k, litim=True, d=d)
    xq, wq = rule(c["rule_q"])
    flow, chan, dmin = oracle.lpa(c["d"], 0.0, 0, 1, c["N"], c["prefactor"], c["reg_kind"], 1, k, xq, wq,
                                  c["rho"], c["u"], c["du"])
    m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
    E2 = k * k + m2
    ok = np.abs(E2) > 1e-9
    ref = c["prefactor"] * 2 * k ** (d + 2) / (d * E2)
    if d == 4 and k == 1.0:                      # the literal number: k^6/(64 pi^2 (k^2+m^2))
        np.testing.assert_allclose(ref[ok], 1 / (64 * PI ** 2 * E2[ok]), rtol=1e-15)
    if d == 3 and k == 1.0:                      # k^5/(6 pi^2 (k^2+m^2))
        np.testing.assert_allclose(ref[ok], 1 / (6 * PI ** 2 * E2[ok]), rtol=1e-15)
    np.testing.assert_allclose(chan[ok], ref[ok], rtol=1e-13)
    both = ok[0] & ok[1]
    np.testing.assert_allclose(flow[both], (3 * ref[0] + ref[1])[both], rtol=1e-12)
    np.testing.assert_allclose(dmin, np.minimum(E2[0], E2[1]) / (k * k), rtol=1e-14, atol=1e-14)


# ----------------------------------------------------------------------------------------
# P3  finite-T Litim (spatial regulator): truncated Matsubara sum, coth + digamma closed form
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("T_over_k", inputs.CONFIG1_TEMPERATURES)
def test_p3_finite_T_litim_coth_closed_form(T_over_k):
    k = 1.0
    c = inputs.config1(T_over_k, n_field=129, k=k, litim=True)
    xq, wq = rule(c["rule_q"])
    T, N = c["T"], c["n_max"]
    assert N == {0.05: 20, 0.1: 10, 0.2: 5, 0.5: 2}[T_over_k]
    flow, chan, dmin = oracle.lpa(3, T, N, 0, 4.0, c["prefactor"], oracle.REG_LITIM, 1, k, xq, wq,
                                  c["rho"], c["u"], c["du"])
    m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
    mp.mp.dps = 30
    checked = 0
    for ch in range(2):
        for f in range(0, 129, 7):
            E2 = k * k + m2[ch, f]
            if E2 <= 1e-3:
                continue
            E = mp.sqrt(E2)
            a = E / (2 * mp.pi * T)
            tail = mp.im(mp.digamma(N + 1 + 1j * a)) / a                       # sum_{n>N} 1/(n^2+a^2)
            S = mp.coth(E / (2 * T)) / (2 * E * T) - 2 / (2 * mp.pi * T) ** 2 * tail
            ref = c["prefactor"] * T * (2 * k ** 5 / 3) * S
            assert abs(chan[ch, f] / float(ref) - 1) < 1e-12
            checked += 1
    assert checked > 20
    # N -> infinity limit quoted in SURVEY P3: k^5 coth(E/2T)/(12 pi^2 E) bounds the truncated sum from above
    E = np.sqrt(k * k + m2[1, -1])
    assert chan[1, -1] < k ** 5 / math.tanh(E / (2 * T)) / (12 * PI ** 2 * E)


# ----------------------------------------------------------------------------------------
# P4  exponential regulator: weight integrals through the m^2 -> infinity limit
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("d,exact", [(4, 3.0), (3, 5 * math.sqrt(PI) / 4)])
def test_p4_exp_regulator_weight_integral_T0(d, exact):
    k, big = 1.0, 1e15
    xq, wq = oracle.gl_rule(64, 0.0, 8.0 * k)
    _, chan, _ = oracle.lpa(d, 0.0, 0, 1, 4.0, 1.0, oracle.REG_EXP_POLY, 1, k, xq, wq,
                            np.zeros(1), np.full(1, big), np.zeros(1))
    assert abs(chan[0, 0] * big / exact - 1) < 1e-12
    # on the config's own interval [0, 6k] the cut costs ~1e-13
    xq, wq = oracle.gl_rule(64, 0.0, 6.0 * k)
    _, chan, _ = oracle.lpa(d, 0.0, 0, 1, 4.0, 1.0, oracle.REG_EXP_POLY, 1, k, xq, wq,
                            np.zeros(1), np.full(1, big), np.zeros(1))
    assert abs(chan[0, 0] * big / exact - 1) < 1e-11


def test_p4_exp_regulator_weight_integral_finite_T():
    # I m^2/(C T) -> sum_n int_0^inf q^2 Rdot(w_n^2 + q^2) dq, each term a Gaussian integral:
    # int q^2 2 e^{-(w^2+q^2)} (1 + w^2 + q^2) dq = e^{-w^2} sqrt(pi) (5/4 + w^2/2)
    k, big, T, N = 1.0, 1e15, 0.2, 5
    xq, wq = oracle.gl_rule(64, 0.0, 8.0)
    _, chan, _ = oracle.lpa(3, T, N, 1, 4.0, 1.0, oracle.REG_EXP_POLY, 1, k, xq, wq,
                            np.zeros(1), np.full(1, big), np.zeros(1))
    ref = sum(math.exp(-(2 * PI * n * T) ** 2) * math.sqrt(PI) * (1.25 + 0.5 * (2 * PI * n * T) ** 2)
              for n in range(-N, N + 1))
    assert abs(chan[0, 0] * big / (T * ref) - 1) < 1e-12
    # spatial argument (reg_arg4d = 0): every Matsubara term carries the same weight 5 sqrt(pi)/4
    _, chan, _ = oracle.lpa(3, T, N, 0, 4.0, 1.0, oracle.REG_EXP_POLY, 1, k, xq, wq,
                            np.zeros(1), np.full(1, big), np.zeros(1))
    assert abs(chan[0, 0] * big / (T * (2 * N + 1) * 5 * math.sqrt(PI) / 4) - 1) < 1e-12


def test_lpa_exp_regulator_vs_adaptive_quadrature():
    # config 0 / config 1 integrands against mpmath adaptive quadrature of the continuum integral
    mp.mp.dps = 25
    k = 1.0
    c = inputs.config0(n_field=9)
    xq, wq = rule(c["rule_q"])
    flow, chan, _ = oracle.lpa(4, 0.0, 0, 1, 4.0, c["prefactor"], 1, 1, k, xq, wq, c["rho"], c["u"], c["du"])
    for f in (3, 5, 8):                                   # regular points (m^2 > -k^2)
        for ch, m2 in enumerate((c["u"][f], c["u"][f] + 2 * c["rho"][f] * c["du"][f])):
            ref = mp.quad(lambda q: q ** 3 * 2 * mp.exp(-q * q) * (1 + q * q) / (q * q + mp.exp(-q * q) + m2),
                          [0, 1, 2, 6]) / (32 * mp.pi ** 2)
            assert abs(chan[ch, f] / float(ref) - 1) < 1e-12
    c = inputs.config1(0.2, n_field=9)
    flow, chan, _ = oracle.lpa(3, c["T"], c["n_max"], 1, 4.0, c["prefactor"], 1, 1, k, xq, wq,
                               c["rho"], c["u"], c["du"])
    f, T = 6, c["T"]
    m2 = c["u"][f]
    ref = 0
    for n in range(-c["n_max"], c["n_max"] + 1):
        w2 = (2 * mp.pi * n * T) ** 2
        ref += mp.quad(lambda q: q * q * 2 * mp.exp(-(w2 + q * q)) * (1 + w2 + q * q)
                       / (w2 + q * q + mp.exp(-(w2 + q * q)) + m2), [0, 1, 2, 6])
    ref *= T / (4 * mp.pi ** 2)
    assert abs(chan[0, f] / float(ref) - 1) < 1e-12
    assert abs(flow[f] - (3 * chan[0, f] + chan[1, f])) < 1e-15 * abs(flow[f])


def test_p11_lpa_terms_even_in_n_and_dmin_sign():
    # dropping the n<0 half and doubling n>0 must give the same sum (terms are even in n)
    c = inputs.config1(0.2, n_field=33)
    xq, wq = rule(c["rule_q"])
    args = (c["prefactor"], 1, 1, 1.0, xq, wq, c["rho"], c["u"], c["du"])
    full = oracle.lpa(3, c["T"], 5, 1, 4.0, *args)[1]
    n0 = oracle.lpa(3, c["T"], 0, 1, 4.0, *args)[1]
    part = [oracle.lpa(3, c["T"], n, 1, 4.0, *args)[1] for n in range(6)]
    # sum_{|n|<=5} = term(0) + 2 sum_{n=1..5} term(n);  term(n) = (S_n - S_{n-1})/2
    regular = (c["u"] > -0.9)
    np.testing.assert_allclose(full[:, regular], (n0 + (part[5] - part[0]))[:, regular], rtol=1e-13)
    # dmin: negative as soon as a node sees D < 0 (reading A4); for m^2 > -min(s+R) it is positive
    _, _, dmin = oracle.lpa(3, c["T"], 5, 1, 4.0, *args)
    assert np.all(dmin[c["u"] < -1.05] < 0)
    assert np.all(dmin[c["u"] > -0.9] > 0)


# ----------------------------------------------------------------------------------------
# P9  dimensional scaling
# ----------------------------------------------------------------------------------------
def test_p9_lpa_scaling_with_k():
    for litim in (False, True):
        a = inputs.config0(n_field=65, k=1.0, litim=litim)
        b = inputs.config0(n_field=65, k=1.7, litim=litim)
        fa = oracle.lpa(4, 0.0, 0, 1, 4.0, a["prefactor"], a["reg_kind"], 1, 1.0, *rule(a["rule_q"]),
                        a["rho"], a["u"], a["du"])[0]
        fb = oracle.lpa(4, 0.0, 0, 1, 4.0, b["prefactor"], b["reg_kind"], 1, 1.7, *rule(b["rule_q"]),
                        b["rho"], b["u"], b["du"])[0]
        # rho ~ k^2, lambda dimensionless, I ~ k^4 in d=4:  int q^3 dq Rdot/(...) ~ k^4
        reg = a["u"] > -0.95
        np.testing.assert_allclose(fb[reg], 1.7 ** 4 * fa[reg], rtol=2e-12)
    a = inputs.config1(0.2, n_field=33, k=1.0)
    b = inputs.config1(0.2, n_field=33, k=1.7)
    assert a["n_max"] == b["n_max"]
    fa = oracle.lpa(3, a["T"], a["n_max"], 1, 4.0, a["prefactor"], 1, 1, 1.0, *rule(a["rule_q"]),
                    a["rho"], a["u"], a["du"])[0]
    fb = oracle.lpa(3, b["T"], b["n_max"], 1, 4.0, b["prefactor"], 1, 1, 1.7, *rule(b["rule_q"]),
                    b["rho"], b["u"], b["du"])[0]
    reg = a["u"] > -0.95
    np.testing.assert_allclose(fb[reg], 1.7 ** 4 * fa[reg], rtol=2e-12)     # T sum_n int q^2 dq ~ k^4


# ----------------------------------------------------------------------------------------
# two-point family (config 2)
# ----------------------------------------------------------------------------------------
def _twopoint(c, xq, wq, xc, wc, **over):
    a = dict(c)
    a.update(over)
    return oracle.loop4d_twopoint(a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], xq, wq, xc, wc,
                                  a["Z"], a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"], a["m2"], a["pext"],
                                  sel=a.get("sel"))


def test_p7_twopoint_p0_litim_closed_form():
    # Litim, Z = 1, p = 0, radial [0,k]: G = 1/(k^2+m^2) everywhere =>
    # out = C S_c coef0 2k^2 (k^4/4)/(k^2+m^2)^3 with S_c = sum_j w_j sqrt(1-c_j^2) -> pi/2
    for k in (1.0, 1.7):
        c = inputs.config2(n_field=17, n_ext=1, k=k)
        xq, wq = oracle.gl_rule(16, 0, k)
        xc, wc = oracle.gl_rule(32, -1, 1)
        out, dmin = _twopoint(c, xq, wq, xc, wc, reg_kind=oracle.REG_LITIM, Z=np.ones(8), interp=1,
                              pext=np.zeros(1), coef=np.array([0.7, 0.4]))
        Sc = float(np.sum(wc * np.sqrt(1 - xc ** 2)))
        assert abs(Sc - PI / 2) < 2e-4                    # GL sees the sqrt end points: algebraic convergence
        E2 = k * k + c["m2"]
        ok = np.abs(E2) > 1e-6
        ref = c["prefactor"] * Sc * 0.7 * 2 * k * k * (k ** 4 / 4) / E2 ** 3
        np.testing.assert_allclose(out[0][ok], ref[ok], rtol=1e-12)
        np.testing.assert_allclose(dmin[0], E2 / (k * k), rtol=1e-13, atol=1e-13)


def test_twopoint_constant_Z_multiplies_s_not_R():
    # Litim, Z = 1.7 (constant table), p = 0: D = 1.7 s + (k^2 - s) + m^2, not 1.7 (s + R)
    mp.mp.dps = 25
    k, m2, Zc = 1.0, 0.8, 1.7
    xq, wq = oracle.gl_rule(48, 0, k)
    xc, wc = oracle.gl_rule(8, -1, 1)
    c = inputs.config2(n_field=1, n_ext=1)
    out, _ = _twopoint(c, xq, wq, xc, wc, reg_kind=oracle.REG_LITIM, Z=np.full(8, Zc), interp=3,
                       pext=np.zeros(1), m2=np.array([m2]), coef=np.array([1.0, 0.0]))
    Sc = float(np.sum(wc * np.sqrt(1 - xc ** 2)))
    ref = mp.quad(lambda q: q ** 3 * 2 / ((Zc - 1) * q * q + 1 + m2) ** 3, [0, 1]) * Sc * c["prefactor"]
    assert abs(out[0, 0] / float(ref) - 1) < 1e-12


def test_twopoint_litim_kinematics_closed_form_angle():
    # Litim, Z = 1, p = 3k > 2k: the shifted line sees s > k^2 => G(s) = 1/(s + m^2), G(q) = 1/(k^2+m^2).
    # Angular integrals in closed form (a = q^2+p^2+m^2, b = 2qp):
    #   J0 = int sqrt(1-c^2)/(a+bc) dc = pi (a - sqrt(a^2-b^2))/b^2,   J1 = int sqrt(1-c^2) c/(a+bc) dc = (pi/2 - a J0)/b
    mp.mp.dps = 25
    k, p, m2, c0, c1 = 1.0, 3.0, 0.6, 0.9, 0.35
    xq, wq = oracle.gl_rule(24, 0, k)
    xc, wc = oracle.gl_rule(1500, -1, 1)
    c = inputs.config2(n_field=1, n_ext=1)
    out, _ = _twopoint(c, xq, wq, xc, wc, reg_kind=oracle.REG_LITIM, Z=np.ones(8), interp=1,
                       pext=np.array([p]), m2=np.array([m2]), coef=np.array([c0, c1]))

    def radial(q):
        a, b = q * q + p * p + m2, 2 * q * p
        J0 = mp.pi * (a - mp.sqrt(a * a - b * b)) / (b * b)
        J1 = (mp.pi / 2 - a * J0) / b
        return q ** 3 * 2 * k * k / (k * k + m2) ** 2 * (c0 * J0 + c1 * q * p / (k * k) * J1)
    ref = c["prefactor"] * mp.quad(radial, [0, k])
    assert abs(out[0, 0] / float(ref) - 1) < 2e-8        # limited by GL(1500) on the sqrt end points
    # a wrong sign of 2 q p c (or of the coef1 term) would change the result at the 1e-2 level:
    wrong = c["prefactor"] * mp.quad(lambda q: q ** 3 * 2 / (1 + m2) ** 2 * (
        c0 * mp.pi * ((q * q + p * p + m2) - mp.sqrt((q * q + p * p + m2) ** 2 - (2 * q * p) ** 2)) / (2 * q * p) ** 2
        - c1 * q * p * ((mp.pi / 2 - (q * q + p * p + m2) * mp.pi * ((q * q + p * p + m2) - mp.sqrt(
            (q * q + p * p + m2) ** 2 - (2 * q * p) ** 2)) / (2 * q * p) ** 2) / (2 * q * p))), [0, k])
    assert abs(float(wrong) / float(ref) - 1) > 1e-3


def test_twopoint_exp_regulator_vs_scipy_dblquad():
    # full config-2 integrand (exp regulator, dressed propagators) against adaptive 2-D quadrature of
    # the continuum integral with the ANALYTIC dressing Z(q) = 1 + 0.3/(1+q^2) (finely tabulated: no noise)
    k, p, m2 = 1.0, 0.7, 0.4
    qt, lo, hi = inputs.table_grid(4096)
    Zt = 1 + 0.3 / (1 + qt ** 2)
    xq, wq = oracle.gl_rule(96, 0, 8)
    xc, wc = oracle.gl_rule(1200, -1, 1)
    c = inputs.config2(n_field=1, n_ext=1)
    out, _ = _twopoint(c, xq, wq, xc, wc, Z=Zt, lnq_lo=lo, lnq_hi=hi, interp=3,
                       pext=np.array([p]), m2=np.array([m2]))

    def G(s):
        return 1.0 / ((1 + 0.3 / (1 + s)) * s + math.exp(-s) + m2)

    def f(cth, q):
        s = q * q + p * p + 2 * q * p * cth
        return (q ** 3 * 2 * math.exp(-q * q) * (1 + q * q) * G(q * q) ** 2
                * math.sqrt(max(1 - cth * cth, 0.0)) * (1 + 0.1 * q * p * cth) * G(s))
    ref, err = integrate.dblquad(f, 0, 8, -1, 1, epsabs=1e-12, epsrel=1e-10)
    ref *= c["prefactor"]
    assert abs(out[0, 0] / ref - 1) < 5e-8


def test_p8_p9_twopoint_linearity_and_scaling():
    c = inputs.config2(n_field=5, n_ext=3)
    xq, wq = rule((32, 0.0, 8.0))
    xc, wc = rule((12, -1.0, 1.0))
    o = lambda coef: _twopoint(c, xq, wq, xc, wc, coef=np.array(coef))[0]
    reg = c["m2"] > -0.5
    np.testing.assert_allclose(o([0.3, -1.1])[:, reg], (0.3 * o([1, 0]) - 1.1 * o([0, 1]))[:, reg], rtol=1e-13)
    # scaling: Z = 1 (dimensionless), everything else ~ k:  out ~ k^0 for d^4q Rdot G^3 (mass dim 4+2-6)
    k = 1.7
    c2 = inputs.config2(n_field=5, n_ext=3, k=k)
    assert np.allclose(c2["pext"], k * c["pext"]) and np.allclose(c2["m2"], k * k * c["m2"])
    a = _twopoint(c, xq, wq, xc, wc, Z=np.ones(8))[0]
    b = _twopoint(c2, k * xq, k * wq, xc, wc, Z=np.ones(8))[0]
    np.testing.assert_allclose(b[:, reg], a[:, reg], rtol=2e-12)


def test_p10_twopoint_quadrature_order_convergence():
    # algebraic convergence of the config's rule towards a brute-force 512 x 512 rule; the paper quotes
    # ~1e-4 for its medium rule 32 x 8 x 8
    c = inputs.config2(n_field=2, n_ext=2)
    c["m2"] = np.array([0.0, 5.0])
    c["pext"] = np.array([0.5, 3.0])
    ref = _twopoint(c, *oracle.gl_rule(512, 0, 8), *oracle.gl_rule(512, -1, 1))[0]
    errs = []
    for nq, nc in ((32, 8), (64, 16), (128, 32), (256, 64)):
        o = _twopoint(c, *oracle.gl_rule(nq, 0, 8), *oracle.gl_rule(nc, -1, 1))[0]
        errs.append(np.max(np.abs(o / ref - 1)))
    assert errs[0] < 5e-3 and errs[2] < 1e-4 and errs[3] < 1e-5
    assert errs[0] > errs[1] > errs[2] > errs[3]


def test_twopoint_sel_matches_full():
    c = inputs.config2(n_field=6, n_ext=4)
    xq, wq = rule((16, 0.0, 8.0))
    xc, wc = rule((8, -1.0, 1.0))
    full, dfull = _twopoint(c, xq, wq, xc, wc)
    sel = np.array([0, 7, 23, 13])
    part, dpart = _twopoint(c, xq, wq, xc, wc, sel=sel)
    assert np.array_equal(part, full.ravel()[sel]) and np.array_equal(dpart, dfull.ravel()[sel])


# ----------------------------------------------------------------------------------------
# three-point family (config 3)
# ----------------------------------------------------------------------------------------
def _threepoint(c, rq, r1, r2, rphi, **over):
    a = dict(c)
    a.update(over)
    return oracle.loop4d_threepoint(a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], *rq, *r1, *r2, *rphi,
                                    a["ZA"], a["Zc"], a["L3"], a["lnq_lo"], a["lnq_hi"], a["interp"],
                                    a["coef"], a["ext"], sel=a.get("sel"), literal_phi=a.get("literal_phi", False))


def _monomial_order(deg):
    return [(a, b, c) for a in range(deg + 1) for b in range(deg + 1 - a) for c in range(deg + 1 - a - b)]


def test_p8_threepoint_monomials_litim_small_momenta():
    # Litim, Z_A = 1, lambda3 = const, all |q +- p| < k: every propagator is 1/k^2, so each unit
    # coefficient vector leaves a pure monomial sum over the quadrature grid, written here with numpy.
    k, lam = 1.3, 0.9
    order = _monomial_order(4)
    assert len(order) == 35 and order[0] == (0, 0, 0) and order[1] == (0, 0, 1) and order[5] == (0, 1, 0)
    rq, r1, r2, rphi = (oracle.gl_rule(6, 0, 0.3 * k), oracle.gl_rule(5, -1, 1), oracle.gl_rule(4, -1, 1),
                        oracle.gl_rule(3, 0, 2 * PI))
    p1, p2, al = 0.25 * k, 0.3 * k, 0.7
    c = inputs.config3(n_p=1, n_alpha=1, k=k)
    base = dict(reg_kind=oracle.REG_LITIM, ZA=np.ones(8), Zc=np.ones(8), L3=np.full(8, lam), interp=1,
                ext=np.array([[p1, p2, al]]))
    q, wq = rq
    c1, w1 = r1
    c2, w2 = r2
    Q, C1, C2 = np.meshgrid(q, c1, c2, indexing="ij")
    W = (wq[:, None, None] * Q ** 3) * (w1[None, :, None] * np.sqrt(1 - C1 ** 2)) * w2[None, None, :] * rphi[1].sum()
    X = Q ** 2 / k ** 2
    Y = Q * p1 * C1 / k ** 2
    Zv = Q * p2 * (math.cos(al) * C1 + math.sin(al) * np.sqrt(1 - C1 ** 2) * C2) / k ** 2
    for idx, (a, b, cc) in enumerate(order):
        coef = np.zeros(35)
        coef[idx] = 1.0
        out, dmin = _threepoint(c, rq, r1, r2, rphi, coef=coef, **base)
        ref = c["prefactor"] * 2 * k * k * (1 / k ** 2) ** 3 * lam ** 3 * np.sum(W * X ** a * Y ** b * Zv ** cc)
        assert abs(out[0] - ref) <= 1e-12 * abs(ref) + 1e-22, (idx, a, b, cc)
        assert abs(dmin[0] - 1.0) < 1e-14
    # linearity (P8)
    kap = c["coef"]
    full = _threepoint(c, rq, r1, r2, rphi, coef=kap, **base)[0][0]
    parts = sum(kap[i] * _threepoint(c, rq, r1, r2, rphi, coef=np.eye(35)[i], **base)[0][0] for i in range(35))
    assert abs(full - parts) < 1e-12 * abs(full)


def test_threepoint_vs_scipy_tplquad():
    # full config-3 integrand against adaptive 3-D quadrature of the continuum integral with the ANALYTIC
    # rational dressings (finely tabulated).  Pins s_a = |q+p1|^2, s_b = |q-p2|^2, s_c, the vertex arguments.
    k = 1.0
    c = inputs.config3(n_p=1, n_alpha=1, n_tab=4096)
    U = inputs.splitmix64_uniform(7, 15)
    aA, aL = 0.5 + U[0:5], 0.5 + U[10:15]
    rat = lambda a, s: (a[0] + a[1] * s + a[2] * s * s) / (1 + a[3] * s + a[4] * s * s)
    p1, p2, al = 0.8, 1.7, 1.1
    kap = c["coef"]
    order = _monomial_order(4)
    GA = lambda s: 1.0 / (rat(aA, s) * s + math.exp(-s))
    sc = p1 * p1 + p2 * p2 + 2 * p1 * p2 * math.cos(al)

    def f(c2, c1, q):
        s1 = math.sqrt(max(1 - c1 * c1, 0.0))
        qp1 = q * p1 * c1
        qp2 = q * p2 * (math.cos(al) * c1 + math.sin(al) * s1 * c2)
        sa, sb = q * q + p1 * p1 + 2 * qp1, q * q + p2 * p2 - 2 * qp2
        lam = rat(aL, (p1 * p1 + q * q + sa) / 3) * rat(aL, (p2 * p2 + q * q + sb) / 3) * rat(aL, (sc + sa + sb) / 3)
        P = sum(kap[i] * (q * q) ** a * qp1 ** b * qp2 ** cc for i, (a, b, cc) in enumerate(order))
        return q ** 3 * 2 * math.exp(-q * q) * (1 + q * q) * GA(q * q) * s1 * GA(sa) * GA(sb) * lam * P
    ref, err = integrate.tplquad(f, 0, 8, -1, 1, -1, 1, epsabs=1e-8, epsrel=1e-6)
    ref *= 2 * PI * c["prefactor"]
    out, _ = _threepoint(c, oracle.gl_rule(64, 0, 8), oracle.gl_rule(400, -1, 1), oracle.gl_rule(24, -1, 1),
                         oracle.gl_rule(4, 0, 2 * PI), ext=np.array([[p1, p2, al]]))
    assert abs(out[0] / ref - 1) < 1e-5


def test_p11_threepoint_phi_axis_is_trivial():
    c = inputs.config3(n_p=2, n_alpha=2)
    rq, r1, r2 = oracle.gl_rule(6, 0, 8), oracle.gl_rule(5, -1, 1), oracle.gl_rule(4, -1, 1)
    a = _threepoint(c, rq, r1, r2, oracle.gl_rule(16, 0, 2 * PI))[0]
    b = _threepoint(c, rq, r1, r2, oracle.gl_rule(3, 0, 2 * PI))[0]
    lit = _threepoint(c, rq, r1, r2, oracle.gl_rule(16, 0, 2 * PI), literal_phi=True)[0]
    np.testing.assert_allclose(a, b, rtol=1e-14)
    np.testing.assert_allclose(a, lit, rtol=1e-14)
    # Z_c is accepted but unused (reading A14)
    z = _threepoint(c, rq, r1, r2, oracle.gl_rule(16, 0, 2 * PI), Zc=np.zeros_like(c["Zc"]))[0]
    assert np.array_equal(a, z)
    # external index order e = (a*32 + b)*8 + g
    cc = inputs.config3(n_p=3, n_alpha=2)
    assert cc["ext"].shape == (18, 3)
    assert cc["ext"][(1 * 3 + 2) * 2 + 1, 0] == cc["ext"][6, 0] and cc["ext"][(1 * 3 + 2) * 2 + 1, 1] == cc["ext"][4, 1]


# ----------------------------------------------------------------------------------------
# Matsubara family (config 4)
# ----------------------------------------------------------------------------------------
def _mats(c, rq, rc, **over):
    a = dict(c)
    a.update(over)
    return oracle.matsubara3d(a["T"], a["n_max"], a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], *rq, *rc,
                              a["Zpsi"], a["Zphi"], a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"],
                              a["m2psi"], a["m2phi"], a["pext"], a["n_jext"], sel=a.get("sel"))


def test_p8_matsubara_monomials_heavy_mass_limit():
    # m_psi^2 = m_phi^2 = M -> infinity: out M^3/(C T) -> sum_n (nu_n nu_j)^a int q^2 Rdot(s_psi) (p q)^b s_psi^c dq
    #   x int c^b dc, with Gaussian radial integrals done by mpmath and int c^b dc = 2/(b+1) (b even) or 0.
    mp.mp.dps = 30
    k, T, n_max, p, j, M = 1.0, 0.3, 2, 0.7, 1, 1e15
    c = inputs.config4(n_field=1, n_p=1, n_jext=2, T_over_k=T)
    rq, rc = oracle.gl_rule(64, 0, 9), oracle.gl_rule(6, -1, 1)
    order = _monomial_order(3)
    assert len(order) == 20
    nuj = (2 * j + 1) * PI * T
    for idx, (a, b, cc) in enumerate(order):
        coef = np.zeros(20)
        coef[idx] = 1.0
        out, _ = _mats(c, rq, rc, n_max=n_max, coef=coef, m2psi=np.array([M]), m2phi=np.array([M]),
                       pext=np.array([p]), n_jext=2)
        got = out[0, j, 0] * M ** 3 / (c["prefactor"] * T)
        ref, scale = mp.mpf(0), mp.mpf(0)                 # odd a: the n <-> -n-1 terms cancel, so bound
        for n in range(-n_max, n_max + 1):                # the error by the sum of |terms|
            nun = (2 * n + 1) * mp.pi * T
            rad = mp.quad(lambda q: q * q * 2 * mp.exp(-(nun ** 2 + q * q)) * (1 + nun ** 2 + q * q)
                          * (p * q) ** b * (nun ** 2 + q * q) ** cc, [0, 1, 3, 9])
            term = (nun * nuj) ** a * rad * (mp.mpf(2) / (b + 1) if b % 2 == 0 else 0)
            ref += term
            scale += abs(term)
        if b % 2:
            assert abs(got) < 1e-12, (idx, a, b, cc)
        else:
            assert abs(got - float(ref)) < 2e-11 * float(scale), (idx, a, b, cc)


def test_matsubara_vs_scipy_dblquad():
    # full config-4 integrand against adaptive 2-D quadrature per Matsubara term, ANALYTIC dressings.
    # Pins r^2 = p^2+q^2-2pqc, m = j - n, the |m| and nbar row selectors, 4-D regulator arguments, G_psi^2 G_phi.
    k, T, n_max, p, j, f = 1.0, 0.15, 3, 0.9, 2, 0
    c = inputs.config4(n_field=1, n_p=1, n_jext=4, n_tab=4096, T_over_k=T)
    U = inputs.splitmix64_uniform(4, 4)
    A_psi, B_psi, A_phi, B_phi = 0.1 + 0.4 * U[0], 0.5 + 1.5 * U[1], 0.1 + 0.4 * U[2], 0.5 + 1.5 * U[3]
    kap = c["coef"]
    order = _monomial_order(3)
    mpsi, mphi = 0.3, 0.5
    nuj = (2 * j + 1) * PI * T
    ref = 0.0
    for n in range(-n_max, n_max + 1):
        nun = (2 * n + 1) * PI * T
        nbar = n if n >= 0 else -n - 1
        m = j - n
        om = 2 * PI * m * T
        nu_row, om_row = (2 * nbar + 1) * PI * T, 2 * PI * abs(m) * T

        def g(cth, q):
            spsi = nun * nun + q * q
            r2 = p * p + q * q - 2 * p * q * cth
            sphi = om * om + r2
            Zp = 1 + A_psi / (1 + B_psi * (q * q + nu_row ** 2))
            Zb = 1 + A_phi / (1 + B_phi * (r2 + om_row ** 2))
            Gpsi = 1 / (Zp * spsi + math.exp(-spsi) + mpsi)
            Gphi = 1 / (Zb * sphi + math.exp(-sphi) + mphi)
            y1, y2, y3 = nun * nuj, p * q * cth, spsi
            P = sum(kap[i] * y1 ** a * y2 ** b * y3 ** cc for i, (a, b, cc) in enumerate(order))
            return q * q * 2 * math.exp(-spsi) * (1 + spsi) * Gpsi ** 2 * P * Gphi
        val, err = integrate.dblquad(g, 0, 10, -1, 1, epsabs=1e-13, epsrel=1e-10)
        ref += val
    ref *= c["prefactor"] * T
    out, _ = _mats(c, oracle.gl_rule(128, 0, 10), oracle.gl_rule(48, -1, 1), n_max=n_max,
                   m2psi=np.array([mpsi]), m2phi=np.array([mphi]), pext=np.array([p]), n_jext=4)
    assert abs(out[0, j, f] / ref - 1) < 1e-8


def test_p11_matsubara_symmetries_and_sel():
    c = inputs.config4(n_field=3, n_p=2, n_jext=3)
    rq, rc = oracle.gl_rule(8, 0, 10), oracle.gl_rule(4, -1, 1)
    full, dfull = _mats(c, rq, rc, n_max=2)
    assert full.shape == (2, 3, 3)
    sel = np.array([0, 5, 17, 9])
    part, dpart = _mats(c, rq, rc, n_max=2, sel=sel)
    assert np.array_equal(part, full.ravel()[sel]) and np.array_equal(dpart, dfull.ravel()[sel])
    # the boson line depends on (j, n) only through |j - n|: permuting the rows of Z_phi above the largest
    # |m| = n_jext-1+n_max that occurs changes nothing, touching row |m| = 4 does
    Zphi = c["Zphi"].copy()
    Zphi[5:] = Zphi[5:][::-1]
    assert np.array_equal(_mats(c, rq, rc, n_max=2, Zphi=Zphi)[0], full)
    Zphi = c["Zphi"].copy()
    Zphi[4] *= 1.01
    changed = _mats(c, rq, rc, n_max=2, Zphi=Zphi)[0]
    assert np.all(changed[:, 2] != full[:, 2]) and np.array_equal(changed[:, :2], full[:, :2])
    # fermion rows: nbar = n (n>=0), -n-1 (n<0): rows 0..n_max only
    Zpsi = c["Zpsi"].copy()
    Zpsi[3:] = 7.0
    assert np.array_equal(_mats(c, rq, rc, n_max=2, Zpsi=Zpsi)[0], full)


def test_p9_matsubara_scaling():
    k = 1.7
    a = inputs.config4(n_field=3, n_p=2, n_jext=2)
    b = inputs.config4(n_field=3, n_p=2, n_jext=2, k=k)
    rq, rc = oracle.gl_rule(16, 0, 10), oracle.gl_rule(6, -1, 1)
    one = np.ones_like(a["Zpsi"])
    oa = _mats(a, rq, rc, Zpsi=one, Zphi=one)[0]
    ob = _mats(b, (k * rq[0], k * rq[1]), rc, Zpsi=one, Zphi=one)[0]
    # T sum int q^2 dq Rdot G^2 G ~ k^(1+3+2-6) = k^0
    np.testing.assert_allclose(ob, oa, rtol=3e-12)


def test_oracle_regression_fixture():
    """The oracle's arithmetic is frozen by tests/golden/oracle_regression.txt (written by the committed script beside it,
    which calls only oracle/): a change of the oracle's numbers has to be deliberate -- regenerate the fixture and say why
    in the commit message.  (Not a pin: the pins are the tests above.)"""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_oracle_regression", os.path.join(here, "make_oracle_regression.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    stored = {}
    for line in open(os.path.join(here, "oracle_regression.txt")):
        if line.startswith("#"):
            continue
        name, idx, hx, _ = line.split(None, 3)
        stored[(name, int(idx))] = float.fromhex(hx)
    n = 0
    for name, vals in mod.cases():
        for i, v in enumerate(np.asarray(vals, dtype=np.float64)):
            ref = stored[(name, i)]
            assert abs(v - ref) <= 1e-14 * abs(ref) + 1e-300, (name, i, v, ref)
            n += 1
    assert n == len(stored) and n >= 30
