"""Pins for the oracle's tolerance yardsticks: `sens` (every family and every mass-derivative twin) and `dmin`
(three-point, 3-D-table and Matsubara families; lpa and two-point dmin are pinned in test_oracle_pins.py).

`sens` decides which outputs are graded by the relative bar and is the only bar for the others,
so a wrong sens -- a condition factor applied twice, a propagator power dropped, |P| instead of the sum of |monomials|
-- must fail here.  What fixes it from outside the oracle:

  S1  positive-term identity: non-negative masses, positive weights, tables and coefficients => every term is positive
      and every condition factor (|D - m2| + |m2|)/|D| is exactly 1, hence sens = out * (1 + sum of propagator powers)
      (1 for the families without a mass term, whose sens carries no condition factor).
  S2  worst-case response: with NEGATIVE masses (all D still positive) scale Z tables and zk by (1 + d), the masses by
      (1 - d) and the prefactor by (1 - 2 d): every first-order contribution has the same sign and the pinned VALUE
      function must move by -d * sens.  This is the definition of sens as a first-order perturbation bound, attained.
  S3  sum of |monomials|: sens is invariant under sign flips of the coefficients and additive in |kappa|.
  S4  a plain numpy restatement on a 3 x 2 x 2-node input with mixed signs (mass, coefficients, nodes).
  S5  sens bounds the response to random relative perturbations of size 1e-9 of every input of the value function.
dmin: closed forms with flat regulators and Z = 1, the monotonicity of s + R(s), and "which propagator sets the minimum".
CPU only.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2412_13043_b200 import inputs

PI = math.pi
EXP, LITIM = 1, 0


def gl(n, a, b):
    return oracle.gl_rule(n, a, b)


# ---------------------------------------------------------------------------------------------------------
# small workloads (positive tables)
# ---------------------------------------------------------------------------------------------------------
def twopoint_args(m2, coef=(1.0, 0.0), zk=1.0, zscale=1.0, prefactor=0.7, pext=(0.3, 2.0), k=1.3):
    c = inputs.config2(n_field=4, n_ext=2, n_q=7, n_c=5, k=k)
    xq, wq = gl(7, 0.0, 8.0 * k)
    xc, wc = gl(5, -1.0, 1.0)
    return dict(prefactor=prefactor, reg_kind=EXP, reg_order=2, k=k, xq=xq, wq=wq, xc=xc, wc=wc, Z=zscale * c["Z"],
                lnq_lo=c["lnq_lo"], lnq_hi=c["lnq_hi"], interp=3, coef=np.array(coef), m2=np.asarray(m2, dtype=float),
                pext=np.array(pext) * k, zk=zk)


def mats_args(m2psi, m2phi, coef=None, zk=1.0, zscale=1.0, prefactor=0.9, k=1.2, reg_kind=EXP, n_max=2, n_jext=2, T=0.21,
              nq=4, nc=3, pext=(0.4, 1.7)):
    c = inputs.config4(n_field=3, n_p=2, n_jext=n_jext, n_q=nq, n_c=nc, k=k)
    xq, wq = gl(nq, 0.0, 4.0 * k)
    xc, wc = gl(nc, -1.0, 1.0)
    if coef is None:                         # P = 0.8 + 0.5 y3 + 0.25 y3^2: positive monomials only (y3 = s_psi / k^2 > 0)
        coef = np.zeros(20)
        coef[idx3(0, 0, 0)], coef[idx3(0, 0, 1)], coef[idx3(0, 0, 2)] = 0.8, 0.5, 0.25
    return dict(T=T * k, n_max=n_max, prefactor=prefactor, reg_kind=reg_kind, reg_order=1, k=k, xq=xq, wq=wq, xc=xc, wc=wc,
                Zpsi=zscale * c["Zpsi"], Zphi=zscale * c["Zphi"], lnq_lo=c["lnq_lo"], lnq_hi=c["lnq_hi"], interp=3,
                coef=np.asarray(coef, dtype=float), m2psi=np.asarray(m2psi, dtype=float), m2phi=np.asarray(m2phi, dtype=float),
                pext=np.array(pext) * k, n_jext=n_jext, zk=zk)


def idx3(a, b, c, deg=3):
    """position of the monomial (a, b, c) in the coefficient order `a outermost, then b, then c, a + b + c <= deg`"""
    i = 0
    for aa in range(deg + 1):
        for bb in range(deg + 1 - aa):
            for cc in range(deg + 1 - aa - bb):
                if (aa, bb, cc) == (a, b, c):
                    return i
                i += 1
    raise ValueError


def threepoint_args(coef, ext=((0.4, 0.9, 0.7), (2.0, 0.3, 2.1)), k=1.1, reg_kind=EXP, ZA=None, L3=None, nq=4, n1=4, n2=3):
    c = inputs.config3(n_p=2, n_alpha=1, n_q=nq, n_c1=n1, n_c2=n2, n_phi=3, k=k)
    xq, wq = gl(nq, 0.0, 6.0 * k)
    x1, w1 = gl(n1, -1.0, 1.0)
    x2, w2 = gl(n2, -1.0, 1.0)
    xp, wp = gl(3, 0.0, 2 * PI)
    e = np.array(ext, dtype=float)
    e[:, :2] *= k
    return dict(prefactor=0.6, reg_kind=reg_kind, reg_order=1, k=k, xq=xq, wq=wq, x1=x1, w1=w1, x2=x2, w2=w2, xphi=xp,
                wphi=wp, ZA=c["ZA"] if ZA is None else ZA, Zc=c["Zc"], L3=c["L3"] if L3 is None else L3,
                lnq_lo=c["lnq_lo"], lnq_hi=c["lnq_hi"], interp=3, coef=np.asarray(coef, dtype=float), ext=e)


def call_two(a, **kw):
    return oracle.loop4d_twopoint(a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], a["xq"], a["wq"], a["xc"], a["wc"],
                                  a["Z"], a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"], a["m2"], a["pext"],
                                  want_sens=True, zk=a["zk"], **kw)


def call_two_dm2(a):
    return oracle.loop4d_twopoint_dm2(a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], a["xq"], a["wq"], a["xc"], a["wc"],
                                      a["Z"], a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"], a["m2"], a["pext"], zk=a["zk"])


def _mats_tuple(a):
    return (a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], a["xq"], a["wq"], a["xc"], a["wc"], a["Zpsi"], a["Zphi"],
            a["lnq_lo"], a["lnq_hi"], a["interp"], a["coef"], a["m2psi"], a["m2phi"], a["pext"], a["n_jext"])


def call_mats(a):
    return oracle.matsubara3d(a["T"], a["n_max"], *_mats_tuple(a), want_sens=True, zk=a["zk"])


def call_mats_mu(a, mu):
    return oracle.matsubara3d_mu(a["T"], a["n_max"], mu, *_mats_tuple(a), want_sens=True, zk=a["zk"])


def call_mats_dm2(a):
    return oracle.matsubara3d_dm2(a["T"], a["n_max"], *_mats_tuple(a), zk=a["zk"])


def call_mats_mu_dm2(a, mu):
    return oracle.matsubara3d_mu_dm2(a["T"], a["n_max"], mu, *_mats_tuple(a), zk=a["zk"])


def call_three(a):
    return oracle.loop4d_threepoint(a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], a["xq"], a["wq"], a["x1"], a["w1"],
                                    a["x2"], a["w2"], a["xphi"], a["wphi"], a["ZA"], a["Zc"], a["L3"], a["lnq_lo"],
                                    a["lnq_hi"], a["interp"], a["coef"], a["ext"], want_sens=True)


def lpa_case(T, u, k=1.4, zk=1.0, prefactor=0.8, d=3, reg_kind=EXP, reg_arg4d=1, n_max=3, nq=6):
    xq, wq = gl(nq, 0.0, 5.0 * k)
    u = np.asarray(u, dtype=float)
    rho = np.linspace(0.1, 0.4, u.size)
    du = np.full(u.size, 0.3)
    return dict(d=d, T=T * k, n_max=n_max if T > 0 else 0, reg_arg4d=reg_arg4d, N=4.0, prefactor=prefactor, reg_kind=reg_kind,
                reg_order=1, k=k, xq=xq, wq=wq, rho=rho, u=u, du=du, zk=zk)


def call_lpa(a):
    return oracle.lpa(a["d"], a["T"], a["n_max"], a["reg_arg4d"], a["N"], a["prefactor"], a["reg_kind"], a["reg_order"],
                      a["k"], a["xq"], a["wq"], a["rho"], a["u"], a["du"], want_sens=True, zk=a["zk"])


def call_lpa_dm2(a):
    return oracle.lpa_dm2(a["d"], a["T"], a["n_max"], a["reg_arg4d"], a["prefactor"], a["reg_kind"], a["reg_order"], a["k"],
                          a["xq"], a["wq"], a["rho"], a["u"], a["du"], zk=a["zk"])


# ---------------------------------------------------------------------------------------------------------
# S1  positive-term identity
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T", [0.0, 0.17])
def test_s1_lpa_positive_terms(T):
    a = lpa_case(T, u=[0.0, 0.4, 2.5])
    flow, chan, dmin, sens = call_lpa(a)
    np.testing.assert_allclose(sens, 2.0 * chan, rtol=1e-13)             # one propagator: 1 + 1
    d, sd = call_lpa_dm2(a)
    np.testing.assert_allclose(sd, 3.0 * np.abs(d), rtol=1e-13)          # 1/D^2: 1 + 2
    assert np.all(d < 0)


def test_s1_lpa_fermion_positive_terms_at_zero_mu():
    a = lpa_case(0.2, u=[0.0, 0.6])
    I, dI, dmin, sens, sens_d = oracle.lpa_fermion(a["d"], a["T"], 2, 0.0, a["prefactor"], a["reg_kind"], a["reg_order"],
                                                   a["k"], a["xq"], a["wq"], a["u"])
    np.testing.assert_allclose(sens, 2.0 * I, rtol=1e-13)
    np.testing.assert_allclose(sens_d, 3.0 * np.abs(dI), rtol=1e-13)


def test_s1_twopoint_positive_terms():
    a = twopoint_args(m2=[0.0, 0.3, 1.0, 7.0])
    out, dmin, sens = call_two(a)
    assert np.all(out > 0)
    np.testing.assert_allclose(sens, 4.0 * out, rtol=1e-13)              # G(q)^2 G(s): 1 + 2 + 1
    d, sd = call_two_dm2(a)
    # -2 G(q)^3 G(s) carries 1 + 3 + 1, -G(q)^2 G(s)^2 carries 1 + 2 + 2: both 5
    np.testing.assert_allclose(sd, 5.0 * np.abs(d), rtol=1e-13)


def test_s1_matsubara_positive_terms():
    a = mats_args(m2psi=[0.0, 0.5, 2.0], m2phi=[0.0, 0.2, 3.0])
    out, dmin, sens = call_mats(a)
    assert np.all(out > 0)
    np.testing.assert_allclose(sens, 4.0 * out, rtol=1e-13)              # G_psi^2 G_phi
    dpsi, dphi, spsi, sphi = call_mats_dm2(a)
    np.testing.assert_allclose(spsi, 5.0 * np.abs(dpsi), rtol=1e-13)     # G_psi^3 G_phi
    np.testing.assert_allclose(sphi, 5.0 * np.abs(dphi), rtol=1e-13)     # G_psi^2 G_phi^2
    # spatial-regulator twin at mu = 0 (real, positive)
    o2, dm2, s2 = call_mats_mu(a, 0.0)
    np.testing.assert_allclose(s2, 4.0 * o2.real, rtol=1e-13)
    assert np.all(o2.imag == 0)
    dp2, df2, sp2, sf2 = call_mats_mu_dm2(a, 0.0)
    np.testing.assert_allclose(sp2, 5.0 * np.abs(dp2), rtol=1e-13)
    np.testing.assert_allclose(sf2, 5.0 * np.abs(df2), rtol=1e-13)


def test_s1_threepoint_families_positive_monomials():
    # monomials with even powers of q.p1 and no q.p2 are positive at every node: sens = out (no condition factor in the
    # families without a mass term)
    coef = np.zeros(35)
    coef[idx3(0, 0, 0, 4)], coef[idx3(1, 0, 0, 4)], coef[idx3(0, 2, 0, 4)], coef[idx3(2, 2, 0, 4)] = 0.7, 0.3, 0.9, 0.2
    a = threepoint_args(coef)
    out, dmin, sens = call_three(a)
    assert np.all(out > 0)
    np.testing.assert_allclose(sens, out, rtol=1e-13)
    # 3-D vertex table twin
    c6 = inputs.config6(n_p=2, n_alpha=1, n_q=4, n_c1=4, n_c2=3, n3=(12, 4, 3), k=a["k"])
    o3, d3, s3 = oracle.loop4d_threepoint_tab3d(a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], a["xq"], a["wq"],
                                                a["x1"], a["w1"], a["x2"], a["w2"], a["wphi"], a["ZA"], a["lnq_lo"],
                                                a["lnq_hi"], a["interp"], c6["v3"], c6["lo3"], c6["hi3"], c6["log3"],
                                                coef, a["ext"], want_sens=True)
    assert np.all(o3 > 0) and np.all(c6["v3"] > 0)
    np.testing.assert_allclose(s3, o3, rtol=1e-13)
    # four-point: monomials in q^2 only
    c5 = inputs.config5(n_s=2, n_ang=1, n_q=3, n_c1=3, n_c2=2, n_phi=3, k=a["k"])
    k4 = np.zeros(70)
    k4[0], k4[35], k4[34], k4[69] = 0.5, 0.4, 0.1, 0.2          # (0,0,0,0) and (3,0,0,0) of both polynomials
    xq, wq = gl(3, 0.0, 6.0 * a["k"])
    x1, w1 = gl(3, -1.0, 1.0)
    x2, w2 = gl(2, -1.0, 1.0)
    o4, d4, s4 = oracle.loop4d_fourpoint(0.6, EXP, 1, a["k"], xq, wq, x1, w1, x2, w2, a["xphi"], a["wphi"], c5["ZA"], c5["Zc"],
                                         c5["L3"], c5["lnq_lo"], c5["lnq_hi"], 3, k4, c5["ext"], want_sens=True)
    np.testing.assert_allclose(s4, o4, rtol=1e-13)


# ---------------------------------------------------------------------------------------------------------
# S2  worst-case first-order response with negative masses
# ---------------------------------------------------------------------------------------------------------
DELTA = 1e-6


def test_s2_twopoint_worst_case_response():
    m2 = np.array([-0.2, -0.45, -0.7]) * 1.3 ** 2              # D = Z s + R + m2 stays positive (Z >= 1, s + R >= k^2)
    a0 = twopoint_args(m2=m2)
    out, dmin, sens = call_two(a0)
    assert np.all(dmin > 0) and np.all(sens > 4.05 * out)      # condition factors > 1 now
    a1 = twopoint_args(m2=m2 * (1 - DELTA), zk=1 + DELTA, zscale=1 + DELTA, prefactor=0.7 * (1 - 2 * DELTA))
    out1, _, _ = call_two(a1)
    np.testing.assert_allclose((out - out1) / DELTA, sens, rtol=2e-4)
    # derivative twin: each of its two products attains its own bound under the same perturbation
    d, sd = call_two_dm2(a0)
    d1, _ = call_two_dm2(a1)
    np.testing.assert_allclose((np.abs(d) - np.abs(d1)) / DELTA, sd, rtol=2e-4)


def test_s2_matsubara_worst_case_response():
    k = 1.2
    mpsi, mphi = np.array([-0.3, -0.1, -0.5]) * k * k, np.array([-0.5, -0.6, -0.05]) * k * k
    a0 = mats_args(mpsi, mphi)
    out, dmin, sens = call_mats(a0)
    assert np.all(dmin > 0) and np.all(sens > 4.05 * out)
    a1 = mats_args(mpsi * (1 - DELTA), mphi * (1 - DELTA), zk=1 + DELTA, zscale=1 + DELTA, prefactor=0.9 * (1 - 2 * DELTA))
    out1, _, _ = call_mats(a1)
    np.testing.assert_allclose((out - out1) / DELTA, sens, rtol=2e-4)
    dpsi, dphi, spsi, sphi = call_mats_dm2(a0)
    dpsi1, dphi1, _, _ = call_mats_dm2(a1)
    np.testing.assert_allclose((np.abs(dpsi) - np.abs(dpsi1)) / DELTA, spsi, rtol=2e-4)
    np.testing.assert_allclose((np.abs(dphi) - np.abs(dphi1)) / DELTA, sphi, rtol=2e-4)
    # spatial-regulator twin (mu = 0): same bound structure
    o, dm, s = call_mats_mu(a0, 0.0)
    o1, _, _ = call_mats_mu(a1, 0.0)
    np.testing.assert_allclose((o.real - o1.real) / DELTA, s, rtol=2e-4)
    dp, df, sp, sf = call_mats_mu_dm2(a0, 0.0)
    dp1, df1, _, _ = call_mats_mu_dm2(a1, 0.0)
    np.testing.assert_allclose((np.abs(dp) - np.abs(dp1)) / DELTA, sp, rtol=2e-4)
    np.testing.assert_allclose((np.abs(df) - np.abs(df1)) / DELTA, sf, rtol=2e-4)


def test_s2_lpa_worst_case_response_through_zk():
    # lpa has no table: D = s + zk R_shape + m2.  With the flat regulator below k (all nodes inside), s + zk (k^2 - s) is
    # linear in zk, so scaling "D - m2" by (1 + d) is reachable exactly by zk -> zk + d (s + zk (k^2 - s))/(k^2 - s) only per
    # node; instead use s -> 0: a rule concentrated at tiny q makes D - m2 = zk k^2 to 1e-8, and zk scales it.
    k = 1.4
    xq, wq = gl(5, 0.0, 1e-4 * k)
    u = np.array([-0.3, -0.6]) * k * k
    base = dict(d=3, T=0.0, n_max=0, reg_arg4d=1, N=4.0, prefactor=0.8, reg_kind=LITIM, reg_order=1, k=k, xq=xq, wq=wq,
                rho=np.array([0.1, 0.2]), u=u, du=np.array([0.0, 0.0]), zk=1.0)
    flow, chan, dmin, sens = call_lpa(base)
    pert = dict(base, u=u * (1 - DELTA), zk=1 + DELTA, prefactor=0.8 * (1 - 2 * DELTA))
    _, chan1, _, _ = call_lpa(pert)
    np.testing.assert_allclose((chan - chan1) / DELTA, sens, rtol=2e-4)
    d, sd = call_lpa_dm2(base)
    d1, _ = call_lpa_dm2(pert)
    np.testing.assert_allclose((np.abs(d) - np.abs(d1)) / DELTA, sd, rtol=2e-4)


# ---------------------------------------------------------------------------------------------------------
# S3  sum of |monomials|
# ---------------------------------------------------------------------------------------------------------
def test_s3_sens_is_invariant_under_coefficient_signs_and_additive_in_abs_kappa():
    rng = np.random.default_rng(5)
    # Matsubara family (20 coefficients)
    kap = rng.uniform(0.2, 1.0, 20)
    sgn = rng.choice([-1.0, 1.0], 20)
    base = mats_args([0.3, 0.1, 0.8], [0.2, 0.9, 0.4], coef=kap)
    _, _, s_pos = call_mats(base)
    o_mix, _, s_mix = call_mats(mats_args([0.3, 0.1, 0.8], [0.2, 0.9, 0.4], coef=kap * sgn))
    np.testing.assert_allclose(s_mix, s_pos, rtol=1e-13)
    assert np.all(s_mix > 1.5 * np.abs(o_mix))                  # the mixed polynomial really cancels
    unit = sum(kap[i] * call_mats(mats_args([0.3, 0.1, 0.8], [0.2, 0.9, 0.4], coef=np.eye(20)[i]))[2] for i in range(20))
    np.testing.assert_allclose(unit, s_pos, rtol=1e-12)
    _, _, s_mu = call_mats_mu(base, 0.4)
    _, _, s_mu_mix = call_mats_mu(mats_args([0.3, 0.1, 0.8], [0.2, 0.9, 0.4], coef=kap * sgn), 0.4)
    np.testing.assert_allclose(s_mu_mix, s_mu, rtol=1e-13)
    # three-point family (35 coefficients)
    kap3 = rng.uniform(0.2, 1.0, 35)
    sgn3 = rng.choice([-1.0, 1.0], 35)
    _, _, s3 = call_three(threepoint_args(kap3))
    o3m, _, s3m = call_three(threepoint_args(kap3 * sgn3))
    np.testing.assert_allclose(s3m, s3, rtol=1e-13)
    assert np.all(s3m > 1.2 * np.abs(o3m))
    unit3 = sum(kap3[i] * call_three(threepoint_args(np.eye(35)[i]))[2] for i in range(35))
    np.testing.assert_allclose(unit3, s3, rtol=1e-12)
    # two-point (2 coefficients)
    _, _, s2 = call_two(twopoint_args([0.2, 0.5], coef=(0.7, 0.4)))
    _, _, s2m = call_two(twopoint_args([0.2, 0.5], coef=(0.7, -0.4)))
    np.testing.assert_allclose(s2m, s2, rtol=1e-13)


# ---------------------------------------------------------------------------------------------------------
# S4  plain numpy restatement on a tiny mixed-sign input
# ---------------------------------------------------------------------------------------------------------
def np_reg(kind, order, k, s, zk=1.0):
    k2 = k * k
    if kind == LITIM:
        return (zk * (k2 - s), zk * 2 * k2) if s < k2 else (0.0, 0.0)
    x = s / k2
    R = k2 * math.exp(-sum(x ** i / i for i in range(1, order + 1)))
    return zk * R, zk * 2 * R * (1 + sum(x ** i for i in range(1, order + 1)))


def test_s4_matsubara_sens_numpy_restatement():
    k = 1.2
    kap = np.array([0.8, -0.5, 0.3, 0.0, -0.7, 0.2, 0.0, 0.0, 0.4, 0.0, -0.6, 0.0, 0.3, 0.0, 0.0, 0.0, 0.5, 0.0, 0.0, -0.2])
    a = mats_args(m2psi=[-0.25 * k * k, 0.4], m2phi=[0.3, -0.35 * k * k], coef=kap, nq=3, nc=2, n_max=1, zk=1.15)
    out, dmin, sens = call_mats(a)
    T, k2 = a["T"], k * k
    mono_idx = [(aa, bb, cc) for aa in range(4) for bb in range(4 - aa) for cc in range(4 - aa - bb)]
    for e, p in enumerate(a["pext"]):
        for j in range(a["n_jext"]):
            for f in range(2):
                tot, val = 0.0, 0.0
                for n in range(-a["n_max"], a["n_max"] + 1):
                    nun, nuj = (2 * n + 1) * PI * T, (2 * j + 1) * PI * T
                    nbar, mabs = (n if n >= 0 else -n - 1), abs(j - n)
                    om = 2 * PI * (j - n) * T
                    for q, wq in zip(a["xq"], a["wq"]):
                        spsi = nun * nun + q * q
                        Rp, Rdp = np_reg(EXP, 1, k, spsi, a["zk"])
                        Dpsi = oracle.table_lookup(a["Zpsi"][nbar], a["lnq_lo"], a["lnq_hi"], 3, q * q) * spsi + Rp + a["m2psi"][f]
                        cpsi = (abs(Dpsi - a["m2psi"][f]) + abs(a["m2psi"][f])) / abs(Dpsi)
                        for c, wc in zip(a["xc"], a["wc"]):
                            r2 = max(p * p + q * q - 2 * p * q * c, 0.0)
                            sphi = om * om + r2
                            Rb, _ = np_reg(EXP, 1, k, sphi, a["zk"])
                            Dphi = oracle.table_lookup(a["Zphi"][mabs], a["lnq_lo"], a["lnq_hi"], 3, r2) * sphi + Rb + a["m2phi"][f]
                            cphi = (abs(Dphi - a["m2phi"][f]) + abs(a["m2phi"][f])) / abs(Dphi)
                            y = (nun * nuj / k2, p * q * c / k2, spsi / k2)
                            monos = [kap[i] * y[0] ** aa * y[1] ** bb * y[2] ** cc for i, (aa, bb, cc) in enumerate(mono_idx)]
                            w = wq * q * q * Rdp / Dpsi ** 2 * wc / Dphi
                            val += w * sum(monos)
                            tot += abs(w) * sum(abs(m) for m in monos) * (1 + 2 * cpsi + cphi)
                np.testing.assert_allclose(out[e, j, f], a["prefactor"] * T * val, rtol=1e-12)
                np.testing.assert_allclose(sens[e, j, f], abs(a["prefactor"]) * T * tot, rtol=1e-12)


def test_s4_lpa_sens_numpy_restatement():
    a = lpa_case(0.23, u=[-0.4, 0.7, -1.1], reg_arg4d=1, n_max=2, zk=0.9)
    flow, chan, dmin, sens = call_lpa(a)
    k, T = a["k"], a["T"]
    for f in range(3):
        for ch, m2 in enumerate((a["u"][f], a["u"][f] + 2 * a["rho"][f] * a["du"][f])):
            tot = 0.0
            for n in range(-2, 3):
                for q, w in zip(a["xq"], a["wq"]):
                    s = (2 * PI * n * T) ** 2 + q * q
                    R, Rd = np_reg(EXP, 1, k, s, a["zk"])
                    D = s + R + m2
                    tot += abs(w * q ** 2 * Rd / D) * (1 + (abs(s + R) + abs(m2)) / abs(D))
            np.testing.assert_allclose(sens[ch, f], a["prefactor"] * T * tot, rtol=1e-12)


# ---------------------------------------------------------------------------------------------------------
# S5  sens bounds the response to random relative perturbations of every input
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(4))
def test_s5_sens_bounds_random_perturbations(seed):
    rng = np.random.default_rng(100 + seed)
    eps = 1e-9
    jit = lambda x: np.asarray(x) * (1 + eps * rng.uniform(-1, 1, np.shape(x)))
    k = 1.2
    kap = rng.uniform(-1, 1, 20)
    mpsi, mphi = rng.uniform(-0.4, 1.0, 3) * k * k, rng.uniform(-0.6, 1.0, 3) * k * k
    a = mats_args(mpsi, mphi, coef=kap)
    out, dmin, sens = call_mats(a)
    b = dict(a, prefactor=float(jit(a["prefactor"])), wq=jit(a["wq"]), wc=jit(a["wc"]), Zpsi=jit(a["Zpsi"]), Zphi=jit(a["Zphi"]),
             coef=jit(kap), m2psi=jit(mpsi), m2phi=jit(mphi), zk=float(jit(1.0)))
    out1, _, _ = call_mats(b)
    # every factor of a term moves by <= eps (tables through at most 4 stencil values with Lagrange weights of modulus
    # <= 1.25: allow 2 x); the bound must hold with that slack, and must not be vacuous
    assert np.all(np.abs(out1 - out) <= 2.5 * eps * sens)
    assert np.max(np.abs(out1 - out) / sens) > 0.02 * eps
    # two-point
    a = twopoint_args(m2=rng.uniform(-0.5, 1.0, 4) * 1.69, coef=(0.8, -0.3))
    out, dmin, sens = call_two(a)
    b = dict(a, prefactor=float(jit(a["prefactor"])), wq=jit(a["wq"]), wc=jit(a["wc"]), Z=jit(a["Z"]), coef=jit(a["coef"]),
             m2=jit(a["m2"]), zk=float(jit(1.0)))
    out1, _, _ = call_two(b)
    assert np.all(np.abs(out1 - out) <= 2.5 * eps * sens)
    # three-point (weights, tables, coefficients)
    a = threepoint_args(rng.uniform(-1, 1, 35))
    out, dmin, sens = call_three(a)
    b = dict(a, wq=jit(a["wq"]), w1=jit(a["w1"]), w2=jit(a["w2"]), coef=jit(a["coef"]), L3=jit(a["L3"]))
    out1, _, _ = call_three(b)
    assert np.all(np.abs(out1 - out) <= 6 * eps * sens)       # three vertex look-ups, two weights, one coefficient


# ---------------------------------------------------------------------------------------------------------
# dmin
# ---------------------------------------------------------------------------------------------------------
def test_dmin_matsubara_closed_forms_and_which_line_sets_it():
    k = 1.2
    ones = np.ones_like(inputs.config4(n_field=3, n_p=2, n_jext=2, n_q=4, n_c=3, k=k)["Zpsi"])
    T = 0.05                                                    # (pi T)^2 + q_min^2 < k^2: the flat regulator is active
    for mpsi, mphi in (([0.3, 0.1, -0.2], [0.5, 0.6, 0.9]),     # fermion line sets the minimum
                       ([0.7, 0.9, 1.4], [0.2, -0.3, 0.05])):   # boson line sets it
        mpsi, mphi = np.array(mpsi) * k * k, np.array(mphi) * k * k
        a = mats_args(mpsi, mphi, reg_kind=LITIM, T=T, pext=(0.4, 0.6))   # |p - q|^2 < k^2 at the first radial node
        a["Zpsi"], a["Zphi"] = ones, ones
        assert (PI * a["T"]) ** 2 + a["xq"][0] ** 2 < k * k and (a["pext"].max() + a["xq"][0]) ** 2 < k * k
        # 4-D flat regulator: D = max(s, k^2) + m2 on both lines; the m = j - n = 0 boson term is in range
        out, dmin, sens = call_mats(a)
        want = (k * k + np.minimum(mpsi, mphi)) / (k * k)
        np.testing.assert_allclose(dmin, np.broadcast_to(want, dmin.shape), rtol=1e-14)
        # spatial flat regulator: D_psi = nu_n^2 + max(q^2, k^2) + m2_psi >= (pi T)^2 + k^2 + m2_psi, D_phi >= k^2 + m2_phi
        o2, dm2, s2 = call_mats_mu(a, 0.0)
        want2 = np.minimum((PI * a["T"]) ** 2 + k * k + mpsi, k * k + mphi) / (k * k)
        np.testing.assert_allclose(dm2, np.broadcast_to(want2, dm2.shape), rtol=1e-14)
        # moving ONLY the mass of the line that sets the minimum moves dmin by that amount; the other mass does not
        shift = 0.01 * k * k
        a_psi = dict(a, m2psi=mpsi - shift)
        a_phi = dict(a, m2phi=mphi - shift)
        d_psi, d_phi = call_mats(a_psi)[1], call_mats(a_phi)[1]
        psi_sets = mpsi < mphi
        np.testing.assert_allclose((dmin - d_psi)[..., psi_sets], shift / (k * k), rtol=1e-10)
        np.testing.assert_allclose((dmin - d_phi)[..., ~psi_sets], shift / (k * k), rtol=1e-10)
        assert np.all((dmin - d_psi)[..., ~psi_sets & (mpsi - shift > mphi)] == 0)
    # mu != 0: dmin = min(|D_psi|, D_phi); |D_psi|^2 = (nu^2 - mu^2 + max(q^2,k^2) + m2)^2 + (2 nu mu)^2 at nu = pi T
    mu = 0.4 * k
    mpsi, mphi = np.array([0.3, 0.1, -0.2]) * k * k, np.array([5.0, 6.0, 9.0]) * k * k
    a = mats_args(mpsi, mphi, reg_kind=LITIM, T=T, pext=(0.4, 0.6))
    a["Zpsi"], a["Zphi"] = ones, ones
    o3, dm3, s3 = call_mats_mu(a, mu)
    nu = PI * a["T"]
    want3 = np.hypot(nu * nu - mu * mu + k * k + mpsi, 2 * nu * mu) / (k * k)
    np.testing.assert_allclose(dm3, np.broadcast_to(want3, dm3.shape), rtol=1e-14)


def test_dmin_threepoint_families():
    k = 1.1
    # (1) flat regulator, Z_A = 1: D = max(s, k^2) -> dmin = 1 as soon as one argument lies below k^2
    nt = inputs.config3(n_p=2, n_alpha=1, n_q=4, n_c1=4, n_c2=3, n_phi=3, k=k)["ZA"].size
    a = threepoint_args(np.ones(35), reg_kind=LITIM, ZA=np.ones(nt))
    out, dmin, sens = call_three(a)
    np.testing.assert_allclose(dmin, 1.0, rtol=1e-15)
    # (2) exponential regulator, Z_A = 1: D(s) = s + k^2 exp(-s/k^2) is increasing in s, so dmin = D(min over nodes of
    #     {q^2, s_a, s_b}); s_a and s_b restated with Cartesian 4-vectors
    a = threepoint_args(np.ones(35), ZA=np.ones(nt), ext=((3.0, 4.0, 0.7), (5.0, 2.5, 2.1)))
    out, dmin, sens = call_three(a)
    for e, (p1, p2, al) in enumerate(a["ext"]):
        P1 = np.array([p1, 0.0, 0.0, 0.0])
        P2 = p2 * np.array([math.cos(al), math.sin(al), 0.0, 0.0])
        smin = np.inf
        for q in a["xq"]:
            for c1 in a["x1"]:
                for c2 in a["x2"]:
                    s1 = math.sqrt(1 - c1 * c1)
                    Q = q * np.array([c1, s1 * c2, s1 * math.sqrt(1 - c2 * c2), 0.0])
                    smin = min(smin, q * q, float((Q + P1) @ (Q + P1)), float((Q - P2) @ (Q - P2)))
        want = (smin + k * k * math.exp(-smin / (k * k))) / (k * k)
        np.testing.assert_allclose(dmin[e], want, rtol=1e-13)
    # (3) dropping one propagator from the minimum would be seen: p1 huge makes s_a large, p2 = the first radial node (nearly parallel) makes s_b the smallest
    a = threepoint_args(np.ones(35), ZA=np.ones(nt), ext=((50.0, a["xq"][0] / k, 1e-3),))
    out, dmin, sens = call_three(a)
    D = lambda s: (s + k * k * math.exp(-s / (k * k))) / (k * k)
    assert dmin[0] < D(a["xq"][0] ** 2) * (1 - 1e-3)            # below what q^2 and s_a alone would give: s_b sets it
    # 3-D-table twin shares the propagators: same dmin on the same inputs
    c6 = inputs.config6(n_p=2, n_alpha=1, n_q=4, n_c1=4, n_c2=3, n3=(12, 4, 3), k=k)
    a = threepoint_args(np.ones(35), ZA=np.ones(nt), ext=((3.0, 4.0, 0.7), (5.0, 2.5, 2.1)))
    _, dmin_1d, _ = call_three(a)
    _, dmin_3d, _ = oracle.loop4d_threepoint_tab3d(a["prefactor"], a["reg_kind"], a["reg_order"], a["k"], a["xq"], a["wq"],
                                                   a["x1"], a["w1"], a["x2"], a["w2"], a["wphi"], a["ZA"], a["lnq_lo"],
                                                   a["lnq_hi"], a["interp"], c6["v3"], c6["lo3"], c6["hi3"], c6["log3"],
                                                   np.ones(35), a["ext"], want_sens=True)
    np.testing.assert_array_equal(dmin_1d, dmin_3d)
