"""Pins of the mass-derivative oracle functions (oracle.lpa_dm2, loop4d_twopoint_dm2, matsubara3d_dm2):
Jacobian support, the paper's "AD" kernels (eq. 27).

What fixes them, independently of the oracle itself:
  D1  derivative of the Litim threshold closed form (T = 0):   dI/dm2 = -C 2 k^(d+2) / (d (k^2+m^2)^2)
  D2  finite-T spatial Litim: mpmath derivative (in E^2) of the coth + digamma closed form of the truncated sum
  D3  exponential regulator, m2 -> inf:  dI/dm2 m^4 / C -> -int q^(d-1) Rdot dq  (= -3 k^6 for d = 4)
  D4  five-point central finite differences of the *value* functions (which carry their own pins in
      test_oracle_pins.py) in the mass argument: catches a wrong power, sign, factor 2 or a swapped mass.
"""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2412_13043_b200 import inputs

PI = math.pi


def rule(r):
    return oracle.gl_rule(*r)


def fd5(fun, h):
    """five-point central difference of fun(delta) at 0: error O(h^4 f^(5))"""
    return (fun(-2 * h) - 8 * fun(-h) + 8 * fun(h) - fun(2 * h)) / (12 * h)


@pytest.mark.parametrize("d,k", [(4, 1.0), (3, 1.0), (4, 1.7)])
def test_d1_litim_threshold_derivative_closed_form(d, k):
    c = inputs.config0(n_field=257, k=k, litim=True, d=d)
    xq, wq = rule(c["rule_q"])
    dchan, _ = oracle.lpa_dm2(c["d"], 0.0, 0, 1, c["prefactor"], c["reg_kind"], 1, k, xq, wq, c["rho"], c["u"], c["du"])
    m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
    E2 = k * k + m2
    ok = np.abs(E2) > 1e-6
    ref = -c["prefactor"] * 2 * k ** (d + 2) / (d * E2 ** 2)
    np.testing.assert_allclose(dchan[ok], ref[ok], rtol=1e-13)


@pytest.mark.parametrize("T_over_k", inputs.CONFIG1_TEMPERATURES)
def test_d2_finite_T_litim_derivative_of_coth_closed_form(T_over_k):
    k = 1.0
    c = inputs.config1(T_over_k, n_field=65, k=k, litim=True)
    xq, wq = rule(c["rule_q"])
    T, N = c["T"], c["n_max"]
    dchan, _ = oracle.lpa_dm2(3, T, N, 0, c["prefactor"], oracle.REG_LITIM, 1, k, xq, wq, c["rho"], c["u"], c["du"])
    m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
    mp.mp.dps = 40

    def S(E2):                                    # sum_{|n|<=N} 1/(w_n^2 + E^2), closed form (pin P3)
        E = mp.sqrt(E2)
        a = E / (2 * mp.pi * T)
        tail = mp.im(mp.digamma(N + 1 + 1j * a)) / a
        return mp.coth(E / (2 * T)) / (2 * E * T) - 2 / (2 * mp.pi * T) ** 2 * tail

    checked = 0
    for ch in range(2):
        for f in range(0, 65, 5):
            E2 = k * k + m2[ch, f]
            if E2 <= 1e-2:
                continue
            ref = c["prefactor"] * T * (2 * k ** 5 / 3) * mp.diff(S, mp.mpf(E2))
            assert abs(dchan[ch, f] / float(ref) - 1) < 1e-11
            checked += 1
    assert checked > 15


@pytest.mark.parametrize("d,exact", [(4, 3.0), (3, 5 * math.sqrt(PI) / 4)])
def test_d3_exp_regulator_heavy_mass_limit(d, exact):
    k, big = 1.0, 1e12
    xq, wq = oracle.gl_rule(64, 0.0, 8.0 * k)
    dchan, _ = oracle.lpa_dm2(d, 0.0, 0, 1, 1.0, oracle.REG_EXP_POLY, 1, k, xq, wq,
                              np.zeros(1), np.full(1, big), np.zeros(1))
    assert abs(dchan[0, 0] * big * big / (-exact) - 1) < 1e-11


@pytest.mark.parametrize("T_over_k", [0.0, 0.2])
def test_d4_lpa_derivative_vs_finite_difference(T_over_k):
    c = inputs.config0(n_field=40) if T_over_k == 0.0 else inputs.config1(T_over_k, n_field=40)
    xq, wq = rule(c["rule_q"])
    args = (c["d"], c["T"], c["n_max"], c["reg_arg4d"])
    dchan, _ = oracle.lpa_dm2(*args, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], xq, wq,
                              c["rho"], c["u"], c["du"])
    _, _, dmin = oracle.lpa(*args, c["N"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], xq, wq,
                            c["rho"], c["u"], c["du"])
    chan = lambda dl: oracle.lpa(*args, c["N"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], xq, wq,
                                 c["rho"], c["u"] + dl, c["du"])[1]
    fd = fd5(chan, 1e-3)
    reg = dmin > 0.2                               # away from the propagator poles (A4): FD error ~ (h/dmin)^4
    assert reg.sum() > 20
    np.testing.assert_allclose(dchan[:, reg], fd[:, reg], rtol=2e-9)


def test_d4_twopoint_derivative_vs_finite_difference():
    c = inputs.config2(n_field=24, n_ext=5, n_q=24, n_c=8)
    xq, wq = rule(c["rule_q"])
    xc, wc = rule(c["rule_c"])
    base = (c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], xq, wq, xc, wc, c["Z"], c["lnq_lo"], c["lnq_hi"],
            c["interp"], c["coef"])
    dout, sens = oracle.loop4d_twopoint_dm2(*base, c["m2"], c["pext"])
    out, dmin = oracle.loop4d_twopoint(*base, c["m2"], c["pext"])
    fd = fd5(lambda dl: oracle.loop4d_twopoint(*base, c["m2"] + dl, c["pext"])[0], 1e-3)
    reg = dmin > 0.2
    assert reg.sum() > 50 and np.all(sens[reg] >= np.abs(dout[reg]))
    np.testing.assert_allclose(dout[reg], fd[reg], rtol=5e-9)
    # sel picks the same numbers
    sel = np.array([0, 7, 24, 119])
    d2, _ = oracle.loop4d_twopoint_dm2(*base, c["m2"], c["pext"], sel=sel)
    assert np.array_equal(d2, dout.ravel()[sel])


def test_d4_matsubara_derivatives_vs_finite_difference():
    c = inputs.config4(n_field=12, n_p=3, n_jext=3, n_q=16, n_c=6)
    c["n_max"] = 3
    xq, wq = rule(c["rule_q"])
    xc, wc = rule(c["rule_c"])
    base = (c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], xq, wq, xc, wc, c["Zpsi"],
            c["Zphi"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"])
    tail = (c["pext"], c["n_jext"])
    dpsi, dphi, spsi, sphi = oracle.matsubara3d_dm2(*base, c["m2psi"], c["m2phi"], *tail)
    out, dmin = oracle.matsubara3d(*base, c["m2psi"], c["m2phi"], *tail)
    fd_psi = fd5(lambda dl: oracle.matsubara3d(*base, c["m2psi"] + dl, c["m2phi"], *tail)[0], 1e-3)
    fd_phi = fd5(lambda dl: oracle.matsubara3d(*base, c["m2psi"], c["m2phi"] + dl, *tail)[0], 1e-3)
    reg = dmin > 0.2
    assert reg.sum() > 50
    scale = np.maximum(np.abs(dpsi), 1e-3 * spsi)     # zero crossings: compare against the size of the terms
    assert np.max(np.abs(dpsi - fd_psi)[reg] / scale[reg]) < 5e-9
    scale = np.maximum(np.abs(dphi), 1e-3 * sphi)
    assert np.max(np.abs(dphi - fd_phi)[reg] / scale[reg]) < 5e-9
    # the two derivatives are different functions (a swapped mass would be caught above; make sure of it)
    assert np.max(np.abs(dpsi - dphi)[reg] / np.abs(dpsi)[reg]) > 1e-2
    sel = np.array([1, 13, 50, 107])
    a, b, _, _ = oracle.matsubara3d_dm2(*base, c["m2psi"], c["m2phi"], *tail, sel=sel)
    assert np.array_equal(a, dpsi.ravel()[sel]) and np.array_equal(b, dphi.ravel()[sel])
