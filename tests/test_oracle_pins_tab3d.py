"""Pins for the 3-D dressing tables of the CPU oracle and the three-point family that uses one (SURVEY 8(f) item 4,
DESIGN.md reading A23; PAPER.md:1860-1896 LinearInterpolator3D with Log x Log x Lin / Log x Lin x Lin coordinates,
PAPER.md:336 the 96 x 8 x 7 vertex grids in (S0, a, s)) against things other than the oracle:
  * trilinear look-up: scipy.interpolate.RegularGridInterpolator (independent library) in coordinate space, exactness
    on multilinear functions, node values, clamps, both coordinate packs;
  * vertex coordinates (S0^2, a, s): hand values, the unit disc under momentum conservation, permutation behaviour;
  * the family: with a table that does not depend on (a, s) and whose S0 axis is the 1-D lambda3 grid shifted by
    ln(2)/2 it must reproduce the pinned 1-D three-point oracle (linear mode) to rounding; with a table that is linear
    in a or s, a numpy restatement with Cartesian 4-vectors.
CPU only."""
import math

import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

import oracle
from paper_2412_13043_b200 import inputs

PI = math.pi


def grid3(n, lo, hi):
    return [np.linspace(lo[a], hi[a], n[a]) for a in range(3)]


@pytest.mark.parametrize("log3", [(1, 0, 0), (1, 1, 0)])
def test_table3d_vs_scipy_regular_grid_interpolator(log3):
    rng = np.random.default_rng(11)
    n = (9, 5, 4)
    lo = [math.log(1e-2), -1.0, -1.0] if log3 == (1, 0, 0) else [math.log(1e-2), math.log(0.1), -1.0]
    hi = [math.log(1e2), 1.0, 1.0] if log3 == (1, 0, 0) else [math.log(1e2), math.log(50.0), 1.0]
    v = rng.uniform(0.5, 1.5, n)
    rgi = RegularGridInterpolator(grid3(n, lo, hi), v, method="linear")
    for _ in range(300):
        c = [rng.uniform(lo[a], hi[a]) for a in range(3)]
        x = [math.exp(2 * c[a]) if log3[a] else c[a] for a in range(3)]       # log axes take the SQUARED momentum
        got = oracle.table3d_lookup(v, lo, hi, log3, *x)
        assert abs(got - float(rgi(c)[0])) <= 1e-13
    # node values and clamps
    g = grid3(n, lo, hi)
    for idx in ((0, 0, 0), (8, 4, 3), (3, 2, 1)):
        c = [g[a][idx[a]] for a in range(3)]
        x = [math.exp(2 * c[a]) if log3[a] else c[a] for a in range(3)]
        assert abs(oracle.table3d_lookup(v, lo, hi, log3, *x) - v[idx]) <= 1e-13
    far_lo = [1e-30 if log3[a] else -7.0 for a in range(3)]
    far_hi = [1e30 if log3[a] else 7.0 for a in range(3)]
    assert oracle.table3d_lookup(v, lo, hi, log3, *far_lo) == v[0, 0, 0]
    assert oracle.table3d_lookup(v, lo, hi, log3, *far_hi) == v[-1, -1, -1]
    assert oracle.table3d_lookup(v, lo, hi, log3, 0.0, far_hi[1], far_lo[2]) == v[0, -1, 0]   # log(0) = -inf clamps low


def test_table3d_exact_on_multilinear_functions():
    n = (7, 8, 7)
    lo, hi = [-2.0, -1.0, -1.0], [3.0, 1.0, 1.0]
    g = np.meshgrid(*grid3(n, lo, hi), indexing="ij")
    f = lambda c0, c1, c2: 0.3 + 0.2 * c0 - 0.1 * c1 + 0.4 * c2 + 0.05 * c0 * c1 - 0.07 * c1 * c2 + 0.02 * c0 * c1 * c2
    v = f(*g)
    rng = np.random.default_rng(2)
    for _ in range(100):
        c = [rng.uniform(lo[a], hi[a]) for a in range(3)]
        got = oracle.table3d_lookup(v, lo, hi, (1, 0, 0), math.exp(2 * c[0]), c[1], c[2])
        assert abs(got - f(*c)) <= 1e-13


def test_vertex_coords_hand_values_and_unit_disc():
    assert oracle.vertex_coords(1.0, 1.0, 1.0) == (0.5, 0.0, 0.0)                 # symmetric point
    S, a, s = oracle.vertex_coords(1.0, 1.0, 4.0)                                # collinear, k3 = -(k1 + k2)
    assert (S, a, s) == (1.0, 0.0, -1.0)
    S, a, s = oracle.vertex_coords(1.0, 1.0, 0.0)                                # k3 = 0
    assert abs(S - 1 / 3) < 1e-16 and a == 0.0 and abs(s - 1.0) < 1e-15
    S, a, s = oracle.vertex_coords(0.0, 3.0, 3.0)                                # k1 = 0: (a, s) = (sqrt3/2, -1/2)
    assert abs(S - 1.0) < 1e-16 and abs(a - math.sqrt(3) / 2) < 1e-15 and abs(s + 0.5) < 1e-15
    assert oracle.vertex_coords(0.0, 0.0, 0.0) == (0.0, 0.0, 0.0)
    rng = np.random.default_rng(4)
    for _ in range(500):                                                          # momentum conservation => unit disc
        k1, k2 = rng.normal(size=4), rng.normal(size=4)
        k3 = -(k1 + k2)
        S, a, s = oracle.vertex_coords(k1 @ k1, k2 @ k2, k3 @ k3)
        assert a * a + s * s <= 1 + 1e-14 and abs(S - (k1 @ k1 + k2 @ k2 + k3 @ k3) / 6) < 1e-15
        S2, a2, s2 = oracle.vertex_coords(k2 @ k2, k1 @ k1, k3 @ k3)              # k1 <-> k2: a -> -a
        assert abs(a2 + a) < 1e-15 and abs(s2 - s) < 1e-15 and S2 == S


def _rules(c, nq=10, n1=8, n2=6, nphi=4):
    return (oracle.gl_rule(nq, *c["rule_q"][1:]), oracle.gl_rule(n1, -1, 1), oracle.gl_rule(n2, -1, 1),
            oracle.gl_rule(nphi, 0, 2 * PI))


def test_tab3d_family_reduces_to_the_pinned_1d_threepoint_oracle():
    """lambda3(S0, a, s) independent of (a, s), S0 axis = the 1-D grid shifted by ln(2)/2 (the 1-D family looks lambda3 up
    at the mean squared leg momentum = 2 S0^2): must equal the 1-D three-point oracle in linear mode."""
    c = inputs.config3(n_p=3, n_alpha=2)
    (xq, wq), (x1, w1), (x2, w2), (xp, wp) = _rules(c)
    L3 = c["L3"]
    v3 = np.repeat(np.repeat(L3[:, None, None], 3, axis=1), 4, axis=2)
    shift = 0.5 * math.log(2.0)
    lo3, hi3 = [c["lnq_lo"] - shift, -1.0, -1.0], [c["lnq_hi"] - shift, 1.0, 1.0]
    o1, d1, s1 = oracle.loop4d_threepoint(c["prefactor"], c["reg_kind"], 1, c["k"], xq, wq, x1, w1, x2, w2, xp, wp,
                                          c["ZA"], c["Zc"], L3, c["lnq_lo"], c["lnq_hi"], 1, c["coef"], c["ext"],
                                          want_sens=True)
    for za_interp in (1,):
        o3, d3, s3 = oracle.loop4d_threepoint_tab3d(c["prefactor"], c["reg_kind"], 1, c["k"], xq, wq, x1, w1, x2, w2, wp,
                                                    c["ZA"], c["lnq_lo"], c["lnq_hi"], za_interp, v3, lo3, hi3, (1, 0, 0),
                                                    c["coef"], c["ext"], want_sens=True)
        assert np.all(np.abs(o3 - o1) <= 1e-12 * s1)
        np.testing.assert_allclose(d3, d1, rtol=1e-14)
        np.testing.assert_allclose(s3, s1, rtol=1e-10)


@pytest.mark.parametrize("axis", [1, 2])
def test_tab3d_family_angle_dependence_vs_cartesian_restatement(axis):
    """A table that is linear in a (or s) and constant otherwise: lambda3 = 1 + 0.3 a (resp. s), exact under trilinear
    interpolation.  Reference: numpy sum over the same grid, legs from Cartesian 4-vectors."""
    c = inputs.config3(n_p=1, n_alpha=1)
    k = c["k"]
    (xq, wq), (x1, w1), (x2, w2), (xp, wp) = _rules(c, 8, 6, 5, 3)
    n = (4, 8, 7)
    lo3, hi3 = [c["lnq_lo"], -1.0, -1.0], [c["lnq_hi"], 1.0, 1.0]
    g = np.meshgrid(*grid3(n, lo3, hi3), indexing="ij")
    v3 = 1.0 + 0.3 * g[axis]
    ZA = np.full(8, 1.1)
    coef = np.random.default_rng(9).uniform(-1, 1, 35)
    p1, p2, al = 0.8, 1.3, 1.1
    out = oracle.loop4d_threepoint_tab3d(c["prefactor"], oracle.REG_EXP_POLY, 1, k, xq, wq, x1, w1, x2, w2, wp,
                                         ZA, c["lnq_lo"], c["lnq_hi"], 1, v3, lo3, hi3, (1, 0, 0), coef,
                                         np.array([[p1, p2, al]]))[0][0]
    P1 = p1 * np.array([1.0, 0, 0, 0])
    P2 = p2 * np.array([math.cos(al), math.sin(al), 0, 0])
    Q, C1, C2 = np.meshgrid(xq, x1, x2, indexing="ij")
    S1 = np.sqrt(1 - C1 ** 2)
    qv = np.stack([Q * C1, Q * S1 * C2, Q * S1 * np.sqrt(1 - C2 ** 2), 0 * Q], axis=-1)    # phi = 0: the integrand is phi-free
    n2 = lambda v: np.sum(v * v, axis=-1)
    sq, sa, sb, sc = n2(qv), n2(qv + P1), n2(qv - P2), float(n2(P1 + P2))
    R = lambda s: k * k * np.exp(-s / (k * k))
    G = lambda s: 1.0 / (1.1 * s + R(s))

    def lam(k1, k2, k3):
        six = k1 + k2 + k3
        coord = math.sqrt(3) * (k2 - k1) / six if axis == 1 else (k1 + k2 - 2 * k3) / six
        return 1.0 + 0.3 * np.clip(coord, -1, 1)
    Lam = lam(p1 * p1, sq, sa) * lam(p2 * p2, sq, sb) * lam(sc, sa, sb)
    P = np.zeros_like(Q)
    idx = 0
    for a in range(5):
        for b in range(5 - a):
            for cc in range(5 - a - b):
                P += coef[idx] * (sq / k ** 2) ** a * ((qv @ P1) / k ** 2) ** b * ((qv @ P2) / k ** 2) ** cc
                idx += 1
    W = (wq * xq ** 3)[:, None, None] * (w1 * np.sqrt(1 - x1 ** 2))[None, :, None] * w2[None, None, :]
    Rd = 2 * k * k * np.exp(-sq / (k * k)) * (1 + sq / (k * k))
    ref = c["prefactor"] * np.sum(wp) * np.sum(W * Rd * G(sq) * G(sa) * G(sb) * Lam * P)
    assert abs(out / ref - 1) < 1e-12
