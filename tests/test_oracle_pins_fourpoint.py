"""Pins for the four-point box family of the CPU oracle (orc_loop4d_fourpoint, DESIGN.md
reading A21) against things other than itself:
  * a Cartesian restatement: the same quadrature sum with every momentum built as a 4-vector in Cartesian components
    and every invariant taken as a numpy dot product (the oracle uses the angle-expanded formulas), tables linear in
    ln q (interpolation exact), both regulators -- fixes u1, u2, u3, s_a, s_b, s_d, s12, s123, the four vertex
    arguments, the monomial order of both polynomials and the ghost term;
  * the measure and the prefactor against a Cartesian-volume quadrature of the CONTINUUM integral d^4q/(2 pi)^4;
  * quadrature-order convergence; phi really matters (a phi-independent shortcut would fail); sel.
CPU only."""
import math

import numpy as np
import pytest

import oracle
from paper_2412_13043_b200 import inputs

PI = math.pi


def vec(p, *angles):
    """4-vector of length p: (cos a, sin a cos b, sin a sin b cos c, sin a sin b sin c)."""
    a, b, c = (list(angles) + [0.0, 0.0, 0.0])[:3]
    return p * np.array([math.cos(a), math.sin(a) * math.cos(b), math.sin(a) * math.sin(b) * math.cos(c),
                         math.sin(a) * math.sin(b) * math.sin(c)])


def monomials4(deg=3):
    return [(a, b, c, d) for a in range(deg + 1) for b in range(deg + 1 - a) for c in range(deg + 1 - a - b)
            for d in range(deg + 1 - a - b - c)]


def reg_np(kind, k, s, zk=1.0):
    if kind == oracle.REG_LITIM:
        return zk * np.where(s < k * k, k * k - s, 0.0)
    return zk * k * k * np.exp(-s / (k * k))


def regdot_np(kind, k, s, zk=1.0, eta=0.0):
    if kind == oracle.REG_LITIM:
        return zk * (np.where(s < k * k, 2 * k * k, 0.0) - eta * np.where(s < k * k, k * k - s, 0.0))
    return zk * (2 * k * k * np.exp(-s / (k * k)) * (1 + s / (k * k)) - eta * k * k * np.exp(-s / (k * k)))


def cartesian_sum(kind, k, rules, lin_tabs, lo, hi, n_tab, coef, ext, prefactor, zk=1.0, eta=0.0):
    """The quadrature sum of reading A21 with Cartesian 4-vectors.  lin_tabs = ((a, b) for Z_A, Z_c, lambda3): tables
    that are linear in the grid coordinate t, v(t) = a + b t, so that any interpolation mode reproduces them exactly."""
    (xq, wq), (x1, w1), (x2, w2), (xp, wp) = rules
    h = (hi - lo) / (n_tab - 1)

    def tab(ab, s):
        t = np.clip((0.5 * np.log(s) - lo) / h, 0.0, n_tab - 1.0)
        return ab[0] + ab[1] * t
    p1, p2, p3, al, be, ga = ext
    P1, P2, P3 = vec(p1), vec(p2, al), vec(p3, be, ga)
    Q, C1, C2, PH = np.meshgrid(xq, x1, x2, xp, indexing="ij")
    S1, S2 = np.sqrt(1 - C1 ** 2), np.sqrt(1 - C2 ** 2)
    qv = np.stack([Q * C1, Q * S1 * C2, Q * S1 * S2 * np.cos(PH), Q * S1 * S2 * np.sin(PH)], axis=-1)
    W = (wq * xq ** 3)[:, None, None, None] * (w1 * np.sqrt(1 - x1 ** 2))[None, :, None, None] * \
        w2[None, None, :, None] * wp[None, None, None, :]
    n2 = lambda v: np.sum(v * v, axis=-1)
    sq, sa, sb, sd = n2(qv), n2(qv + P1), n2(qv + P1 + P2), n2(qv + P1 + P2 + P3)
    u = [qv @ P1, qv @ P2, qv @ P3]
    p4sq = float(n2(P1 + P2 + P3))
    GA = lambda s: 1.0 / (tab(lin_tabs[0], s) * s + reg_np(kind, k, s, zk))
    Gc = lambda s: 1.0 / (tab(lin_tabs[1], s) * s + reg_np(kind, k, s, zk))
    L = lambda s: tab(lin_tabs[2], s)
    lam = L((sq + p1 * p1 + sa) / 3) * L((sa + p2 * p2 + sb) / 3) * L((sb + p3 * p3 + sd) / 3) * L((sd + p4sq + sq) / 3)
    PA = np.zeros_like(Q)
    Pc = np.zeros_like(Q)
    for idx, (a, b, c, d) in enumerate(monomials4()):
        mono = (sq / k ** 2) ** a * (u[0] / k ** 2) ** b * (u[1] / k ** 2) ** c * (u[2] / k ** 2) ** d
        PA += coef[idx] * mono
        Pc += coef[35 + idx] * mono
    F = GA(sq) * GA(sa) * GA(sb) * GA(sd) * lam * PA + Gc(sq) * Gc(sa) * Gc(sb) * Gc(sd) * Pc
    return prefactor * np.sum(W * regdot_np(kind, k, sq, zk, eta) * F)


def small_rules(nq=7, n1=6, n2=5, nphi=6, qmax=4.0):
    return (oracle.gl_rule(nq, 0, qmax), oracle.gl_rule(n1, -1, 1), oracle.gl_rule(n2, -1, 1),
            oracle.gl_rule(nphi, 0, 2 * PI))


def run(c, rules, ext, coef, tabs, kind=oracle.REG_EXP_POLY, interp=3, **kw):
    (xq, wq), (x1, w1), (x2, w2), (xp, wp) = rules
    return oracle.loop4d_fourpoint(c["prefactor"], kind, 1, c["k"], xq, wq, x1, w1, x2, w2, xp, wp, *tabs,
                                   c["lnq_lo"], c["lnq_hi"], interp, coef, np.atleast_2d(ext), **kw)


@pytest.mark.parametrize("kind", [oracle.REG_EXP_POLY, oracle.REG_LITIM])
@pytest.mark.parametrize("interp", [1, 3])
def test_fourpoint_vs_cartesian_restatement(kind, interp):
    c = inputs.config5(n_s=1, n_ang=1)
    n_tab = c["ZA"].size
    t = np.arange(n_tab, dtype=np.float64)
    lin = ((1.2, 0.004), (0.8, -0.002), (0.9, 0.003))
    tabs = [a + b * t for a, b in lin]
    rng = np.random.default_rng(5)
    rules = small_rules()
    for ext in ([0.7, 1.1, 0.4, 0.9, 2.1, 0.6], [3.0, 0.2, 1.5, 2.8, 0.3, 4.0], [1e-3, 2.0, 2.0, 1.0, 1.0, 1.0]):
        coef = rng.uniform(-1, 1, 70)
        out, dmin, sens = run(c, rules, ext, coef, tabs, kind=kind, interp=interp, want_sens=True, zk=1.2, eta=0.1)
        ref = cartesian_sum(kind, c["k"], rules, lin, c["lnq_lo"], c["lnq_hi"], n_tab, coef, ext, c["prefactor"],
                            zk=1.2, eta=0.1)
        assert abs(out[0] - ref) <= 1e-13 * sens[0], (ext, out[0], ref)
        assert sens[0] >= abs(out[0])


def test_fourpoint_unit_monomials_and_linearity():
    """Each of the 70 coefficients on its own against the Cartesian sum (index order of both polynomials)."""
    c = inputs.config5(n_s=1, n_ang=1)
    n_tab = c["ZA"].size
    lin = ((1.0, 0.0), (1.3, 0.0), (1.0, 0.0))
    tabs = [np.full(n_tab, a) for a, _ in lin]
    rules = small_rules(5, 4, 4, 5, 2.0)
    ext = [0.6, 0.9, 0.5, 1.0, 0.8, 2.0]
    total = 0.0
    kap = np.linspace(-1, 1, 70)
    for i in range(70):
        e = np.zeros(70)
        e[i] = 1.0
        out = run(c, rules, ext, e, tabs)[0][0]
        ref = cartesian_sum(oracle.REG_EXP_POLY, c["k"], rules, lin, c["lnq_lo"], c["lnq_hi"], n_tab, e, ext,
                            c["prefactor"])
        assert abs(out - ref) <= 1e-12 * abs(ref) + 1e-300, i
        total += kap[i] * out
    full = run(c, rules, ext, kap, tabs)[0][0]
    assert abs(full - total) <= 1e-12 * np.sum(np.abs(kap)) * abs(full)


def test_fourpoint_measure_against_cartesian_volume_quadrature():
    """C sum_q w q^3 ... sqrt(1-c1^2) dc1 dc2 dphi against int d^4q/(2 pi)^4 on a Cartesian tensor grid (Gauss-Legendre
    in every Cartesian component; the integrand is smooth and decays like e^{-q^2}).  Constant tables: no interpolation."""
    c = inputs.config5(n_s=1, n_ang=1)
    n_tab = c["ZA"].size
    k = c["k"]
    zA, zc, l3 = 1.1, 0.9, 1.2
    tabs = [np.full(n_tab, v) for v in (zA, zc, l3)]
    rng = np.random.default_rng(3)
    coef = rng.uniform(-1, 1, 70)
    ext = [0.8, 0.5, 0.6, 1.1, 0.7, 1.9]
    # sqrt(1-c1^2) at the end points of the c1 rule converges algebraically (~n1^-3): a long c1 rule for this check
    rules = (oracle.gl_rule(64, 0, 7.0), oracle.gl_rule(160, -1, 1), oracle.gl_rule(24, -1, 1),
             oracle.gl_rule(24, 0, 2 * PI))
    out = run(c, rules, ext, coef, tabs)[0][0]
    # continuum, Cartesian: 48^4 nodes on [-5.5, 5.5]^4 (the insertion decays like e^{-q^2}), one slab at a time
    n = 48
    x, w = oracle.gl_rule(n, -5.5, 5.5)
    P1, P2, P3 = vec(ext[0]), vec(ext[1], ext[3]), vec(ext[2], ext[4], ext[5])
    Y = np.stack(np.meshgrid(x, x, x, indexing="ij"), axis=-1).reshape(-1, 3)
    Wy = np.prod(np.stack(np.meshgrid(w, w, w, indexing="ij"), axis=-1).reshape(-1, 3), axis=1)
    n2 = lambda v: np.sum(v * v, axis=-1)
    R = lambda s: k * k * np.exp(-s / (k * k))
    GA = lambda s: 1.0 / (zA * s + R(s))
    Gc = lambda s: 1.0 / (zc * s + R(s))
    ref = 0.0
    for i in range(n):
        X = np.concatenate([np.full((Y.shape[0], 1), x[i]), Y], axis=1)
        sq, sa, sb, sd = n2(X), n2(X + P1), n2(X + P1 + P2), n2(X + P1 + P2 + P3)
        u = [X @ P1, X @ P2, X @ P3]
        PA = np.zeros_like(sq)
        Pc = np.zeros_like(sq)
        for idx, (a, b, cc, d) in enumerate(monomials4()):
            mono = (sq / k ** 2) ** a * (u[0] / k ** 2) ** b * (u[1] / k ** 2) ** cc * (u[2] / k ** 2) ** d
            PA += coef[idx] * mono
            Pc += coef[35 + idx] * mono
        F = GA(sq) * GA(sa) * GA(sb) * GA(sd) * l3 ** 4 * PA + Gc(sq) * Gc(sa) * Gc(sb) * Gc(sd) * Pc
        Rd = 2 * k * k * np.exp(-sq / (k * k)) * (1 + sq / (k * k))
        ref += w[i] * np.sum(Wy * Rd * F)
    ref /= (2 * PI) ** 4
    assert abs(c["prefactor"] - 1 / (2 * PI) ** 4) < 1e-18
    assert abs(out / ref - 1) < 2e-6, (out, ref)


def test_fourpoint_convergence_phi_dependence_and_sel():
    c = inputs.config5(n_s=2, n_ang=2, n_tab=128)
    tabs = (c["ZA"], c["Zc"], c["L3"])
    ext = c["ext"]
    lo_rules = small_rules(12, 8, 6, 6, 8.0)
    hi_rules = small_rules(48, 20, 14, 14, 8.0)
    vh_rules = small_rules(64, 28, 18, 18, 8.0)
    o_lo, o_hi, o_vh = (run(c, r, ext, c["coef"], tabs)[0] for r in (lo_rules, hi_rules, vh_rules))
    err_lo, err_hi = np.abs(o_lo / o_vh - 1), np.abs(o_hi / o_vh - 1)
    assert np.all(err_hi < 2e-3) and np.median(err_hi) < np.median(err_lo)
    # phi matters: a single phi node (the phi-independent shortcut) is far off for an ext with gamma-dependence
    one_phi = (hi_rules[0], hi_rules[1], hi_rules[2], (np.array([PI]), np.array([2 * PI])))
    o_1 = run(c, one_phi, ext, c["coef"], tabs)[0]
    assert np.max(np.abs(o_1 / o_hi - 1)) > 1e-3
    # gamma -> -gamma mirrors the third axis = the shift phi -> phi + pi of the loop angle: the continuum integral is
    # invariant, the 14-node phi rule up to its (tiny) quadrature error
    ext_m = ext.copy()
    ext_m[:, 5] *= -1
    o_m, _, sens = run(c, hi_rules, ext_m, c["coef"], tabs, want_sens=True)
    assert np.all(np.abs(o_m - o_hi) <= 1e-9 * sens)        # some outputs cancel by many digits: sens is the yardstick
    assert np.any(o_m != o_hi)
    # sel
    sel = np.array([3, 0])
    o_s, d_s = run(c, lo_rules, ext, c["coef"], tabs, sel=sel)
    np.testing.assert_array_equal(o_s, o_lo[sel])
