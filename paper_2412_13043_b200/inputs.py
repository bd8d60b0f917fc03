"""Seeded synthetic inputs for the five BASELINE.json workloads (numpy only).

This module holds NONE of the method's arithmetic: no quadrature nodes, no regulators,
no interpolation, no integrands.  It only writes down the *inputs* a caller of the
library would supply -- field grids, masses, external-momentum grids, dressing tables,
polynomial coefficients, and the (order, interval) of each quadrature rule -- with the
shapes and value distributions of the paper's workloads (log momentum grids of ~100
points over several decades; radial x 1-3 angle quadrature,
PAPER.md:357, 1030; dressings as log-grid tables and per-Matsubara-index stacks,
PAPER.md:1854-1905).  Both the CUDA tests/bench and the CPU oracle tests draw from it,
so the two sides see bit-identical inputs without sharing any numerical code.

Random numbers: SplitMix64 counter-based stream, U_i = (mix(seed + (i+1)*GOLDEN) >> 11) * 2^-53,
draws consumed in the order stated per config.
"""
import math

import numpy as np

_M64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15

LN_Q_LO = math.log(1e-4)   # dressing grid: q/k in [1e-4, 2e2], reading A9
LN_Q_HI = math.log(2e2)
LAMBDA = 10.0              # u(rho) = LAMBDA (rho - KAPPA k^2)
KAPPA = 0.5

REG_LITIM = 0
REG_EXP_POLY = 1


def splitmix64_uniform(seed, count, offset=0):
    """count doubles in [0,1) from the SplitMix64 stream of `seed`, starting at draw `offset`."""
    out = np.empty(count, dtype=np.float64)
    for i in range(count):
        z = (seed + (offset + i + 1) * _GOLDEN) & _M64
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
        z ^= z >> 31
        out[i] = (z >> 11) * (1.0 / 9007199254740992.0)
    return out


def field_grid(n_field, k=1.0):
    """rho uniform in [0, 2] k^2, endpoints included; u = LAMBDA (rho - KAPPA k^2); u' = LAMBDA."""
    if n_field == 1:
        rho = np.array([0.0])
    else:
        rho = 2.0 * k * k * np.arange(n_field, dtype=np.float64) / (n_field - 1)
    u = LAMBDA * (rho - KAPPA * k * k)
    du = np.full(n_field, LAMBDA)
    return rho, u, du


def logspace(lo, hi, n):
    """n points 10^(a + (b-a) e/(n-1)), endpoints included (reading A3)."""
    a, b = math.log10(lo), math.log10(hi)
    if n == 1:
        return np.array([lo], dtype=np.float64)
    return 10.0 ** (a + (b - a) * np.arange(n, dtype=np.float64) / (n - 1))


def table_grid(n_q, k=1.0):
    """(q_i, lnq_lo, lnq_hi): uniform grid in ln q over [1e-4, 2e2] k."""
    lo, hi = LN_Q_LO + math.log(k), LN_Q_HI + math.log(k)
    lnq = lo + (hi - lo) * np.arange(n_q, dtype=np.float64) / (n_q - 1)
    return np.exp(lnq), lo, hi


def config0(n_field=1024, n_q=64, k=1.0, litim=False, d=4):
    """LPA O(N) flow RHS, T=0, d=4, N=4 (BASELINE.json configs[0])."""
    rho, u, du = field_grid(n_field, k)
    pref = {4: 1.0 / (32.0 * math.pi ** 2), 3: 1.0 / (4.0 * math.pi ** 2)}.get(d, 1.0)
    return dict(name="cfg0_lpa_T0", d=d, T=0.0, n_max=0, reg_arg4d=1, N=4.0,
                prefactor=pref,
                reg_kind=REG_LITIM if litim else REG_EXP_POLY, reg_order=1, k=k,
                rule_q=(n_q, 0.0, (1.0 if litim else 6.0) * k),
                rho=rho, u=u, du=du)


def config1(T_over_k, n_field=4096, n_q=64, k=1.0, litim=False):
    """LPA O(N) flow RHS at finite T, d=3+Matsubara (BASELINE.json configs[1]); one temperature."""
    rho, u, du = field_grid(n_field, k)
    T = T_over_k * k
    n_max = int(math.ceil(6.0 * k / (2.0 * math.pi * T)))
    return dict(name="cfg1_lpa_T%g" % T_over_k, d=3, T=T, n_max=n_max,
                reg_arg4d=0 if litim else 1, N=4.0,
                prefactor=1.0 / (4.0 * math.pi ** 2),
                reg_kind=REG_LITIM if litim else REG_EXP_POLY, reg_order=1, k=k,
                rule_q=(n_q, 0.0, (1.0 if litim else 6.0) * k),
                rho=rho, u=u, du=du)


CONFIG1_TEMPERATURES = (0.05, 0.1, 0.2, 0.5)


def config2(n_field=256, n_ext=64, n_q=128, n_c=32, n_tab=128, k=1.0, seed=2, interp=3):
    """Momentum-dependent two-point loop in 4D at T=0 (BASELINE.json configs[2])."""
    _, u, _ = field_grid(n_field, k)
    qt, lo, hi = table_grid(n_tab, k)
    U = splitmix64_uniform(seed, n_tab)
    Z = 1.0 + 0.3 / (1.0 + (qt / k) ** 2) + 1e-3 * (2.0 * U - 1.0)
    return dict(name="cfg2_twopoint", family=0, prefactor=1.0 / (4.0 * math.pi ** 3),
                reg_kind=REG_EXP_POLY, reg_order=1, k=k,
                rule_q=(n_q, 0.0, 8.0 * k), rule_c=(n_c, -1.0, 1.0),
                Z=Z, lnq_lo=lo, lnq_hi=hi, interp=interp,
                coef=np.array([1.0, 0.1]),
                m2=u, pext=logspace(1e-3 * k, 1e2 * k, n_ext))


def _rational(qt, k, a):
    t = (qt / k) ** 2
    return (a[0] + a[1] * t + a[2] * t * t) / (1.0 + a[3] * t + a[4] * t * t)


def config3(n_p=32, n_alpha=8, n_q=96, n_c1=32, n_c2=16, n_phi=16, n_tab=128, k=1.0, seed=7, interp=3):
    """Three-point vertex loop in 4D at T=0 (BASELINE.json configs[3])."""
    qt, lo, hi = table_grid(n_tab, k)
    U = splitmix64_uniform(seed, 15 + 35)
    ZA = _rational(qt, k, 0.5 + U[0:5])
    Zc = _rational(qt, k, 0.5 + U[5:10])
    L3 = _rational(qt, k, 0.5 + U[10:15])
    coef = 2.0 * U[15:50] - 1.0
    p = logspace(1e-2 * k, 1e2 * k, n_p)
    alpha = math.pi * (np.arange(n_alpha, dtype=np.float64) + 0.5) / n_alpha
    ext = np.empty((n_p, n_p, n_alpha, 3))
    ext[..., 0] = p[:, None, None]
    ext[..., 1] = p[None, :, None]
    ext[..., 2] = alpha[None, None, :]
    return dict(name="cfg3_threepoint", family=1, prefactor=1.0 / (2.0 * math.pi) ** 4,
                reg_kind=REG_EXP_POLY, reg_order=1, k=k,
                rule_q=(n_q, 0.0, 8.0 * k), rule_c1=(n_c1, -1.0, 1.0), rule_c2=(n_c2, -1.0, 1.0),
                rule_phi=(n_phi, 0.0, 2.0 * math.pi),
                ZA=ZA, Zc=Zc, L3=L3, lnq_lo=lo, lnq_hi=hi, interp=interp,
                coef=coef, ext=ext.reshape(-1, 3), ext_outer=n_p)  # product grid: |p1| outermost


def config5(n_s=16, n_ang=8, n_q=96, n_c1=32, n_c2=16, n_phi=16, n_tab=128, k=1.0, seed=11, interp=3):
    """Four-point box loop in 4D at T=0 with genuine three-angle kinematics and a ghost loop (SURVEY 8(f) item 3,
    DESIGN.md reading A21; not a BASELINE.json config).  Quadrature and tables as config 3; externals: n_s scales S
    log-spaced in [1e-2, 1e2] k with (|p1|, |p2|, |p3|) = (S, 0.7 S, 1.3 S), times n_ang seeded angle triples
    (alpha, beta, gamma) in (0.1 pi, 0.9 pi)."""
    qt, lo, hi = table_grid(n_tab, k)
    U = splitmix64_uniform(seed, 15 + 70 + 3 * n_ang)
    ZA = _rational(qt, k, 0.5 + U[0:5])
    Zc = _rational(qt, k, 0.5 + U[5:10])
    L3 = _rational(qt, k, 0.5 + U[10:15])
    coef = 2.0 * U[15:85] - 1.0
    ang = math.pi * (0.1 + 0.8 * U[85:85 + 3 * n_ang].reshape(n_ang, 3))
    S = logspace(1e-2 * k, 1e2 * k, n_s)
    ext = np.empty((n_s, n_ang, 6))
    ext[..., 0] = S[:, None]
    ext[..., 1] = 0.7 * S[:, None]
    ext[..., 2] = 1.3 * S[:, None]
    ext[..., 3:6] = ang[None, :, :]
    return dict(name="cfg5_fourpoint", family=2, prefactor=1.0 / (2.0 * math.pi) ** 4,
                reg_kind=REG_EXP_POLY, reg_order=1, k=k,
                rule_q=(n_q, 0.0, 8.0 * k), rule_c1=(n_c1, -1.0, 1.0), rule_c2=(n_c2, -1.0, 1.0),
                rule_phi=(n_phi, 0.0, 2.0 * math.pi),
                ZA=ZA, Zc=Zc, L3=L3, lnq_lo=lo, lnq_hi=hi, interp=interp,
                coef=coef, ext=ext.reshape(-1, 6))


def config6(n_p=32, n_alpha=8, n_q=96, n_c1=32, n_c2=16, n_phi=16, n_tab=128, n3=(96, 8, 7), k=1.0, seed=13, interp=3):
    """Three-point vertex loop with a 3-D vertex dressing table lambda3(S0, a, s) (DESIGN.md reading
    A23; not a BASELINE.json config).  Externals, quadrature, Z_A and the polynomial as config 3 (own seed); the vertex
    table has the paper's 96 x 8 x 7 shape: S0 log-spaced over the 1-D grid's range, a and s uniform in
    [-1, 1];  lambda3 = X(S0) (1 + c1 a^2 + c2 s + c3 a s) with X the rational function of config 3 and c_i seeded."""
    c = config3(n_p=n_p, n_alpha=n_alpha, n_q=n_q, n_c1=n_c1, n_c2=n_c2, n_phi=n_phi, n_tab=n_tab, k=k, seed=seed,
                interp=interp)
    U = splitmix64_uniform(seed + 1000, 8)
    lo, hi = c["lnq_lo"], c["lnq_hi"]
    S0 = np.exp(np.linspace(lo, hi, n3[0]))
    a = np.linspace(-1.0, 1.0, n3[1])
    s_ = np.linspace(-1.0, 1.0, n3[2])
    X = _rational(S0, k, 0.5 + U[0:5])
    c1, c2, c3 = 0.3 * (U[5] - 0.5), 0.3 * (U[6] - 0.5), 0.3 * (U[7] - 0.5)
    v3 = X[:, None, None] * (1.0 + c1 * a[None, :, None] ** 2 + c2 * s_[None, None, :] + c3 * a[None, :, None] * s_[None, None, :])
    c.update(name="cfg6_threepoint3d", family=3, v3=np.ascontiguousarray(v3), lo3=(lo, -1.0, -1.0), hi3=(hi, 1.0, 1.0),
             log3=(1, 0, 0))   # ext_outer = n_p from config 3: the externals are a product grid
    del c["L3"], c["Zc"]
    return c


def config4(n_field=512, n_p=64, n_jext=16, n_q=96, n_c=24, n_tab=128, n_freq=64,
            T_over_k=0.15, cut=10.0, k=1.0, seed=4, interp=3):
    """Finite-T momentum-dependent loop, quark-meson-like (BASELINE.json configs[4])."""
    rho, u, _ = field_grid(n_field, k)
    T = T_over_k * k
    n_max = int(math.ceil(cut * k / (2.0 * math.pi * T)))
    qt, lo, hi = table_grid(n_tab, k)
    U = splitmix64_uniform(seed, 4 + 20)
    A_psi, B_psi = 0.1 + 0.4 * U[0], 0.5 + 1.5 * U[1]
    A_phi, B_phi = 0.1 + 0.4 * U[2], 0.5 + 1.5 * U[3]
    iota = np.arange(n_freq, dtype=np.float64)
    nu = (2.0 * iota + 1.0) * math.pi * T
    om = 2.0 * iota * math.pi * T
    Zpsi = 1.0 + A_psi / (1.0 + B_psi * (qt[None, :] ** 2 + nu[:, None] ** 2) / (k * k))
    Zphi = 1.0 + A_phi / (1.0 + B_phi * (qt[None, :] ** 2 + om[:, None] ** 2) / (k * k))
    return dict(name="cfg4_matsubara3d", T=T, n_max=n_max, prefactor=1.0 / (4.0 * math.pi ** 2),
                reg_kind=REG_EXP_POLY, reg_order=1, k=k,
                rule_q=(n_q, 0.0, cut * k), rule_c=(n_c, -1.0, 1.0),
                Zpsi=np.ascontiguousarray(Zpsi), Zphi=np.ascontiguousarray(Zphi),
                lnq_lo=lo, lnq_hi=hi, interp=interp,
                coef=2.0 * U[4:24] - 1.0,
                m2psi=rho.copy(), m2phi=u,
                pext=logspace(1e-2 * k, 20.0 * k, n_p), n_jext=n_jext)


def make_rules(c, gen):
    """gen(n, a, b) -> (x, w), the caller's node generator (the library's dfrg_quad_nodes or the oracle's);
    returns {axis: (x, w)} for every rule_* entry of the workload."""
    return {key[5:]: gen(*val) for key, val in c.items() if key.startswith("rule_")}
