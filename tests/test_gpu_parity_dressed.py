"""GPU parity for the dressed regulator (reading A20):  R = zk R_shape,
Rdot = zk (Rdot_shape - eta R_shape) in every kernel, against the pinned oracle (tests/test_oracle_pins_dressed.py)
on the same nodes; plus the (1 - eta/(d+2)) closed form straight against the CUDA path."""
import numpy as np
import pytest

from paper_2412_13043_b200 import inputs

from helpers import assert_parity, gpu_run, make_rules, oracle_run, oracle_run_dm2

pytestmark = pytest.mark.gpu

ZK, ETA = 1.3, 0.27


def nodes(n, a, b):
    from paper_2412_13043_b200 import binding as B
    return B.dfrg_quad_nodes(n, a, b)


def dressed(c, zk=ZK, eta=ETA, **over):
    c = dict(c)
    c["reg_zk"], c["reg_eta"] = zk, eta
    c.update(over)
    return c


def both(c, sel=None):
    R = make_rules(c, nodes)
    g = gpu_run(c, R)
    o = oracle_run(c, R, sel=sel)
    gout = g["out"] if sel is None else g["out"].ravel()[sel]
    rep = assert_parity(gout, o["out"], o["dmin"], o["sens"], c["name"] + "_dressed")
    assert rep["n_regular"] > 0
    return g, o, R


@pytest.mark.parametrize("order", [1, 8])
def test_lpa_dressed(order):
    both(dressed(inputs.config0(n_field=333, n_q=40), reg_order=order))
    both(dressed(inputs.config1(0.2, n_field=200, n_q=33), reg_order=order))
    both(dressed(inputs.config1(0.5, n_field=64, litim=True)))


def test_lpa_eta_closed_form_on_gpu():
    for d in (3, 4):
        c = dressed(inputs.config0(n_field=257, litim=True, d=d), zk=1.0, eta=0.4)
        g = gpu_run(c, make_rules(c, nodes))
        m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
        E2 = 1.0 + m2
        ok = np.abs(E2) > 1e-3
        ref = c["prefactor"] * 2.0 / d * (1 - 0.4 / (d + 2)) / E2
        assert np.max(np.abs(g["chan"][ok] / ref[ok] - 1)) < 1e-10


def test_twopoint_dressed_with_derivative():
    c = dressed(inputs.config2(n_field=150, n_ext=5, n_q=37, n_c=8))
    g, o, R = both(c)
    gd = gpu_run(c, R, want_d=True)
    d, s = oracle_run_dm2(c, R)["dout"]
    assert_parity(gd["dout"], d, o["dmin"], s, "twopoint_dressed_dm2")
    both(dressed(inputs.config2(n_field=64, n_ext=3, n_q=24, n_c=6), reg_kind=0))       # Litim


@pytest.mark.parametrize("ext_outer", [0, 1])
def test_threepoint_dressed(ext_outer):
    c = dressed(inputs.config3(n_p=3, n_alpha=2, n_q=16, n_c1=8, n_c2=4))
    if not ext_outer:
        c["ext_outer"] = 0                      # general kernel
    both(c)
    c2 = dressed(inputs.config3(n_p=2, n_alpha=2, n_q=12, n_c1=6, n_c2=4), reg_kind=0)  # Litim
    if not ext_outer:
        c2["ext_outer"] = 0
    both(c2)
    c3 = dressed(inputs.config3(n_p=2, n_alpha=1, n_q=12, n_c1=6, n_c2=4), reg_order=3)
    if not ext_outer:
        c3["ext_outer"] = 0
    both(c3)


@pytest.mark.parametrize("shape", [dict(n_field=260, n_p=2, n_jext=2, n_q=16, n_c=8),      # moment path (11, 2)
                                   dict(n_field=130, n_p=2, n_jext=3, n_q=12, n_c=6)])     # generic path
def test_matsubara_dressed(shape):
    c = dressed(inputs.config4(**shape))
    g, o, R = both(c)
    gd = gpu_run(c, R, want_d=True)
    od = oracle_run_dm2(c, R)
    for key in ("dpsi", "dphi"):
        assert_parity(gd[key], od[key][0], o["dmin"], od[key][1], "mats_dressed_" + key)
