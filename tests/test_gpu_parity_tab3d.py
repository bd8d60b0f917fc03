"""GPU parity for the three-point family with a 3-D vertex dressing table (DFRG_LOOP_THREEPOINT_TAB3D; SURVEY 8(f)
item 4, reading A23) against the pinned oracle (tests/test_oracle_pins_tab3d.py) on the same nodes."""
import numpy as np
import pytest

from paper_2412_13043_b200 import inputs

from helpers import assert_dmin, assert_parity, gpu_run, make_rules, oracle_run

pytestmark = pytest.mark.gpu


def nodes(n, a, b):
    from paper_2412_13043_b200 import binding as B
    return B.dfrg_quad_nodes(n, a, b)


def both(c, sel=None, host=False):
    R = make_rules(c, nodes)
    g = gpu_run(c, R, host=host)
    o = oracle_run(c, R, sel=sel)
    gout, gdm = (g["out"], g["dmin"]) if sel is None else (g["out"].ravel()[sel], g["dmin"].ravel()[sel])
    rep = assert_parity(gout, o["out"], o["dmin"], o["sens"], c["name"])
    assert_dmin(gdm, o["dmin"], scale=1.0 + float(np.max(np.abs(o["dmin"]))))
    return g, o, rep


@pytest.mark.parametrize("shape", [dict(n_p=1, n_alpha=1, n_q=3, n_c1=2, n_c2=2, n3=(2, 2, 2)),
                                   dict(n_p=3, n_alpha=2, n_q=16, n_c1=8, n_c2=4, n3=(96, 8, 7)),
                                   dict(n_p=14, n_alpha=12, n_q=7, n_c1=5, n_c2=3, n3=(33, 5, 9)),     # more outputs than SMs
                                   dict(n_p=2, n_alpha=2, n_q=40, n_c1=9, n_c2=6, n3=(128, 12, 8))])   # 12288-entry table
def test_tab3d_small(shape):
    c = inputs.config6(**shape)
    g, _, _ = both(c)                               # product-grid kernels (ext_outer = n_p, checked on the device)
    c["ext_outer"] = 0
    g0, _, _ = both(c)                              # general kernel
    if int(np.prod(shape["n3"])) <= 6000:           # (larger tables do not fit beside the product-grid tables: general kernel)
        assert not np.array_equal(g["out"], g0["out"]) or g["out"].size <= 2
    c["ext_outer"] = shape["n_p"]
    c["ext"] = c["ext"].copy()
    c["ext"][-1, 1] *= 1.5                          # the promise is broken: the device check must send it to the general kernel
    gb, _, _ = both(c)
    c["ext_outer"] = 0
    gb0, _, _ = both(c)
    assert np.array_equal(gb["out"], gb0["out"])


def test_tab3d_regulators_coordinate_packs_host_and_edges():
    base = dict(n_p=2, n_alpha=2, n_q=12, n_c1=6, n_c2=4)
    c = inputs.config6(**base)
    c["reg_kind"] = 0
    both(c)
    c = inputs.config6(k=1.7, interp=1, **base)
    c["reg_order"] = 8
    c["reg_zk"], c["reg_eta"] = 1.3, 0.27
    both(c)
    c = inputs.config6(**base)                      # a linear S0 axis (Lin x Lin x Lin is allowed: is_log per axis)
    c["log3"] = (0, 0, 0)
    c["lo3"], c["hi3"] = (0.0, -1.0, -1.0), (50.0, 1.0, 1.0)
    both(c)
    c = inputs.config6(**base)                      # angle axes narrower than the unit disc: clamps on both sides
    c["lo3"], c["hi3"] = (c["lo3"][0], -0.5, -0.25), (c["hi3"][0], 0.5, 0.75)
    g, _, _ = both(c)
    h, _, _ = both(c, host=True)
    assert np.array_equal(g["out"], h["out"])
    c = inputs.config6(n_p=1, n_alpha=1, n_q=12, n_c1=6, n_c2=4)
    c["ext_outer"] = 0
    c["ext"] = np.array([[0.0, 0.0, 1.0], [1e-5, 1e3, 0.0], [2.0, 2.0, np.pi]])     # S0 -> 0, far off the table, p2 = -p1
    both(c)


def test_tab3d_full_size():
    """The paper-shaped workload in full (cfg3's 8192 external configurations and 96 x 32 x 16 x 16 quadrature, 96 x 8 x 7
    vertex table) on the product-grid kernels, every output against the oracle (~6 s on 16 host cores)."""
    c = inputs.config6()
    g, o, rep = both(c)
    assert g["out"].shape == (8192,) and np.all(np.isfinite(g["out"])) and rep["n_regular"] >= 8190
