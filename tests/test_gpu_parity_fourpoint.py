"""GPU parity for the four-point box family (DFRG_LOOP_FOURPOINT, reading A21) against
the pinned oracle (tests/test_oracle_pins_fourpoint.py) on the same nodes: small cases that span several work units
and ragged chunks, every regulator path, both interpolation modes, dmin, the host entry point, edge momenta, and the
full-size quadrature (96 x 32 x 16 x 16 nodes per output) on a few outputs."""
import numpy as np
import pytest

from paper_2412_13043_b200 import inputs

from helpers import assert_dmin, assert_parity, gpu_run, make_rules, oracle_run

pytestmark = pytest.mark.gpu


def nodes(n, a, b):
    from paper_2412_13043_b200 import binding as B
    return B.dfrg_quad_nodes(n, a, b)


def both(c, host=False, want_dmin=True):
    R = make_rules(c, nodes)
    g = gpu_run(c, R, host=host, want_dmin=want_dmin)
    o = oracle_run(c, R)
    rep = assert_parity(g["out"], o["out"], o["dmin"], o["sens"], c["name"])
    if want_dmin:
        assert_dmin(g["dmin"], o["dmin"], scale=1.0 + float(np.max(np.abs(o["dmin"]))))
    return g, o, rep


@pytest.mark.parametrize("shape", [dict(n_s=1, n_ang=1, n_q=3, n_c1=2, n_c2=2, n_phi=3),
                                   dict(n_s=3, n_ang=2, n_q=13, n_c1=7, n_c2=5, n_phi=6),      # ragged chunks (512 / 5)
                                   dict(n_s=2, n_ang=3, n_q=24, n_c1=10, n_c2=16, n_phi=9),
                                   dict(n_s=5, n_ang=40, n_q=6, n_c1=4, n_c2=3, n_phi=4)])    # more outputs than SMs
def test_fourpoint_small(shape):
    _, _, rep = both(inputs.config5(**shape))
    assert rep["n_regular"] >= rep["n"] - 2


def test_fourpoint_regulators_interp_and_dressing():
    base = dict(n_s=2, n_ang=2, n_q=12, n_c1=6, n_c2=4, n_phi=5)
    c = inputs.config5(**base)
    c["reg_kind"] = 0                                   # flat regulator
    both(c)
    c = inputs.config5(**base)
    c["reg_order"] = 8                                  # the paper's default shape s_8
    both(c)
    c = inputs.config5(interp=1, **base)
    both(c)
    c = inputs.config5(k=1.7, **base)
    c["reg_zk"], c["reg_eta"] = 1.3, 0.27
    both(c)


def test_fourpoint_without_dmin_and_host_entry_point():
    c = inputs.config5(n_s=2, n_ang=2, n_q=10, n_c1=6, n_c2=4, n_phi=5)
    g0, _, _ = both(c, want_dmin=False)
    g1, _, _ = both(c, want_dmin=True)
    np.testing.assert_array_equal(g0["out"], g1["out"])          # deterministic, dmin does not touch the sums
    g2, _, _ = both(c, host=True)
    np.testing.assert_array_equal(g2["out"], g1["out"])


def test_fourpoint_edge_momenta():
    c = inputs.config5(n_s=1, n_ang=1, n_q=12, n_c1=6, n_c2=4, n_phi=6)
    c["ext"] = np.array([[0.0, 0.0, 0.0, 1.0, 1.0, 1.0],        # all externals vanish: s_a = s_b = s_d = q^2
                         [1e-4, 1e-4, 1e-4, 0.0, 0.0, 0.0],     # collinear
                         [5e2, 5e2, 5e2, 3.0, 2.0, 1.0],        # far above the table: clamp high
                         [1.0, 1.0, 1.0, np.pi, 0.0, 0.0]])     # p2 = -p1, p3 parallel to p1
    both(c)


def test_fourpoint_full_config5():
    """The bench workload in full: 128 outputs x 786 432 distinct nodes (quadrature as BASELINE config 3), ~2 s of oracle."""
    c = inputs.config5()
    _, _, rep = both(c)
    assert rep["n"] == 128 and rep["max_rel_regular"] <= 1e-12
