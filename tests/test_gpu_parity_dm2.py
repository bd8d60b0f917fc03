"""GPU parity of the mass-derivative outputs (Jacobian support; include/dfrg.h "Mass derivatives") against the
oracle's *_dm2 functions, element by element on the same nodes.  Same bars as the values:
regular outputs (oracle dmin >= 1e-6, no cancellation) <= 1e-12 relative, every output |diff| <= 1e-14 sens."""
import os

import numpy as np
import pytest

from paper_2412_13043_b200 import binding as B
from paper_2412_13043_b200 import inputs

from helpers import assert_parity, gpu_run, make_rules, oracle_run, oracle_run_dm2

pytestmark = pytest.mark.gpu


def nodes(n, a, b):
    from paper_2412_13043_b200 import binding as B
    return B.dfrg_quad_nodes(n, a, b)


def check(c, keys, sel=None, what=""):
    """values unchanged by asking for derivatives (bitwise); derivatives against the oracle"""
    R = make_rules(c, nodes)
    g = gpu_run(c, R, want_d=True)
    g0 = gpu_run(c, R)
    assert np.array_equal(g["out"], g0["out"], equal_nan=True) and np.array_equal(g["dmin"], g0["dmin"], equal_nan=True)
    o = oracle_run(c, R, sel=sel)
    od = oracle_run_dm2(c, R, sel=sel)
    reps = {}
    for key in keys:
        val, sens = od[key]
        got = g[key] if sel is None else g[key].ravel()[sel]
        dmin = o["dmin"] if key != "dchan" else np.stack([o["dmin"]] * 2)
        reps[key] = assert_parity(got, val, dmin, sens, what + ":" + key)
        assert reps[key]["n_regular"] > 0 or reps[key]["n"] <= 2
    return g, reps


@pytest.mark.parametrize("T,n_field,n_q", [(0.0, 1, 5), (0.0, 1000, 64), (0.2, 777, 33), (0.05, 130, 64)])
def test_lpa_dchan(T, n_field, n_q):
    c = inputs.config0(n_field=n_field, n_q=n_q) if T == 0.0 else inputs.config1(T, n_field=n_field, n_q=n_q)
    check(c, ["dchan"], what="lpa_dm2_T%g" % T)


def test_lpa_dchan_litim_closed_form():
    for d in (3, 4):
        c = inputs.config0(n_field=513, litim=True, d=d)
        g = gpu_run(c, make_rules(c, nodes), want_d=True)
        m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
        E2 = 1.0 + m2
        ok = np.abs(E2) > 1e-3
        ref = -c["prefactor"] * 2.0 / (d * E2 ** 2)
        assert np.max(np.abs(g["dchan"][ok] / ref[ok] - 1)) < 1e-10


@pytest.mark.parametrize("n_field,n_ext,n_q,n_c,interp", [(1, 1, 3, 2, 3), (130, 3, 33, 9, 3), (300, 2, 40, 7, 1)])
def test_twopoint_dout_small(n_field, n_ext, n_q, n_c, interp):
    c = inputs.config2(n_field=n_field, n_ext=n_ext, n_q=n_q, n_c=n_c, interp=interp)
    check(c, ["dout"], what="twopoint_dm2_%d_%d" % (n_field, n_ext))


def test_twopoint_dout_full_config2():
    g, reps = check(inputs.config2(), ["dout"], what="cfg2_dm2_full")
    assert reps["dout"]["n"] == 16384


@pytest.mark.parametrize("n_field,n_p,n_jext,n_q,n_c,n_max,interp", [(1, 1, 1, 3, 2, 0, 3), (100, 3, 3, 24, 8, 3, 3),
                                                                      (300, 2, 2, 17, 5, 2, 3), (600, 1, 2, 12, 6, 1, 1),
                                                                      (1100, 3, 2, 13, 5, 11, 3), (257, 5, 2, 150, 4, 2, 1)])
def test_matsubara_derivatives_small(n_field, n_p, n_jext, n_q, n_c, n_max, interp):
    # shapes of both paths: moment kernel (compiled (n_max, n_jext) pairs) and the generic kernel
    c = inputs.config4(n_field=n_field, n_p=n_p, n_jext=n_jext, n_q=n_q, n_c=n_c, interp=interp)
    c["n_max"] = n_max
    what = "mats_dm2_%d_%d_%d_%d_%d_%d" % (n_field, n_p, n_jext, n_q, n_c, n_max)
    g, _ = check(c, ["dpsi", "dphi"], what=what)
    c["path"] = B.M3_ROW_STREAMING
    g2, _ = check(c, ["dpsi", "dphi"], what=what + "_generic")
    c["path"] = 0


def test_matsubara_derivatives_full_config4_sampled():
    c = inputs.config4()
    sel = np.arange(0, 64 * 16 * 512, 521)               # 1007 outputs over all (p, j, f) residues
    g, reps = check(c, ["dpsi", "dphi"], sel=sel, what="cfg4_dm2_sampled")
    assert g["dpsi"].shape == (64, 16, 512)


def test_host_entry_points_return_the_same_derivatives():
    for c, keys in ((inputs.config1(0.2, n_field=100), ["dchan"]),
                    (inputs.config2(n_field=140, n_ext=3, n_q=24, n_c=8), ["dout"]),
                    (inputs.config4(n_field=70, n_p=2, n_jext=2, n_q=12, n_c=6), ["dpsi", "dphi"])):
        R = make_rules(c, nodes)
        d = gpu_run(c, R, want_d=True)
        h = gpu_run(c, R, host=True, want_d=True)
        for key in keys + ["out"]:
            assert np.array_equal(d[key], h[key], equal_nan=True), (c["name"], key)


def test_threepoint_rejects_a_derivative_pointer():
    import torch
    from paper_2412_13043_b200 import binding as B
    c = inputs.config3(n_p=1, n_alpha=1, n_q=4, n_c1=3, n_c2=2)
    R = make_rules(c, nodes)
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a)).cuda()
    rr = {k_: (up(v[0]), up(v[1])) for k_, v in R.items()}
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    with pytest.raises(B.DfrgError):
        B.dfrg_integrate_loop4d(B.LOOP_THREEPOINT, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rr["q"],
                                rr["c1"], rr["c2"], rr["phi"], (up(c["ZA"]), up(c["Zc"]), up(c["L3"])), c["lnq_lo"],
                                c["lnq_hi"], c["interp"], up(c["coef"]), None, up(c["ext"]), out, dout_dm2=out)
