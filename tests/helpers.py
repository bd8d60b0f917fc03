"""Shared test plumbing: run one workload dict (paper_2412_13043_b200.inputs) through the CPU oracle
or through the CUDA library, and the parity criterion of DESIGN.md ("Parity bar")."""
import numpy as np

import oracle  # noqa: F401
from oracle.harness import (COND_MAX, REGULAR_DMIN, RTOL, SENS_EPS, _dress, kind_of, oracle_run,  # noqa: F401
                            oracle_run_dm2, parity_report)
from paper_2412_13043_b200 import inputs  # noqa: F401
from paper_2412_13043_b200.inputs import make_rules  # noqa: F401


CANARY = -7.25e77       # sentinel around every output buffer of gpu_run(..., canary=True)
CANARY_PAD = 64


def gpu_run(c, R, host=False, want_dmin=True, want_d=False, canary=False):
    """Runs the workload through the C ABI (device entry point on torch CUDA tensors, or the *_host entry
    point on numpy arrays).  -> dict(out=, dmin=, [chan=], [dchan= | dout= | dpsi=, dphi=]) of numpy arrays.
    canary=True (device entry points): every output lives inside a larger buffer whose margins hold a sentinel; the
    margins are checked after the call (an out-of-bounds write of the library fails the test)."""
    import torch
    from paper_2412_13043_b200 import binding as B
    guards = []

    if host:
        up = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        new = lambda *shape: np.full(shape, np.nan)
        down = lambda a: a
    else:
        up = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()
        down = lambda a: a.cpu().numpy()

        def new(*shape):
            if not canary:
                return torch.full(shape, float("nan"), dtype=torch.float64, device="cuda")
            n = int(np.prod(shape))
            big = torch.full((n + 2 * CANARY_PAD,), CANARY, dtype=torch.float64, device="cuda")
            big[CANARY_PAD:CANARY_PAD + n] = float("nan")
            guards.append((big, n))
            return big[CANARY_PAD:CANARY_PAD + n].view(*shape)
    rule = lambda key: (up(R[key][0]), up(R[key][1]))
    kd = kind_of(c)
    res = {}
    dress = dict(reg_zk=c.get("reg_zk", 1.0), reg_eta=c.get("reg_eta", 0.0))
    if kd == "lpa":
        nf = c["rho"].size
        flow, chan, dmin = new(nf), new(2, nf), new(nf) if want_dmin else None
        dchan = new(2, nf) if want_d else None
        fn = B.dfrg_integrate_lpa_host if host else B.dfrg_integrate_lpa
        fn(c["d"], c["T"], c["n_max"], c["reg_arg4d"], c["N"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
           rule("q"), up(c["rho"]), up(c["u"]), up(c["du"]), flow, chan, dmin, dchan=dchan,
           statistics=c.get("statistics", 0), mu=c.get("mu", 0.0) if c.get("statistics", 0) == 1 else 0.0,
           fermion_reg=c.get("fermion_reg", 0), **dress)
        res = dict(out=flow, chan=chan, dmin=dmin, dchan=dchan)
    elif kd == "twopoint":
        out = new(c["pext"].size, c["m2"].size)
        dmin = new(c["pext"].size, c["m2"].size) if want_dmin else None
        dout = new(c["pext"].size, c["m2"].size) if want_d else None
        fn = B.dfrg_integrate_loop4d_host if host else B.dfrg_integrate_loop4d
        fn(B.LOOP_TWOPOINT, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rule("q"), rule("c"), None, None,
           (up(c["Z"]),), c["lnq_lo"], c["lnq_hi"], c["interp"], up(c["coef"]), up(c["m2"]), up(c["pext"]), out, dmin,
           dout_dm2=dout, **dress)
        res = dict(out=out, dmin=dmin, dout=dout)
    elif kd == "threepoint3d":
        ne = c["ext"].shape[0]
        out, dmin = new(ne), new(ne) if want_dmin else None
        fn = B.dfrg_integrate_loop4d_host if host else B.dfrg_integrate_loop4d
        fn(B.LOOP_THREEPOINT_TAB3D, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rule("q"), rule("c1"),
           rule("c2"), rule("phi"), (up(c["ZA"]),), c["lnq_lo"], c["lnq_hi"], c["interp"], up(c["coef"]), None,
           up(c["ext"]), out, dmin, tab3d=(up(c["v3"]), c["lo3"], c["hi3"], c["log3"]),
           ext_outer=c.get("ext_outer", 0), **dress)
        res = dict(out=out, dmin=dmin)
    elif kd == "fourpoint":
        ne = c["ext"].shape[0]
        out, dmin = new(ne), new(ne) if want_dmin else None
        fn = B.dfrg_integrate_loop4d_host if host else B.dfrg_integrate_loop4d
        fn(B.LOOP_FOURPOINT, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rule("q"), rule("c1"),
           rule("c2"), rule("phi"), (up(c["ZA"]), up(c["Zc"]), up(c["L3"])), c["lnq_lo"], c["lnq_hi"], c["interp"],
           up(c["coef"]), None, up(c["ext"]), out, dmin, **dress)
        res = dict(out=out, dmin=dmin)
    elif kd == "threepoint":
        ne = c["ext"].shape[0]
        out, dmin = new(ne), new(ne) if want_dmin else None
        fn = B.dfrg_integrate_loop4d_host if host else B.dfrg_integrate_loop4d
        fn(B.LOOP_THREEPOINT, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rule("q"), rule("c1"),
           rule("c2"), rule("phi"), (up(c["ZA"]), up(c["Zc"]), up(c["L3"])), c["lnq_lo"], c["lnq_hi"], c["interp"],
           up(c["coef"]), None, up(c["ext"]), out, dmin, ext_outer=c.get("ext_outer", 0), **dress)
        res = dict(out=out, dmin=dmin)
    else:
        shape = (c["pext"].size, c["n_jext"], c["m2psi"].size)
        out, dmin = new(*shape), new(*shape) if want_dmin else None
        dpsi, dphi = (new(*shape), new(*shape)) if want_d else (None, None)
        spatial = c.get("reg_arg4d", 1) == 0
        out_im = new(*shape) if spatial else None
        fn = B.dfrg_integrate_matsubara3d_host if host else B.dfrg_integrate_matsubara3d
        fn(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rule("q"), rule("c"),
           up(c["Zpsi"]), up(c["Zphi"]), c["lnq_lo"], c["lnq_hi"], c["interp"], up(c["coef"]), up(c["m2psi"]),
           up(c["m2phi"]), up(c["pext"]), c["n_jext"], out, dmin, dout_dm2_psi=dpsi, dout_dm2_phi=dphi,
           reg_arg4d=c.get("reg_arg4d", 1), mu=c.get("mu", 0.0) if spatial else 0.0, out_im=out_im,
           path=c.get("path", 0), fermion_reg=c.get("fermion_reg", 0), **dress)
        res = dict(out=out, dmin=dmin, dpsi=dpsi, dphi=dphi, out_im=out_im)
    if not host:
        torch.cuda.synchronize()
    for big, n in guards:
        edge = torch.cat([big[:CANARY_PAD], big[CANARY_PAD + n:]]).cpu().numpy()
        assert np.all(edge == CANARY), "the library wrote outside an output buffer (%s)" % c["name"]
    return {k_: (None if v is None else down(v)) for k_, v in res.items() if v is not None or k_ == "dmin"}


def assert_parity(gpu, orc, dmin_orc, sens, what=""):
    rep = parity_report(gpu, orc, dmin_orc, sens)
    msg = {k_: v for k_, v in rep.items() if not k_.startswith("_")}
    assert rep["n_nonfinite_gpu_only"] == 0, (what, msg)
    assert rep["max_rel_regular"] <= RTOL, (what, msg)
    assert rep["max_sens_ratio_regular"] <= SENS_EPS, (what, msg)
    assert rep["max_sens_ratio_singular"] <= SENS_EPS, (what, msg)
    return msg


def assert_dmin(gpu_dmin, orc_dmin, scale=1.0):
    """dmin is a min over the same node set on both sides; the sides differ by the rounding of D0 only."""
    g, o = np.asarray(gpu_dmin).ravel(), np.asarray(orc_dmin).ravel()
    assert np.all(np.abs(g - o) <= 1e-12 * (scale + np.abs(o))), float(np.max(np.abs(g - o)))
