"""Shared test plumbing: run one workload dict (paper_2412_13043_b200.inputs) through the CPU oracle
or through the CUDA library, and the parity criterion of DESIGN.md ("Parity bar")."""
import numpy as np

import oracle
from paper_2412_13043_b200 import inputs  # noqa: F401

REGULAR_DMIN = 1e-6      # an output is regular iff the oracle's dmin >= this (reading A4) ...
COND_MAX = 1e4           # ... and its terms do not cancel by more than this: sens / |out| <= COND_MAX
RTOL = 1e-12             # north_star: relative error <= 1e-12 per output on the same nodes (regular outputs)
SENS_EPS = 1e-14         # every output, regular or not: |gpu - oracle| <= SENS_EPS * sens (condition-aware bound)


def kind_of(c):
    n = c["name"]
    return "lpa" if n.startswith(("cfg0", "cfg1")) else n.split("_", 1)[1]


def make_rules(c, gen):
    """gen(n, a, b) -> (x, w); returns {axis: (x, w)} for every rule_* entry of the workload."""
    return {key[5:]: gen(*val) for key, val in c.items() if key.startswith("rule_")}


def _dress(c):
    """Dressed-regulator parameters of a workload (reading A20); absent = plain shapes."""
    return dict(zk=c.get("reg_zk", 1.0), eta=c.get("reg_eta", 0.0))


def oracle_run(c, R, sel=None):
    """-> (out, dmin, sens); lpa: out = flow[n_field], extra channels under key 'chan' are returned via dict."""
    kd = kind_of(c)
    if kd == "lpa" and c.get("statistics", 0) == 1:     # fermionic loop at chemical potential (reading A22)
        m2 = np.stack([c["u"], c["u"] + 2.0 * c["rho"] * c["du"]])
        I, dI, dm, sn, snd = oracle.lpa_fermion(c["d"], c["T"], c["n_max"], c.get("mu", 0.0), c["prefactor"], c["reg_kind"],
                                                c["reg_order"], c["k"], *R["q"], m2.ravel(), **_dress(c))
        I, dm, sn = (a.reshape(2, -1) for a in (I, dm, sn))
        return dict(out=(c["N"] - 1.0) * I[0] + I[1], chan=I, dmin=np.minimum(dm[0], dm[1]),
                    sens=abs(c["N"] - 1.0) * sn[0] + sn[1], sens_chan=sn)
    if kd == "matsubara3d" and c.get("reg_arg4d", 1) == 0:   # spatial regulators / chemical potential (reading A24)
        out, dmin, sens = oracle.matsubara3d_mu(c["T"], c["n_max"], c.get("mu", 0.0), c["prefactor"], c["reg_kind"],
                                                c["reg_order"], c["k"], *R["q"], *R["c"], c["Zpsi"], c["Zphi"],
                                                c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["m2psi"], c["m2phi"],
                                                c["pext"], c["n_jext"], sel=sel, want_sens=True, **_dress(c))
        return dict(out=out, dmin=dmin, sens=sens)
    if kd == "lpa":
        flow, chan, dmin, sens = oracle.lpa(c["d"], c["T"], c["n_max"], c["reg_arg4d"], c["N"], c["prefactor"],
                                            c["reg_kind"], c["reg_order"], c["k"], *R["q"], c["rho"], c["u"], c["du"],
                                            want_sens=True, **_dress(c))
        return dict(out=flow, chan=chan, dmin=dmin, sens=(c["N"] - 1.0) * sens[0] + sens[1], sens_chan=sens)
    if kd == "twopoint":
        out, dmin, sens = oracle.loop4d_twopoint(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *R["q"], *R["c"],
                                                 c["Z"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["m2"],
                                                 c["pext"], sel=sel, want_sens=True, **_dress(c))
    elif kd == "threepoint3d":
        out, dmin, sens = oracle.loop4d_threepoint_tab3d(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *R["q"],
                                                         *R["c1"], *R["c2"], R["phi"][1], c["ZA"], c["lnq_lo"],
                                                         c["lnq_hi"], c["interp"], c["v3"], c["lo3"], c["hi3"], c["log3"],
                                                         c["coef"], c["ext"], sel=sel, want_sens=True, **_dress(c))
    elif kd == "fourpoint":
        out, dmin, sens = oracle.loop4d_fourpoint(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *R["q"],
                                                  *R["c1"], *R["c2"], *R["phi"], c["ZA"], c["Zc"], c["L3"],
                                                  c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["ext"],
                                                  sel=sel, want_sens=True, **_dress(c))
    elif kd == "threepoint":
        out, dmin, sens = oracle.loop4d_threepoint(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *R["q"],
                                                   *R["c1"], *R["c2"], *R["phi"], c["ZA"], c["Zc"], c["L3"],
                                                   c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["ext"],
                                                   sel=sel, want_sens=True, **_dress(c))
    else:
        out, dmin, sens = oracle.matsubara3d(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
                                             *R["q"], *R["c"], c["Zpsi"], c["Zphi"], c["lnq_lo"], c["lnq_hi"],
                                             c["interp"], c["coef"], c["m2psi"], c["m2phi"], c["pext"], c["n_jext"],
                                             sel=sel, want_sens=True, **_dress(c))
    return dict(out=out, dmin=dmin, sens=sens)


def oracle_run_dm2(c, R, sel=None):
    """Mass derivatives from the oracle: dict of (value, sens) arrays keyed like gpu_run(..., want_d=True)."""
    kd = kind_of(c)
    if kd == "lpa":
        d, s = oracle.lpa_dm2(c["d"], c["T"], c["n_max"], c["reg_arg4d"], c["prefactor"], c["reg_kind"], c["reg_order"],
                              c["k"], *R["q"], c["rho"], c["u"], c["du"], **_dress(c))
        return dict(dchan=(d, s))
    if kd == "twopoint":
        d, s = oracle.loop4d_twopoint_dm2(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *R["q"], *R["c"],
                                          c["Z"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["m2"], c["pext"],
                                          sel=sel, **_dress(c))
        return dict(dout=(d, s))
    assert kd == "matsubara3d"
    a, b, sa, sb = oracle.matsubara3d_dm2(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
                                          *R["q"], *R["c"], c["Zpsi"], c["Zphi"], c["lnq_lo"], c["lnq_hi"], c["interp"],
                                          c["coef"], c["m2psi"], c["m2phi"], c["pext"], c["n_jext"], sel=sel, **_dress(c))
    return dict(dpsi=(a, sa), dphi=(b, sb))


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
           statistics=c.get("statistics", 0), mu=c.get("mu", 0.0) if c.get("statistics", 0) == 1 else 0.0, **dress)
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
           path=c.get("path", 0), **dress)
        res = dict(out=out, dmin=dmin, dpsi=dpsi, dphi=dphi, out_im=out_im)
    if not host:
        torch.cuda.synchronize()
    for big, n in guards:
        edge = torch.cat([big[:CANARY_PAD], big[CANARY_PAD + n:]]).cpu().numpy()
        assert np.all(edge == CANARY), "the library wrote outside an output buffer (%s)" % c["name"]
    return {k_: (None if v is None else down(v)) for k_, v in res.items() if v is not None or k_ == "dmin"}


def parity_report(gpu, orc, dmin_orc, sens):
    """Element-by-element comparison.  Regular outputs (oracle dmin >= REGULAR_DMIN and sens/|out| <= COND_MAX):
    relative error.  All outputs: |diff| / sens.  Returns a dict of worst cases; assert_parity() applies the bars."""
    gpu, orc, dmin_orc, sens = (np.asarray(a, dtype=np.float64).ravel() for a in (gpu, orc, dmin_orc, sens))
    with np.errstate(divide="ignore", invalid="ignore"):
        cond = np.where(orc != 0, sens / np.abs(orc), np.inf)
    regular = (dmin_orc >= REGULAR_DMIN) & (cond <= COND_MAX)
    diff = np.abs(gpu - orc)
    both_nonfinite = ~np.isfinite(gpu) & ~np.isfinite(orc)
    with np.errstate(divide="ignore", invalid="ignore"):
        rel = np.where(orc != 0, diff / np.abs(orc), np.where(diff == 0, 0.0, np.inf))
        ratio = np.where(diff == 0, 0.0, diff / sens)      # 0/0: both sides are exactly zero (e.g. Rdot = 0 at every node)
    # a non-finite value on one side only is a failure whatever the class of the output (NaN would otherwise drop out of
    # every maximum below); non-finite on both sides (an exactly vanishing denominator: inf in the oracle, NaN here) is none
    ratio = np.where(both_nonfinite, 0.0, np.where(np.isfinite(ratio), ratio, np.inf))
    rel = np.where(both_nonfinite, 0.0, np.where(np.isfinite(rel), rel, np.inf))
    rep = dict(n=gpu.size, n_regular=int(regular.sum()), n_singular=int((~regular).sum()),
               n_pole=int((dmin_orc < REGULAR_DMIN).sum()), n_cancelling=int(((dmin_orc >= REGULAR_DMIN) & ~regular).sum()),
               max_rel_regular=float(rel[regular].max()) if regular.any() else 0.0,
               max_sens_ratio_regular=float(ratio[regular].max()) if regular.any() else 0.0,
               max_sens_ratio_singular=float(ratio[~regular].max()) if (~regular).any() else 0.0,
               max_rel_cancelling=float(rel[(dmin_orc >= REGULAR_DMIN) & ~regular].max())
               if ((dmin_orc >= REGULAR_DMIN) & ~regular).any() else 0.0,
               n_nonfinite_gpu=int((~np.isfinite(gpu)).sum()), n_nonfinite_oracle=int((~np.isfinite(orc)).sum()),
               n_nonfinite_gpu_only=int((~np.isfinite(gpu) & np.isfinite(orc)).sum()))
    rep["_rel"] = rel
    rep["_regular"] = regular
    return rep


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
