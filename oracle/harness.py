"""Runs a workload dict (the seeded inputs of paper_2412_13043_b200.inputs, passed in by the caller) through the CPU
oracle, and the parity criterion of DESIGN.md ("Parity bar").  TEST INFRASTRUCTURE like the rest of oracle/: used by
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --full / --impl reference legs only.  Imports nothing
from the CUDA package."""
import numpy as np

from . import binding as oracle

REGULAR_DMIN = 1e-6      # an output is regular iff the oracle's dmin >= this (reading A4) ...
COND_MAX = 1e4           # ... and its terms do not cancel by more than this: sens / |out| <= COND_MAX
RTOL = 1e-12             # north_star: relative error <= 1e-12 per output on the same nodes (regular outputs)
SENS_EPS = 1e-14         # every output, regular or not: |gpu - oracle| <= SENS_EPS * sens (condition-aware bound)


def kind_of(c):
    n = c["name"]
    return "lpa" if n.startswith(("cfg0", "cfg1")) else n.split("_", 1)[1]


def _dress(c):
    """Dressed-regulator parameters of a workload (reading A20); absent = plain shapes."""
    return dict(zk=c.get("reg_zk", 1.0), eta=c.get("reg_eta", 0.0))


def _fdress(c):
    """... plus the fermionic-regulator switch of the families with a fermion line (reading A25)."""
    return dict(freg=c.get("fermion_reg", 0), **_dress(c))


def oracle_run(c, R, sel=None):
    """-> (out, dmin, sens); lpa: out = flow[n_field], extra channels under key 'chan' are returned via dict."""
    kd = kind_of(c)
    if kd == "lpa" and c.get("statistics", 0) == 1:     # fermionic loop at chemical potential (reading A22)
        m2 = np.stack([c["u"], c["u"] + 2.0 * c["rho"] * c["du"]])
        I, dI, dm, sn, snd = oracle.lpa_fermion(c["d"], c["T"], c["n_max"], c.get("mu", 0.0), c["prefactor"], c["reg_kind"],
                                                c["reg_order"], c["k"], *R["q"], m2.ravel(), **_fdress(c))
        I, dm, sn = (a.reshape(2, -1) for a in (I, dm, sn))
        return dict(out=(c["N"] - 1.0) * I[0] + I[1], chan=I, dmin=np.minimum(dm[0], dm[1]),
                    sens=abs(c["N"] - 1.0) * sn[0] + sn[1], sens_chan=sn)
    if kd == "matsubara3d" and c.get("reg_arg4d", 1) == 0:   # spatial regulators / chemical potential (reading A24)
        out, dmin, sens = oracle.matsubara3d_mu(c["T"], c["n_max"], c.get("mu", 0.0), c["prefactor"], c["reg_kind"],
                                                c["reg_order"], c["k"], *R["q"], *R["c"], c["Zpsi"], c["Zphi"],
                                                c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["m2psi"], c["m2phi"],
                                                c["pext"], c["n_jext"], sel=sel, want_sens=True, **_fdress(c))
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
                                             sel=sel, want_sens=True, **_fdress(c))
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
                                          c["coef"], c["m2psi"], c["m2phi"], c["pext"], c["n_jext"], sel=sel, **_fdress(c))
    return dict(dpsi=(a, sa), dphi=(b, sb))


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


