"""Writes tests/golden/oracle_regression.txt: values of the CPU oracle on small seeded workloads.

Calls only `oracle/` and the seeded input recipes (`paper_2412_13043_b200/inputs.py`, no method arithmetic).  The stored
values are NOT a pin of the oracle (its pins are in tests/test_oracle_pins*.py); they freeze its arithmetic so that a later
change to it is deliberate: tests/test_oracle_pins.py::test_oracle_regression_fixture compares to 1e-14 relative.

    python tests/golden/make_oracle_regression.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2412_13043_b200 import inputs  # noqa: E402


def cases():
    """-> list of (name, 1-D array of values)"""
    out = []
    gl = oracle.gl_rule
    c = inputs.config0(n_field=9)
    flow, chan, dmin = oracle.lpa(c["d"], c["T"], c["n_max"], c["reg_arg4d"], c["N"], c["prefactor"], c["reg_kind"],
                                  c["reg_order"], c["k"], *gl(*c["rule_q"]), c["rho"], c["u"], c["du"])
    out.append(("cfg0_flow", flow[[0, 4, 8]]))
    c = inputs.config1(0.2, n_field=9)
    flow, chan, dmin = oracle.lpa(c["d"], c["T"], c["n_max"], c["reg_arg4d"], c["N"], c["prefactor"], c["reg_kind"],
                                  c["reg_order"], c["k"], *gl(*c["rule_q"]), c["rho"], c["u"], c["du"])
    out.append(("cfg1_T0.2_flow", flow[[0, 4, 8]]))
    I, dI, _, _, _ = oracle.lpa_fermion(3, 0.1, 8, 0.4, 1.0, oracle.REG_EXP_POLY, 1, 1.0, *gl(32, 0, 6), np.array([0.3, 2.0]))
    out.append(("lpa_fermion_mu0.4", np.concatenate([I, dI])))
    c = inputs.config2(n_field=5, n_ext=3, n_q=24, n_c=8)
    o, _ = oracle.loop4d_twopoint(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *gl(*c["rule_q"]), *gl(*c["rule_c"]),
                                  c["Z"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["m2"], c["pext"])
    out.append(("cfg2_out", o[:, [2, 4]].ravel()))
    c = inputs.config3(n_p=2, n_alpha=2, n_q=12, n_c1=6, n_c2=4, n_phi=3)
    r = [gl(*c["rule_" + a]) for a in ("q", "c1", "c2", "phi")]
    o, _ = oracle.loop4d_threepoint(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *r[0], *r[1], *r[2], *r[3],
                                    c["ZA"], c["Zc"], c["L3"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["ext"])
    out.append(("cfg3_out", o[[0, 3, 5, 7]]))
    c = inputs.config5(n_s=2, n_ang=1, n_q=8, n_c1=5, n_c2=4, n_phi=5)
    r = [gl(*c["rule_" + a]) for a in ("q", "c1", "c2", "phi")]
    o, _ = oracle.loop4d_fourpoint(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *r[0], *r[1], *r[2], *r[3],
                                   c["ZA"], c["Zc"], c["L3"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["ext"])
    out.append(("cfg5_out", o))
    c = inputs.config6(n_p=2, n_alpha=1, n_q=8, n_c1=5, n_c2=4, n_phi=3)
    r = [gl(*c["rule_" + a]) for a in ("q", "c1", "c2", "phi")]
    o, _ = oracle.loop4d_threepoint_tab3d(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *r[0], *r[1], *r[2], r[3][1],
                                          c["ZA"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["v3"], c["lo3"], c["hi3"],
                                          c["log3"], c["coef"], c["ext"])
    out.append(("cfg6_out", o))
    c = inputs.config4(n_field=4, n_p=2, n_jext=2, n_q=10, n_c=6)
    c["n_max"] = 3
    a = (c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], *gl(*c["rule_q"]), *gl(*c["rule_c"]), c["Zpsi"], c["Zphi"],
         c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["m2psi"], c["m2phi"], c["pext"], c["n_jext"])
    o, _ = oracle.matsubara3d(c["T"], c["n_max"], *a)
    out.append(("cfg4_out", o[:, :, 3].ravel()))
    o, _ = oracle.matsubara3d_mu(c["T"], c["n_max"], 0.3, *a)
    out.append(("cfg4_mu0.3_re", o[:, :, 3].real.ravel()))
    out.append(("cfg4_mu0.3_im", o[:, :, 3].imag.ravel()))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt")
    with open(path, "w") as fh:
        fh.write("# written by tests/golden/make_oracle_regression.py (calls only oracle/ and the seeded input recipes)\n")
        fh.write("# name index value(hex float) value(repr)\n")
        for name, vals in cases():
            for i, v in enumerate(np.asarray(vals, dtype=np.float64)):
                fh.write("%s %d %s %r\n" % (name, i, float(v).hex(), float(v)))
    print("wrote", path)
