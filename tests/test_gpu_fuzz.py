"""Seeded shape fuzzing of every family through the C ABI against the oracle, with sentinel margins around every
output buffer (tests/helpers.py: gpu_run(canary=True)): ragged sizes, sizes of 1, sizes around the tile and chunk
boundaries of the kernels (32 / 128 / 256 / 512 field points, 512-node chunks, 148 CTAs), both interpolation modes and
all regulator paths.  compute-sanitizer is not available on this pool; an out-of-bounds write that lands in a margin,
or a wrong index that changes a value, fails here."""
import os

import numpy as np
import pytest

from paper_2412_13043_b200 import inputs

from helpers import assert_parity, gpu_run, make_rules, oracle_run, oracle_run_dm2

pytestmark = pytest.mark.gpu


def nodes(n, a, b):
    from paper_2412_13043_b200 import binding as B
    return B.dfrg_quad_nodes(n, a, b)


def pick(rng, *choices):
    return choices[int(rng.integers(len(choices)))]


def draw(rng):
    fam = pick(rng, "lpa0", "lpa1", "lpaF", "two", "three", "four", "tab3d", "mats", "matsmu")
    edge_f = lambda: int(pick(rng, 1, 2, 31, 32, 33, 127, 128, 129, 255, 256, 257, 300, 511, 513, int(rng.integers(1, 700))))
    if fam == "lpa0":
        c = inputs.config0(n_field=edge_f(), n_q=int(rng.integers(1, 70)), d=int(pick(rng, 3, 4)))
    elif fam == "lpa1":
        c = inputs.config1(float(pick(rng, 0.05, 0.1, 0.2, 0.5)), n_field=edge_f(), n_q=int(rng.integers(1, 70)))
    elif fam == "lpaF":                              # fermionic loop at chemical potential: spatial regulator
        c = inputs.config1(float(pick(rng, 0.05, 0.1, 0.2, 0.5)), n_field=edge_f(), n_q=int(rng.integers(1, 70)))
        c["reg_arg4d"], c["statistics"], c["mu"] = 0, 1, float(pick(rng, 0.0, 0.3, 0.9))
        c["N"] = float(pick(rng, 1.0, 4.0))
    elif fam == "two":
        c = inputs.config2(n_field=edge_f(), n_ext=int(rng.integers(1, 9)), n_q=int(rng.integers(1, 50)),
                           n_c=int(rng.integers(1, 20)), interp=int(pick(rng, 1, 3)))
    elif fam == "three":
        c = inputs.config3(n_p=int(rng.integers(1, 5)), n_alpha=int(rng.integers(1, 4)), n_q=int(rng.integers(1, 20)),
                           n_c1=int(rng.integers(1, 9)), n_c2=int(rng.integers(1, 7)), n_phi=int(rng.integers(1, 5)),
                           interp=int(pick(rng, 1, 3)))
        if rng.integers(2):
            c["ext_outer"] = 0
    elif fam == "four":
        c = inputs.config5(n_s=int(rng.integers(1, 4)), n_ang=int(rng.integers(1, 4)), n_q=int(rng.integers(1, 12)),
                           n_c1=int(rng.integers(1, 7)), n_c2=int(rng.integers(1, 9)), n_phi=int(rng.integers(1, 7)),
                           interp=int(pick(rng, 1, 3)))
    elif fam == "tab3d":
        c = inputs.config6(n_p=int(rng.integers(1, 4)), n_alpha=int(rng.integers(1, 4)), n_q=int(rng.integers(1, 16)),
                           n_c1=int(rng.integers(1, 8)), n_c2=int(rng.integers(1, 6)),
                           n3=(int(rng.integers(2, 40)), int(rng.integers(2, 9)), int(rng.integers(2, 9))),
                           interp=int(pick(rng, 1, 3)))
        if rng.integers(2):
            c["ext_outer"] = 0
    else:
        n_jext = int(pick(rng, 1, 2, 3, 5, 8, 16, 17, 33))
        n_max = int(pick(rng, 0, 1, 2, 3, 7, 11))
        c = inputs.config4(n_field=edge_f(), n_p=int(rng.integers(1, 4)), n_jext=n_jext, n_q=int(rng.integers(1, 14)),
                           n_c=int(pick(rng, 1, 3, 4, 6, 8, 16)), interp=int(pick(rng, 1, 3)))
        c["n_max"] = n_max
        if fam == "matsmu":                          # spatial regulators; mu = 0 runs the real kernels, mu != 0 the complex one
            c["reg_arg4d"], c["mu"] = 0, float(pick(rng, 0.0, 0.35, -0.8))
            if c["mu"] != 0.0 and n_jext > 32:
                c["mu"] = 0.0
    reg = pick(rng, "exp1", "exp1", "exp3", "litim")
    if reg == "litim":
        c["reg_kind"] = 0
    elif reg == "exp3":
        c["reg_order"] = 3
    if rng.integers(3) == 0:
        c["reg_zk"], c["reg_eta"] = 1.0 + 0.5 * float(rng.random()), float(rng.random()) - 0.3
    if fam in ("lpaF", "mats", "matsmu") and rng.integers(2):
        c["fermion_reg"] = 1                         # fermion line regulated with RF / RFdot (reading A25)
    return fam, c


N_SEEDS = int(os.environ.get("DFRG_FUZZ_SEEDS", "400"))      # a longer soak: DFRG_FUZZ_SEEDS=2000 python -m pytest tests/test_gpu_fuzz.py


@pytest.mark.parametrize("seed", range(N_SEEDS))
def test_fuzz_shapes_against_oracle_with_canaries(seed):
    rng = np.random.default_rng(1000 + seed)
    fam, c = draw(rng)
    R = make_rules(c, nodes)
    want_d = fam in ("lpa0", "lpa1", "two", "mats") and bool(rng.integers(2))
    g = gpu_run(c, R, want_d=want_d, canary=True)
    o = oracle_run(c, R)
    what = "%s %s seed %d" % (c["name"], fam, seed)
    if fam == "matsmu":                              # complex result: both parts against the same yardstick
        assert_parity(g["out"], o["out"].real, o["dmin"], o["sens"], what + " re")
        assert_parity(g["out_im"], o["out"].imag, o["dmin"], o["sens"], what + " im")
        return
    assert_parity(g["out"], o["out"], o["dmin"], o["sens"], what)
    if want_d:
        od = oracle_run_dm2(c, R)
        for key, (val, sens) in od.items():
            dm = np.stack([o["dmin"]] * 2) if key == "dchan" else o["dmin"]
            assert_parity(g[key], val, dm, sens, "%s %s seed %d" % (c["name"], key, seed))
