"""dfrg_integrate_twopoint_noalloc: the two-point loop for callers that cannot allocate device memory.

Who needs it: a host program that has handed all device memory to its own allocator, a thread that must never wait on
the CUDA driver's allocation lock, a job under a device-memory cap.  The regular entry point (dfrg_integrate_loop4d)
takes the scratch of its kernels from a memory pool that may have to grow; this one keeps the scratch in a fixed
8 MiB array inside libdfrg.so and allocates nothing, at the price of a size limit (DFRG_ESCRATCH beyond it).

What is checked here: its outputs (values, mass derivatives, dmin) against those of the regular entry point on the same
inputs -- they run the same kernels with the same launch plan, so they must agree bit for bit, which is inside the
1e-12 parity bar the other GPU tests use -- on calls made back to back without clearing anything in between (the array
keeps what the previous, differently shaped call left in it), and that an oversized call is refused with nothing written.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It does not depend on what ran before it (fresh process or not)."""
import ctypes as C

import numpy as np
import pytest

from paper_2412_13043_b200 import binding as B
from paper_2412_13043_b200 import inputs

from helpers import RTOL, make_rules


def _nodes(n, a, b):
    return B.dfrg_quad_nodes(n, a, b)


def _both_paths(c, want_d, want_dmin):
    """Runs the workload through dfrg_integrate_loop4d and through dfrg_integrate_twopoint_noalloc on the same device
    tensors -> ((out, dout, dmin) of the regular path, the same of the no-allocation path) as numpy arrays (None = not asked)."""
    import torch
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    R = make_rules(c, _nodes)
    rq, rc = (up(R["q"][0]), up(R["q"][1])), (up(R["c"][0]), up(R["c"][1]))
    Z, coef, m2, pext = up(c["Z"]), up(c["coef"]), up(c["m2"]), up(c["pext"])
    shape = (c["pext"].size, c["m2"].size)
    new = lambda want: torch.full(shape, float("nan"), dtype=torch.float64, device="cuda") if want else None
    ref = (new(True), new(want_d), new(want_dmin))
    got = (new(True), new(want_d), new(want_dmin))
    B.dfrg_integrate_loop4d(B.LOOP_TWOPOINT, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rq, rc, None, None,
                            (Z,), c["lnq_lo"], c["lnq_hi"], c["interp"], coef, m2, pext, ref[0], ref[2], dout_dm2=ref[1])
    B.dfrg_integrate_twopoint_noalloc(c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rq, rc, Z, c["lnq_lo"],
                                      c["lnq_hi"], c["interp"], coef, m2, pext, got[0], got[2], dout_dm2=got[1])
    torch.cuda.synchronize()
    down = lambda t: None if t is None else t.cpu().numpy()
    return tuple(map(down, ref)), tuple(map(down, got))


def _assert_same(ref, got, what):
    for name, r, g in zip(("out", "dout_dm2", "dmin"), ref, got):
        if r is None:
            assert g is None
            continue
        assert np.all(np.isfinite(r)), "%s %s: regular path not finite" % (what, name)
        assert np.all(np.isfinite(g)), "%s %s: a NaN of the output's initial fill survived or was produced" % (what, name)
        rel = np.max(np.abs(g - r) / np.maximum(np.abs(r), 1e-300))
        assert rel <= RTOL, "%s %s: max rel %.3e" % (what, name, rel)          # the bar of the parity tests
        assert np.array_equal(g, r), "%s %s: same kernels, same plan: must be bit-identical" % (what, name)


@pytest.mark.gpu
def test_noalloc_matches_regular_path_on_calls_in_a_row():
    # three calls back to back, nothing cleared in between: a ragged small case (two field tiles, short last tile, 37
    # radial nodes in chunks of 8), then BASELINE.json config 2 in full with derivatives (which overwrites most of what
    # the first call left), then the small case again on top of the big call's leftovers, without dmin / derivatives
    small = inputs.config2(n_field=300, n_ext=5, n_q=37, n_c=7)
    ref, got = _both_paths(small, want_d=True, want_dmin=True)
    _assert_same(ref, got, "small, first call")
    first_small = got
    ref, got = _both_paths(inputs.config2(), want_d=True, want_dmin=True)
    assert got[0].shape == (64, 256)
    _assert_same(ref, got, "cfg2, second call")
    ref, got = _both_paths(small, want_d=False, want_dmin=False)
    _assert_same(ref, got, "small, third call")
    assert np.array_equal(got[0], first_small[0])      # values do not depend on whether derivatives / dmin were asked for


@pytest.mark.gpu
def test_noalloc_refuses_what_does_not_fit_and_writes_nothing():
    import torch
    # 4096 field points x 300 momenta with derivatives: the partial sums alone are 2 * 4096 * 300 * 8 B = 19.7 MB > 8 MiB
    c = inputs.config2(n_field=4096, n_ext=300, n_q=16, n_c=8)
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    R = make_rules(c, _nodes)
    rq, rc = (up(R["q"][0]), up(R["q"][1])), (up(R["c"][0]), up(R["c"][1]))
    out = torch.full((300, 4096), -3.5, dtype=torch.float64, device="cuda")
    dout = torch.full((300, 4096), -3.5, dtype=torch.float64, device="cuda")
    args = (c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], rq, rc, up(c["Z"]), c["lnq_lo"], c["lnq_hi"],
            c["interp"], up(c["coef"]), up(c["m2"]), up(c["pext"]))
    with pytest.raises(B.DfrgError) as err:
        B.dfrg_integrate_twopoint_noalloc(*args, out, None, dout_dm2=dout)
    assert err.value.status == B.DFRG_ESCRATCH and "scratch" in str(err.value)
    torch.cuda.synchronize()
    assert bool((out == -3.5).all()) and bool((dout == -3.5).all())
    # the regular entry point serves the same call
    B.dfrg_integrate_loop4d(B.LOOP_TWOPOINT, *args[:6], None, None, (args[6],), *args[7:], out, None, dout_dm2=dout)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all()) and bool(torch.isfinite(dout).all())


def test_noalloc_validates_before_touching_the_device():
    # fake non-null pointers, as tests/test_abi_cpu.py: rejected without dereferencing anything and without a GPU
    from paper_2412_13043_b200 import build as dfrg_build
    dfrg_build.build()
    lib = B.lib()
    p = 0x1000
    reg = B.Regulator(B.REG_EXP_POLY, 1, 1.0, 1.0, 0.0)
    rule = B.Rule(p, p, 8)
    tab = B.Table(p, 16, 1, -3.0, 3.0, 3)
    f = lib.dfrg_integrate_twopoint_noalloc

    def desc(family=B.LOOP_TWOPOINT, n_coef=2):
        D = B.Loop4dDesc()
        D.family, D.prefactor, D.reg, D.q, D.cos1, D.coef, D.n_coef = family, 1.0, reg, rule, rule, p, n_coef
        D.tab[0] = tab
        return D
    assert f(None, 4, p, 2, p, p, None, None) == B.DFRG_EINVAL
    assert f(C.byref(desc(family=B.LOOP_THREEPOINT)), 4, p, 2, p, p, None, None) == B.DFRG_EINVAL   # two-point only
    assert f(C.byref(desc(n_coef=3)), 4, p, 2, p, p, None, None) == B.DFRG_EINVAL
    assert f(C.byref(desc()), 0, p, 2, p, p, None, None) == B.DFRG_EINVAL
    assert f(C.byref(desc()), 4, None, 2, p, p, None, None) == B.DFRG_EINVAL
    assert f(C.byref(desc()), 4, p, 2, p, None, None, None) == B.DFRG_EINVAL
    assert b"scratch" in lib.dfrg_strerror(B.DFRG_ESCRATCH)
    assert B.NOALLOC_SCRATCH_BYTES == 8 * 1024 * 1024
