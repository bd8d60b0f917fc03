"""GPU parity for the Matsubara family with spatial regulators and at finite chemical potential (dfrg_mats3d_desc::
reg_arg4d = 0, mu, out_im, reading A24) against the pinned oracle
(tests/test_oracle_pins_matsubara_mu.py) on the same nodes: real and imaginary parts, dmin, every moment-kernel shape
class, the symmetric-pair and plain moment loops, the host entry point, and mu = 0 through the real kernels."""
import numpy as np
import pytest

import oracle
from paper_2412_13043_b200 import binding as B
from paper_2412_13043_b200 import inputs

from helpers import RTOL, SENS_EPS, assert_dmin

pytestmark = pytest.mark.gpu


def run(c, mu, host=False, want_dmin=True, want_im=True):
    import torch
    from paper_2412_13043_b200 import binding as B
    xq, wq = B.dfrg_quad_nodes(*c["rule_q"])
    xc, wc = B.dfrg_quad_nodes(*c["rule_c"])
    shape = (c["pext"].size, c["n_jext"], c["m2psi"].size)
    if host:
        up = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        new = lambda: np.full(shape, np.nan)
        fn, down = B.dfrg_integrate_matsubara3d_host, (lambda a: a)
    else:
        up = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()
        new = lambda: torch.full(shape, float("nan"), dtype=torch.float64, device="cuda")
        fn, down = B.dfrg_integrate_matsubara3d, (lambda a: a.cpu().numpy())
    out, out_im, dmin = new(), (new() if want_im else None), (new() if want_dmin else None)
    fn(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], (up(xq), up(wq)), (up(xc), up(wc)),
       up(c["Zpsi"]), up(c["Zphi"]), c["lnq_lo"], c["lnq_hi"], c["interp"], up(c["coef"]), up(c["m2psi"]),
       up(c["m2phi"]), up(c["pext"]), c["n_jext"], out, dmin, reg_arg4d=0, mu=mu, out_im=out_im,
       reg_zk=c.get("reg_zk", 1.0), reg_eta=c.get("reg_eta", 0.0), path=c.get("path", 0))
    if not host:
        torch.cuda.synchronize()
    o, odm, osens = oracle.matsubara3d_mu(c["T"], c["n_max"], mu, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
                                          xq, wq, xc, wc, c["Zpsi"], c["Zphi"], c["lnq_lo"], c["lnq_hi"], c["interp"],
                                          c["coef"], c["m2psi"], c["m2phi"], c["pext"], c["n_jext"], want_sens=True,
                                          zk=c.get("reg_zk", 1.0), eta=c.get("reg_eta", 0.0))
    g = down(out) + 1j * (down(out_im) if want_im else 0.0)
    return g, (None if dmin is None else down(dmin)), o, odm, osens


def check(g, gdm, o, odm, sens, what):
    """The bars of DESIGN.md section 5 on the real and the imaginary part separately: each part's error against
    SENS_EPS * sens (every output) and against RTOL * |out| (regular outputs; |out| = modulus of the complex value)."""
    assert not np.any(~np.isfinite(g) & np.isfinite(o)), what
    regular = (odm >= 1e-6) & (sens <= 1e4 * np.abs(o))
    assert regular.sum() > 0.5 * regular.size or regular.size < 16, what     # (a lone field point at rho = 0 is a pole output)
    for part in (np.real, np.imag):
        diff = np.abs(part(g) - part(o))
        assert np.all(diff <= SENS_EPS * sens), (what, part.__name__, float(np.max(diff / sens)))
        if regular.any():
            assert np.max(diff[regular] / np.abs(o[regular])) <= RTOL, (what, part.__name__)
    if gdm is not None:
        assert_dmin(gdm, odm, scale=1.0 + float(np.max(odm)))


@pytest.mark.parametrize("n_field,n_p,n_jext,n_q,n_c,n_max,mu", [(1, 1, 1, 3, 2, 0, 0.3), (300, 2, 3, 9, 8, 3, 0.4),
                                                                 (530, 2, 5, 7, 6, 4, 0.9), (100, 3, 16, 5, 16, 11, 0.25),
                                                                 (64, 1, 32, 4, 4, 5, 0.6), (260, 2, 2, 12, 24, 11, -0.5)])
def test_matsubara_mu_parity(n_field, n_p, n_jext, n_q, n_c, n_max, mu):
    c = inputs.config4(n_field=n_field, n_p=n_p, n_jext=n_jext, n_q=n_q, n_c=n_c)
    c["n_max"] = n_max
    g, gdm, o, odm, sens = run(c, mu)
    check(g, gdm, o, odm, sens, "mats_mu_%d_%d_%d_%d_%d_%d" % (n_field, n_p, n_jext, n_q, n_c, n_max))
    assert np.any(g.imag != 0)


def test_matsubara_mu_regulators_interp_dressing_and_options():
    import os
    base = dict(n_field=140, n_p=2, n_jext=3, n_q=10, n_c=8)
    c = inputs.config4(**base)
    c["n_max"] = 3
    c["reg_kind"] = 0                                              # flat spatial regulator
    check(*run(c, 0.35), "mats_mu_litim")
    c = inputs.config4(interp=1, k=1.7, **base)
    c["n_max"] = 2
    c["reg_order"] = 3
    c["reg_zk"], c["reg_eta"] = 1.3, 0.27
    check(*run(c, 0.5), "mats_mu_dressed")
    c = inputs.config4(**base)
    c["n_max"] = 3
    g, gdm, o, odm, sens = run(c, 0.35)
    c["path"] = B.M3_PLAIN_MOMENTS
    g2, _, _, _, _ = run(c, 0.35)
    c["path"] = 0
    check(g2, None, o, odm, sens, "mats_mu_plain_loop")
    assert not np.array_equal(g, g2)
    g3, _, _, _, _ = run(c, 0.35, want_dmin=False)
    assert np.array_equal(g, g3)
    g4, gdm4, _, _, _ = run(c, 0.35, host=True)
    assert np.array_equal(g, g4) and np.array_equal(gdm, gdm4)
    gm, _, om, _, _ = run(c, -0.35)
    assert np.array_equal(gm, np.conj(g))                          # mu -> -mu conjugates, bit for bit


@pytest.mark.parametrize("shape", [dict(n_field=300, n_p=2, n_jext=3, n_q=9, n_c=8, n_max=3),      # specialised kernel
                                   dict(n_field=130, n_p=2, n_jext=5, n_q=7, n_c=5, n_max=2),      # any-shape kernel
                                   dict(n_field=90, n_p=1, n_jext=40, n_q=5, n_c=4, n_max=3)])     # row-streaming kernel
def test_matsubara_spatial_regulators_mu0_through_the_real_kernels(shape):
    n_max = shape.pop("n_max")
    c = inputs.config4(**shape)
    c["n_max"] = n_max
    g, gdm, o, odm, sens = run(c, 0.0)
    assert np.all(g.imag == 0) and np.all(o.imag == 0)             # out_im is zero-filled
    check(g, gdm, o, odm, sens, "mats_spatial_mu0")
    g2, _, _, _, _ = run(c, 0.0, want_im=False)
    assert np.array_equal(g.real, g2.real)


def test_matsubara_mu_shared_memory_limit_is_reported():
    from paper_2412_13043_b200 import binding as B
    c = inputs.config4(n_field=64, n_p=1, n_jext=32, n_q=4, n_c=4)
    c["n_max"] = 20                                  # 32 x 41 complex beta' entries x 2 stages + H columns > 220 KB
    with pytest.raises(B.DfrgError) as err:
        run(c, 0.6)
    assert err.value.status == B.DFRG_EUNSUPPORTED


def test_matsubara_mu_full_config4_sampled():
    """BASELINE config 4's sizes (64 p x 16 j x 512 field points, 23 x 96 x 24 nodes) at mu = 0.3 k, oracle on a
    deterministic sample of outputs."""
    import torch
    from paper_2412_13043_b200 import binding as B
    c = inputs.config4()
    mu = 0.3
    xq, wq = B.dfrg_quad_nodes(*c["rule_q"])
    xc, wc = B.dfrg_quad_nodes(*c["rule_c"])
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    shape = (c["pext"].size, c["n_jext"], c["m2psi"].size)
    out, out_im, dmin = (torch.empty(shape, dtype=torch.float64, device="cuda") for _ in range(3))
    B.dfrg_integrate_matsubara3d(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
                                 (up(xq), up(wq)), (up(xc), up(wc)), up(c["Zpsi"]), up(c["Zphi"]), c["lnq_lo"],
                                 c["lnq_hi"], c["interp"], up(c["coef"]), up(c["m2psi"]), up(c["m2phi"]), up(c["pext"]),
                                 c["n_jext"], out, dmin, reg_arg4d=0, mu=mu, out_im=out_im)
    torch.cuda.synchronize()
    sel = np.arange(0, 64 * 16 * 512, 1021)
    o, odm, sens = oracle.matsubara3d_mu(c["T"], c["n_max"], mu, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
                                         xq, wq, xc, wc, c["Zpsi"], c["Zphi"], c["lnq_lo"], c["lnq_hi"], c["interp"],
                                         c["coef"], c["m2psi"], c["m2phi"], c["pext"], c["n_jext"], sel=sel,
                                         want_sens=True)
    g = (out.cpu().numpy() + 1j * out_im.cpu().numpy()).ravel()[sel]
    check(g, dmin.cpu().numpy().ravel()[sel], o, odm, sens, "cfg4_mu_full_sampled")


def run_dm2(c, mu, host=False):
    import torch
    from paper_2412_13043_b200 import binding as B
    xq, wq = B.dfrg_quad_nodes(*c["rule_q"])
    xc, wc = B.dfrg_quad_nodes(*c["rule_c"])
    shape = (c["pext"].size, c["n_jext"], c["m2psi"].size)
    if host:
        up = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        new = lambda: np.full(shape, np.nan)
        fn, down = B.dfrg_integrate_matsubara3d_host, (lambda a: a)
    else:
        up = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()
        new = lambda: torch.full(shape, float("nan"), dtype=torch.float64, device="cuda")
        fn, down = B.dfrg_integrate_matsubara3d, (lambda a: a.cpu().numpy())
    bufs = [new() for _ in range(6)]
    fn(c["T"], c["n_max"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], (up(xq), up(wq)), (up(xc), up(wc)),
       up(c["Zpsi"]), up(c["Zphi"]), c["lnq_lo"], c["lnq_hi"], c["interp"], up(c["coef"]), up(c["m2psi"]),
       up(c["m2phi"]), up(c["pext"]), c["n_jext"], bufs[0], None, reg_arg4d=0, mu=mu, out_im=bufs[1],
       dout_dm2_psi=bufs[2], dout_dm2_psi_im=bufs[3], dout_dm2_phi=bufs[4], dout_dm2_phi_im=bufs[5])
    if not host:
        torch.cuda.synchronize()
    b = [down(x) for x in bufs]
    args = (c["T"], c["n_max"], mu, c["prefactor"], c["reg_kind"], c["reg_order"], c["k"], xq, wq, xc, wc, c["Zpsi"],
            c["Zphi"], c["lnq_lo"], c["lnq_hi"], c["interp"], c["coef"], c["m2psi"], c["m2phi"], c["pext"], c["n_jext"])
    o, odm, sens = oracle.matsubara3d_mu(*args, want_sens=True)
    dpsi, dphi, spsi, sphi = oracle.matsubara3d_mu_dm2(*args)
    return (b[0] + 1j * b[1], b[2] + 1j * b[3], b[4] + 1j * b[5]), (o, dpsi, dphi), (sens, spsi, sphi), odm


@pytest.mark.parametrize("n_field,n_p,n_jext,n_q,n_c,n_max,mu", [(300, 2, 3, 9, 8, 3, 0.4), (130, 2, 5, 7, 5, 2, 0.7),
                                                                 (300, 2, 3, 9, 8, 3, 0.0), (130, 2, 5, 7, 5, 2, 0.0),
                                                                 (90, 1, 40, 5, 4, 3, 0.0)])
def test_matsubara_mu_mass_derivatives(n_field, n_p, n_jext, n_q, n_c, n_max, mu):
    # mu != 0: complex kernel, modes 1 and 2; mu = 0: spatial regulators through the real kernels (specialised, any-shape,
    # row-streaming), imaginary parts zero-filled
    c = inputs.config4(n_field=n_field, n_p=n_p, n_jext=n_jext, n_q=n_q, n_c=n_c)
    c["n_max"] = n_max
    g, o, sens, odm = run_dm2(c, mu)
    for gi, oi, si, name in zip(g, o, sens, ("value", "dpsi", "dphi")):
        diff = np.abs(gi - oi)
        assert np.all(diff <= SENS_EPS * si), (name, float(np.max(diff / si)))
        regular = (odm >= 1e-6) & (si <= 1e4 * np.abs(oi))
        assert np.max(diff[regular] / np.abs(oi[regular])) <= RTOL, name
        if mu == 0.0:
            assert np.all(gi.imag == 0)
    if n_jext <= 5 and n_field == 130:
        h, _, _, _ = run_dm2(c, mu, host=True)
        assert all(np.array_equal(a, b) for a, b in zip(g, h))


def test_matsubara_mu_static_and_runtime_pair_enumeration_agree():
    """(n_max, n_jext) = (11, 16) takes the complex kernel whose pair code is enumerated at compile time; forced through the
    run-time enumeration (DFRG_M3_PATH=moment-generic) it must give the same sums (same order per accumulator: bit for bit)."""
    import os
    c = inputs.config4(n_field=300, n_p=2, n_jext=16, n_q=6, n_c=8)
    g, gdm, o, odm, sens = run(c, 0.3)
    check(g, gdm, o, odm, sens, "mats_mu_static_11_16")
    c["path"] = B.M3_ANY_SHAPE
    g2, _, _, _, _ = run(c, 0.3)
    c["path"] = 0
    assert np.array_equal(g, g2)
