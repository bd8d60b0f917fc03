"""GPU parity for fermion lines regulated with the fermionic regulator RF / RFdot (dfrg_lpa_desc::fermion_reg,
dfrg_mats3d_desc::fermion_reg, reading A25) against the pinned oracle
(tests/test_oracle_pins_fermion_reg.py) on the same nodes: the fermionic LPA loop, and the Matsubara family through
every kernel path (specialised and any-shape moment kernels, row-streaming kernel, complex kernel at mu != 0), values,
dmin and mass derivatives; the flat fermionic threshold function straight against the CUDA path."""
import numpy as np
import pytest

import oracle
from paper_2412_13043_b200 import inputs

from helpers import RTOL, SENS_EPS, assert_dmin, assert_parity, gpu_run, make_rules, oracle_run, oracle_run_dm2
from test_gpu_parity_fermion import check, run as run_lpa

pytestmark = pytest.mark.gpu


def run_lpa_freg(c, mu, **dress):
    """test_gpu_parity_fermion.run with fermion_reg = 1 on both sides."""
    import torch
    from paper_2412_13043_b200 import binding as B
    xq, wq = B.dfrg_quad_nodes(*c["rule_q"])
    nf = c["rho"].size
    up = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    new = lambda *s: torch.full(s, float("nan"), dtype=torch.float64, device="cuda")
    flow, chan, dmin, dchan = new(nf), new(2, nf), new(nf), new(2, nf)
    B.dfrg_integrate_lpa(c["d"], c["T"], c["n_max"], 0, c["N"], c["prefactor"], c["reg_kind"], c["reg_order"], c["k"],
                         (up(xq), up(wq)), up(c["rho"]), up(c["u"]), up(c["du"]), flow, chan, dmin, dchan=dchan,
                         statistics=B.STAT_FERMION, mu=mu, reg_zk=dress.get("zk", 1.0), reg_eta=dress.get("eta", 0.0),
                         fermion_reg=1)
    torch.cuda.synchronize()
    m2 = np.stack([c["u"], c["u"] + 2 * c["rho"] * c["du"]])
    I, dI, dm, sens, sens_d = oracle.lpa_fermion(c["d"], c["T"], c["n_max"], mu, c["prefactor"], c["reg_kind"],
                                                 c["reg_order"], c["k"], xq, wq, m2.ravel(), freg=1, **dress)
    shp = lambda a: a.reshape(2, nf)
    g = dict(flow=flow.cpu().numpy(), chan=chan.cpu().numpy(), dmin=dmin.cpu().numpy(), dchan=dchan.cpu().numpy())
    o = dict(chan=shp(I), dchan=shp(dI), dmin=shp(dm), sens=shp(sens), sens_d=shp(sens_d))
    return g, o, m2


@pytest.mark.parametrize("T,mu,n_field,n_q,zk,eta", [(0.2, 0.0, 33, 17, 1.0, 0.0), (0.1, 0.4, 700, 64, 1.3, 0.27),
                                                     (0.05, 0.9, 100, 40, 0.7, -0.1)])
def test_fermion_lpa_fermionic_regulator_parity(T, mu, n_field, n_q, zk, eta):
    c = inputs.config1(T, n_field=n_field, n_q=n_q)
    g, o, _ = run_lpa_freg(c, mu, zk=zk, eta=eta)
    check(g, o, c["N"])
    c = inputs.config1(T, n_field=n_field, n_q=n_q, litim=True)
    c["reg_order"] = 8
    g, o, _ = run_lpa_freg(c, mu, zk=zk, eta=eta)
    check(g, o, c["N"])


def test_fermion_lpa_undressed_fermionic_regulator_is_the_bosonic_one():
    c = inputs.config1(0.1, n_field=130, n_q=32)
    g1, o1, _ = run_lpa_freg(c, 0.4)
    g0, o0, _ = run_lpa(c, 0.4)
    assert np.all(np.abs(g1["chan"] - g0["chan"]) <= SENS_EPS * o0["sens"])


def test_fermionic_threshold_function_on_gpu():
    """Flat fermionic regulator, zk = 1, eta != 0, radial [0,k], ONE Matsubara pair n in {-1, 0}:
    I = C T (2 k^5/3)(1 - eta/4) 2 Re 1/((pi T + i mu)^2 + k^2 + m2) in closed form (<= 1e-10: north_star)."""
    T, mu, eta, k = 0.25, 0.3, 0.4, 1.0
    c = inputs.config1(T, n_field=200, n_q=16, litim=True)
    c["n_max"] = 0
    g, o, m2 = run_lpa_freg(c, mu, eta=eta)
    D = (np.pi * T + 1j * mu) ** 2 + k * k + m2
    ref = c["prefactor"] * T * (2.0 * k ** 5 / 3.0) * (1 - eta / 4.0) * 2 * (1 / D).real
    ok = np.abs(D) > 0.05
    assert np.max(np.abs(g["chan"][ok] / ref[ok] - 1)) <= 1e-10


def mats_cfg(n_field, n_p, n_jext, n_q, n_c, n_max, **kw):
    c = inputs.config4(n_field=n_field, n_p=n_p, n_jext=n_jext, n_q=n_q, n_c=n_c)
    c["n_max"] = n_max
    c["fermion_reg"] = 1
    c.update(kw)
    return c


@pytest.mark.parametrize("shape", [(300, 2, 3, 9, 8, 3), (260, 2, 16, 7, 8, 11), (130, 2, 5, 7, 5, 2), (90, 1, 40, 5, 4, 3)])
@pytest.mark.parametrize("litim", [False, True])
def test_matsubara_fermionic_regulator_parity_4d(shape, litim):
    """4-D regulator argument (the BASELINE config 4 reading) through the specialised moment kernels ((3,3), (11,16)), the
    any-shape moment kernel and the row-streaming kernel (n_jext = 40)."""
    from paper_2412_13043_b200 import binding as B
    c = mats_cfg(*shape, reg_zk=1.2, reg_eta=0.15)
    if litim:
        c["reg_kind"] = oracle.REG_LITIM
    R = make_rules(c, B.dfrg_quad_nodes)
    o = oracle_run(c, R)
    for path in (0, B.M3_ANY_SHAPE, B.M3_ROW_STREAMING):
        g = gpu_run(dict(c, path=path), R, want_d=True, canary=True)
        assert_parity(g["out"], o["out"], o["dmin"], o["sens"], "freg path %d" % path)
        assert_dmin(g["dmin"], o["dmin"])
        if path == 0:
            od = oracle_run_dm2(c, R)
            for key in ("dpsi", "dphi"):
                d, s = od[key]
                assert np.all(np.abs(g[key] - d) <= SENS_EPS * s), key
    # and it is not the bosonic regularisation of the same line
    g0 = gpu_run(dict(c, fermion_reg=0), R)
    assert np.max(np.abs(g0["out"] / o["out"] - 1)) > 1e-4


@pytest.mark.parametrize("mu", [0.0, 0.45])
@pytest.mark.parametrize("shape", [(300, 2, 3, 9, 8, 3), (260, 2, 16, 7, 8, 11), (130, 2, 5, 7, 5, 2)])
def test_matsubara_fermionic_regulator_parity_spatial_and_mu(shape, mu):
    """Spatial regulators; mu != 0: the complex kernel (run-time and compile-time pair enumeration)."""
    from paper_2412_13043_b200 import binding as B
    c = mats_cfg(*shape, reg_zk=0.8, reg_eta=0.1, reg_arg4d=0, mu=mu)
    R = make_rules(c, B.dfrg_quad_nodes)
    o = oracle_run(c, R)
    g = gpu_run(c, R, canary=True)
    got = g["out"] + 1j * g["out_im"]
    for part in (np.real, np.imag):
        diff = np.abs(part(got) - part(o["out"]))
        assert np.all(diff <= SENS_EPS * o["sens"]), (mu, part.__name__, float(np.max(diff / o["sens"])))
    regular = (o["dmin"] >= 1e-6) & (o["sens"] <= 1e4 * np.abs(o["out"]))
    assert np.max(np.abs(got - o["out"])[regular] / np.abs(o["out"])[regular]) <= RTOL
    assert_dmin(g["dmin"], o["dmin"])
    if mu == 0.0:
        assert np.all(g["out_im"] == 0)


def test_matsubara_undressed_fermionic_regulator_with_unit_Zpsi_is_the_bosonic_one():
    from paper_2412_13043_b200 import binding as B
    c = mats_cfg(130, 2, 3, 9, 8, 3)
    c["Zpsi"] = np.ones_like(c["Zpsi"])
    R = make_rules(c, B.dfrg_quad_nodes)
    g1 = gpu_run(c, R)
    g0 = gpu_run(dict(c, fermion_reg=0), R)
    o0 = oracle_run(dict(c, fermion_reg=0), R)
    assert np.all(np.abs(g1["out"] - g0["out"]) <= SENS_EPS * o0["sens"])


def test_fermion_reg_validation():
    from paper_2412_13043_b200 import binding as B
    c = mats_cfg(4, 1, 1, 4, 4, 1, fermion_reg=2)
    R = make_rules(c, B.dfrg_quad_nodes)
    with pytest.raises(B.DfrgError) as e:
        gpu_run(c, R)
    assert e.value.status == B.DFRG_EINVAL
    c = inputs.config1(0.2, n_field=8, n_q=8)
    c["fermion_reg"] = 1                      # bosonic statistics: the switch must be 0
    R = make_rules(c, B.dfrg_quad_nodes)
    with pytest.raises(B.DfrgError) as e:
        gpu_run(c, R)
    assert e.value.status == B.DFRG_EINVAL
