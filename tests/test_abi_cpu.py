"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/dfrg.h declares,
dfrg_quad_nodes (host-side S1) agrees with the oracle's generator, and argument validation
returns the documented status codes before anything touches a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
from paper_2412_13043_b200 import binding as B
from paper_2412_13043_b200 import build as dfrg_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    dfrg_build.build()
    return B.lib()


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "dfrg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(dfrg_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert lib.dfrg_version() == 100
    assert lib.dfrg_strerror(0) == b"ok" and b"invalid" in lib.dfrg_strerror(-1)


def test_struct_layouts_match_header_sizes(tmp_path):
    # compile include/dfrg.h as plain C and compare sizeof / offsetof with the ctypes mirrors
    import subprocess
    src = tmp_path / "sz.c"
    src.write_text("""#include <stdio.h>
#include <stddef.h>
#include "dfrg.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu ", sizeof(dfrg_regulator), sizeof(dfrg_rule), sizeof(dfrg_table),
         sizeof(dfrg_lpa_desc), sizeof(dfrg_loop4d_desc), sizeof(dfrg_mats3d_desc));
  printf("%zu %zu %zu %zu\\n", offsetof(dfrg_lpa_desc, q), offsetof(dfrg_loop4d_desc, tab),
         offsetof(dfrg_loop4d_desc, n_coef), offsetof(dfrg_mats3d_desc, tab_phi));
  return 0;
}
""")
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(v) for v in subprocess.check_output([str(exe)]).split()]
    want = [C.sizeof(B.Regulator), C.sizeof(B.Rule), C.sizeof(B.Table), C.sizeof(B.LpaDesc), C.sizeof(B.Loop4dDesc),
            C.sizeof(B.Mats3dDesc), B.LpaDesc.q.offset, B.Loop4dDesc.tab.offset, B.Loop4dDesc.n_coef.offset,
            B.Mats3dDesc.tab_phi.offset]
    assert got == want


@pytest.mark.parametrize("n", [1, 2, 3, 5, 16, 24, 32, 64, 96, 127, 128, 512])
def test_quad_nodes_match_oracle_generator(lib, n):
    for a, b in ((-1.0, 1.0), (0.0, 6.0), (0.0, 2 * np.pi)):
        x, w = B.dfrg_quad_nodes(n, a, b)
        xo, wo = oracle.gl_rule(n, a, b)
        scale = max(abs(a), abs(b))
        assert np.all(np.abs(x - xo) <= 4 * np.finfo(float).eps * scale)          # <= 4 ulp of the interval scale
        assert np.all(np.abs(w - wo) <= 4 * np.finfo(float).eps * np.abs(wo))
        assert np.all(np.diff(x) > 0) and np.all(w > 0)
        assert abs(w.sum() - (b - a)) <= 1e-14 * (b - a) * max(1, n / 32)


def test_quad_nodes_validation(lib):
    x = np.empty(4)
    w = np.empty(4)
    q = lib.dfrg_quad_nodes
    assert q(0, 0, -1.0, 1.0, x.ctypes.data, w.ctypes.data) == B.DFRG_EINVAL
    assert q(0, 4, 1.0, 1.0, x.ctypes.data, w.ctypes.data) == B.DFRG_EINVAL
    assert q(1, 4, -1.0, 1.0, x.ctypes.data, w.ctypes.data) == B.DFRG_EINVAL
    assert q(0, 4, -1.0, 1.0, None, w.ctypes.data) == B.DFRG_EINVAL
    assert q(0, 5000, -1.0, 1.0, x.ctypes.data, w.ctypes.data) == B.DFRG_EINVAL
    assert q(0, 4, -1.0, 1.0, x.ctypes.data, w.ctypes.data) == B.DFRG_OK


def test_integrators_validate_before_touching_the_device(lib):
    # fake non-null pointers: validation must reject these calls without dereferencing anything
    p = 0x1000
    reg = B.Regulator(B.REG_EXP_POLY, 1, 1.0, 1.0, 0.0)
    rule = B.Rule(p, p, 8)
    D = B.LpaDesc(4, 0.0, 0, 1, 4.0, 1.0, reg, rule)
    f = lib.dfrg_integrate_lpa
    assert f(None, 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    assert f(C.byref(D), 0, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    assert f(C.byref(D), 4, None, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(4, -1.0, 0, 1, 4.0, 1.0, reg, rule)
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(4, 0.0, 0, 1, 4.0, 1.0, B.Regulator(1, 1, 0.0, 1.0, 0.0), rule)
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(4, 0.0, 0, 1, 4.0, 1.0, B.Regulator(7, 1, 1.0, 1.0, 0.0), rule)
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(4, 0.0, 0, 1, 4.0, 1.0, B.Regulator(1, 1, 1.0), rule)            # zk = 0 (zero-initialised): rejected
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(3, 0.1, 4, 1, 4.0, 1.0, reg, rule, None, B.STAT_FERMION, 0.3)    # fermions + mu: spatial regulator only
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(3, 0.0, 4, 0, 4.0, 1.0, reg, rule, None, B.STAT_FERMION, 0.3)    # fermionic frequencies need T > 0
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(3, 0.1, 4, 0, 4.0, 1.0, reg, rule, None, B.STAT_BOSON, 0.3)      # no chemical potential for bosons
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(3, 0.1, 4, 0, 4.0, 1.0, reg, rule, None, 7, 0.0)
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    bad = B.LpaDesc(9, 0.0, 0, 1, 4.0, 1.0, reg, rule)
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EUNSUPPORTED
    # batched temperatures: host arrays, 1 <= n_T <= 16, every entry validated like a single call
    fb = lib.dfrg_integrate_lpa_batch
    Tv, nv = (C.c_double * 17)(*([0.1] * 17)), (C.c_int * 17)(*([3] * 17))
    Db = B.LpaDesc(3, 0.0, 0, 1, 4.0, 1.0, reg, rule)
    assert fb(C.byref(Db), 0, Tv, nv, 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    assert fb(C.byref(Db), 2, None, nv, 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    assert fb(C.byref(Db), 17, Tv, nv, 4, p, p, p, p, None, None, None) == B.DFRG_EUNSUPPORTED
    Tv[1] = -0.5
    assert fb(C.byref(Db), 2, Tv, nv, 4, p, p, p, p, None, None, None) == B.DFRG_EINVAL
    Tv[1], nv[1] = 0.1, 100000
    assert fb(C.byref(Db), 2, Tv, nv, 4, p, p, p, p, None, None, None) == B.DFRG_EUNSUPPORTED
    bad = B.LpaDesc(3, 0.1, 4000, 1, 4.0, 1.0, reg, rule)
    assert f(C.byref(bad), 4, p, p, p, p, None, None, None) == B.DFRG_EUNSUPPORTED

    T3 = B.Table * 3
    tab = B.Table(p, 128, 1, -9.0, 5.0, 3)
    g = lib.dfrg_integrate_loop4d
    D2 = B.Loop4dDesc(B.LOOP_TWOPOINT, 1.0, reg, rule, rule, B.Rule(None, None, 0), B.Rule(None, None, 0),
                      T3(tab, tab, tab), p, 2)
    assert g(C.byref(D2), 0, p, 4, p, p, None, None) == B.DFRG_EINVAL           # n_field < 1
    D2.n_coef = 3
    assert g(C.byref(D2), 4, p, 4, p, p, None, None) == B.DFRG_EINVAL           # wrong n_coef
    D2.n_coef = 2
    D2.tab[0].interp = 2
    assert g(C.byref(D2), 4, p, 4, p, p, None, None) == B.DFRG_EINVAL           # interp not in {1,3}
    D2.tab[0].interp = 3
    D2.tab[0].n_q = 3
    assert g(C.byref(D2), 4, p, 4, p, p, None, None) == B.DFRG_EINVAL           # cubic needs n_q >= 4
    D2.tab[0].n_q = 128
    D2.tab[0].lnq_hi = -9.0
    assert g(C.byref(D2), 4, p, 4, p, p, None, None) == B.DFRG_EINVAL           # lnq_hi <= lnq_lo
    D2.tab[0].lnq_hi = 5.0
    D2.q.n = 4096
    D2.cos1.n = 64
    assert g(C.byref(D2), 4, p, 4, p, p, None, None) == B.DFRG_EUNSUPPORTED     # beyond shared memory
    D3 = B.Loop4dDesc(B.LOOP_THREEPOINT, 1.0, reg, rule, rule, rule, rule, T3(tab, tab, tab), p, 34)
    assert g(C.byref(D3), 0, None, 4, p, p, None, None) == B.DFRG_EINVAL        # n_coef != 35
    D3.n_coef = 35
    assert g(C.byref(D3), 3, None, 4, p, p, None, None) == B.DFRG_EINVAL        # three-point has no field axis
    D3.family = 5
    assert g(C.byref(D3), 0, None, 4, p, p, None, None) == B.DFRG_EINVAL
    D3.family = B.LOOP_FOURPOINT
    assert g(C.byref(D3), 0, None, 4, p, p, None, None) == B.DFRG_EINVAL        # four-point needs n_coef == 70
    D3.n_coef = 70
    big = B.Rule(p, p, 600)
    D5 = B.Loop4dDesc(B.LOOP_FOURPOINT, 1.0, reg, rule, rule, big, rule, T3(tab, tab, tab), p, 70)
    assert g(C.byref(D5), 0, None, 4, p, p, None, None) == B.DFRG_EUNSUPPORTED  # cos2 rule longer than a CTA

    i3, d3 = C.c_int * 3, C.c_double * 3
    t3 = B.Table3D(p, i3(96, 8, 7), d3(-9.0, -1.0, -1.0), d3(5.0, 1.0, 1.0), i3(1, 0, 0))
    D6 = B.Loop4dDesc(B.LOOP_THREEPOINT_TAB3D, 1.0, reg, rule, rule, rule, rule, T3(tab, tab, tab), p, 35, 0, None, t3)
    assert g(C.byref(D6), 1, None, 4, p, p, None, None) == B.DFRG_EINVAL        # no field axis
    D6.tab3d.n[1] = 1
    assert g(C.byref(D6), 0, None, 4, p, p, None, None) == B.DFRG_EINVAL        # every axis needs >= 2 points
    D6.tab3d.n[1] = 8
    D6.tab3d.hi[2] = -1.0
    assert g(C.byref(D6), 0, None, 4, p, p, None, None) == B.DFRG_EINVAL        # empty axis range
    D6.tab3d.hi[2] = 1.0
    D6.tab3d.n[0] = 4000
    assert g(C.byref(D6), 0, None, 4, p, p, None, None) == B.DFRG_EUNSUPPORTED  # table beyond the shared-memory budget
    D6.tab3d.n[0] = 96
    D6.tab3d.v = None
    assert g(C.byref(D6), 0, None, 4, p, p, None, None) == B.DFRG_EINVAL

    h = lib.dfrg_integrate_matsubara3d
    stack = B.Table(p, 128, 64, -9.0, 5.0, 3)
    D4 = B.Mats3dDesc(0.15, 11, 1.0, reg, rule, rule, stack, stack, p, 20, None, None, 1, 0.0, None, None, None)
    assert h(C.byref(D4), 4, p, p, 2, p, 0, p, None, None) == B.DFRG_EINVAL     # n_jext < 1
    assert h(C.byref(D4), 4, p, p, 2, p, 60, p, None, None) == B.DFRG_EINVAL    # needs rows up to 60-1+11 > 63
    D4.T = 0.0
    assert h(C.byref(D4), 4, p, p, 2, p, 4, p, None, None) == B.DFRG_EINVAL     # T must be > 0
    D4.T = 0.15
    D4.n_coef = 19
    assert h(C.byref(D4), 4, p, p, 2, p, 4, p, None, None) == B.DFRG_EINVAL


def test_no_cpu_fallback_without_gpu(lib):
    """On a box without a GPU a well-formed call must fail loudly (DFRG_ECUDA / EUNSUPPORTED), never compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    x, w = B.dfrg_quad_nodes(8, 0.0, 6.0)
    rho = np.linspace(0, 2, 4)
    flow = np.full(4, np.nan)
    with pytest.raises(B.DfrgError):
        B.dfrg_integrate_lpa_host(4, 0.0, 0, 1, 4.0, 1.0, B.REG_EXP_POLY, 1, 1.0, (x, w), rho, rho.copy(), rho.copy(), flow)
    assert np.all(np.isnan(flow))


def test_matsubara_n_max_domains(lib):
    """Quadraturex0 (domain scales with k) and Quadratureq0 (fixed domain); BASELINE.json's
    N_max = ceil(6k/(2 pi T)) = 20, 10, 5, 2 for T/k = 0.05, 0.1, 0.2, 0.5 and ceil(10k/(2 pi T)) = 11 for T = 0.15k."""
    for T, want in ((0.05, 20), (0.1, 10), (0.2, 5), (0.5, 2)):
        assert B.dfrg_matsubara_n_max(B.DOMAIN_X0, T, 1.0, 6.0) == want
        assert B.dfrg_matsubara_n_max(B.DOMAIN_X0, 1.7 * T, 1.7, 6.0) == want      # scales with k
        assert B.dfrg_matsubara_n_max(B.DOMAIN_Q0, T, 1.0, 6.0) == want
        assert B.dfrg_matsubara_n_max(B.DOMAIN_Q0, T, 0.01, 6.0) == want            # fixed domain: independent of k
    assert B.dfrg_matsubara_n_max(B.DOMAIN_X0, 0.15, 1.0, 10.0) == 11
    assert B.dfrg_matsubara_n_max(B.DOMAIN_Q0, 0.15, 1.0, 0.0) == 0
    for bad in ((0, 0.0, 1.0, 6.0), (0, 0.1, 0.0, 6.0), (0, 0.1, 1.0, -1.0), (5, 0.1, 1.0, 6.0), (1, 1e-12, 1.0, 1e3)):
        assert lib.dfrg_matsubara_n_max(*bad) == B.DFRG_EINVAL
    from paper_2412_13043_b200 import inputs
    for T in inputs.CONFIG1_TEMPERATURES:
        assert inputs.config1(T)["n_max"] == B.dfrg_matsubara_n_max(B.DOMAIN_X0, T, 1.0, 6.0)
    assert inputs.config4()["n_max"] == B.dfrg_matsubara_n_max(B.DOMAIN_X0, 0.15, 1.0, 10.0)


def test_constant_tables_are_what_the_generator_writes():
    """csrc/fm_tables.inc (the constants of the device log / exp) is generated: regenerate and compare, and check two entries
    against closed forms (mpmath)."""
    import subprocess
    import sys
    import mpmath as mp
    gen = os.path.join(ROOT, "paper_2412_13043_b200", "csrc", "gen_fm_tables.py")
    assert subprocess.run([sys.executable, gen, "--check"]).returncode == 0
    txt = open(os.path.join(ROOT, "paper_2412_13043_b200", "csrc", "fm_tables.inc")).read()
    body = txt.split("kFmExp[64] = {")[1].split("}")[0]
    vals = [float.fromhex(t.strip()) for t in body.split(",") if t.strip()]
    mp.mp.dps = 40
    assert len(vals) == 64 and vals[0] == 1.0 and vals[32] == float(mp.sqrt(2))
    body = txt.split("kLg2Log[1024] = {")[1].split("}")[0]
    vals = [float.fromhex(t.strip()) for t in body.split(",") if t.strip()]
    assert len(vals) == 1024
    for j in (0, 255, 511):
        inv = 1.0 / (1.0 + (j + 0.5) / 512.0)
        assert vals[2 * j] == inv and vals[2 * j + 1] == float(mp.log(mp.mpf(inv)))
