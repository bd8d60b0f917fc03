"""ctypes wrapper around oracle/dfrg_oracle.cpp (test infrastructure; see oracle/__init__.py)."""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dfrg_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

REG_LITIM = 0
REG_EXP_POLY = 1

_lib = None


def build(force=False):
    """g++ -O2 -fopenmp; no fast-math (libm exp/log, IEEE order of operations)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c++17", "-ffp-contract=off",
               "-o", _LIB, _SRC]
        subprocess.check_call(cmd)
    return _LIB


_dp = C.POINTER(C.c_double)
_lp = C.POINTER(C.c_longlong)


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _arr(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_table_lookup.restype = C.c_double
        _lib.orc_table_lookup.argtypes = [_dp, C.c_int, C.c_double, C.c_double, C.c_int, C.c_double]
        _lib.orc_regulator.restype = None
        _lib.orc_regulator.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, _dp, _dp]
        _lib.orc_regulator_fermion.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, _dp, _dp]
        _lib.orc_gl_rule.argtypes = [C.c_int, C.c_double, C.c_double, _dp, _dp]
        _lib.orc_lpa.argtypes = [C.c_int, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double,
                                 C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                 C.c_int, _dp, _dp, C.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        _lib.orc_loop4d_twopoint.argtypes = [C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                             C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                             _dp, C.c_int, C.c_double, C.c_double, C.c_int,
                                             _dp, C.c_int, C.c_int, _dp, C.c_int, _dp,
                                             C.c_longlong, _lp, _dp, _dp, _dp]
        _lib.orc_loop4d_threepoint.argtypes = [C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                               C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                               C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                               _dp, _dp, _dp, C.c_int, C.c_double, C.c_double, C.c_int,
                                               _dp, C.c_int, C.c_int, _dp,
                                               C.c_longlong, _lp, C.c_int, _dp, _dp, _dp]
        _lib.orc_lpa_fermion.argtypes = [C.c_int, C.c_double, C.c_int, C.c_double, C.c_double,
                                         C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                         C.c_int, _dp, _dp, C.c_int, _dp, _dp, _dp, _dp, _dp, _dp]
        _ip = C.POINTER(C.c_int)
        _lib.orc_table3d_lookup.restype = C.c_double
        _lib.orc_table3d_lookup.argtypes = [_dp, _ip, _dp, _dp, _ip, C.c_double, C.c_double, C.c_double]
        _lib.orc_vertex_coords.restype = None
        _lib.orc_vertex_coords.argtypes = [C.c_double, C.c_double, C.c_double, _dp, _dp, _dp]
        _lib.orc_loop4d_threepoint_tab3d.argtypes = [C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                                     C.c_int, _dp, _dp, C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                                     C.c_int, _dp,
                                                     _dp, C.c_int, C.c_double, C.c_double, C.c_int,
                                                     _dp, _ip, _dp, _dp, _ip,
                                                     _dp, C.c_int, C.c_int, _dp,
                                                     C.c_longlong, _lp, _dp, _dp, _dp]
        _lib.orc_loop4d_fourpoint.argtypes = [C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                              C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                              C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                              _dp, _dp, _dp, C.c_int, C.c_double, C.c_double, C.c_int,
                                              _dp, C.c_int, C.c_int, _dp,
                                              C.c_longlong, _lp, _dp, _dp, _dp]
        _lib.orc_matsubara3d.argtypes = [C.c_double, C.c_int, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                         C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                         _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int,
                                         _dp, C.c_int, C.c_int, _dp, _dp, C.c_int, _dp, C.c_int,
                                         C.c_longlong, _lp, _dp, _dp, _dp]
        _lib.orc_matsubara3d_mu.argtypes = [C.c_double, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double,
                                            C.c_double, C.c_double, C.c_int,
                                            C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                            _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int,
                                            _dp, C.c_int, C.c_int, _dp, _dp, C.c_int, _dp, C.c_int,
                                            C.c_longlong, _lp, _dp, _dp, _dp, _dp]
        _lib.orc_matsubara3d_mu_dm2.argtypes = [C.c_double, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double,
                                                C.c_double, C.c_double, C.c_int,
                                                C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                                _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int,
                                                _dp, C.c_int, C.c_int, _dp, _dp, C.c_int, _dp, C.c_int,
                                                C.c_longlong, _lp, _dp, _dp, _dp, _dp, _dp, _dp]
        _lib.orc_lpa_dm2.argtypes = [C.c_int, C.c_double, C.c_int, C.c_int, C.c_double,
                                     C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                     C.c_int, _dp, _dp, C.c_int, _dp, _dp, _dp, _dp, _dp]
        _lib.orc_loop4d_twopoint_dm2.argtypes = [C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                                 C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                                 _dp, C.c_int, C.c_double, C.c_double, C.c_int,
                                                 _dp, C.c_int, C.c_int, _dp, C.c_int, _dp,
                                                 C.c_longlong, _lp, _dp, _dp]
        _lib.orc_matsubara3d_dm2.argtypes = [C.c_double, C.c_int, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                             C.c_int, _dp, _dp, C.c_int, _dp, _dp,
                                             _dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int,
                                             _dp, C.c_int, C.c_int, _dp, _dp, C.c_int, _dp, C.c_int,
                                             C.c_longlong, _lp, _dp, _dp, _dp, _dp]
    return _lib


def num_threads():
    return int(_load().orc_num_threads())


def set_num_threads(n):
    _load().orc_set_num_threads(int(n))


def gl_rule(n, a, b):
    x = np.empty(n)
    w = np.empty(n)
    rc = _load().orc_gl_rule(int(n), float(a), float(b), _d(x), _d(w))
    if rc:
        raise ValueError("orc_gl_rule: bad arguments")
    return x, w


def regulator(kind, order, k, s, zk=1.0, eta=0.0):
    R = C.c_double()
    Rd = C.c_double()
    _load().orc_regulator(int(kind), int(order), float(k), float(zk), float(eta), float(s), C.byref(R), C.byref(Rd))
    return R.value, Rd.value


def regulator_fermion(kind, order, k, s, zk=1.0, eta=0.0):
    """(RF, RFdot) of reading A25 at the squared momentum s."""
    R = C.c_double()
    Rd = C.c_double()
    _load().orc_regulator_fermion(int(kind), int(order), float(k), float(zk), float(eta), float(s), C.byref(R), C.byref(Rd))
    return R.value, Rd.value


def table_lookup(v, lnq_lo, lnq_hi, interp, s):
    v = _arr(v)
    return float(_load().orc_table_lookup(_d(v), int(v.size), float(lnq_lo), float(lnq_hi), int(interp), float(s)))


def _sel(sel):
    if sel is None:
        return 0, None, None
    sel = np.ascontiguousarray(sel, dtype=np.int64)
    return int(sel.size), sel.ctypes.data_as(_lp), sel


def lpa(d, T, n_max, reg_arg4d, N, prefactor, reg_kind, reg_order, k, xq, wq, rho, u, du, want_sens=False, zk=1.0, eta=0.0):
    """Returns (flow[n_field], chan[2, n_field], dmin[n_field]) (+ sens[2, n_field] if want_sens)."""
    xq, wq, rho, u, du = map(_arr, (xq, wq, rho, u, du))
    nf = rho.size
    flow = np.empty(nf)
    chan = np.empty((2, nf))
    dmin = np.empty(nf)
    sens = np.empty((2, nf))
    rc = _load().orc_lpa(int(d), float(T), int(n_max), int(reg_arg4d), float(N), float(prefactor),
                         int(reg_kind), int(reg_order), float(k), float(zk), float(eta), int(xq.size), _d(xq), _d(wq),
                         int(nf), _d(rho), _d(u), _d(du), _d(flow), _d(chan), _d(dmin), _d(sens))
    if rc:
        raise ValueError("orc_lpa: bad arguments")
    return (flow, chan, dmin, sens) if want_sens else (flow, chan, dmin)


def lpa_fermion(d, T, n_max, mu, prefactor, reg_kind, reg_order, k, xq, wq, m2, zk=1.0, eta=0.0, freg=0):
    """Fermionic LPA loop at chemical potential mu (spatial regulator).  Returns (I, dI, dmin, sens, sens_d), each [m2.size]."""
    xq, wq, m2 = map(_arr, (xq, wq, m2))
    I, dI, dmin, sens, sens_d = (np.empty(m2.shape) for _ in range(5))
    rc = _load().orc_lpa_fermion(int(d), float(T), int(n_max), float(mu), float(prefactor),
                                 int(reg_kind), int(reg_order), float(k), float(zk), float(eta), int(freg),
                                 int(xq.size), _d(xq), _d(wq), int(m2.size), _d(m2),
                                 _d(I), _d(dI), _d(dmin), _d(sens), _d(sens_d))
    if rc:
        raise ValueError("orc_lpa_fermion: bad arguments")
    return I, dI, dmin, sens, sens_d


def loop4d_twopoint(prefactor, reg_kind, reg_order, k, xq, wq, xc, wc, Z, lnq_lo, lnq_hi, interp,
                    coef, m2, pext, sel=None, want_sens=False, zk=1.0, eta=0.0):
    """Returns (out, dmin): shape [n_ext, n_field], or [n_sel] for flat indices e*n_field+f in sel."""
    xq, wq, xc, wc, Z, coef, m2, pext = map(_arr, (xq, wq, xc, wc, Z, coef, m2, pext))
    ns, selp, _keep = _sel(sel)
    shape = (ns,) if sel is not None else (pext.size, m2.size)
    out = np.empty(shape)
    dmin = np.empty(shape)
    sens = np.empty(shape)
    rc = _load().orc_loop4d_twopoint(float(prefactor), int(reg_kind), int(reg_order), float(k), float(zk), float(eta),
                                     int(xq.size), _d(xq), _d(wq), int(xc.size), _d(xc), _d(wc),
                                     _d(Z), int(Z.size), float(lnq_lo), float(lnq_hi), int(interp),
                                     _d(coef), int(coef.size), int(m2.size), _d(m2), int(pext.size), _d(pext),
                                     ns, selp, _d(out), _d(dmin), _d(sens))
    if rc:
        raise ValueError("orc_loop4d_twopoint: bad arguments")
    return (out, dmin, sens) if want_sens else (out, dmin)


def loop4d_threepoint(prefactor, reg_kind, reg_order, k, xq, wq, x1, w1, x2, w2, xphi, wphi,
                      ZA, Zc, L3, lnq_lo, lnq_hi, interp, coef, ext, sel=None, literal_phi=False, want_sens=False, zk=1.0, eta=0.0):
    """ext: [n_ext, 3] = (|p1|, |p2|, alpha).  Returns (out[n_ext or n_sel], dmin)."""
    xq, wq, x1, w1, x2, w2, xphi, wphi, ZA, Zc, L3, coef, ext = map(
        _arr, (xq, wq, x1, w1, x2, w2, xphi, wphi, ZA, Zc, L3, coef, ext))
    n_ext = ext.size // 3
    ns, selp, _keep = _sel(sel)
    n_out = ns if sel is not None else n_ext
    out = np.empty(n_out)
    dmin = np.empty(n_out)
    sens = np.empty(n_out)
    rc = _load().orc_loop4d_threepoint(float(prefactor), int(reg_kind), int(reg_order), float(k), float(zk), float(eta),
                                       int(xq.size), _d(xq), _d(wq), int(x1.size), _d(x1), _d(w1),
                                       int(x2.size), _d(x2), _d(w2), int(xphi.size), _d(xphi), _d(wphi),
                                       _d(ZA), _d(Zc), _d(L3), int(ZA.size), float(lnq_lo), float(lnq_hi),
                                       int(interp), _d(coef), int(coef.size), int(n_ext), _d(ext),
                                       ns, selp, int(bool(literal_phi)), _d(out), _d(dmin), _d(sens))
    if rc:
        raise ValueError("orc_loop4d_threepoint: bad arguments")
    return (out, dmin, sens) if want_sens else (out, dmin)


def _tab3d(v3, lo3, hi3, log3):
    v3 = _arr(v3)
    assert v3.ndim == 3
    n3 = np.ascontiguousarray(v3.shape, dtype=np.int32)
    lo3, hi3 = _arr(lo3), _arr(hi3)
    log3 = np.ascontiguousarray(log3, dtype=np.int32)
    ip = lambda a: a.ctypes.data_as(C.POINTER(C.c_int))
    return v3, n3, lo3, hi3, log3, (_d(v3), ip(n3), _d(lo3), _d(hi3), ip(log3))


def table3d_lookup(v3, lo3, hi3, log3, x0, x1, x2):
    """Trilinear look-up in a 3-D table v3[n0, n1, n2]; logarithmic axes take the squared momentum."""
    *_keep, args = _tab3d(v3, lo3, hi3, log3)
    return float(_load().orc_table3d_lookup(*args, float(x0), float(x1), float(x2)))


def vertex_coords(k1sq, k2sq, k3sq):
    """(S0^2, a, s) of a three-point function with squared leg momenta k1sq, k2sq, k3sq."""
    S, a, s = C.c_double(), C.c_double(), C.c_double()
    _load().orc_vertex_coords(float(k1sq), float(k2sq), float(k3sq), C.byref(S), C.byref(a), C.byref(s))
    return S.value, a.value, s.value


def loop4d_threepoint_tab3d(prefactor, reg_kind, reg_order, k, xq, wq, x1, w1, x2, w2, wphi, ZA, lnq_lo, lnq_hi, interp,
                            v3, lo3, hi3, log3, coef, ext, sel=None, want_sens=False, zk=1.0, eta=0.0):
    """Three-point loop with the vertex dressing from a 3-D table l3(S0^2, a, s).  Returns (out, dmin[, sens])."""
    xq, wq, x1, w1, x2, w2, wphi, ZA, coef, ext = map(_arr, (xq, wq, x1, w1, x2, w2, wphi, ZA, coef, ext))
    *_keep, targs = _tab3d(v3, lo3, hi3, log3)
    n_ext = ext.size // 3
    ns, selp, _keep2 = _sel(sel)
    n_out = ns if sel is not None else n_ext
    out, dmin, sens = np.empty(n_out), np.empty(n_out), np.empty(n_out)
    rc = _load().orc_loop4d_threepoint_tab3d(float(prefactor), int(reg_kind), int(reg_order), float(k), float(zk),
                                             float(eta), int(xq.size), _d(xq), _d(wq), int(x1.size), _d(x1), _d(w1),
                                             int(x2.size), _d(x2), _d(w2), int(wphi.size), _d(wphi),
                                             _d(ZA), int(ZA.size), float(lnq_lo), float(lnq_hi), int(interp),
                                             *targs, _d(coef), int(coef.size), int(n_ext), _d(ext),
                                             ns, selp, _d(out), _d(dmin), _d(sens))
    if rc:
        raise ValueError("orc_loop4d_threepoint_tab3d: bad arguments")
    return (out, dmin, sens) if want_sens else (out, dmin)


def loop4d_fourpoint(prefactor, reg_kind, reg_order, k, xq, wq, x1, w1, x2, w2, xphi, wphi,
                     ZA, Zc, L3, lnq_lo, lnq_hi, interp, coef, ext, sel=None, want_sens=False, zk=1.0, eta=0.0):
    """ext: [n_ext, 6] = (|p1|, |p2|, |p3|, alpha, beta, gamma); coef: 70 = [gluon box | ghost box].
    Returns (out[n_ext or n_sel], dmin)."""
    xq, wq, x1, w1, x2, w2, xphi, wphi, ZA, Zc, L3, coef, ext = map(
        _arr, (xq, wq, x1, w1, x2, w2, xphi, wphi, ZA, Zc, L3, coef, ext))
    n_ext = ext.size // 6
    ns, selp, _keep = _sel(sel)
    n_out = ns if sel is not None else n_ext
    out = np.empty(n_out)
    dmin = np.empty(n_out)
    sens = np.empty(n_out)
    rc = _load().orc_loop4d_fourpoint(float(prefactor), int(reg_kind), int(reg_order), float(k), float(zk), float(eta),
                                      int(xq.size), _d(xq), _d(wq), int(x1.size), _d(x1), _d(w1),
                                      int(x2.size), _d(x2), _d(w2), int(xphi.size), _d(xphi), _d(wphi),
                                      _d(ZA), _d(Zc), _d(L3), int(ZA.size), float(lnq_lo), float(lnq_hi),
                                      int(interp), _d(coef), int(coef.size), int(n_ext), _d(ext),
                                      ns, selp, _d(out), _d(dmin), _d(sens))
    if rc:
        raise ValueError("orc_loop4d_fourpoint: bad arguments")
    return (out, dmin, sens) if want_sens else (out, dmin)


def matsubara3d(T, n_max, prefactor, reg_kind, reg_order, k, xq, wq, xc, wc, Zpsi, Zphi,
                lnq_lo, lnq_hi, interp, coef, m2psi, m2phi, pext, n_jext, sel=None, want_sens=False, zk=1.0, eta=0.0, freg=0):
    """Zpsi, Zphi: [n_freq, n_q].  Returns (out, dmin): [n_p, n_jext, n_field] or [n_sel]
    for flat indices (e*n_jext + j)*n_field + f in sel."""
    xq, wq, xc, wc, Zpsi, Zphi, coef, m2psi, m2phi, pext = map(
        _arr, (xq, wq, xc, wc, Zpsi, Zphi, coef, m2psi, m2phi, pext))
    assert Zpsi.ndim == 2 and Zpsi.shape == Zphi.shape
    nfreq, tnq = Zpsi.shape
    ns, selp, _keep = _sel(sel)
    shape = (ns,) if sel is not None else (pext.size, int(n_jext), m2psi.size)
    out = np.empty(shape)
    dmin = np.empty(shape)
    sens = np.empty(shape)
    rc = _load().orc_matsubara3d(float(T), int(n_max), float(prefactor), int(reg_kind), int(reg_order), float(k), float(zk), float(eta), int(freg),
                                 int(xq.size), _d(xq), _d(wq), int(xc.size), _d(xc), _d(wc),
                                 _d(Zpsi), _d(Zphi), int(tnq), int(nfreq), float(lnq_lo), float(lnq_hi), int(interp),
                                 _d(coef), int(coef.size), int(m2psi.size), _d(m2psi), _d(m2phi),
                                 int(pext.size), _d(pext), int(n_jext), ns, selp, _d(out), _d(dmin), _d(sens))
    if rc:
        raise ValueError("orc_matsubara3d: bad arguments")
    return (out, dmin, sens) if want_sens else (out, dmin)


def matsubara3d_mu(T, n_max, mu, prefactor, reg_kind, reg_order, k, xq, wq, xc, wc, Zpsi, Zphi,
                   lnq_lo, lnq_hi, interp, coef, m2psi, m2phi, pext, n_jext, sel=None, want_sens=False, zk=1.0, eta=0.0, freg=0):
    """Matsubara family at chemical potential mu with spatial regulators.  Returns (out complex128, dmin[, sens])."""
    xq, wq, xc, wc, Zpsi, Zphi, coef, m2psi, m2phi, pext = map(
        _arr, (xq, wq, xc, wc, Zpsi, Zphi, coef, m2psi, m2phi, pext))
    nfreq, tnq = Zpsi.shape
    ns, selp, _keep = _sel(sel)
    shape = (ns,) if sel is not None else (pext.size, int(n_jext), m2psi.size)
    o_re, o_im, dmin, sens = (np.empty(shape) for _ in range(4))
    rc = _load().orc_matsubara3d_mu(float(T), int(n_max), float(mu), float(prefactor), int(reg_kind), int(reg_order),
                                    float(k), float(zk), float(eta), int(freg),
                                    int(xq.size), _d(xq), _d(wq), int(xc.size), _d(xc), _d(wc),
                                    _d(Zpsi), _d(Zphi), int(tnq), int(nfreq), float(lnq_lo), float(lnq_hi), int(interp),
                                    _d(coef), int(coef.size), int(m2psi.size), _d(m2psi), _d(m2phi),
                                    int(pext.size), _d(pext), int(n_jext), ns, selp, _d(o_re), _d(o_im), _d(dmin),
                                    _d(sens))
    if rc:
        raise ValueError("orc_matsubara3d_mu: bad arguments")
    out = o_re + 1j * o_im
    return (out, dmin, sens) if want_sens else (out, dmin)


def matsubara3d_mu_dm2(T, n_max, mu, prefactor, reg_kind, reg_order, k, xq, wq, xc, wc, Zpsi, Zphi,
                       lnq_lo, lnq_hi, interp, coef, m2psi, m2phi, pext, n_jext, sel=None, zk=1.0, eta=0.0, freg=0):
    """Mass derivatives of matsubara3d_mu.  Returns (dpsi, dphi, sens_psi, sens_phi), dpsi / dphi complex128."""
    xq, wq, xc, wc, Zpsi, Zphi, coef, m2psi, m2phi, pext = map(
        _arr, (xq, wq, xc, wc, Zpsi, Zphi, coef, m2psi, m2phi, pext))
    nfreq, tnq = Zpsi.shape
    ns, selp, _keep = _sel(sel)
    shape = (ns,) if sel is not None else (pext.size, int(n_jext), m2psi.size)
    a_re, a_im, b_re, b_im, sa, sb = (np.empty(shape) for _ in range(6))
    rc = _load().orc_matsubara3d_mu_dm2(float(T), int(n_max), float(mu), float(prefactor), int(reg_kind),
                                        int(reg_order), float(k), float(zk), float(eta), int(freg),
                                        int(xq.size), _d(xq), _d(wq), int(xc.size), _d(xc), _d(wc),
                                        _d(Zpsi), _d(Zphi), int(tnq), int(nfreq), float(lnq_lo), float(lnq_hi),
                                        int(interp), _d(coef), int(coef.size), int(m2psi.size), _d(m2psi), _d(m2phi),
                                        int(pext.size), _d(pext), int(n_jext), ns, selp,
                                        _d(a_re), _d(a_im), _d(b_re), _d(b_im), _d(sa), _d(sb))
    if rc:
        raise ValueError("orc_matsubara3d_mu_dm2: bad arguments")
    return a_re + 1j * a_im, b_re + 1j * b_im, sa, sb


# ---- mass derivatives (Jacobian support) ------------------------------------------------------------
def lpa_dm2(d, T, n_max, reg_arg4d, prefactor, reg_kind, reg_order, k, xq, wq, rho, u, du, zk=1.0, eta=0.0):
    """Returns (dchan[2, n_field], sens[2, n_field]): dI/dm2 at the pion and sigma masses."""
    xq, wq, rho, u, du = map(_arr, (xq, wq, rho, u, du))
    nf = rho.size
    dchan = np.empty((2, nf))
    sens = np.empty((2, nf))
    rc = _load().orc_lpa_dm2(int(d), float(T), int(n_max), int(reg_arg4d), float(prefactor),
                             int(reg_kind), int(reg_order), float(k), float(zk), float(eta), int(xq.size), _d(xq), _d(wq),
                             int(nf), _d(rho), _d(u), _d(du), _d(dchan), _d(sens))
    if rc:
        raise ValueError("orc_lpa_dm2: bad arguments")
    return dchan, sens


def loop4d_twopoint_dm2(prefactor, reg_kind, reg_order, k, xq, wq, xc, wc, Z, lnq_lo, lnq_hi, interp,
                        coef, m2, pext, sel=None, zk=1.0, eta=0.0):
    """Returns (dout, sens): d out[e][f] / d m2[f], shape [n_ext, n_field] or [n_sel]."""
    xq, wq, xc, wc, Z, coef, m2, pext = map(_arr, (xq, wq, xc, wc, Z, coef, m2, pext))
    ns, selp, _keep = _sel(sel)
    shape = (ns,) if sel is not None else (pext.size, m2.size)
    dout = np.empty(shape)
    sens = np.empty(shape)
    rc = _load().orc_loop4d_twopoint_dm2(float(prefactor), int(reg_kind), int(reg_order), float(k), float(zk), float(eta),
                                         int(xq.size), _d(xq), _d(wq), int(xc.size), _d(xc), _d(wc),
                                         _d(Z), int(Z.size), float(lnq_lo), float(lnq_hi), int(interp),
                                         _d(coef), int(coef.size), int(m2.size), _d(m2), int(pext.size), _d(pext),
                                         ns, selp, _d(dout), _d(sens))
    if rc:
        raise ValueError("orc_loop4d_twopoint_dm2: bad arguments")
    return dout, sens


def matsubara3d_dm2(T, n_max, prefactor, reg_kind, reg_order, k, xq, wq, xc, wc, Zpsi, Zphi,
                    lnq_lo, lnq_hi, interp, coef, m2psi, m2phi, pext, n_jext, sel=None, zk=1.0, eta=0.0, freg=0):
    """Returns (dpsi, dphi, sens_psi, sens_phi): d out / d m2_psi[f] and d out / d m2_phi[f]."""
    xq, wq, xc, wc, Zpsi, Zphi, coef, m2psi, m2phi, pext = map(
        _arr, (xq, wq, xc, wc, Zpsi, Zphi, coef, m2psi, m2phi, pext))
    nfreq, tnq = Zpsi.shape
    ns, selp, _keep = _sel(sel)
    shape = (ns,) if sel is not None else (pext.size, int(n_jext), m2psi.size)
    dpsi, dphi, spsi, sphi = (np.empty(shape) for _ in range(4))
    rc = _load().orc_matsubara3d_dm2(float(T), int(n_max), float(prefactor), int(reg_kind), int(reg_order), float(k), float(zk), float(eta), int(freg),
                                     int(xq.size), _d(xq), _d(wq), int(xc.size), _d(xc), _d(wc),
                                     _d(Zpsi), _d(Zphi), int(tnq), int(nfreq), float(lnq_lo), float(lnq_hi),
                                     int(interp), _d(coef), int(coef.size), int(m2psi.size), _d(m2psi), _d(m2phi),
                                     int(pext.size), _d(pext), int(n_jext), ns, selp, _d(dpsi), _d(dphi), _d(spsi),
                                     _d(sphi))
    if rc:
        raise ValueError("orc_matsubara3d_dm2: bad arguments")
    return dpsi, dphi, spsi, sphi
