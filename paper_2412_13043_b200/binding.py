"""Thin ctypes binding of the C ABI in include/dfrg.h -- argument marshalling only.

Same names as the C entry points.  Device entry points take torch CUDA tensors (float64,
contiguous) and enqueue on torch's current stream; `*_host` entry points take numpy arrays or
pinned CPU tensors.  There is no CPU fallback: if libdfrg.so is missing or a call fails, it raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdfrg.so")

DFRG_OK, DFRG_EINVAL, DFRG_EUNSUPPORTED, DFRG_ECUDA, DFRG_ENOMEM, DFRG_ESCRATCH = 0, -1, -2, -3, -4, -5
NOALLOC_SCRATCH_BYTES = 8 * 1024 * 1024   # DFRG_NOALLOC_SCRATCH_BYTES of include/dfrg.h
REG_LITIM, REG_EXP_POLY = 0, 1
STAT_BOSON, STAT_FERMION = 0, 1
DOMAIN_X0, DOMAIN_Q0 = 0, 1
LOOP_TWOPOINT, LOOP_THREEPOINT, LOOP_FOURPOINT, LOOP_THREEPOINT_TAB3D = 0, 1, 2, 3
# dfrg_mats3d_desc::path bits (kernel-path selection; 0 = the library's own choice)
M3_AUTO, M3_ROW_STREAMING, M3_ANY_SHAPE, M3_PLAIN_MOMENTS, M3_ONE_FIELD, M3_GROUPS_4, M3_GROUPS_7 = 0, 1, 2, 4, 8, 16, 32
RULE_GAUSS_LEGENDRE = 0

EXPORTS = (
    "dfrg_strerror", "dfrg_last_cuda_error", "dfrg_version", "dfrg_shutdown", "dfrg_quad_nodes",
    "dfrg_matsubara_n_max",
    "dfrg_integrate_lpa", "dfrg_integrate_lpa_host", "dfrg_integrate_lpa_batch", "dfrg_integrate_lpa_batch_host",
    "dfrg_integrate_loop4d", "dfrg_integrate_loop4d_host", "dfrg_integrate_twopoint_noalloc",
    "dfrg_integrate_matsubara3d", "dfrg_integrate_matsubara3d_host",
)

_vp = C.c_void_p


class Regulator(C.Structure):
    _fields_ = [("kind", C.c_int), ("order", C.c_int), ("k", C.c_double), ("zk", C.c_double), ("eta", C.c_double)]


class Rule(C.Structure):
    _fields_ = [("x", _vp), ("w", _vp), ("n", C.c_int)]


class Table(C.Structure):
    _fields_ = [("v", _vp), ("n_q", C.c_int), ("n_freq", C.c_int), ("lnq_lo", C.c_double), ("lnq_hi", C.c_double),
                ("interp", C.c_int)]


class Table3D(C.Structure):
    _fields_ = [("v", _vp), ("n", C.c_int * 3), ("lo", C.c_double * 3), ("hi", C.c_double * 3), ("is_log", C.c_int * 3)]


class LpaDesc(C.Structure):
    _fields_ = [("d", C.c_int), ("T", C.c_double), ("n_max", C.c_int), ("reg_arg4d", C.c_int), ("N", C.c_double),
                ("prefactor", C.c_double), ("reg", Regulator), ("q", Rule), ("dchan", _vp),
                ("statistics", C.c_int), ("mu", C.c_double), ("fermion_reg", C.c_int)]


class Loop4dDesc(C.Structure):
    _fields_ = [("family", C.c_int), ("prefactor", C.c_double), ("reg", Regulator),
                ("q", Rule), ("cos1", Rule), ("cos2", Rule), ("phi", Rule),
                ("tab", Table * 3), ("coef", _vp), ("n_coef", C.c_int), ("ext_outer", C.c_int),
                ("dout_dm2", _vp), ("tab3d", Table3D)]


class Mats3dDesc(C.Structure):
    _fields_ = [("T", C.c_double), ("n_max", C.c_int), ("prefactor", C.c_double), ("reg", Regulator),
                ("q", Rule), ("cos1", Rule), ("tab_psi", Table), ("tab_phi", Table),
                ("coef", _vp), ("n_coef", C.c_int), ("dout_dm2_psi", _vp), ("dout_dm2_phi", _vp),
                ("reg_arg4d", C.c_int), ("mu", C.c_double), ("out_im", _vp),
                ("dout_dm2_psi_im", _vp), ("dout_dm2_phi_im", _vp), ("path", C.c_int), ("fermion_reg", C.c_int)]


class DfrgError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = lib().dfrg_strerror(status).decode()
        if status == DFRG_ECUDA:
            msg += " [cudaError %d]" % lib().dfrg_last_cuda_error()
        super().__init__("%s: %s (%d)" % (where, msg, status))


_lib = None


def lib():
    """Loads libdfrg.so (built by `python -m paper_2412_13043_b200.build`); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libdfrg.so not built: run `python -m paper_2412_13043_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.dfrg_strerror.restype = C.c_char_p
        L.dfrg_strerror.argtypes = [C.c_int]
        L.dfrg_shutdown.restype = None
        L.dfrg_matsubara_n_max.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
        L.dfrg_quad_nodes.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, _vp, _vp]
        L.dfrg_integrate_lpa.argtypes = [C.POINTER(LpaDesc), C.c_int, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
        L.dfrg_integrate_lpa_host.argtypes = [C.POINTER(LpaDesc), C.c_int, _vp, _vp, _vp, _vp, _vp, _vp]
        L.dfrg_integrate_lpa_batch.argtypes = [C.POINTER(LpaDesc), C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_int,
                                               _vp, _vp, _vp, _vp, _vp, _vp, _vp]
        L.dfrg_integrate_lpa_batch_host.argtypes = [C.POINTER(LpaDesc), C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int),
                                                    C.c_int, _vp, _vp, _vp, _vp, _vp, _vp]
        L.dfrg_integrate_loop4d.argtypes = [C.POINTER(Loop4dDesc), C.c_int, _vp, C.c_int, _vp, _vp, _vp, _vp]
        L.dfrg_integrate_loop4d_host.argtypes = [C.POINTER(Loop4dDesc), C.c_int, _vp, C.c_int, _vp, _vp, _vp]
        L.dfrg_integrate_twopoint_noalloc.argtypes = [C.POINTER(Loop4dDesc), C.c_int, _vp, C.c_int, _vp, _vp, _vp, _vp]
        L.dfrg_integrate_matsubara3d.argtypes = [C.POINTER(Mats3dDesc), C.c_int, _vp, _vp, C.c_int, _vp, C.c_int,
                                                 _vp, _vp, _vp]
        L.dfrg_integrate_matsubara3d_host.argtypes = [C.POINTER(Mats3dDesc), C.c_int, _vp, _vp, C.c_int, _vp,
                                                      C.c_int, _vp, _vp]
        _lib = L
    return _lib


def _check(status, where):
    if status != DFRG_OK:
        raise DfrgError(status, where)


def _ptr(a, device):
    """Address of a float64 contiguous array: torch CUDA tensor (device=True) or numpy / CPU tensor."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if device:
            raise TypeError("device entry point got a numpy array")
        if a.dtype != np.float64 or not a.flags.c_contiguous:
            raise TypeError("need a contiguous float64 array")
        return a.ctypes.data
    import torch
    if not isinstance(a, torch.Tensor) or a.dtype != torch.float64 or not a.is_contiguous():
        raise TypeError("need a contiguous float64 tensor")
    if a.is_cuda != bool(device):
        raise TypeError("tensor is on the wrong side of the boundary (cuda=%s, expected %s)" % (a.is_cuda, device))
    return a.data_ptr()


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


def _rule(xw, device):
    if xw is None:
        return Rule(None, None, 0)
    x, w = xw
    return Rule(_ptr(x, device), _ptr(w, device), int(x.numel() if hasattr(x, "numel") else x.size))


def _table(v, lnq_lo, lnq_hi, interp, device):
    if v is None:
        return Table(None, 0, 0, 0.0, 0.0, 0)
    shape = tuple(v.shape)
    n_freq, n_q = (1, shape[0]) if len(shape) == 1 else shape
    return Table(_ptr(v, device), int(n_q), int(n_freq), float(lnq_lo), float(lnq_hi), int(interp))


# ---- S1 -------------------------------------------------------------------------------------------
def dfrg_quad_nodes(n, a, b, rule_kind=RULE_GAUSS_LEGENDRE):
    """Host-side Gauss-Legendre rule: returns (x, w) numpy arrays."""
    x = np.empty(max(int(n), 0))
    w = np.empty(max(int(n), 0))
    _check(lib().dfrg_quad_nodes(int(rule_kind), int(n), float(a), float(b), x.ctypes.data, w.ctypes.data),
           "dfrg_quad_nodes")
    return x, w


def dfrg_matsubara_n_max(domain, T, k, extent):
    """Number of Matsubara terms on either side for a time-direction cut-off (Quadraturex0 / Quadratureq0)."""
    n = lib().dfrg_matsubara_n_max(int(domain), float(T), float(k), float(extent))
    if n < 0:
        raise DfrgError(n, "dfrg_matsubara_n_max")
    return n


# ---- LPA ------------------------------------------------------------------------------------------
def _lpa_desc(d, T, n_max, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, device, dchan=None, reg_zk=1.0, reg_eta=0.0,
              statistics=STAT_BOSON, mu=0.0, fermion_reg=0):
    return LpaDesc(int(d), float(T), int(n_max), int(reg_arg4d), float(N), float(prefactor),
                   Regulator(int(reg_kind), int(reg_order), float(k), float(reg_zk), float(reg_eta)), _rule(rule_q, device),
                   _ptr(dchan, device), int(statistics), float(mu), int(fermion_reg))


def dfrg_integrate_lpa(d, T, n_max, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, rho, u, du,
                       flow, chan=None, dmin=None, dchan=None, reg_zk=1.0, reg_eta=0.0, statistics=STAT_BOSON, mu=0.0,
                       fermion_reg=0):
    """dchan (optional, [2, n_field]): dI/dm2 per channel (include/dfrg.h, "Mass derivatives")."""
    D = _lpa_desc(d, T, n_max, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, True, dchan, reg_zk, reg_eta, statistics, mu, fermion_reg)
    _check(lib().dfrg_integrate_lpa(C.byref(D), int(rho.numel()), _ptr(rho, True), _ptr(u, True), _ptr(du, True),
                                    _ptr(flow, True), _ptr(chan, True), _ptr(dmin, True), _stream()),
           "dfrg_integrate_lpa")
    return flow


def dfrg_integrate_lpa_batch(d, Ts, n_maxs, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, rho, u, du,
                             flow, chan=None, dmin=None, dchan=None, reg_zk=1.0, reg_eta=0.0, statistics=STAT_BOSON, mu=0.0,
                             fermion_reg=0):
    """Several temperatures in one launch: flow [n_T, n_field], chan / dchan [n_T, 2, n_field], dmin [n_T, n_field]."""
    n_T = len(Ts)
    assert len(n_maxs) == n_T
    D = _lpa_desc(d, 0.0, 0, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, True, dchan, reg_zk, reg_eta, statistics,
                  mu, fermion_reg)
    Tv = (C.c_double * n_T)(*[float(t) for t in Ts])
    nv = (C.c_int * n_T)(*[int(n) for n in n_maxs])
    _check(lib().dfrg_integrate_lpa_batch(C.byref(D), n_T, Tv, nv, int(rho.numel()), _ptr(rho, True), _ptr(u, True),
                                          _ptr(du, True), _ptr(flow, True), _ptr(chan, True), _ptr(dmin, True), _stream()),
           "dfrg_integrate_lpa_batch")
    return flow


def dfrg_integrate_lpa_batch_host(d, Ts, n_maxs, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, rho, u, du,
                                  flow, chan=None, dmin=None, dchan=None, reg_zk=1.0, reg_eta=0.0, statistics=STAT_BOSON, mu=0.0,
                                  fermion_reg=0):
    """dfrg_integrate_lpa_batch on host (numpy) arrays."""
    n_T = len(Ts)
    D = _lpa_desc(d, 0.0, 0, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, False, dchan, reg_zk, reg_eta, statistics,
                  mu, fermion_reg)
    Tv = (C.c_double * n_T)(*[float(t) for t in Ts])
    nv = (C.c_int * n_T)(*[int(n) for n in n_maxs])
    n_field = rho.numel() if hasattr(rho, "numel") else rho.size
    _check(lib().dfrg_integrate_lpa_batch_host(C.byref(D), n_T, Tv, nv, int(n_field), _ptr(rho, False), _ptr(u, False),
                                               _ptr(du, False), _ptr(flow, False), _ptr(chan, False), _ptr(dmin, False)),
           "dfrg_integrate_lpa_batch_host")
    return flow


def dfrg_integrate_lpa_host(d, T, n_max, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, rho, u, du,
                            flow, chan=None, dmin=None, dchan=None, reg_zk=1.0, reg_eta=0.0, statistics=STAT_BOSON, mu=0.0,
                       fermion_reg=0):
    D = _lpa_desc(d, T, n_max, reg_arg4d, N, prefactor, reg_kind, reg_order, k, rule_q, False, dchan, reg_zk, reg_eta, statistics, mu, fermion_reg)
    n_field = rho.numel() if hasattr(rho, "numel") else rho.size
    _check(lib().dfrg_integrate_lpa_host(C.byref(D), int(n_field), _ptr(rho, False), _ptr(u, False),
                                         _ptr(du, False), _ptr(flow, False), _ptr(chan, False), _ptr(dmin, False)),
           "dfrg_integrate_lpa_host")
    return flow


# ---- loop4d ---------------------------------------------------------------------------------------
def _loop4d_desc(family, prefactor, reg_kind, reg_order, k, rule_q, rule_c1, rule_c2, rule_phi, tabs, lnq_lo,
                 lnq_hi, interp, coef, device, ext_outer=0, dout_dm2=None, reg_zk=1.0, reg_eta=0.0, tab3d=None):
    T3 = Table * 3
    if tab3d is None:
        t3d = Table3D(None, (C.c_int * 3)(), (C.c_double * 3)(), (C.c_double * 3)(), (C.c_int * 3)())
    else:
        v3, lo3, hi3, log3 = tab3d
        t3d = Table3D(_ptr(v3, device), (C.c_int * 3)(*[int(x) for x in v3.shape]), (C.c_double * 3)(*map(float, lo3)),
                      (C.c_double * 3)(*map(float, hi3)), (C.c_int * 3)(*map(int, log3)))
    tt = [_table(t, lnq_lo, lnq_hi, interp, device) for t in tabs] + [_table(None, 0, 0, 0, device)] * (3 - len(tabs))
    n_coef = coef.numel() if hasattr(coef, "numel") else coef.size
    return Loop4dDesc(int(family), float(prefactor), Regulator(int(reg_kind), int(reg_order), float(k), float(reg_zk), float(reg_eta)),
                      _rule(rule_q, device), _rule(rule_c1, device), _rule(rule_c2, device), _rule(rule_phi, device),
                      T3(*tt), _ptr(coef, device), int(n_coef), int(ext_outer), _ptr(dout_dm2, device), t3d)


def _n(a):
    return 0 if a is None else int(a.numel() if hasattr(a, "numel") else a.size)


def dfrg_integrate_loop4d(family, prefactor, reg_kind, reg_order, k, rule_q, rule_c1, rule_c2, rule_phi, tabs,
                          lnq_lo, lnq_hi, interp, coef, m2, ext, out, dmin=None, ext_outer=0, dout_dm2=None, reg_zk=1.0, reg_eta=0.0, tab3d=None):
    """two-point: tabs=(Z,), m2=[n_field], ext=[n_ext] -> out [n_ext, n_field];
    three-point: tabs=(Z_A, Z_c, lambda3), m2=None, ext=[n_ext, 3] -> out [n_ext]; ext_outer: dfrg_loop4d_desc;
    four-point: tabs=(Z_A, Z_c, lambda3), m2=None, ext=[n_ext, 6], coef[70] -> out [n_ext];
    three-point with a 3-D vertex table: tabs=(Z_A,), tab3d=(v3[n0,n1,n2], lo3, hi3, is_log3), ext=[n_ext, 3]."""
    D = _loop4d_desc(family, prefactor, reg_kind, reg_order, k, rule_q, rule_c1, rule_c2, rule_phi, tabs, lnq_lo,
                     lnq_hi, interp, coef, True, ext_outer, dout_dm2, reg_zk, reg_eta, tab3d)
    n_ext = _n(ext) // {LOOP_TWOPOINT: 1, LOOP_THREEPOINT: 3, LOOP_FOURPOINT: 6, LOOP_THREEPOINT_TAB3D: 3}[family]
    _check(lib().dfrg_integrate_loop4d(C.byref(D), _n(m2), _ptr(m2, True), n_ext, _ptr(ext, True),
                                       _ptr(out, True), _ptr(dmin, True), _stream()), "dfrg_integrate_loop4d")
    return out


def dfrg_integrate_twopoint_noalloc(prefactor, reg_kind, reg_order, k, rule_q, rule_c1, Z, lnq_lo, lnq_hi, interp, coef,
                                    m2, ext, out, dmin=None, dout_dm2=None, reg_zk=1.0, reg_eta=0.0):
    """Two-point loop without any device allocation inside the library (include/dfrg.h, dfrg_integrate_twopoint_noalloc):
    for hosts that may not call cudaMalloc -- all memory owned by another allocator, allocation-lock-free threads, jobs
    under a memory cap.  The kernels' scratch is a fixed NOALLOC_SCRATCH_BYTES array inside libdfrg.so; a call that needs
    more raises DfrgError with status DFRG_ESCRATCH.  Same arguments and bit-identical results as the two-point case of
    dfrg_integrate_loop4d.  One array per device: do not let two such calls overlap on the GPU.  Make the first call on a
    device outside stream capture (it looks the array's address up)."""
    D = _loop4d_desc(LOOP_TWOPOINT, prefactor, reg_kind, reg_order, k, rule_q, rule_c1, None, None, (Z,), lnq_lo, lnq_hi,
                     interp, coef, True, 0, dout_dm2, reg_zk, reg_eta, None)
    _check(lib().dfrg_integrate_twopoint_noalloc(C.byref(D), _n(m2), _ptr(m2, True), _n(ext), _ptr(ext, True),
                                                 _ptr(out, True), _ptr(dmin, True), _stream()),
           "dfrg_integrate_twopoint_noalloc")
    return out


def dfrg_integrate_loop4d_host(family, prefactor, reg_kind, reg_order, k, rule_q, rule_c1, rule_c2, rule_phi, tabs,
                               lnq_lo, lnq_hi, interp, coef, m2, ext, out, dmin=None, ext_outer=0, dout_dm2=None, reg_zk=1.0, reg_eta=0.0, tab3d=None):
    D = _loop4d_desc(family, prefactor, reg_kind, reg_order, k, rule_q, rule_c1, rule_c2, rule_phi, tabs, lnq_lo,
                     lnq_hi, interp, coef, False, ext_outer, dout_dm2, reg_zk, reg_eta, tab3d)
    n_ext = _n(ext) // {LOOP_TWOPOINT: 1, LOOP_THREEPOINT: 3, LOOP_FOURPOINT: 6, LOOP_THREEPOINT_TAB3D: 3}[family]
    _check(lib().dfrg_integrate_loop4d_host(C.byref(D), _n(m2), _ptr(m2, False), n_ext, _ptr(ext, False),
                                            _ptr(out, False), _ptr(dmin, False)), "dfrg_integrate_loop4d_host")
    return out


# ---- matsubara3d ----------------------------------------------------------------------------------
def _mats_desc(T, n_max, prefactor, reg_kind, reg_order, k, rule_q, rule_c, Zpsi, Zphi, lnq_lo, lnq_hi, interp, coef,
               device, dpsi=None, dphi=None, reg_zk=1.0, reg_eta=0.0, reg_arg4d=1, mu=0.0, out_im=None,
               dpsi_im=None, dphi_im=None, path=0, fermion_reg=0):
    return Mats3dDesc(float(T), int(n_max), float(prefactor), Regulator(int(reg_kind), int(reg_order), float(k), float(reg_zk), float(reg_eta)),
                      _rule(rule_q, device), _rule(rule_c, device),
                      _table(Zpsi, lnq_lo, lnq_hi, interp, device), _table(Zphi, lnq_lo, lnq_hi, interp, device),
                      _ptr(coef, device), _n(coef), _ptr(dpsi, device), _ptr(dphi, device),
                      int(reg_arg4d), float(mu), _ptr(out_im, device), _ptr(dpsi_im, device), _ptr(dphi_im, device),
                      int(path), int(fermion_reg))


def dfrg_integrate_matsubara3d(T, n_max, prefactor, reg_kind, reg_order, k, rule_q, rule_c, Zpsi, Zphi, lnq_lo,
                               lnq_hi, interp, coef, m2psi, m2phi, pext, n_jext, out, dmin=None,
                               dout_dm2_psi=None, dout_dm2_phi=None, reg_zk=1.0, reg_eta=0.0, reg_arg4d=1, mu=0.0, out_im=None,
                               dout_dm2_psi_im=None, dout_dm2_phi_im=None, path=0, fermion_reg=0):
    """out: [n_p, n_jext, n_field].  reg_arg4d=0: spatial regulators; mu != 0 (needs reg_arg4d=0 and out_im): complex result,
    out = real part, out_im = imaginary part (include/dfrg.h, dfrg_mats3d_desc::mu)."""
    D = _mats_desc(T, n_max, prefactor, reg_kind, reg_order, k, rule_q, rule_c, Zpsi, Zphi, lnq_lo, lnq_hi, interp,
                   coef, True, dout_dm2_psi, dout_dm2_phi, reg_zk, reg_eta, reg_arg4d, mu, out_im, dout_dm2_psi_im, dout_dm2_phi_im,
                   path, fermion_reg)
    _check(lib().dfrg_integrate_matsubara3d(C.byref(D), _n(m2psi), _ptr(m2psi, True), _ptr(m2phi, True), _n(pext),
                                            _ptr(pext, True), int(n_jext), _ptr(out, True), _ptr(dmin, True),
                                            _stream()), "dfrg_integrate_matsubara3d")
    return out


def dfrg_integrate_matsubara3d_host(T, n_max, prefactor, reg_kind, reg_order, k, rule_q, rule_c, Zpsi, Zphi, lnq_lo,
                                    lnq_hi, interp, coef, m2psi, m2phi, pext, n_jext, out, dmin=None,
                               dout_dm2_psi=None, dout_dm2_phi=None, reg_zk=1.0, reg_eta=0.0, reg_arg4d=1, mu=0.0, out_im=None,
                               dout_dm2_psi_im=None, dout_dm2_phi_im=None, path=0, fermion_reg=0):
    D = _mats_desc(T, n_max, prefactor, reg_kind, reg_order, k, rule_q, rule_c, Zpsi, Zphi, lnq_lo, lnq_hi, interp,
                   coef, False, dout_dm2_psi, dout_dm2_phi, reg_zk, reg_eta, reg_arg4d, mu, out_im, dout_dm2_psi_im, dout_dm2_phi_im,
                   path, fermion_reg)
    _check(lib().dfrg_integrate_matsubara3d_host(C.byref(D), _n(m2psi), _ptr(m2psi, False), _ptr(m2phi, False),
                                                 _n(pext), _ptr(pext, False), int(n_jext), _ptr(out, False),
                                                 _ptr(dmin, False)), "dfrg_integrate_matsubara3d_host")
    return out
