"""ctypes access to libdfrg_probe.so: bench.py's FP64 peak probe (bench_probe/fp64_probe.cu).  A measurement aid,
not part of the library: the product ABI (include/dfrg.h, libdfrg.so, binding.py) does not contain it."""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdfrg_probe.so")
_lib = None


def _load():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libdfrg_probe.so not built: run `python -m paper_2412_13043_b200.build`")
        _lib = C.CDLL(LIB_PATH)
        _lib.dfrg_probe_fp64_peak.argtypes = [C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
        _lib.dfrg_probe_fp64_issue.argtypes = [C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    return _lib


def fp64_issue_model(sink, n_iter=20000):
    """Times 8 DFMA chains per thread with K instructions of another pipe interleaved per 8 DFMA (bench_probe/fp64_probe.cu).
    Returns {"base_ms": t(K=0), "int_add": {K: t/t0}, "cvt_f64": {...}, "lds128": {...}}.  int_add ratios (16 + K)/16 = 1.25, 1.5
    would mean an FP64 warp instruction holds the issue port for two cycles; ratios of 1 that other instructions issue in its
    shadow."""
    import torch
    lib = _load()
    st = torch.cuda.current_stream().cuda_stream

    def t(kind, k):
        for rep in range(2):           # the first launch of each instantiation is the warm-up
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            rc = lib.dfrg_probe_fp64_issue(int(n_iter), kind, k, sink.data_ptr(), st)
            b.record()
            b.synchronize()
            if rc != 0:
                raise RuntimeError("dfrg_probe_fp64_issue failed (%d)" % rc)
        return a.elapsed_time(b)
    t0 = t(0, 0)
    return {"base_ms": t0, "int_add": {k: t(0, k) / t0 for k in (4, 8)}, "cvt_f64": {k: t(1, k) / t0 for k in (2, 4, 8)},
            "lds128": {k: t(2, k) / t0 for k in (2, 4, 8)}, "mufu_rcp64h": {k: t(3, k) / t0 for k in (1, 2, 4)}}


def fp64_peak(n_iter, ctas_per_sm, sink):
    """Enqueues the register-only DFMA kernel on torch's current stream; returns the FP64 flops it executes.
    sink: torch CUDA tensor of at least one double."""
    import torch
    flops = C.c_double()
    rc = _load().dfrg_probe_fp64_peak(int(n_iter), int(ctas_per_sm), sink.data_ptr(), C.byref(flops),
                                   torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError("dfrg_probe_fp64_peak failed (%d)" % rc)
    return flops.value
