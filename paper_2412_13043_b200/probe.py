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
        _lib.dfrg_probe_fp64_issue.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    return _lib


def fp64_issue_model(sink, n_iter=20000):
    """Times 8 DFMA chains with 0, 4 and 8 interleaved integer adds per 8 DFMA (bench_probe/fp64_probe.cu).  Returns
    {"ms": [t0, t4, t8], "ratio": [1, t4/t0, t8/t0]}: (16 + K)/16 = 1.25, 1.5 means an FP64 warp instruction holds the issue
    port for two cycles and every other instruction for one."""
    import torch
    lib = _load()
    st = torch.cuda.current_stream().cuda_stream
    ms = []
    for k in (0, 4, 8):
        for rep in range(2):           # the first launch of each instantiation is the warm-up
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            rc = lib.dfrg_probe_fp64_issue(int(n_iter), k, sink.data_ptr(), st)
            b.record()
            b.synchronize()
            if rc != 0:
                raise RuntimeError("dfrg_probe_fp64_issue failed (%d)" % rc)
        ms.append(a.elapsed_time(b))
    return {"ms": ms, "ratio": [t / ms[0] for t in ms]}


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
