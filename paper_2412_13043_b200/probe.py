"""ctypes access to libdfrg_probe.so: bench.py's FP64 peak probe (bench_probe/fp64_probe.cu).  A measurement aid,
not part of the library: the product ABI (include/dfrg.h, libdfrg.so, binding.py) does not contain it."""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdfrg_probe.so")
_lib = None


def fp64_peak(n_iter, ctas_per_sm, sink):
    """Enqueues the register-only DFMA kernel on torch's current stream; returns the FP64 flops it executes.
    sink: torch CUDA tensor of at least one double."""
    global _lib
    import torch
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libdfrg_probe.so not built: run `python -m paper_2412_13043_b200.build`")
        _lib = C.CDLL(LIB_PATH)
        _lib.dfrg_probe_fp64_peak.argtypes = [C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
    flops = C.c_double()
    rc = _lib.dfrg_probe_fp64_peak(int(n_iter), int(ctas_per_sm), sink.data_ptr(), C.byref(flops),
                                   torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError("dfrg_probe_fp64_peak failed (%d)" % rc)
    return flops.value
