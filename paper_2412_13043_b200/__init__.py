"""dfrg on B200: momentum-loop integrals of fRG flow equations (arxiv 2412.13043, sec. 5.3.2).

`inputs`  -- seeded synthetic workloads (numpy only, no method arithmetic).
`binding` -- thin ctypes binding of the C-ABI library csrc/libdfrg.so (see include/dfrg.h);
             imported lazily so that `inputs` can be used on a box without CUDA.
"""
__all__ = ["inputs", "binding"]


def __getattr__(name):
    if name in ("binding", "inputs"):
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
