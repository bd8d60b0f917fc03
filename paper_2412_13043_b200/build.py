"""Builds csrc/*.cu into paper_2412_13043_b200/libdfrg.so for sm_100a (in-tree; nvcc cross-compiles without a GPU),
and bench_probe/fp64_probe.cu into libdfrg_probe.so (bench.py's FP64 peak probe: a measurement aid, not part of the library).

    python -m paper_2412_13043_b200.build [--force] [--verbose]

One nvcc per translation unit, side by side; a translation unit is recompiled only if it, or a header it includes
(transitively), is newer than its object file.
"""
import glob
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdfrg.so")
PROBE_SRC = os.path.join(HERE, "bench_probe", "fp64_probe.cu")
PROBE_LIB = os.path.join(HERE, "libdfrg_probe.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "--fmad=true", "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps(path, seen=None):
    """path and every quoted #include reachable from it."""
    seen = set() if seen is None else seen
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    for inc in re.findall(r'^\s*#\s*include\s+"([^"]+)"', open(path).read(), flags=re.M):
        _deps(os.path.normpath(os.path.join(os.path.dirname(path), inc)), seen)
    return seen


def _obj(src):
    return os.path.join(CSRC, os.path.basename(src)[:-3] + ".o")


def _tu_stale(src):
    obj = _obj(src)
    if not os.path.exists(obj):
        return True
    t = os.path.getmtime(obj)
    return any(os.path.getmtime(d) > t for d in _deps(src))


def stale():
    if not os.path.exists(LIB) or not os.path.exists(PROBE_LIB):
        return True
    if os.path.getmtime(PROBE_SRC) > os.path.getmtime(PROBE_LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(_tu_stale(s) or os.path.getmtime(_obj(s)) > t for s in sources())


def build(force=False, verbose=False):
    if not force and not stale():
        return LIB
    from concurrent.futures import ThreadPoolExecutor

    todo = [s for s in sources() if force or _tu_stale(s)]

    def compile_one(src):
        return src, subprocess.run([NVCC, *FLAGS, "-c", src, "-o", _obj(src)], capture_output=True, text=True)

    logs = []
    if todo:
        with ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as pool:
            for src, r in pool.map(compile_one, todo):   # one nvcc per translation unit, side by side
                logs.append(r.stderr)
                if r.returncode != 0:
                    sys.stderr.write(r.stdout + r.stderr)
                    raise RuntimeError("nvcc failed on %s" % src)
    objs = [_obj(s) for s in sources()]
    r = subprocess.run([NVCC, "-shared", "-o", LIB, *objs, "-lcudart"], capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_SRC) > os.path.getmtime(PROBE_LIB):
        r = subprocess.run([NVCC, *FLAGS, "-shared", PROBE_SRC, "-o", PROBE_LIB, "-lcudart"], capture_output=True, text=True)
        logs.append(r.stderr)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed on %s" % PROBE_SRC)
    if verbose:
        sys.stderr.write("".join(logs))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
