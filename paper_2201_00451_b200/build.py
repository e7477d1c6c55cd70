"""Build the C-ABI shared library (include/fstat.h) in-tree with nvcc for sm_100a.

The FFT pass kernels are instantiated in several translation units (csrc/fft_unit.cu compiled once per FFT_UNIT
value); the objects are compiled in parallel into build/ and only those whose sources changed are recompiled."""
from __future__ import annotations

import concurrent.futures
import os
import re
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(HERE, "..", "include")
OBJ_DIR = os.path.join(HERE, "build")
LIB_PATH = os.path.join(HERE, "libfstat_b200.so")
N_FFT_UNITS = 8        # 0-5: FFT pass kernels, 6: fused sky + pass 1, 7: single cooperative kernel
# (object name, source, extra flags)
UNITS = [("fstat_capi", "fstat_capi.cu", [])] + [(f"fft_unit{u}", "fft_unit.cu", [f"-DFFT_UNIT={u}"]) for u in range(N_FFT_UNITS)]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
CFLAGS = ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found")


def have_nvcc() -> bool:
    try:
        _nvcc()
        return True
    except RuntimeError:
        return False


def _deps(src: str, seen=None):
    """The source file and every header it includes with quotes, recursively."""
    seen = set() if seen is None else seen
    path = os.path.normpath(src)
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    for inc in re.findall(r'^\s*#include\s+"([^"]+)"', open(path).read(), flags=re.M):
        _deps(os.path.join(os.path.dirname(path), inc), seen)
    return seen


def _obj_path(name: str) -> str:
    return os.path.join(OBJ_DIR, name + ".o")


def _obj_stale(name: str, src: str) -> bool:
    obj = _obj_path(name)
    if not os.path.exists(obj):
        return True
    t = os.path.getmtime(obj)
    return any(os.path.getmtime(d) > t for d in _deps(os.path.join(CSRC, src)) | {os.path.abspath(__file__)})


def is_stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    deps = set()
    for _, src, _ in UNITS:
        deps |= _deps(os.path.join(CSRC, src))
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB_PATH
    # one builder at a time (torchrun starts several ranks in the same tree); the others wait and reuse the result
    import fcntl
    with open(LIB_PATH + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and not is_stale():
            return LIB_PATH
        return _build_locked(force, verbose)


def _compile(nvcc: str, name: str, src: str, flags, verbose: bool):
    cmd = [nvcc] + ARCH + CFLAGS + (["-Xptxas", "-v"] if verbose else []) + list(flags) + ["-c", os.path.join(CSRC, src), "-o", _obj_path(name)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    return name, r


def _build_locked(force: bool, verbose: bool) -> str:
    nvcc = _nvcc()
    os.makedirs(OBJ_DIR, exist_ok=True)
    todo = [(n, s, f) for (n, s, f) in UNITS if force or _obj_stale(n, s)]
    with concurrent.futures.ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as ex:
        for name, r in ex.map(lambda u: _compile(nvcc, u[0], u[1], u[2], verbose), todo):
            if verbose:
                sys.stderr.write(f"==== {name}\n{r.stderr}")
            if r.returncode != 0:
                raise RuntimeError(f"nvcc failed on {name}:\n" + r.stdout + r.stderr)
    tmp = LIB_PATH + ".tmp.%d" % os.getpid()
    cmd = [nvcc] + ARCH + ["-shared", "-cudart", "static", "-o", tmp] + [_obj_path(n) for n, _, _ in UNITS]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc link failed:\n" + r.stdout + r.stderr)
    os.replace(tmp, LIB_PATH)                      # atomic: a concurrent dlopen never sees a half-written file
    return LIB_PATH


if __name__ == "__main__":
    print(build_library(force="-f" in sys.argv or "-v" in sys.argv, verbose="-v" in sys.argv))
