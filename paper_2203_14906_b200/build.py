"""Build libpab.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2203_14906_b200.build [--force] [--verbose]

The library is several translation units (csrc/pab_api.cu + csrc/pab_tu_*.cu, one per kernel family), compiled in
parallel into csrc/../build/*.o and linked into one shared object; only units whose sources changed are recompiled.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "libpab.so")
_COMMON = ["pab_types.h", "pab_launch.h", "pab_plan.h", os.path.join("..", "..", "include", "pab.h")]
_KERNEL = _COMMON + ["pab_math.cuh", "pab_pipe.cuh"]
# translation unit -> the files it includes
UNITS = {
    "pab_api.cu": _COMMON + ["pab_run.inl"],
    "pab_tu_direct.cu": _KERNEL + ["pab_kernels.cuh"],
    "pab_tu_staged.cu": _KERNEL + ["pab_staged.cuh"],
    "pab_tu_staged_gen.cu": _KERNEL + ["pab_staged.cuh"],
    "pab_tu_cached.cu": _KERNEL + ["pab_cache.cuh"],
    "pab_tu_diag.cu": _KERNEL + ["pab_diag.cuh"],
    "pab_tu_nearest.cu": _KERNEL + ["pab_nearest.cuh"],
    "pab_tu_post.cu": _KERNEL + ["pab_post.cuh", "pab_metrics.cuh"],
    "pab_tu_peaks.cu": [os.path.join("..", "..", "include", "pab.h")],
}
SOURCES = list(UNITS)
DEPS = sorted({d for u, ds in UNITS.items() for d in [u] + ds})
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libpab.so cannot be built (there is no CPU fallback)")


def _mtime(name: str) -> float:
    return os.path.getmtime(os.path.join(CSRC, name))


def _obj(unit: str) -> str:
    return os.path.join(OBJ, os.path.splitext(unit)[0] + ".o")


def _unit_stale(unit: str) -> bool:
    o = _obj(unit)
    if not os.path.exists(o):
        return True
    t = os.path.getmtime(o)
    return any(_mtime(d) > t for d in [unit] + UNITS[unit])


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(_mtime(d) > t for d in DEPS)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    import fcntl
    with open(LIB + ".lock", "w") as lock:            # several ranks may get here at once: one builds, the rest wait
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and not is_stale():
            return LIB
        return _build_locked(force, verbose)


def _compile(unit: str, verbose: bool) -> None:
    cmd = [nvcc_path()] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", _obj(unit), os.path.join(CSRC, unit)]
    subprocess.check_call(cmd)


def _build_locked(force: bool, verbose: bool) -> str:
    os.makedirs(OBJ, exist_ok=True)
    todo = [u for u in SOURCES if force or _unit_stale(u)]
    with ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as pool:
        list(pool.map(lambda u: _compile(u, verbose), todo))
    subprocess.check_call([nvcc_path(), "-shared", "-cudart", "static", "-o", LIB] + [_obj(u) for u in SOURCES])
    return LIB


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
