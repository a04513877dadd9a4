"""Build step: compile csrc/*.cu into libhicr_b200.so for sm_100a with nvcc (in-tree), and
csrc/hicr_pyext.c (CPython entry points of the calls of a step) into _hicr_step.*.so with gcc.

``python -m paper_2509_01425_b200.build [--force]`` or ``build()`` from Python.  nvcc
cross-compiles without a GPU; the .so is git-ignored but travels to the GPU box.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess
import sys
import sysconfig

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhicr_b200.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
PYEXT_SRC = os.path.join(CSRC, "hicr_pyext.c")
PYEXT = os.path.join(HERE, "_hicr_step" + (sysconfig.get_config_var("EXT_SUFFIX") or ".so"))

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-Wall,-Wextra",
    "-shared",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: cannot build libhicr_b200.so (there is no CPU fallback)")


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + sorted(glob.glob(os.path.join(INCLUDE, "*.h")))


def is_stale() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(PYEXT):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(PYEXT))
    return any(os.path.getmtime(f) > t for f in _deps() + [PYEXT_SRC])


def _build_pyext() -> str:
    """The CPython extension links against the library beside it (rpath $ORIGIN)."""
    tmp = PYEXT + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-shared", "-fPIC", "-Wall", "-Wextra", "-I", sysconfig.get_paths()["include"], "-I", INCLUDE,
           "-o", tmp, PYEXT_SRC, "-L", HERE, "-l:" + os.path.basename(LIB), "-Wl,-rpath,$ORIGIN"]
    try:
        subprocess.check_call(cmd)
        os.replace(tmp, PYEXT)
    finally:
        if os.path.exists(tmp):
            os.remove(tmp)
    return PYEXT


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every CUDA source into one shared library; returns its path."""
    if not force and not is_stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-I", INCLUDE, "-o", tmp] + sources()
    try:
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    finally:
        if os.path.exists(tmp):
            os.remove(tmp)
    _build_pyext()
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
