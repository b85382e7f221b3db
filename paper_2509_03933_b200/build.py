"""Builds the C-ABI shared library ``libtdma.so`` in-tree with nvcc for sm_100a.

The library has no torch types anywhere; it links the CUDA runtime statically, so it loads
next to PyTorch's own runtime and shares the device's primary context (streams and device
pointers interoperate).  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libtdma.so")
# translation unit -> the headers it includes (a unit is recompiled when any of them is newer)
_TDMA_H = os.path.join("..", "..", "include", "tdma.h")
UNITS = {
    "tdma_plan.cu": ["tdma_stage_kernels.cuh", "tdma_fused.cuh", "tdma_fused_tma.cuh", "tdma_shared.h", "tdma_staged.h", _TDMA_H],
    "tdma_staged.cu": ["tdma_fused_tma.cuh", "tdma_staged.h"],
    "tdma_shared.cu": ["tdma_shared_tma.cuh", "tdma_fused_tma.cuh", "tdma_shared.h"],
    "tdma_shared_lines.cu": ["tdma_shared.h"],
    "tdma_probe.cu": [_TDMA_H],
    "tdma_slab.cu": ["tdma_stage_kernels.cuh", "tdma_staged.h", _TDMA_H],
    "tdma_static.cu": ["tdma_stage_kernels.cuh", _TDMA_H],
}
OBJ_DIR = os.path.join(CSRC, "build")

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC",
    # fp64 division and sqrt stay IEEE; FMA contraction is allowed (default); no fast-math
    "--ftz=false", "--prec-div=true", "--prec-sqrt=true",
]
LINK_FLAGS = ["-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC"]


def nvcc_path() -> str:
    cand = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(cand):
        raise RuntimeError("nvcc not found; the CUDA extension cannot be built")
    return cand


def _newer(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps if os.path.exists(d))


def _obj(unit: str) -> str:
    return os.path.join(OBJ_DIR, os.path.splitext(unit)[0] + ".o")


def _unit_deps(unit: str):
    return [os.path.join(CSRC, f) for f in [unit] + UNITS[unit]] + [os.path.abspath(__file__)]


def _stale() -> bool:
    return any(_newer(LIB_PATH, _unit_deps(u)) for u in UNITS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu -> objects (in parallel, only the stale ones) -> libtdma.so.  Returns the path."""
    if not force and not _stale():
        return LIB_PATH
    os.makedirs(OBJ_DIR, exist_ok=True)
    nvcc = nvcc_path()
    procs = []
    for unit in UNITS:
        if not force and not _newer(_obj(unit), _unit_deps(unit)):
            continue
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-c", os.path.join(CSRC, unit), "-o", _obj(unit)]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)))
    for cmd, pr in procs:
        _, err = pr.communicate()
        if pr.returncode != 0:
            raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), err))
        if verbose:
            print(err)
    tmp = LIB_PATH + ".tmp.%d" % os.getpid()
    cmd = [nvcc] + LINK_FLAGS + ["-o", tmp] + [_obj(u) for u in UNITS]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (" ".join(cmd), res.stderr))
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
