"""Build step: compile csrc/mlp_pipe.cu into csrc/libmlp_pipe.so with nvcc for sm_100a.

`python -m paper_2607_07862_b200.build` (or `__graft_entry__.build()`).  The library is built
IN-TREE so that it travels with the repository snapshot to the GPU box; nvcc cross-compiles
without a GPU.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(CSRC, "libmlp_pipe.so")
SOURCES = ["mlp_pipe.cu"]
HEADERS = ["kernel.cuh", "ptx.cuh", os.path.join("..", "..", "include", "mlp_pipe.h")]

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-shared", "-Xcompiler", "-fPIC",
    "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found (set NVCC=/path/to/nvcc)")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    """Compile the C-ABI library if it is missing or older than its sources; return its path."""
    if not force and not needs_build():
        return LIB
    # MLP_PIPE_DEBUG_HOOKS=1: developer build whose planner reads MLP_PIPE_BOUNDS_<l> / MLP_PIPE_NO_RASTER / MLP_PIPE_DEBUG
    hooks = ["-DMLP_PIPE_DEBUG_HOOKS"] if os.environ.get("MLP_PIPE_DEBUG_HOOKS") == "1" else []
    cmd = [_nvcc()] + NVCC_FLAGS + hooks + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if verbose:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose=True))
