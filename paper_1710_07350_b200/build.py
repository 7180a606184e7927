"""Build libelg.so (hand-written CUDA for sm_100a) in-tree with nvcc.  No JIT cache, no torch extension:
the result is a plain C-ABI shared library next to this file (see include/elg.h)."""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "csrc", "elg.cu")
DEPS = [SRC, os.path.join(_HERE, "csrc", "elg_kernels.cuh"),
        os.path.join(os.path.dirname(_HERE), "include", "elg.h")]
LIB = os.path.join(_HERE, "libelg.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-fmad=false",                       # arithmetic specification: only explicit fma() fuses
    "-shared", "-Xcompiler", "-fPIC",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found (set NVCC or add /usr/local/cuda/bin to PATH)")


def build(force: bool = False, verbose: bool = False, out: str = LIB, extra=()) -> str:
    """Compile libelg.so.  `extra` / `out` build tuning variants (-DELG_COMPACT_WARPS=..., see elg_kernels.cuh)."""
    newest = max(os.path.getmtime(p) for p in DEPS)
    if not force and os.path.exists(out) and os.path.getmtime(out) >= newest:
        return out
    cmd = [nvcc_path()] + NVCC_FLAGS + list(extra) + (["-Xptxas", "-v"] if verbose else []) + [SRC, "-o", out]
    subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    print(build(force=True, verbose=True))
