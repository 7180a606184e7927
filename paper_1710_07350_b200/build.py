"""Build libelg.so (hand-written CUDA for sm_100a) in-tree with nvcc.  No JIT cache, no torch extension:
the result is a plain C-ABI shared library next to this file (see include/elg.h).

Staleness is decided by CONTENT, not by modification time: the SHA-256 of the sources and the compiler flags is kept
in a sidecar file next to the library (file times do not survive a copy to another machine; a hash does).  A library
whose sidecar does not match the sources is never loaded: it is rebuilt, and if that is impossible the caller gets the
error."""
from __future__ import annotations

import hashlib
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


def source_hash(extra=()) -> str:
    h = hashlib.sha256()
    for p in DEPS:
        with open(p, "rb") as f:
            h.update(f.read())
        h.update(b"\0")
    h.update(" ".join(NVCC_FLAGS + list(extra)).encode())
    return h.hexdigest()


def is_current(out: str = LIB, extra=()) -> bool:
    """True when `out` exists and was built from exactly the present sources and flags."""
    side = out + ".hash"
    if not (os.path.exists(out) and os.path.exists(side)):
        return False
    with open(side) as f:
        return f.read().strip() == source_hash(extra)


def build(force: bool = False, verbose: bool = False, out: str = LIB, extra=()) -> str:
    """Compile libelg.so unless it is current.  `extra` / `out` build tuning variants (-D..., see elg_kernels.cuh).
    Raises if the compiler is missing or the compilation fails: a stale library is never returned."""
    if not force and is_current(out, extra):
        return out
    cmd = [nvcc_path()] + NVCC_FLAGS + list(extra) + (["-Xptxas", "-v"] if verbose else []) + [SRC, "-o", out + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(out + ".tmp", out)
    with open(out + ".hash", "w") as f:
        f.write(source_hash(extra) + "\n")
    return out


if __name__ == "__main__":
    print(build(force=True, verbose=True))
