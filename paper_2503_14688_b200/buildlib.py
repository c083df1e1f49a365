"""Build the CUDA library in-tree: csrc/*.cu -> paper_2503_14688_b200/liblattice.so (sm_100a).

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the working tree.
"""
from __future__ import annotations

import os
import subprocess

_PKG = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_PKG)
SO_PATH = os.path.join(_PKG, "liblattice.so")
SOURCES = [os.path.join(_PKG, "csrc", "lattice.cu")]
HEADERS = sorted(os.path.join(_PKG, "csrc", n) for n in os.listdir(os.path.join(_PKG, "csrc")) if n.endswith(".cuh"))
HEADERS.append(os.path.join(_ROOT, "include", "lattice.h"))

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(SO_PATH):
        return True
    t = os.path.getmtime(SO_PATH)
    return any(os.path.getmtime(p) > t for p in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile liblattice.so if it is missing or older than its sources; return its path.

    Safe under torchrun (every rank calls this): an exclusive file lock serialises the check and
    the compile, nvcc writes to a temporary file in the same directory and the finished library is
    moved into place with os.replace(), so no process ever dlopens a half-written file."""
    import fcntl
    with open(SO_PATH + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not needs_build():
                return SO_PATH
            tmp = f"{SO_PATH}.{os.getpid()}.tmp"
            cmd = [nvcc(), *NVCC_FLAGS, "-I", os.path.join(_ROOT, "include"), "-o", tmp, *SOURCES]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
                print(" ".join(cmd))
            try:
                subprocess.run(cmd, check=True)
                os.replace(tmp, SO_PATH)
            finally:
                if os.path.exists(tmp):
                    os.unlink(tmp)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return SO_PATH


if __name__ == "__main__":
    print(build(force=True, verbose=True))
