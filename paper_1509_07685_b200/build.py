"""Builds the C-ABI library libdks_poisson.so (sm_100a only) in-tree with nvcc.

    python -m paper_1509_07685_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so sits beside this file so that it travels to the GPU box
with the repo snapshot (it is git-ignored: the history stays source-only).
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libdks_poisson.so")
SOURCES = [os.path.join(CSRC, "dks_poisson.cu")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "--fmad=true",
    "-cudart", "shared",
]


def _deps():
    return SOURCES + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(INCLUDE, "*.h"))


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    import fcntl
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    with open(LIB + ".lock", "w") as lock:             # several ranks may import the package at once
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and not stale():                  # another process built it while this one waited
            return LIB
        tmp = f"{LIB}.{os.getpid()}.tmp"
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-I", INCLUDE] + SOURCES + ["-o", tmp]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError("nvcc failed building libdks_poisson.so")
        os.replace(tmp, LIB)                           # atomic: no process ever maps a half-written library
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
