"""Builds the CPU oracle shared libraries (test infrastructure; never on the product path).

    python -m oracle.build

produces oracle/liboracle_ld.so (REAL = long double: parity reference values) and
oracle/liboracle_d.so (REAL = double: the timed CPU baseline) from oracle/poisson_oracle.c.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "poisson_oracle.c")
LIBS = {"ld": os.path.join(HERE, "liboracle_ld.so"), "d": os.path.join(HERE, "liboracle_d.so")}


def _stale(lib: str) -> bool:
    return (not os.path.exists(lib)) or os.path.getmtime(lib) < os.path.getmtime(SRC)


def build(force: bool = False) -> dict:
    for kind, lib in LIBS.items():
        if not force and not _stale(lib):
            continue
        # -ffp-contract=off / no -ffast-math: IEEE arithmetic exactly as written.
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-Wall", "-Wextra", SRC, "-o", lib, "-lm"]
        if kind == "ld":
            cmd.insert(1, "-DORACLE_LD")
        subprocess.run(cmd, check=True)
    return LIBS


if __name__ == "__main__":
    build(force="--force" in sys.argv)
    print("\n".join(LIBS.values()))
