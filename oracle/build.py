"""Builds the CPU oracle shared libraries (test infrastructure; never on the product path).

    python -m oracle.build

produces oracle/liboracle_ld.so (REAL = long double: parity reference values) and
oracle/liboracle_d.so (REAL = double: the timed CPU baseline) from oracle/poisson_oracle.c and oracle/field_ops_oracle.c.
ORACLE_SANITIZE=1 adds -fsanitize=address,undefined (used by the sanitizer run recorded under profiles/) and writes to
liboracle_ld_san.so / liboracle_d_san.so instead, so that an instrumented (several times slower) library can never be what a
later run without the variable loads -- bench.py times the plain build as its CPU baseline.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "poisson_oracle.c"), os.path.join(HERE, "field_ops_oracle.c")]
SANITIZE = os.environ.get("ORACLE_SANITIZE") == "1"
_SUFFIX = "_san" if SANITIZE else ""
LIBS = {"ld": os.path.join(HERE, f"liboracle_ld{_SUFFIX}.so"), "d": os.path.join(HERE, f"liboracle_d{_SUFFIX}.so")}


def _stale(lib: str) -> bool:
    return (not os.path.exists(lib)) or any(os.path.getmtime(lib) < os.path.getmtime(src) for src in SRCS)


def build(force: bool = False) -> dict:
    for kind, lib in LIBS.items():
        if not force and not _stale(lib):
            continue
        # -ffp-contract=off / no -ffast-math: IEEE arithmetic exactly as written.
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-Wall", "-Wextra"] + SRCS + ["-o", lib, "-lm"]
        if kind == "ld":
            cmd.insert(1, "-DORACLE_LD")
        if SANITIZE:
            cmd[1:1] = ["-fsanitize=address,undefined", "-fno-omit-frame-pointer", "-g"]
        subprocess.run(cmd, check=True)
    return LIBS


if __name__ == "__main__":
    build(force="--force" in sys.argv)
    print("\n".join(LIBS.values()))
