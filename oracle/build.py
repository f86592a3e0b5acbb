"""Build the oracle shared libraries (serial and OpenMP) with g++.

    python -m oracle.build

-ffp-contract=off keeps the canonical evaluation order of the sensor
free of FMA contraction.  Building the checker is not using it.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "streams_oracle.cpp")
OUT = os.path.join(HERE, "build")
FLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-shared", "-fPIC", "-Wall", "-Wno-unknown-pragmas"]


def lib_path(kind: str) -> str:
    return os.path.join(OUT, f"liboracle_{kind}.so")


def build(force: bool = False) -> None:
    os.makedirs(OUT, exist_ok=True)
    for kind, extra in (("serial", []), ("omp", ["-fopenmp"])):
        out = lib_path(kind)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(SRC):
            continue
        subprocess.check_call(["g++", *FLAGS, *extra, SRC, "-o", out])


if __name__ == "__main__":
    build(force=True)
    print("built", lib_path("serial"), lib_path("omp"))
