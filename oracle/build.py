"""Build the CPU oracle shared library (TEST INFRASTRUCTURE; see oracle/lbm_oracle.cpp header)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["lbm_oracle.cpp"]
HEADERS = ["jets.hpp", "systems.hpp", "mms_fields.hpp"]
LIB = os.path.join(HERE, "liblbm_oracle.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    # -O3, no -ffast-math, no -march=native (the .so may travel to another host): keep IEEE semantics; -ffp-contract=off so the arithmetic is exactly as written
    cmd = ["g++", "-std=c++17", "-O3", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-o", LIB + ".tmp"] + [os.path.join(HERE, s) for s in SOURCES]
    if verbose:
        print(" ".join(cmd))
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
