"""Build the CPU oracle shared library (TEST INFRASTRUCTURE; see oracle/lbm_oracle.cpp header)."""
from __future__ import annotations

import fcntl
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["lbm_oracle.cpp"]
HEADERS = ["jets.hpp", "systems.hpp", "mms_fields.hpp"]
LIB = os.path.join(HERE, "liblbm_oracle.so")


STAMP = LIB + ".stamp"


def _source_hash() -> str:
    h = hashlib.sha256()
    for f in sorted(SOURCES + HEADERS):
        with open(os.path.join(HERE, f), "rb") as fh:
            h.update(f.encode()); h.update(fh.read())
    return h.hexdigest()


def needs_build() -> bool:
    """By content, not by mtime (a copied snapshot keeps no meaningful mtimes)."""
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as fh:
        return fh.read().strip() != _source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and not needs_build():
            return LIB
        return _build_locked(verbose)


def _build_locked(verbose: bool) -> str:
    # -O3, no -ffast-math, no -march=native (the .so may travel to another host): keep IEEE semantics; -ffp-contract=off so the arithmetic is exactly as written
    cmd = ["g++", "-std=c++17", "-O3", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-o", f"{LIB}.{os.getpid()}.tmp"] + [os.path.join(HERE, s) for s in SOURCES]
    if verbose:
        print(" ".join(cmd))
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(f"{LIB}.{os.getpid()}.tmp", LIB)
    with open(STAMP, "w") as fh:
        fh.write(_source_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
