"""In-tree build of liblbmk.so (the C-ABI library of include/lbmk.h) with nvcc for sm_100a.

One translation unit per system (sys_*.cu) plus the API (lbmk_api.cu), compiled in parallel, linked into
`paper_2607_05668_b200/liblbmk.so`.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import concurrent.futures as cf
import fcntl
import hashlib
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblbmk.so")
UNITS = ["lbmk_api", "sys_advection2d", "sys_burgers2d", "sys_swe2d", "sys_euler2d", "sys_adr2d", "sys_nsf3d", "sys_mhd3d",
         "sys_urf2d", "sys_maxwell2d", "sys_allencahn2d", "sys_inse2d", "sys_elasticity2d", "sys_nsf2d",
         "sys_swe2d_bathy", "sys_hcnsf3d", "sys_mhd2d"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: liblbmk.so cannot be built (there is no CPU fallback)")
    return p


def _deps():
    out = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".h"))]
    out.append(os.path.join(os.path.dirname(HERE), "include", "lbmk.h"))
    return out


STAMP = LIB + ".stamp"     # content hash of the sources the library was built from; travels with the .so (git-ignored like it)


def _source_hash() -> str:
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for p in sorted(_deps()):
        h.update(os.path.basename(p).encode())
        with open(p, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def needs_build() -> bool:
    """By CONTENT, not by mtime: a snapshot copied to another box (gpurun) keeps no meaningful mtimes, and rebuilding there would
    cost a minute per process and race between the ranks of a torchrun launch."""
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as fh:
        return fh.read().strip() != _source_hash()


def _compile(unit: str) -> str:
    src = os.path.join(CSRC, unit + ".cu")
    obj = os.path.join(OBJ, unit + ".o")
    log = os.path.join(OBJ, unit + ".ptxas.log")
    r = subprocess.run([_nvcc()] + NVCC_FLAGS + ["-c", src, "-o", obj], capture_output=True, text=True)
    with open(log, "w") as fh:
        fh.write(r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {unit}:\n{r.stdout}\n{r.stderr}")
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    with open(os.path.join(OBJ, ".lock"), "w") as lock:          # one builder at a time (ranks of one launch, parallel test workers)
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and not needs_build():                       # another process built it while this one waited
            return LIB
        with cf.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
            objs = list(ex.map(_compile, UNITS))
        tmp = f"{LIB}.{os.getpid()}.tmp"
        cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs
        if verbose:
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
        with open(STAMP, "w") as fh:
            fh.write(_source_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
