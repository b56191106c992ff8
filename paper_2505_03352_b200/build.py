"""Build step of the CUDA library: nvcc, sm_100a only, in-tree (``libepsgrad.so`` next to
this file, so that the built library travels with the repository snapshot)."""
from __future__ import annotations

import glob
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libepsgrad.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))
                  + glob.glob(os.path.join(INCLUDE, "*.h")))


def source_hash() -> str:
    """sha256 (first 16 hex digits) over the CUDA sources and the ABI header: names the build that a profile was taken on"""
    import hashlib
    h = hashlib.sha256()
    for path in sources():
        h.update(os.path.basename(path).encode())
        with open(path, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def nvcc_path() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the epsgrad CUDA library cannot be built (there is no CPU path)")


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the translation units of csrc/ (plan.cu, launch.cu, hostpath.cu, optimizer.cu, noalloc.cu) into libepsgrad.so; returns its path."""
    if not force and not stale():
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    units = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    cmd = [nvcc_path(), *NVCC_FLAGS, "--threads", str(len(units)), "-I", INCLUDE, "-o", tmp, *units, "-ldl"]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd, cwd=CSRC)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
