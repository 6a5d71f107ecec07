"""Compile csrc/*.cu into paper_2402_00665_b200/libbvh_b200.so for sm_100a (nvcc, in-tree).

The library links the static CUDA runtime and has no torch or Python dependency: it is a plain C-ABI
shared object (include/bvh_b200.h).  ``python -m paper_2402_00665_b200.build`` rebuilds it.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libbvh_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "--fmad=false",            # no FMA contraction anywhere: fp32 results must match the oracle bit for bit
    "-Xcompiler", "-fPIC", "-shared",
    "--threads", "0",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(_HERE, "..", "include", "*.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, out: str | None = None, extra: list[str] | None = None) -> str:
    """Build the library.  ``out``/``extra`` (another output path, extra nvcc flags such as -DBVH_SCAN_LEAVES=8)
    are for tuning sweeps; the product is the default build."""
    target = out or LIB
    if force or out or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = target + f".tmp{os.getpid()}"
        cmd = [nvcc, *NVCC_FLAGS, *(extra or []), *(["-Xptxas", "-v"] if verbose else []), *sources(), "-o", tmp]
        subprocess.check_call(cmd)
        os.replace(tmp, target)
    return target


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
