"""Builds paper_2311_18561_b200/libpvg.so (CUDA kernels + C ABI) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpvg.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++20",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--expt-relaxed-constexpr"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return (glob.glob(os.path.join(CSRC, "*")) +
            [os.path.join(os.path.dirname(HERE), "include", "pvg.h"), os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False, out: str = LIB, defines=()) -> str:
    """Compile csrc/*.cu into `out`. `defines` (e.g. ["PVG_OSL_THREADS=256"]) are for tuning builds."""
    if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(d) for d in _deps()):
        return out
    tmp = out + f".tmp{os.getpid()}"
    cmd = ([NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + [f"-D{d}" for d in defines]
           + ["-o", tmp] + sources())
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)
    return out


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
