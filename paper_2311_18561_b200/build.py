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

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ARCH + ["-O3", "-lineinfo", "-std=c++20", "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]
# round2.cu launches kernels from the device: it alone is compiled as relocatable device code and device-linked against
# the device runtime (the rest of the library is not: -rdc costs the frame's main kernels 10-50 %)
RDC_SOURCES = ("round2.cu",)


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
    objdir = out + f".obj{os.getpid()}"
    os.makedirs(objdir, exist_ok=True)
    extra = (["-Xptxas", "-v"] if verbose else []) + [f"-D{d}" for d in defines]
    objs, rdc_objs = [], []
    try:
        for src in sources():
            obj = os.path.join(objdir, os.path.basename(src) + ".o")
            rdc = os.path.basename(src) in RDC_SOURCES
            subprocess.run([NVCC] + FLAGS + extra + (["-rdc=true"] if rdc else []) + ["-c", "-o", obj, src], check=True)
            (rdc_objs if rdc else objs).append(obj)
        dlink = os.path.join(objdir, "dlink.o")
        subprocess.run([NVCC] + ARCH + ["-Xcompiler", "-fPIC", "-dlink", "-o", dlink] + rdc_objs + ["-lcudadevrt"], check=True)
        subprocess.run([NVCC] + ARCH + ["-shared", "-cudart", "static", "-o", tmp] + objs + rdc_objs + [dlink, "-lcudadevrt"],
                       check=True)
    finally:
        for f in glob.glob(os.path.join(objdir, "*")):
            os.unlink(f)
        os.rmdir(objdir)
    os.replace(tmp, out)
    return out


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
