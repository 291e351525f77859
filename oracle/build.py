"""Builds oracle/libpvg_oracle.so with g++ (TEST INFRASTRUCTURE, not product code).

Flags follow BASELINE.md section 2: -O2 -ffp-contract=off, no fast-math, OpenMP.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pvg_oracle.cpp")
LIB = os.path.join(HERE, "libpvg_oracle.so")


def build(force: bool = False) -> str:
    """PVG_ORACLE_LIB names an alternative library to load instead (the sanitizer build below)."""
    alt = os.environ.get("PVG_ORACLE_LIB")
    if alt:
        return alt
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC",
           "-Wall", "-Wextra", "-o", tmp, SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


def build_sanitized(out: str) -> str:
    """AddressSanitizer + UndefinedBehaviorSanitizer build of the oracle. Run the CPU pins on it:
        python -m oracle.build sanitize /tmp/libpvg_oracle_asan.so
        LD_PRELOAD=$(g++ -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 PVG_ORACLE_LIB=/tmp/libpvg_oracle_asan.so \
            python -m pytest tests/test_oracle_pins.py tests/test_oracle_golden.py -q
    (the interpreter is not instrumented, so the runtime is preloaded and leak checking, which would report CPython's
    own allocations, is off)."""
    cmd = ["g++", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
           "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", out, SRC]
    subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    import sys
    if len(sys.argv) == 3 and sys.argv[1] == "sanitize":
        print(build_sanitized(sys.argv[2]))
    else:
        print(build(force=True))
