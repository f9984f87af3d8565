"""Build the CPU oracle (oracle/libhepo.so) with gcc.  TEST INFRASTRUCTURE ONLY.

-ffp-contract=off and no -ffast-math keep the exact-class float32 expressions one IEEE op per
node.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hepo.c")
HDR = os.path.join(HERE, "hepo.h")
LIB = os.path.join(HERE, "libhepo.so")
# -fopenmp only serves hepo_analysis_chain_omp (the all-cores timing leg); every other function is serial
CFLAGS = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(LIB) >= newest:
            return LIB
    cmd = [*CFLAGS, "-shared", "-fPIC", SRC, "-o", LIB + ".tmp", "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


def build_sanitized(out_dir: str) -> str:
    """The same sources under AddressSanitizer + UndefinedBehaviorSanitizer (tests/test_oracle_sanitizers.py).
    Load it into a process whose first library is libasan (LD_PRELOAD of `asan_runtime()`)."""
    lib = os.path.join(out_dir, "libhepo_san.so")
    cmd = [*CFLAGS, "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer",
           "-shared", "-fPIC", SRC, "-o", lib, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return lib


def asan_runtime() -> str:
    return subprocess.run(["gcc", "-print-file-name=libasan.so"], check=True, capture_output=True, text=True).stdout.strip()


if __name__ == "__main__":
    print(build(force=True))
