"""Build libmcrt_b200.so (hand-written CUDA for sm_100a) in-tree with nvcc."""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = os.path.join(HERE, "csrc", "mcrt.cu")
HDR = os.path.join(ROOT, "include", "mcrt.h")
LIBDIR = os.path.join(HERE, "lib")
OUT = os.path.join(LIBDIR, "libmcrt_b200.so")

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-fmad=false",  # arithmetic contract with the oracle: no FMA contraction of the fp64 trajectory math
    "-Xcompiler", "-fPIC", "-shared",
]


def nvcc_path() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built")


def build(force: bool = False, extra_flags=(), verbose: bool = False) -> str:
    os.makedirs(LIBDIR, exist_ok=True)
    deps = [SRC, HDR, __file__] + [os.path.join(HERE, "csrc", f) for f in os.listdir(os.path.join(HERE, "csrc"))]
    newest = max(os.path.getmtime(f) for f in deps)
    if (not force) and os.path.exists(OUT) and os.path.getmtime(OUT) >= newest:
        return OUT
    cmd = [nvcc_path(), *NVCC_FLAGS, *extra_flags, "-I", os.path.join(ROOT, "include"), "-o", OUT, SRC]
    if verbose:
        print(" ".join(cmd))
    subprocess.run(cmd, check=True)
    return OUT


if __name__ == "__main__":
    flags = [a for a in sys.argv[1:] if a not in ("--force", "-v")]
    print(build(force="--force" in sys.argv, extra_flags=flags, verbose="-v" in sys.argv))
