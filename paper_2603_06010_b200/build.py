"""Builds the in-tree CUDA library (libtdlike.so) and the C oracle helpers, if any.

    python -m paper_2603_06010_b200.build [--force] [--verbose]

nvcc cross-compiles for sm_100a without a GPU.  The .so is git-ignored but travels to the GPU
box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIBDIR = os.path.join(HERE, "lib")
LIB = os.path.join(LIBDIR, "libtdlike.so")
PROBE_LIB = os.path.join(LIBDIR, "libtdprobe.so")   # bench-only (include/tdprobe.h), separate from the product library
PROBE_SRC = os.path.join(CSRC, "probe", "tdprobe.cu")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--expt-relaxed-constexpr", "-split-compile", "0",
]


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cu"))


def deps():
    out = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if os.path.isfile(os.path.join(CSRC, f))]
    out.append(os.path.join(os.path.dirname(HERE), "include", "tdlike.h"))
    return out


def up_to_date() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(PROBE_LIB):
        return False
    t = os.path.getmtime(LIB)
    inc = os.path.join(os.path.dirname(HERE), "include", "tdprobe.h")
    return (all(os.path.getmtime(p) <= t for p in deps())
            and all(os.path.getmtime(p) <= os.path.getmtime(PROBE_LIB) for p in (PROBE_SRC, inc)))


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    os.makedirs(LIBDIR, exist_ok=True)
    for srcs, lib in ((sources(), LIB), ([PROBE_SRC], PROBE_LIB)):
        cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + srcs + ["-o", lib]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
