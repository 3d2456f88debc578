"""Builds libwri.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2410_18429_b200.build [--force]

The .so lands next to this file so that it travels with the repo snapshot to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libwri.so")
SOURCES = [os.path.join(CSRC, "wri_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "wri_kernels.cuh"), os.path.join(CSRC, "wri_pass.cuh"),
                  os.path.join(os.path.dirname(_HERE), "include", "wri.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-fmad=true", "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]
# IEEE fp32 arithmetic with FMA contraction: no --use_fast_math (denormals are kept, divisions are
# exact); the data path has neither divisions nor transcendentals, so nothing is lost.


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + ".%d.tmp" % os.getpid()
        cmd = [nvcc()] + NVCC_FLAGS + ["-o", tmp] + SOURCES
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
