"""Build liblm.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2510_02135_b200.build [--force]

The .so lands next to this file so that it travels with the repo snapshot; it is git-ignored.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblm.so")
SOURCES = [os.path.join(CSRC, "lm_api.cu"), os.path.join(CSRC, "lm_static.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("rpy_pair.cuh", "rpy_small.cuh", "steric_pair.cuh", "vector_kernels.cuh", "lm_common.cuh", "tridiag_host.h",
                                                    "lanczos_host.h", "lm_handle.cuh", "lm_apply.cuh", "lm_lanczos.cuh", "lm_bd.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "lm.h")]
# measurement helper of bench.py (FMA-pipe peak probe): its own library, not part of liblm.so
PROBE_LIB = os.path.join(HERE, "liblm_probe.so")
PROBE_SOURCES = [os.path.join(CSRC, "fma_probe.cu")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-shared", "-Xcompiler", "-fPIC",
    "-cudart", "static",
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
        subprocess.run(cmd, check=True)
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_LIB) < os.path.getmtime(PROBE_SOURCES[0]):
        subprocess.run([nvcc()] + NVCC_FLAGS + ["-o", PROBE_LIB] + PROBE_SOURCES, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
