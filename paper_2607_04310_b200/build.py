"""Builds paper_2607_04310_b200/libpsdf.so in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpsdf.so")
SOURCES = ["psdf_api.cu"]
DEPS = ["psdf_api.cu", "psdf_kernels.cuh", "psdf_device.cuh", "psdf_pack.h", "psdf_pack_kernels.cuh", "psdf_cull_kernels.cuh", "psdf_reduce_kernels.cuh", "../../include/psdf.h", "../../include/psdf_bench.h"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
# PSDF_NVCC_EXTRA="-DPSDF_TUNING": a measurement build in which the PSDF_BD / PSDF_CHUNKS / PSDF_BRANCHES /
# PSDF_NO_ZERO_COPY sweep knobs are read from the environment (they do not exist in the product build)
EXTRA = os.environ.get("PSDF_NVCC_EXTRA", "").split()
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xptxas=-v", "-Xcompiler", "-fPIC", "-shared",
         "-cudart", "static"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [NVCC] + FLAGS + EXTRA + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        print(r.stdout[-20000:])
        print(r.stderr[-20000:])
    r.check_returncode()
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
