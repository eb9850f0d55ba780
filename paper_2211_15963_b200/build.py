"""Builds the CUDA library in-tree: nvcc, sm_100a only, -fmad=false (arithmetic contract)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdb_b200.so")
SOURCES = ["db_step.cu", "db_gen.cu", "db_api.cu", "db_bold.cu", "db_raster.cu"]
PROBE_LIB = os.path.join(HERE, "libdb_probe.so")      # bench-only measurement helper, not part of the product ABI
PROBE_SOURCES = ["db_probe.cu"]
HEADERS = ["db_device.cuh", "db_philox.cuh", "db_host.h", os.path.join("..", "..", "include", "db_b200.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-fmad=false", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--threads", "4",
]


def _stale(lib: str = LIB, sources=None) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    files = [os.path.join(CSRC, f) for f in (SOURCES + HEADERS if sources is None else sources)]
    return any(os.path.getmtime(f) > t for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, *NVCC_FLAGS, "-o", LIB, *[os.path.join(CSRC, f) for f in SOURCES]]
        if verbose:
            cmd.insert(1, "-Xptxas")
            cmd.insert(2, "-v")
        subprocess.check_call(cmd)
    if force or _stale(PROBE_LIB, PROBE_SOURCES):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.check_call([nvcc, *NVCC_FLAGS, "-o", PROBE_LIB, *[os.path.join(CSRC, f) for f in PROBE_SOURCES]])
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
