"""Builds libpccl.so (the C-ABI library of include/pccl.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpccl.so")
SOURCES = ["pccl_api.cu"]
DEPS = ["pccl_api.cu", "pccl_device.cuh", "pccl_loop1.cuh", "pccl_loop2.cuh", "pccl_sweep.cuh", "pccl_bfs.cuh", os.path.join("..", "..", "include", "pccl.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-pthread", "-shared", "-Xptxas", "-v", "-ldl",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libpccl.so cannot be built")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if missing or older than its sources.  Returns the path of libpccl.so."""
    if force or stale():
        tmp = LIB + f".tmp{os.getpid()}"
        extra = os.environ.get("PCCL_NVCC_EXTRA", "").split()   # e.g. -DPCCL_DEBUG_CU, -DPCCL_A2_PROFILE, -DPCCL_BFS_PROFILE
        cmd = [nvcc_path(), *NVCC_FLAGS, *extra, "-o", tmp, *[os.path.join(CSRC, s) for s in SOURCES]]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            print(" ".join(cmd))
            print(res.stdout)
            print(res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed building libpccl.so")
        with open(os.path.join(_HERE, "build_ptxas.log"), "w") as f:
            f.write(" ".join(cmd) + "\n" + res.stderr)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
