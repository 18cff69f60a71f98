"""Build the CUDA library in-tree: csrc/*.cu -> libdpstokes.so (nvcc, sm_100a only)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdpstokes.so")
SOURCES = ["plan.cu", "transfer.cu", "solve.cu", "solve_pair.cu", "fft.cu", "lanczos.cu"]
HEADERS = [os.path.join(CSRC, "common.cuh"), os.path.join(CSRC, "solve_common.cuh"), os.path.join(CSRC, "fft_engine.cuh"), os.path.join(CSRC, "fft_radix.cuh"), os.path.join(os.path.dirname(HERE), "include", "dp.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--extended-lambda", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    objs = []
    procs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + HEADERS):
            cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    if force or procs or _stale(LIB, objs):
        cuda_lib = "/usr/local/cuda/lib64"
        cmd = [_nvcc(), "-shared", "-o", LIB + ".tmp"] + objs + ["-L" + cuda_lib, "-lcufft", "-Xlinker", "-rpath," + cuda_lib]
        subprocess.check_call(cmd)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
