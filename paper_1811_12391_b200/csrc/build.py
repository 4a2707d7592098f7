"""Build libdos.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python paper_1811_12391_b200/csrc/build.py [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["dos_api.cu", "dos_kernels.cu", "dos_sweep_umma.cu", "dos_sweep_ffma.cu", "dos_static.cu"]
HEADERS = ["dos_internal.h", "dos_kernels.h", "dos_sm100.cuh", os.path.join("..", "..", "include", "dos.h")]
LIB = os.path.join(HERE, "libdos.so")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-Xcompiler", "-fPIC"]
STD = {"dos_sweep_umma.cu": "-std=c++20"}     # templated lambdas; nvcc 12.9 breaks on libstdc++ 13 headers of dos_api.cu under C++20


def build(force: bool = False, verbose: bool = False) -> str:
    deps = [os.path.join(HERE, f) for f in SOURCES + HEADERS]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs, procs = [], []
    for src in SOURCES:
        obj = os.path.join(HERE, src.replace(".cu", ".o"))
        objs.append(obj)
        cmd = [nvcc] + FLAGS + [STD.get(src, "-std=c++17")] + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(HERE, src), "-o", obj]
        procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    subprocess.check_call([nvcc, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
