"""Builds bench_aids/libgenga_bench_aids.so (nvcc, sm_100a, in-tree; cross-compiles without a GPU)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "fp64_rate.cu")
LIB = os.path.join(HERE, "libgenga_bench_aids.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        subprocess.check_call([NVCC, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                               "--fmad=false", "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", SRC, "-o", LIB])
    return LIB


if __name__ == "__main__":
    print(build(force=True))
