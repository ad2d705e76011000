"""Builds paper_2201_10058_b200/libgenga_kick.so (the C-ABI library of include/genga_kick.h) with
nvcc for sm_100a, in-tree.  nvcc cross-compiles without a GPU.  Usage: python -m paper_2201_10058_b200.build"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgenga_kick.so")
SOURCES = [os.path.join(CSRC, "genga_kick.cu"), os.path.join(CSRC, "genga_step.cu"), os.path.join(CSRC, "genga_group.cu"), os.path.join(CSRC, "genga_bs.cu"), os.path.join(CSRC, "genga_senc.cu"),
           os.path.join(CSRC, "genga_kick_plan.cpp")]
DEPENDS = SOURCES + [os.path.join(CSRC, "genga_kick_kernels.cuh"), os.path.join(CSRC, "genga_kick_variants.h"),
                     os.path.join(CSRC, "genga_kick_sort.cuh"), os.path.join(CSRC, "genga_kick_ctx.h"),
                     os.path.join(CSRC, "genga_step_kernels.cuh"), os.path.join(CSRC, "genga_group_kernels.cuh"), os.path.join(CSRC, "genga_bs_kernels.cuh"), os.path.join(CSRC, "genga_senc_kernels.cuh"),
                     os.path.join(os.path.dirname(HERE), "include", "genga_senc.h"),
                     os.path.join(os.path.dirname(HERE), "include", "genga_bs.h"),
                     os.path.join(os.path.dirname(HERE), "include", "genga_group.h"),
                     os.path.join(os.path.dirname(HERE), "include", "genga_step.h"),
                     os.path.join(os.path.dirname(HERE), "include", "genga_kick.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
# --fmad=false: no contraction the source does not spell out (the kernels write every fma() themselves)
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "--fmad=false",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def build(force: bool = False, verbose: bool = False) -> str:
    stale = force or not os.path.exists(LIB) or any(os.path.getmtime(LIB) < os.path.getmtime(d) for d in DEPENDS)
    if stale:
        cmd = [NVCC, *FLAGS, *(["-Xptxas", "-v"] if verbose else []), *SOURCES, "-o", LIB]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=bool(os.environ.get("VERBOSE"))))
