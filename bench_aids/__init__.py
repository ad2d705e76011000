"""Bench-side helpers (not part of the product library): bench.py's FP64 roofline probe.

    python -m bench_aids.build        # nvcc, sm_100a, in-tree (also done by __graft_entry__.build())"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libgenga_bench_aids.so")
_lib = None


def fp64_rate(pattern: int, iters: int = 4096, reps: int = 5, stream: int = 0) -> float:
    """DFMAs per second of independent chains with the given register-operand pattern (fp64_rate.cu)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m bench_aids.build`")
        _lib = C.CDLL(LIB_PATH)
        _lib.bench_fp64_rate.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.POINTER(C.c_double)]
        _lib.bench_fp64_rate.restype = C.c_int
    r = C.c_double()
    rc = _lib.bench_fp64_rate(int(pattern), int(iters), int(reps), C.c_void_p(int(stream)), C.byref(r))
    if rc != 0:
        raise RuntimeError(f"bench_fp64_rate failed with code {rc}")
    return float(r.value)
