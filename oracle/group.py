"""ctypes marshalling for genga_group_oracle.c (grouping of close-encounter pairs into connected
components).  TEST INFRASTRUCTURE ONLY; see the C header."""
import ctypes as C
from dataclasses import dataclass
import numpy as np

from . import oracle as _kick

_ready = False


@dataclass
class Groups:
    group_of: np.ndarray     # [N] smallest body index of the body's group, -1: in no pair
    members: np.ndarray      # [n_members] sorted by (group, body)
    offsets: np.ndarray      # [n_groups + 1]
    n_groups: int
    n_members: int
    max_size: int


def group(n: int, pairs) -> Groups:
    global _ready
    lib = _kick._L()
    if not _ready:
        i64, p = C.c_int64, C.c_void_p
        lib.genga_oracle_group.restype = i64
        lib.genga_oracle_group.argtypes = [i64, p, i64, p, p, p, C.POINTER(i64), C.POINTER(i64)]
        _ready = True
    pr = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
    assert pr.size == 0 or (pr.min() >= 0 and pr.max() < n)
    group_of = np.empty(n, dtype=np.int32)
    members = np.empty(max(n, 1), dtype=np.int32)
    offsets = np.empty(n + 1, dtype=np.int32)
    nm, mx = C.c_int64(0), C.c_int64(0)
    ng = lib.genga_oracle_group(n, pr.ctypes.data, pr.shape[0], group_of.ctypes.data, members.ctypes.data,
                                offsets.ctypes.data, C.byref(nm), C.byref(mx))
    return Groups(group_of=group_of, members=members[:nm.value].copy(), offsets=offsets[:ng + 1].copy(),
                  n_groups=int(ng), n_members=int(nm.value), max_size=int(mx.value))
