"""ctypes marshalling for genga_detect_oracle.c (close-encounter detection after the Kepler drift, App. A
PAPER.md:989; reading G16).  TEST INFRASTRUCTURE ONLY; see the C header."""
import ctypes as C
from dataclasses import dataclass
import numpy as np

from . import oracle as _kick

_ready = False


def _L():
    global _ready
    lib = _kick._L()
    if not _ready:
        d, i64, p = C.c_double, C.c_int64, C.c_void_p
        lib.genga_oracle_hermite_min.restype = d
        lib.genga_oracle_hermite_min.argtypes = [d, d, d, d, p]
        lib.genga_oracle_detect.restype = i64
        lib.genga_oracle_detect.argtypes = [i64, p, p, p, p, p, d, d, p, i64, p, p, p, p]
        _ready = True
    return lib


def hermite_min(d0, m0, d1, m1):
    """(min over [0, 1] of the cubic Hermite interpolant, its location tau)."""
    tau = C.c_double(0.0)
    v = _L().genga_oracle_hermite_min(float(d0), float(m0), float(d1), float(m1), C.byref(tau))
    return float(v), float(tau.value)


@dataclass
class DetectResult:
    enc: np.ndarray        # [n_pairs] bool: the candidate is a close-encounter pair of this step
    border: np.ndarray     # [n_pairs] bool: within 1e-12 of the threshold
    d2min: np.ndarray      # [n_pairs] minimum of the interpolated squared separation
    count: np.ndarray      # [N] encounter pairs per body
    pairs: np.ndarray      # [total, 2] the encounter pairs, in the order of the candidate list


def detect(pos0, vel0, pos1, vel1, rc_row, h, pairs, enc_factor=1.0):
    pos0, vel0, pos1, vel1 = (np.ascontiguousarray(a, dtype=np.float64) for a in (pos0, vel0, pos1, vel1))
    rc = np.ascontiguousarray(rc_row, dtype=np.float64).reshape(-1)
    n = pos0.shape[1]
    pr = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
    assert rc.size == n and (pr.size == 0 or (pr.min() >= 0 and pr.max() < n))
    m = max(len(pr), 1)
    enc = np.zeros(m, dtype=np.int8); border = np.zeros(m, dtype=np.int8); d2 = np.zeros(m)
    count = np.zeros(n, dtype=np.int32)
    tot = _L().genga_oracle_detect(n, pos0.ctypes.data, vel0.ctypes.data, pos1.ctypes.data, vel1.ctypes.data,
                                   rc.ctypes.data, float(enc_factor), float(h), pr.ctypes.data, len(pr),
                                   enc.ctypes.data, border.ctypes.data, d2.ctypes.data, count.ctypes.data)
    e = enc[:len(pr)].astype(bool)
    assert int(tot) == int(e.sum())
    return DetectResult(enc=e, border=border[:len(pr)].astype(bool), d2min=d2[:len(pr)], count=count, pairs=pr[e])
