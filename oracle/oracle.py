"""ctypes marshalling for genga_kick_oracle.c (TEST INFRASTRUCTURE ONLY; see the C header)."""
import ctypes as C
from dataclasses import dataclass
import numpy as np

from . import build as _build

_lib = None


def lib_path() -> str:
    return _build.build()


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(lib_path())
        d, i32, i64, p = C.c_double, C.c_int32, C.c_int64, C.c_void_p
        lib.genga_oracle_K_of_y.restype = d
        lib.genga_oracle_K_of_y.argtypes = [d]
        lib.genga_oracle_K.restype = d
        lib.genga_oracle_K.argtypes = [d, d]
        lib.genga_oracle_weight.restype = d
        lib.genga_oracle_weight.argtypes = [d, p, C.c_int]
        lib.genga_oracle_weight_bs.restype = d
        lib.genga_oracle_weight_bs.argtypes = [d, p, C.c_int]
        lib.genga_oracle_num_threads.restype = C.c_int
        lib.genga_oracle_kick.restype = C.c_int
        lib.genga_oracle_kick.argtypes = [i32, i32, i32, d, d, p, p, p, p, i64, p, p, p, p, i32, p, i64, p]
        lib.genga_oracle_kick_tp.restype = C.c_int
        lib.genga_oracle_kick_tp.argtypes = [i32, i32, i32, i32, d, d, p, p, p, p, i64, p, p, p, p, i32, p, i64, p]
        lib.genga_oracle_kick_list.restype = C.c_int
        lib.genga_oracle_kick_list.argtypes = [i32, i32, i32, i32, d, d, p, p, p, p, i64, p, p, p, p, p]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_L().genga_oracle_num_threads())


def K_of_y(y: float) -> float:
    return float(_L().genga_oracle_K_of_y(float(y)))


def K(r: float, rc: float) -> float:
    return float(_L().genga_oracle_K(float(r), float(rc)))


def weight(r: float, rc_rows, level: int) -> float:
    rc = np.ascontiguousarray(rc_rows, dtype=np.float64)
    assert rc.size >= level + 1
    return float(_L().genga_oracle_weight(float(r), rc.ctypes.data, int(level)))


def weight_bs(r: float, rc_rows, nlevels: int) -> float:
    rc = np.ascontiguousarray(rc_rows, dtype=np.float64)
    assert rc.size >= nlevels
    return float(_L().genga_oracle_weight_bs(float(r), rc.ctypes.data, int(nlevels)))


@dataclass
class OracleResult:
    rows: np.ndarray        # [nrows] body indices evaluated
    acc: np.ndarray         # [3, nrows]
    S: np.ndarray           # [3, nrows]  sum_j |term| per component
    count: np.ndarray       # [nrows] partners per body
    partners: list          # list of int32 arrays (ascending j), one per row
    border: np.ndarray      # [nb, 2] borderline (i, j) pairs, |r/(f rc) - 1| <= 1e-12
    coincident: bool        # a distinct pair with r2 == 0 was met (outside the domain)


def kick(pos, mass, rcrit, n_massive, n_test=0, level=0, G=1.0, enc_factor=1.0, rows=None, maxp=64, tp_mode=1):
    """Evaluate the oracle for ``rows`` (default: every body).  Arrays as in SURVEY.md 8(b).
    tp_mode 1: test particles exert no force (TP 1); 2: they act on the massive bodies (TP 2)."""
    n = int(n_massive) + int(n_test)
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    rcrit = np.ascontiguousarray(rcrit, dtype=np.float64).reshape(-1, n)
    assert pos.shape == (3, n) and mass.shape == (n,) and rcrit.shape[0] >= level + 1
    rows = np.arange(n, dtype=np.int32) if rows is None else np.ascontiguousarray(rows, dtype=np.int32)
    nr = rows.size
    acc = np.zeros((3, nr)); S = np.zeros((3, nr)); count = np.zeros(nr, dtype=np.int32)
    bcap = 1 << 16
    border = np.zeros((bcap, 2), dtype=np.int32)
    nb = C.c_int64(0)
    while True:
        part = np.full((nr, maxp), -1, dtype=np.int32)
        nb.value = 0
        rc = _L().genga_oracle_kick_tp(int(n_massive), int(n_test), int(tp_mode), int(level), float(G), float(enc_factor),
                                    pos.ctypes.data, mass.ctypes.data, rcrit.ctypes.data,
                                    rows.ctypes.data, nr, acc.ctypes.data, S.ctypes.data, count.ctypes.data,
                                    part.ctypes.data, int(maxp), border.ctypes.data, bcap, C.byref(nb))
        mx = int(count.max()) if nr else 0
        if mx <= maxp:
            break
        maxp = mx                      # second pass with room for the longest partner list
    partners = [part[q, :count[q]].copy() for q in range(nr)]
    return OracleResult(rows=rows, acc=acc, S=S, count=count, partners=partners,
                        border=border[:min(nb.value, bcap)].copy(), coincident=(rc != 0))


def pair_set(res: OracleResult, n_massive: int) -> np.ndarray:
    """The encounter pair list implied by the partner lists, as sorted rows (lo, hi), each unordered
    pair once (reading G11).  With rows = all bodies this is the full list; with a subset it is the
    set of pairs that contain at least one evaluated body."""
    out = set()
    for q, i in enumerate(res.rows.tolist()):
        for j in res.partners[q].tolist():
            out.add((i, j) if i < j else (j, i))
    arr = np.array(sorted(out), dtype=np.int32).reshape(-1, 2)
    return arr


@dataclass
class ListKickResult:
    acc: np.ndarray         # [3, N]
    S: np.ndarray           # [3, N]
    count: np.ndarray       # [N] level-L partners among the listed pairs
    enc: np.ndarray         # [n_pairs] bool: the pair is a level-L encounter pair
    border: np.ndarray      # [n_pairs] bool: within 1e-12 of the threshold
    coincident: bool


def kick_list(pos, mass, rcrit, n_massive, n_test, pairs, level=1, G=1.0, enc_factor=1.0, tp_mode=1):
    """KickS (App. A): the level-`level` kick over the pairs of a list + their level pre-check."""
    n = int(n_massive) + int(n_test)
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    rcrit = np.ascontiguousarray(rcrit, dtype=np.float64).reshape(-1, n)
    pr = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
    assert rcrit.shape[0] >= level + 1 and (pr.size == 0 or (pr.min() >= 0 and pr.max() < n))
    acc = np.zeros((3, n)); S = np.zeros((3, n)); count = np.zeros(n, dtype=np.int32)
    enc = np.zeros(max(len(pr), 1), dtype=np.int8); border = np.zeros(max(len(pr), 1), dtype=np.int8)
    rc = _L().genga_oracle_kick_list(int(n_massive), int(n_test), int(tp_mode), int(level), float(G), float(enc_factor),
                                     pos.ctypes.data, mass.ctypes.data, rcrit.ctypes.data, pr.ctypes.data, len(pr),
                                     acc.ctypes.data, S.ctypes.data, count.ctypes.data, enc.ctypes.data,
                                     border.ctypes.data)
    return ListKickResult(acc=acc, S=S, count=count, enc=enc[:len(pr)].astype(bool), border=border[:len(pr)].astype(bool),
                          coincident=(rc != 0))
