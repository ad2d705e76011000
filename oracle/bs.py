"""ctypes marshalling for genga_bs_oracle.c (Bulirsch-Stoer integration of close-encounter groups).
TEST INFRASTRUCTURE ONLY; see the C header."""
import ctypes as C
from dataclasses import dataclass
import numpy as np

from . import oracle as _kick

_ready = False


def _L():
    global _ready
    lib = _kick._L()
    if not _ready:
        d, i32, p = C.c_double, C.c_int32, C.c_void_p
        lib.genga_oracle_bs_group.restype = C.c_int
        lib.genga_oracle_bs_group.argtypes = [i32, i32, d, d, d, d, p, p, p, p, p]
        lib.genga_oracle_bs_group_tp.restype = C.c_int
        lib.genga_oracle_bs_group_tp.argtypes = [i32, i32, d, d, d, d, p, p, p, p, p, p, i32]
        _ready = True
    return lib


@dataclass
class BsStats:
    accepted: int
    rejected: int
    force_evaluations: int
    failed: bool


def bs_group(pos, vel, mass, rcrit_rows, G, m_star, dt, tol, is_tp=None, tp_mode=1):
    """One group.  pos, vel [3, n] (the group's bodies), mass [n], rcrit_rows [nlevels, n].
    is_tp [n] bool: semi-active test particles (sec. 8.1): they feel the massive bodies, act on them
    only with tp_mode = 2, and never feel each other; None: fully interactive.
    Returns (pos, vel, BsStats) after dt."""
    pos = np.asarray(pos, dtype=np.float64); vel = np.asarray(vel, dtype=np.float64)
    n = pos.shape[1]
    q = np.ascontiguousarray(pos.T).copy(); v = np.ascontiguousarray(vel.T).copy()      # body-major [n, 3]
    m = np.ascontiguousarray(mass, dtype=np.float64)
    rc = np.ascontiguousarray(np.asarray(rcrit_rows, dtype=np.float64).reshape(-1, n))
    st = np.zeros(3, dtype=np.int64)
    if is_tp is None:
        fail = _L().genga_oracle_bs_group(n, rc.shape[0], float(G), float(m_star), float(dt), float(tol), m.ctypes.data,
                                          rc.ctypes.data, q.ctypes.data, v.ctypes.data, st.ctypes.data)
    else:
        tp = np.ascontiguousarray(is_tp, dtype=np.int8)
        fail = _L().genga_oracle_bs_group_tp(n, rc.shape[0], float(G), float(m_star), float(dt), float(tol), m.ctypes.data,
                                             rc.ctypes.data, q.ctypes.data, v.ctypes.data, st.ctypes.data, tp.ctypes.data,
                                             int(tp_mode))
    return np.ascontiguousarray(q.T), np.ascontiguousarray(v.T), BsStats(int(st[0]), int(st[1]), int(st[2]), bool(fail))


def bs(pos_in, vel_in, mass, rcrit, members, offsets, G, m_star, dt, tol, pos, vel, nlevels=1, max_group=None,
       n_massive=None, tp_mode=1):
    """All groups: members / offsets as genga_group writes them.  pos_in, vel_in: the state before the Kepler
    drift; pos, vel: arrays to update (copies are returned) -- only the members of integrated groups change.
    Groups larger than max_group are skipped (returned in the list `skipped`).
    n_massive: bodies from this index on are semi-active test particles (None: all fully interactive)."""
    pos, vel = np.array(pos, dtype=np.float64, copy=True), np.array(vel, dtype=np.float64, copy=True)
    rc = np.asarray(rcrit, dtype=np.float64).reshape(-1, pos.shape[1])[:nlevels]
    skipped, stats = [], []
    for g in range(len(offsets) - 1):
        idx = np.asarray(members[offsets[g]:offsets[g + 1]])
        if max_group is not None and idx.size > max_group:
            skipped.append(g)
            continue
        q, v, st = bs_group(pos_in[:, idx], vel_in[:, idx], np.asarray(mass)[idx], rc[:, idx], G, m_star, dt, tol,
                            is_tp=None if n_massive is None else idx >= n_massive, tp_mode=tp_mode)
        pos[:, idx], vel[:, idx] = q, v
        stats.append(st)
    return pos, vel, stats, skipped
