"""ctypes marshalling for genga_step_oracle.c and the composition of one hybrid step without the
Bulirsch-Stoer branch (App. A).  TEST INFRASTRUCTURE ONLY; see the C header."""
import ctypes as C
from dataclasses import dataclass
import numpy as np

from . import oracle as _kick

_ready = False


def _L():
    global _ready
    lib = _kick._L()
    if not _ready:
        d, i32, i64, p = C.c_double, C.c_int32, C.c_int64, C.c_void_p
        lib.genga_oracle_rcrit.restype = i64
        lib.genga_oracle_rcrit.argtypes = [i64, p, p, p, d, d, d, d, i32, d, d, p]
        lib.genga_oracle_hc.restype = None
        lib.genga_oracle_hc.argtypes = [i64, p, p, p, d, d, p]
        lib.genga_oracle_fg.restype = i64
        lib.genga_oracle_fg.argtypes = [i64, p, p, d, d]
        _ready = True
    return lib


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def rcrit(pos, vel, mass, m_star, G, dt, substeps=2.0, nrows=1, n1=3.0, n2=0.4):
    """eq. 5 rows [nrows, N].  Returns (rows, number of unbound bodies)."""
    pos, vel, mass = _c(pos), _c(vel), _c(mass)
    n = mass.size
    out = np.zeros((nrows, n))
    bad = _L().genga_oracle_rcrit(n, pos.ctypes.data, vel.ctypes.data, mass.ctypes.data, float(m_star), float(G),
                                  float(dt), float(substeps), int(nrows), float(n1), float(n2), out.ctypes.data)
    return out, int(bad)


def hc(pos, vel, mass, m_star, dt):
    """eq. 4.  Returns (new positions, sum_j m_j v_j)."""
    q, vel, mass = _c(pos).copy(), _c(vel), _c(mass)
    p = np.zeros(3)
    _L().genga_oracle_hc(mass.size, q.ctypes.data, vel.ctypes.data, mass.ctypes.data, float(m_star), float(dt),
                         p.ctypes.data)
    return q, p


def fg(pos, vel, mu, dt):
    """Kepler drift (eq. 2's two-body part).  Returns (q, v, number of unbound bodies)."""
    q, v = _c(pos).copy(), _c(vel).copy()
    bad = _L().genga_oracle_fg(q.shape[1], q.ctypes.data, v.ctypes.data, float(mu), float(dt))
    return q, v, int(bad)


@dataclass
class StepResult:
    pos: np.ndarray          # [3, N] after the step
    vel: np.ndarray          # [3, N]
    rcrit: np.ndarray        # [1, N] the row Rcrit(dt) produced at the start of the step
    first: _kick.OracleResult    # the first Kick(dt/2) + pre-check (its pair list is the step's candidate list)
    second: _kick.OracleResult   # the closing Kick(dt/2)
    unbound: int


def step(pos, vel, mass, n_massive, n_test, m_star, G, dt, enc_factor=1.0, n1=3.0, n2=0.4):
    """Rcrit(dt); Kick(dt/2) + pre-check; HC(dt/2); FG(dt); HC(dt/2); Kick(dt/2)   (App. A, no encounters
    resolved: the Bulirsch-Stoer branch is off this path)."""
    q, v, mass = _c(pos).copy(), _c(vel).copy(), _c(mass)
    rc, bad0 = rcrit(q, v, mass, m_star, G, dt, 2.0, 1, n1, n2)
    k1 = _kick.kick(q, mass, rc, n_massive, n_test, level=0, G=G, enc_factor=enc_factor)
    v = v + (0.5 * dt) * k1.acc
    q, _ = hc(q, v, mass, m_star, 0.5 * dt)
    q, v, bad1 = fg(q, v, G * m_star, dt)
    q, _ = hc(q, v, mass, m_star, 0.5 * dt)
    k2 = _kick.kick(q, mass, rc, n_massive, n_test, level=0, G=G, enc_factor=enc_factor)
    v = v + (0.5 * dt) * k2.acc
    return StepResult(pos=q, vel=v, rcrit=rc, first=k1, second=k2, unbound=bad0 + bad1)


@dataclass
class HybridStepResult:
    pos: np.ndarray
    vel: np.ndarray
    rcrit: np.ndarray
    first: _kick.OracleResult
    groups: object           # oracle.group.Groups of the first kick's pair list
    skipped: list            # groups larger than max_group (left at their Kepler-drifted state)
    unbound: int


def hybrid_step(pos, vel, mass, n_massive, n_test, m_star, G, dt, tol=1e-12, enc_factor=1.0, n1=3.0, n2=0.4,
                max_group=None):
    """The complete scheme of App. A, every candidate pair of the pre-check treated as an encounter
    pair (no separate detection: PAPER.md gives no criterion, and a pair that never enters its critical radius has
    W_BS = 0, so integrating it is only extra work):
        Rcrit(dt); Kick(dt/2) + pre-check; HC(dt/2); FG(dt); grouping; Bulirsch-Stoer(dt) on the groups, from the
        state before FG; HC(dt/2); Kick(dt/2)."""
    from . import group as _group, bs as _bs
    q, v, mass = _c(pos).copy(), _c(vel).copy(), _c(mass)
    n = q.shape[1]
    rc, bad0 = rcrit(q, v, mass, m_star, G, dt, 2.0, 1, n1, n2)
    k1 = _kick.kick(q, mass, rc, n_massive, n_test, level=0, G=G, enc_factor=enc_factor, maxp=256)
    v = v + (0.5 * dt) * k1.acc
    q, _ = hc(q, v, mass, m_star, 0.5 * dt)
    q_in, v_in = q.copy(), v.copy()
    q, v, bad1 = fg(q, v, G * m_star, dt)
    gr = _group.group(n, _kick.pair_set(k1, n_massive))
    q, v, _, skipped = _bs.bs(q_in, v_in, mass, rc, gr.members, gr.offsets, G, m_star, dt, tol, q, v, nlevels=1,
                              max_group=max_group)
    q, _ = hc(q, v, mass, m_star, 0.5 * dt)
    k2 = _kick.kick(q, mass, rc, n_massive, n_test, level=0, G=G, enc_factor=enc_factor, maxp=256)
    v = v + (0.5 * dt) * k2.acc
    return HybridStepResult(pos=q, vel=v, rcrit=rc, first=k1, groups=gr, skipped=skipped, unbound=bad0 + bad1)
