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
    bs_totals: tuple = (0, 0, 0, 0)   # step-size control of the Bulirsch-Stoer phase: accepted, rejected, force evaluations, groups


def hybrid_step(pos, vel, mass, n_massive, n_test, m_star, G, dt, tol=1e-12, enc_factor=1.0, n1=3.0, n2=0.4,
                max_group=None, tp_mode=1):
    """The complete scheme of App. A, every candidate pair of the pre-check treated as an encounter
    pair (no separate detection: PAPER.md gives no criterion, and a pair that never enters its critical radius has
    W_BS = 0, so integrating it is only extra work):
        Rcrit(dt); Kick(dt/2) + pre-check; HC(dt/2); FG(dt); grouping; Bulirsch-Stoer(dt) on the groups, from the
        state before FG; HC(dt/2); Kick(dt/2)."""
    from . import group as _group, bs as _bs
    q, v, mass = _c(pos).copy(), _c(vel).copy(), _c(mass)
    n = q.shape[1]
    rc, bad0 = rcrit(q, v, mass, m_star, G, dt, 2.0, 1, n1, n2)
    tpn = n_massive if n_test > 0 else None                # bodies from here on are semi-active particles
    k1 = _kick.kick(q, mass, rc, n_massive, n_test, level=0, G=G, enc_factor=enc_factor, maxp=256, tp_mode=tp_mode)
    v = v + (0.5 * dt) * k1.acc
    q, _ = hc(q, v, mass, m_star, 0.5 * dt)
    q_in, v_in = q.copy(), v.copy()
    q, v, bad1 = fg(q, v, G * m_star, dt)
    gr = _group.group(n, _kick.pair_set(k1, n_massive))
    q, v, bstats, skipped = _bs.bs(q_in, v_in, mass, rc, gr.members, gr.offsets, G, m_star, dt, tol, q, v, nlevels=1,
                                   max_group=max_group, n_massive=tpn, tp_mode=tp_mode)
    q, _ = hc(q, v, mass, m_star, 0.5 * dt)
    k2 = _kick.kick(q, mass, rc, n_massive, n_test, level=0, G=G, enc_factor=enc_factor, maxp=256, tp_mode=tp_mode)
    v = v + (0.5 * dt) * k2.acc
    return HybridStepResult(pos=q, vel=v, rcrit=rc, first=k1, groups=gr, skipped=skipped, unbound=bad0 + bad1,
                            bs_totals=_bs_totals(bstats))


def _bs_totals(stats):
    """(accepted macro steps, rejected attempts, force evaluations, groups) summed over a list of BsStats: the record
    of the step-size control a kernel's genga_bs_totals is compared with."""
    return (sum(s.accepted for s in stats), sum(s.rejected for s in stats), sum(s.force_evaluations for s in stats),
            len(stats))


@dataclass
class MultilevelStepResult:
    pos: np.ndarray
    vel: np.ndarray
    rcrit: np.ndarray        # [slevels, N]: row 0 of Rcrit(dt); rows >= 1 as the LAST RcritS of each level left them
    first: _kick.OracleResult
    stats: np.ndarray        # [slevels, 4] per level, summed over its sub-steps: candidate pairs, close-encounter pairs,
                             # groups handed to Bulirsch-Stoer, bodies in them
    unbound: int
    bs_totals: tuple = (0, 0, 0, 0)   # step-size control of all Bulirsch-Stoer calls: accepted, rejected, force evaluations, groups


def multilevel_step(pos, vel, mass, n_massive, n_test, m_star, G, dt, slevels=2, substeps=2, tol=1e-12, enc_factor=1.0,
                    n1=3.0, n2=0.4, detect=True, max_group=None, tp_mode=1):
    """The multi-level scheme of App. A, written as printed there:

        Rcrit(dt); Kick(dt/2) + pre-check; HC(dt/2); FG(dt)
        if candidates: close-encounter detection
        if SLevels > 1:  if close-encounters: SEnc(dt, 1.0, 0)
        else:            if close-encounters: grouping; Bulirsch-Stoer(dt)
        HC(dt/2); Kick(dt/2)

        SEnc(dt, ds, SLevel):  groupS;  SLevel += 1;  ds *= substeps
          for s in range(substeps):
            RcritS();  KickS(dt/ds/2);  FGS(dt/ds);  close-encounter detection
            if close-encounters:
              if SLevel < SLevels - 1: SEnc(dt, ds, SLevel)
              else: grouping; Bulirsch-Stoer(dt/ds)
            KickS(dt/ds/2)

    Readings (G17): level l >= 1 works on the close-encounter pairs of level l-1 (groupS) and on the bodies in
    them ("the relevant bodies"); those bodies restart from their state BEFORE the upper level's drift (as the
    Bulirsch-Stoer phase does, G15), which the sub-steps replace; RcritS writes row l of eq. 5 at dt/substeps^l from the
    current velocities; KickS is the level-l kick of eq. 63 over the listed pairs with its level-l
    pre-check; the Bulirsch-Stoer phase of the deepest level carries W_BS = prod_{k < SLevels} (1 - K_k).
    detect=False: every candidate of a pre-check counts as a close-encounter pair (as hybrid_step does).
    tp_mode: the test-particle mode of every kick and of the Bulirsch-Stoer phase (sec. 8.1)."""
    from . import group as _group, bs as _bs, detect as _det
    q, v, mass = _c(pos).copy(), _c(vel).copy(), _c(mass)
    n = q.shape[1]
    mu = G * m_star
    rc = np.zeros((slevels, n))
    row, bad = rcrit(q, v, mass, m_star, G, dt, 2.0, 1, n1, n2)
    rc[0] = row[0]
    stats = np.zeros((slevels, 4), dtype=np.int64)
    unbound = [bad]
    bs_all = []

    def encounters(level, q0, v0, q1, v1, h, cand):
        enc = _det.detect(q0, v0, q1, v1, rc[level], h, cand, enc_factor=1.0).pairs if detect else cand
        stats[level, 0] += len(cand); stats[level, 1] += len(enc)
        return enc, _group.group(n, enc)

    def bulirsch_stoer(level, q0, v0, h, gr, q, v):
        q, v, bstats, skipped = _bs.bs(q0, v0, mass, rc, gr.members, gr.offsets, G, m_star, h, tol, q, v, nlevels=level + 1,
                                       max_group=max_group, n_massive=n_massive if n_test > 0 else None, tp_mode=tp_mode)
        bs_all.extend(bstats)
        stats[level, 2] += gr.n_groups - len(skipped)
        stats[level, 3] += len(gr.members) - sum(int(gr.offsets[g + 1] - gr.offsets[g]) for g in skipped)
        return q, v

    def senc(q, v, level, pairs_up, bodies):                # `level` is the level being entered (SLevel += 1)
        h = dt / float(substeps) ** level                   # dt / ds
        for s in range(substeps):
            row, _ = rcrit(q, v, mass, m_star, G, h, 2.0, 1, n1, n2)                    # RcritS
            rc[level, bodies] = row[0, bodies]
            ks = _kick.kick_list(q, mass, rc[:level + 1], n_massive, n_test, pairs_up, level=level, G=G,
                                 enc_factor=enc_factor, tp_mode=tp_mode)                 # KickS(dt/ds/2)
            v = v + (0.5 * h) * ks.acc
            q0, v0 = q.copy(), v.copy()
            qf, vf, b1 = fg(q, v, mu, h)                                                 # FGS(dt/ds)
            q[:, bodies], v[:, bodies] = qf[:, bodies], vf[:, bodies]
            enc, gr = encounters(level, q0, v0, q, v, h, pairs_up[ks.enc])
            if len(enc):
                if level < slevels - 1:
                    b = np.asarray(gr.members)
                    q[:, b], v[:, b] = q0[:, b], v0[:, b]
                    q, v = senc(q, v, level + 1, enc, b)
                else:
                    q, v = bulirsch_stoer(level, q0, v0, h, gr, q, v)
            ks = _kick.kick_list(q, mass, rc[:level + 1], n_massive, n_test, pairs_up, level=level, G=G,
                                 enc_factor=enc_factor, tp_mode=tp_mode)                 # KickS(dt/ds/2)
            v = v + (0.5 * h) * ks.acc
        return q, v

    k1 = _kick.kick(q, mass, rc[:1], n_massive, n_test, level=0, G=G, enc_factor=enc_factor, maxp=256, tp_mode=tp_mode)
    v = v + (0.5 * dt) * k1.acc
    q, _ = hc(q, v, mass, m_star, 0.5 * dt)
    q_in, v_in = q.copy(), v.copy()
    q, v, bad1 = fg(q, v, mu, dt)
    unbound.append(bad1)
    enc, gr = encounters(0, q_in, v_in, q, v, dt, _kick.pair_set(k1, n_massive))
    if len(enc):
        if slevels > 1:
            b = np.asarray(gr.members)
            q[:, b], v[:, b] = q_in[:, b], v_in[:, b]
            q, v = senc(q, v, 1, enc, b)
        else:
            q, v = bulirsch_stoer(0, q_in, v_in, dt, gr, q, v)
    q, _ = hc(q, v, mass, m_star, 0.5 * dt)
    k2 = _kick.kick(q, mass, rc[:1], n_massive, n_test, level=0, G=G, enc_factor=enc_factor, maxp=256, tp_mode=tp_mode)
    v = v + (0.5 * dt) * k2.acc
    return MultilevelStepResult(pos=q, vel=v, rcrit=rc, first=k1, stats=stats, unbound=sum(unbound),
                                bs_totals=_bs_totals(bs_all))


def steps(pos, vel, mass, n_massive, n_test, m_star, G, dt, n_steps, slevels=0, **kw):
    """n_steps consecutive steps: the definition of what genga_steps computes IS the repetition of the single step
    (App. A, `n_steps` times) -- merging the closing kick of a step with the opening kick of the next
    is a device-side economy that must not change the result beyond rounding.  slevels = 0: `step` (no encounter
    branch); slevels >= 1: `multilevel_step` (kw: substeps, tol, detect, ...).  Returns the list of per-step results."""
    q, v = _c(pos).copy(), _c(vel).copy()
    out = []
    for _ in range(n_steps):
        if slevels == 0:
            r = step(q, v, mass, n_massive, n_test, m_star, G, dt, **{k: w for k, w in kw.items() if k in ("enc_factor", "n1", "n2")})
        else:
            r = multilevel_step(q, v, mass, n_massive, n_test, m_star, G, dt, slevels=slevels, **kw)
        q, v = r.pos, r.vel
        out.append(r)
    return out
