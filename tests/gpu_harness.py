"""Helpers of the -m gpu parity tests: run the CUDA path through the C-ABI binding on a KickInputs,
and compare it with the CPU oracle under north_star's acceptance rule."""
from dataclasses import dataclass
import numpy as np


@dataclass
class GpuResult:
    acc: np.ndarray        # [3, N]
    pairs: np.ndarray      # [min(total, capacity), 2] as written (arbitrary order)
    counts: np.ndarray     # [N]
    total: int
    vel: np.ndarray = None
    status: int = 0
    launches: int = 0


def run_gpu(ki, level=None, capacity=1 << 20, with_vel=False, host=False, kick=None, rcrit=None, order_mode=0,
            tp_mode=1):
    import torch
    from paper_2201_10058_b200 import GengaKick
    level = ki.level if level is None else level
    n = ki.n
    own = kick is None
    if own:
        kick = GengaKick(ki.n_massive, ki.n_test, max_level=level, pair_capacity=capacity, G=ki.G,
                         enc_factor=ki.enc_factor, order_mode=order_mode, tp_mode=tp_mode)
    dev = "cpu" if host else "cuda"
    t = lambda a, dt=torch.float64: torch.from_numpy(np.array(a, copy=True)).to(dt).to(dev).contiguous()
    pos, mass = t(ki.pos), t(ki.mass)
    rc = t(ki.rcrit[:level + 1] if rcrit is None else rcrit)
    vel = t(ki.vel) if with_vel else None
    acc = torch.full((3, n), float("nan"), dtype=torch.float64, device=dev)
    pairs = torch.full((max(capacity, 1), 2), -7, dtype=torch.int32, device=dev)
    npairs = torch.full((n + 1,), -7, dtype=torch.int32, device=dev)
    if host:
        kick.kick_host(pos, vel, mass, rc, level, ki.dt, acc, pairs if capacity else None, npairs)
    else:
        kick.set_stream(torch.cuda.current_stream().cuda_stream)
        kick.kick(pos, vel, mass, rc, level, ki.dt, acc, pairs if capacity else None, npairs)
        torch.cuda.synchronize()
    npn = npairs.cpu().numpy()
    total = int(npn[n])
    res = GpuResult(acc=acc.cpu().numpy(), pairs=pairs.cpu().numpy()[:min(total, capacity)].copy(),
                    counts=npn[:n].copy(), total=total, vel=None if vel is None else vel.cpu().numpy(),
                    status=kick.status(), launches=kick.launch_count())
    if own:
        kick.free()
    return res


def sorted_pairs(pairs):
    p = np.asarray(pairs, dtype=np.int64).reshape(-1, 2)
    if p.size == 0:
        return p
    order = np.lexsort((p[:, 1], p[:, 0]))
    return p[order]


def compare(gpu, orc, n_massive, tol=1e-13, rows=None, check_pairs=True):
    """north_star's rule.  `orc` is an oracle.OracleResult for `rows` (None = all bodies).
    Returns a dict of diagnostics; raises AssertionError on a violation."""
    import oracle
    rows = np.arange(gpu.acc.shape[1]) if rows is None else np.asarray(rows)
    a_g = gpu.acc[:, rows]
    err = np.abs(a_g - orc.acc)
    bound = tol * orc.S
    # a body with no contributing partner has S = 0 and must get exactly 0
    bad = err > bound
    assert not bad.any(), (f"acceleration outside {tol:g} * sum|term|: {int(bad.sum())} components, "
                           f"worst ratio {np.max(err[bad] / np.maximum(bound[bad], 1e-300)):.3g}")
    ratio = float(np.max(np.where(orc.S > 0, err / np.maximum(orc.S, 1e-300), 0.0))) if err.size else 0.0
    border = {tuple(sorted(p)) for p in orc.border.tolist()}
    n_border_diff = 0
    if check_pairs:
        want = {tuple(p) for p in oracle.pair_set(orc, n_massive).tolist()}
        got_all = [tuple(p) for p in gpu.pairs.tolist()]
        assert len(got_all) == len(set(got_all)), "a pair was emitted twice"
        assert all(p[0] < p[1] for p in got_all), "a pair row is not (lo, hi)"
        rowset = set(rows.tolist())
        got = {p for p in got_all if p[0] in rowset or p[1] in rowset}
        diff = got ^ want
        assert diff <= border, f"pair sets differ outside the 1e-12 band: {sorted(diff - border)[:10]}"
        n_border_diff = len(diff)
        cdiff = np.nonzero(gpu.counts[rows] != orc.count)[0]
        touched = {b for p in diff for b in p}
        assert all(int(rows[q]) in touched for q in cdiff), "per-body encounter counts differ"
        if rows.size == gpu.acc.shape[1]:
            assert gpu.total == len(got_all) or gpu.total > len(got_all)
    return dict(max_err_over_S=ratio, borderline=len(border), borderline_mismatch=n_border_diff)
