"""Pins of the detection oracle (oracle/genga_detect_oracle.c; App. A; reading G16) against what
the mathematics fixes.  The CHOICE of the criterion is unpinned by the paper (the header says so); what is pinned here
is that the oracle computes the minimum of the cubic Hermite interpolant of the squared separation, and the decision
and bookkeeping that follow from it."""
import numpy as np
import pytest
from scipy.interpolate import CubicHermiteSpline


@pytest.fixture(scope="module")
def det(oracle_mod):
    return oracle_mod.detect


def test_uniform_relative_motion_gives_the_exact_closest_approach(det):
    """Straight-line relative motion: r^2(t) is a parabola, which the cubic Hermite interpolant reproduces exactly, so
    the minimum is the textbook closest approach |d x u| / |u| (or an end point if the approach is outside the step)."""
    rng = np.random.default_rng(5)
    for k in range(200):
        d = rng.normal(size=3); u = rng.normal(size=3); h = rng.uniform(0.2, 3.0)
        t_star = -np.dot(d, u) / np.dot(u, u)
        d0 = np.dot(d, d); d1 = np.dot(d + h * u, d + h * u)
        m0 = h * 2 * np.dot(d, u); m1 = h * 2 * np.dot(d + h * u, u)
        got, tau = det.hermite_min(d0, m0, d1, m1)
        if 0 < t_star < h:
            want = np.dot(np.cross(d, u), np.cross(d, u)) / np.dot(u, u)
            assert abs(tau - t_star / h) < 1e-9
        else:
            want = min(d0, d1)
        assert abs(got - want) <= 1e-12 * max(d0, d1)


def test_minimum_against_a_dense_scan_of_scipys_hermite_spline(det):
    rng = np.random.default_rng(6)
    tt = np.linspace(0.0, 1.0, 20001)
    inner = 0
    for k in range(300):
        d0, d1 = rng.uniform(0.1, 2.0, size=2)
        m0, m1 = rng.normal(scale=3.0, size=2)
        sp = CubicHermiteSpline([0.0, 1.0], [d0, d1], [m0, m1])
        scan = sp(tt)
        got, tau = det.hermite_min(d0, m0, d1, m1)
        assert got <= scan.min() + 1e-12 and abs(got - scan.min()) < 2e-7 * (abs(m0) + abs(m1) + 1)
        assert abs(sp(tau) - got) < 1e-12 * (abs(got) + d0 + d1 + abs(m0) + abs(m1))     # the value IS on the interpolant
        inner += 0 < tau < 1
    assert 50 < inner < 290          # both branches were exercised


def test_interpolation_conditions_and_degenerate_cases(det):
    # monotone: minimum at an end point
    assert det.hermite_min(1.0, 0.5, 2.0, 0.5) == (1.0, 0.0)
    assert det.hermite_min(2.0, -0.5, 1.0, -0.5) == (1.0, 1.0)
    # symmetric dip: p = d0 + m0 t + b t^2 with m1 = -m0, d1 = d0  =>  tau = 1/2, p = d0 + m0/4
    v, tau = det.hermite_min(1.0, -2.0, 1.0, 2.0)
    assert tau == 0.5 and v == 0.5
    # a bump (interior MAXIMUM only): the end points decide
    v, tau = det.hermite_min(1.0, 2.0, 1.0, -2.0)
    assert v == 1.0 and tau in (0.0, 1.0)
    # time reversal: (d0, m0, d1, m1) -> (d1, -m1, d0, -m0) has the same minimum at 1 - tau
    rng = np.random.default_rng(7)
    for k in range(100):
        d0, d1 = rng.uniform(0.1, 2.0, size=2); m0, m1 = rng.normal(scale=3.0, size=2)
        v1, t1 = det.hermite_min(d0, m0, d1, m1); v2, t2 = det.hermite_min(d1, -m1, d0, -m0)
        assert abs(v1 - v2) < 1e-13 * (d0 + d1 + abs(m0) + abs(m1)) and (abs(t1 + t2 - 1) < 1e-9 or abs(v1 - min(d0, d1)) < 1e-13)


def _flyby(n_pairs, seed, h=2.0):
    """n_pairs independent two-body fly-bys on straight lines (states before / after consistent with uniform motion)."""
    rng = np.random.default_rng(seed)
    n = 2 * n_pairs
    pos0 = rng.normal(size=(3, n)); vel = rng.normal(scale=0.3, size=(3, n))
    # partner j = i + n_pairs starts close to i
    pos0[:, n_pairs:] = pos0[:, :n_pairs] + rng.normal(scale=0.4, size=(3, n_pairs))
    pos1 = pos0 + h * vel
    pairs = np.stack([np.arange(n_pairs), np.arange(n_pairs) + n_pairs], 1).astype(np.int32)
    return pos0, vel, pos1, vel.copy(), pairs, h


def test_decision_counts_and_symmetry(det):
    pos0, vel0, pos1, vel1, pairs, h = _flyby(500, 11)
    n = pos0.shape[1]
    rc = np.full(n, 0.3)
    r = det.detect(pos0, vel0, pos1, vel1, rc, h, pairs)
    # the textbook decision for straight lines
    d = pos0[:, pairs[:, 1]] - pos0[:, pairs[:, 0]]; u = vel0[:, pairs[:, 1]] - vel0[:, pairs[:, 0]]
    t = np.clip(-(d * u).sum(0) / (u * u).sum(0), 0.0, h)
    want = ((d + t * u) ** 2).sum(0) < 0.09
    clear = np.abs(np.sqrt(((d + t * u) ** 2).sum(0)) / 0.3 - 1) > 1e-9
    assert np.array_equal(r.enc[clear], want[clear]) and 50 < r.enc.sum() < 450
    # misses at BOTH end points but inside in between exist, and are found
    ends = np.minimum((d * d).sum(0), ((d + h * u) ** 2).sum(0)) >= 0.09
    assert (r.enc & ends).sum() > 5
    # counts: every body is in at most one pair here
    cnt = np.zeros(n, dtype=np.int32); np.add.at(cnt, r.pairs.reshape(-1), 1)
    assert np.array_equal(cnt, r.count) and r.count.sum() == 2 * r.enc.sum() and len(r.pairs) == r.enc.sum()
    # i <-> j
    r2 = det.detect(pos0, vel0, pos1, vel1, rc, h, pairs[:, ::-1])
    assert np.array_equal(r.enc, r2.enc) and np.array_equal(r.d2min, r2.d2min)
    # pair radius is max(rc_i, rc_j) (reading G2), scaled by enc_factor
    rc2 = rc.copy(); rc2[: n // 2] = 0.0
    assert np.array_equal(det.detect(pos0, vel0, pos1, vel1, rc2, h, pairs).enc, r.enc)
    wide = det.detect(pos0, vel0, pos1, vel1, rc, h, pairs, enc_factor=2.0)
    assert np.array_equal(wide.enc, det.detect(pos0, vel0, pos1, vel1, 2 * rc, h, pairs).enc) and wide.enc.sum() > r.enc.sum()
    # empty list
    e = det.detect(pos0, vel0, pos1, vel1, rc, h, np.zeros((0, 2), dtype=np.int32))
    assert e.enc.size == 0 and e.count.sum() == 0


def test_kepler_drifted_pairs_are_a_subset_of_candidates_and_contain_both_end_point_sets(det, oracle_mod):
    """On a disk: with the states before / after FG, every candidate that is inside its critical radius at either end of
    the drift is an encounter pair (p(0) = d0, p(1) = d1 are in the minimum), and no pair is invented."""
    import genga_inputs as gi
    ki = gi.make_config(0, n=1500)
    st = oracle_mod.step
    q1, v1, _ = st.fg(ki.pos, ki.vel, ki.G * 1.0, ki.dt)
    wide = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n, 0, level=0, G=ki.G, enc_factor=3.0, maxp=256)
    cand = oracle_mod.pair_set(wide, ki.n)
    r = det.detect(ki.pos, ki.vel, q1, v1, ki.rcrit[0], ki.dt, cand)
    rc = np.maximum(ki.rcrit[0][cand[:, 0]], ki.rcrit[0][cand[:, 1]])
    d0 = np.sqrt(((ki.pos[:, cand[:, 0]] - ki.pos[:, cand[:, 1]]) ** 2).sum(0))
    d1 = np.sqrt(((q1[:, cand[:, 0]] - q1[:, cand[:, 1]]) ** 2).sum(0))
    at_ends = (d0 < rc * (1 - 1e-9)) | (d1 < rc * (1 - 1e-9))
    assert at_ends.sum() > 20 and r.enc[at_ends].all()
    assert r.enc.sum() < len(cand)                                   # the pre-check over-selects, detection prunes
    assert (r.enc & ~at_ends).sum() >= 0 and np.all(r.d2min[r.enc] < rc[r.enc] ** 2)
