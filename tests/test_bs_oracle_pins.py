"""Pins of oracle/genga_bs_oracle.c (Bulirsch-Stoer integration of a close-encounter group) against the
solution of the differential equation it integrates -- closed forms, a conserved quantity, an independent
library integrator on an independently written right-hand side -- NOT against the oracle itself.  CPU only."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import genga_inputs as gi

G = gi.G_AU_DAY_MSUN
U = 2.0 ** -53


@pytest.fixture(scope="module")
def bs(oracle_mod):
    return oracle_mod.bs


def _two(a=(1.0, 1.0), e=(0.05, 0.08), M=(0.3, 0.3), dM=0.0):
    a = np.array(a); e = np.array(e); z = np.zeros(2)
    return gi.elements_to_cartesian(a, e, z + 0.01, z, z + 1.0, np.array(M) + np.array([0.0, dM]), G)


def test_far_pair_follows_kepler(bs, oracle_mod):
    """Outside each other's critical radius W_BS = 1 - K = 0: each body on its Kepler orbit (closed-form FG oracle)."""
    pos, vel = _two(a=(1.0, 1.6), M=(0.3, 2.0))
    m = np.array([3e-6, 1e-6]); rc = np.full((1, 2), 0.02)
    for dt in (6.0, -6.0, 40.0):
        q, v, st = bs.bs_group(pos, vel, m, rc, G, 1.0, dt, 1e-13)
        qf, vf, _ = oracle_mod.step.fg(pos, vel, G, dt)
        assert not st.failed and st.accepted >= 1
        assert np.max(np.abs(q - qf)) < 2e-12 and np.max(np.abs(v - vf)) < 2e-12 * np.abs(vel).max() * 10


def test_deep_encounter_conserves_the_newtonian_energy(bs):
    """Inside 0.1 r_crit K = 0, W_BS = 1: Sun (fixed centre) + two bodies with full mutual gravity.  The energy
    sum(m v^2/2 - G m m_star/r) - G m1 m2 / r12 is conserved by the exact flow; the integrator keeps it to ~tol."""
    pos, vel = _two(e=(0.05, 0.05), dM=2e-3)                   # 2e-3 AU apart on the same orbit
    m = np.array([3e-7, 2e-7]); rc = np.full((1, 2), 0.2)       # 0.1 rc = 2e-2 AU >> separation

    def energy(q, v):
        r = np.sqrt((q ** 2).sum(0)); d = np.sqrt(((q[:, 0] - q[:, 1]) ** 2).sum())
        return (0.5 * m * (v ** 2).sum(0) - G * m / r).sum() - G * m[0] * m[1] / d, d

    e0, d0 = energy(pos, vel)
    assert d0 < 0.1 * 0.2 / 5
    for tol in (1e-10, 1e-13):
        q, v, st = bs.bs_group(pos, vel, m, rc, G, 1.0, 6.0, tol)
        e1, d1 = energy(q, v)
        assert not st.failed and d1 < 0.1 * 0.2
        assert abs(e1 - e0) < 50 * tol * abs(e0)
    # the mutual term matters: without it (far-pair rule) the relative motion differs
    qk, vk, _ = bs.bs_group(pos, vel, m, np.full((1, 2), 1e-9), G, 1.0, 6.0, 1e-13)
    assert np.max(np.abs(qk - q)) > 1e-9


def _rhs(t, y, m, rc, nlev):
    """Independent numpy right-hand side: Kepler term + sum_j G m_j prod_k(1 - K_k) d / r^3."""
    n = m.size
    q = y[:3 * n].reshape(n, 3); v = y[3 * n:].reshape(n, 3)
    acc = -G * q / (np.sqrt((q ** 2).sum(1)) ** 3)[:, None]
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            d = q[j] - q[i]
            r = np.sqrt(d @ d)
            w = 1.0
            for k in range(nlev):
                c = max(rc[k, i], rc[k, j])
                yy = (r - 0.1 * c) / (0.9 * c)
                K = 0.0 if yy <= 0 else 1.0 if yy >= 1 else yy * yy / (2 * yy * yy - 2 * yy + 1)
                w *= 1.0 - K
            acc[i] += G * m[j] * w * d / r ** 3
    return np.concatenate([v.ravel(), acc.ravel()])


@pytest.mark.parametrize("nlev", [1, 2])
def test_in_band_group_against_dop853(bs, nlev):
    """Three bodies whose separations sweep the changeover band during the step, against scipy's DOP853 (rtol 1e-13)
    on the right-hand side above."""
    a = np.array([1.0, 1.0, 1.0]); e = np.array([0.02, 0.03, 0.025]); z = np.zeros(3)
    pos, vel = gi.elements_to_cartesian(a, e, z + 0.01, z, z + 1.0, np.array([0.30, 0.31, 0.295]), G)
    m = np.array([3e-6, 1e-6, 2e-6])
    rc = np.stack([np.full(3, 0.03), np.full(3, 0.015)])[:nlev]
    d01 = np.sqrt(((pos[:, 0] - pos[:, 1]) ** 2).sum())
    assert 0.1 * 0.03 < d01 < 0.03                               # inside the band of K_0
    dt = 6.0
    q, v, st = bs.bs_group(pos, vel, m, rc, G, 1.0, dt, 1e-13)
    y0 = np.concatenate([pos.T.ravel(), vel.T.ravel()])
    sol = solve_ivp(_rhs, (0.0, dt), y0, method="DOP853", rtol=1e-13, atol=1e-18, args=(m, rc, nlev))
    qs = sol.y[:9, -1].reshape(3, 3).T; vs = sol.y[9:, -1].reshape(3, 3).T
    assert not st.failed
    assert np.max(np.abs(q - qs)) < 5e-12 and np.max(np.abs(v - vs)) < 5e-12 * np.abs(vel).max() * 10
    # and the encounter does change the orbit (the test would pass trivially otherwise)
    qf = bs.bs_group(pos, vel, m, np.full((nlev, 3), 1e-9), G, 1.0, dt, 1e-13)[0]
    assert np.max(np.abs(q - qf)) > 1e-9


def test_reversibility_and_tolerance_scaling(bs):
    pos, vel = _two(dM=8e-3)
    m = np.array([3e-6, 2e-6]); rc = np.full((1, 2), 0.03)
    q, v, st = bs.bs_group(pos, vel, m, rc, G, 1.0, 6.0, 1e-13)
    qb, vb, _ = bs.bs_group(q, v, m, rc, G, 1.0, -6.0, 1e-13)
    assert np.max(np.abs(qb - pos)) < 1e-11 and np.max(np.abs(vb - vel)) < 1e-12
    # looser tolerance: fewer force evaluations, larger deviation from the tight result, but within ~tol
    ql, vl, sl = bs.bs_group(pos, vel, m, rc, G, 1.0, 6.0, 1e-8)
    assert sl.force_evaluations < st.force_evaluations
    assert np.max(np.abs(ql - q)) < 1e-6
    # a massless member feels the others and moves nobody
    m0 = np.array([3e-6, 0.0])
    q0, v0, _ = bs.bs_group(pos, vel, m0, rc, G, 1.0, 6.0, 1e-13)
    qk, vk, _ = bs.bs_group(pos[:, :1], vel[:, :1], m0[:1], rc[:, :1], G, 1.0, 6.0, 1e-13)
    assert np.max(np.abs(q0[:, 0] - qk[:, 0])) < 1e-13


# ------------------------------------------------------------------------------- test-particle modes in a group (sec. 8.1)
def _tp_group(m_a=1e-9, m_b=1e-9, sep=1e-4):
    """A massive body M on a Kepler orbit and two semi-active particles a, b next to it, `sep` apart from each other."""
    pos, vel = gi.elements_to_cartesian(np.array([1.0]), np.array([0.05]), np.array([0.01]), np.zeros(1), np.zeros(1),
                                        np.array([0.4]), G)
    q = np.repeat(pos, 3, axis=1); v = np.repeat(vel, 3, axis=1)
    q[:, 1] += (0.010, 0.002, 0.0005); q[:, 2] = q[:, 1] + (sep, 0.0, 0.0)
    v[:, 1] += (0.0, 2e-5, 0.0); v[:, 2] += (0.0, 2e-5, 1e-6)
    mass = np.array([1e-5, m_a, m_b])
    rc = np.full((1, 3), 0.05)
    return q, v, mass, rc


def test_semi_active_particles_in_a_group(bs, oracle_mod):
    """Fig. 14 inside the Bulirsch-Stoer phase.  TP 1: nobody feels a particle -- the massive body
    stays on its Kepler orbit and each particle moves as in its own two-body group with it.  TP 2: a particle acts on
    the massive body exactly as a fully interactive body does, and particles still do not feel each other."""
    dt, tol = 1.0, 1e-13
    q, v, mass, rc = _tp_group()
    tp = np.array([False, True, True])
    # --- TP 1
    q1, v1, st = bs.bs_group(q, v, mass, rc, G, 1.0, dt, tol, is_tp=tp, tp_mode=1)
    assert not st.failed
    qk, vk, _ = oracle_mod.step.fg(q[:, :1], v[:, :1], G, dt)
    assert np.abs(q1[:, 0] - qk[:, 0]).max() < 1e-13 and np.abs(v1[:, 0] - vk[:, 0]).max() < 1e-14
    for p in (1, 2):
        qs, vs, _ = bs.bs_group(q[:, [0, p]], v[:, [0, p]], mass[[0, p]], rc[:, [0, p]], G, 1.0, dt, tol,
                                is_tp=np.array([False, True]), tp_mode=1)
        assert np.abs(q1[:, p] - qs[:, 1]).max() < 1e-12 and np.abs(v1[:, p] - vs[:, 1]).max() < 1e-13
    # the massive body does act on the particles: they leave their own Kepler orbits
    qa, va, _ = oracle_mod.step.fg(q[:, 1:], v[:, 1:], G, dt)
    assert np.abs(q1[:, 1:] - qa).max() > 1e-8
    # --- TP 2 on a pair (massive, particle) = the fully interactive pair
    q2, v2, _ = bs.bs_group(q[:, :2], v[:, :2], mass[:2], rc[:, :2], G, 1.0, dt, tol, is_tp=tp[:2], tp_mode=2)
    qf, vf, _ = bs.bs_group(q[:, :2], v[:, :2], mass[:2], rc[:, :2], G, 1.0, dt, tol)
    assert np.array_equal(q2, qf) and np.array_equal(v2, vf)
    qh, vh, _ = bs.bs_group(q[:, :2], v[:, :2], np.array([1e-5, 1e-6]), rc[:, :2], G, 1.0, dt, tol, is_tp=tp[:2], tp_mode=2)
    assert np.abs(qh[:, 0] - qk[:, 0]).max() > 1e-10                          # the particle moves the massive body
    # --- particles never feel each other: what b does to a, fully interactive vs TP 2 (heavy particles, 1e-4 AU apart)
    q, v, mass, rc = _tp_group(m_a=1e-7, m_b=1e-7)
    alone, _, _ = bs.bs_group(q[:, :2], v[:, :2], mass[:2], rc[:, :2], G, 1.0, dt, tol)
    full, _, _ = bs.bs_group(q, v, mass, rc, G, 1.0, dt, tol)
    semi, _, _ = bs.bs_group(q, v, mass, rc, G, 1.0, dt, tol, is_tp=tp, tp_mode=2)
    d_full = np.abs(full[:, 1] - alone[:, 1]).max(); d_semi = np.abs(semi[:, 1] - alone[:, 1]).max()
    assert d_full > 1e-6 and d_semi < 1e-4 * d_full
    # is_tp all False = fully interactive, bit for bit
    same, _, _ = bs.bs_group(q, v, mass, rc, G, 1.0, dt, tol, is_tp=np.zeros(3, bool), tp_mode=2)
    assert np.array_equal(same, full)


def test_large_group_force_sum_order_only_enters_the_rounding(bs):
    """The oracle sums a body's pair terms in member order.  What the mathematics fixes: the result does not depend on
    that order beyond rounding (a permutation of the members changes every running sum) -- which is why a kernel may
    sum in any order it likes and is compared under a tolerance -- and a group deep inside every critical radius
    (K = 0, W_BS = 1) conserves the Newtonian energy of Sun (fixed) + bodies to the tolerance."""
    n = 320
    rng = np.random.default_rng(23)
    ang = 2 * np.pi * np.arange(n) / n
    pos = np.stack([np.cos(ang), np.sin(ang), 1e-3 * rng.normal(size=n)])
    vk = np.sqrt(G)
    vel = np.stack([-vk * np.sin(ang), vk * np.cos(ang), np.zeros(n)]) * (1 + 1e-3 * rng.normal(size=n))
    mass = np.full(n, 1e-7)
    rc = np.full((1, n), 50.0)                    # every pair is inside 0.1 r_crit: K = 0

    def energy(q, v):
        e = 0.5 * (mass * (v * v).sum(0)).sum() - (G * mass / np.sqrt((q * q).sum(0))).sum()
        for i in range(n):
            d = np.sqrt(((q[:, i + 1:] - q[:, i:i + 1]) ** 2).sum(0))
            e -= (G * mass[i] * mass[i + 1:] / d).sum()
        return e

    q1, v1, st = bs.bs_group(pos, vel, mass, rc, G, 1.0, 20.0, 1e-12)
    assert not st.failed and abs(energy(q1, v1) / energy(pos, vel) - 1) < 1e-11
    perm = rng.permutation(n)
    q2, v2, _ = bs.bs_group(pos[:, perm], vel[:, perm], mass[perm], rc[:, perm], G, 1.0, 20.0, 1e-12)
    assert np.abs(q2 - q1[:, perm]).max() < 1e-11 and np.abs(v2 - v1[:, perm]).max() < 1e-12
    assert not np.array_equal(q2, q1[:, perm])                    # (the order does enter the rounding)
    # the bodies do feel each other: without the pair terms (W_BS = 0) the result differs visibly
    q3, _, _ = bs.bs_group(pos, vel, mass, np.full((1, n), 1e-9), G, 1.0, 20.0, 1e-12)
    assert np.abs(q3 - q1).max() > 1e-8
