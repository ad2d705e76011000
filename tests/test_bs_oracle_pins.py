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
