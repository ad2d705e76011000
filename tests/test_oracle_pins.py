"""Pins P1-P10 of SURVEY.md section 8(c): the CPU oracle against what the paper and the mathematics
fix, NOT against itself.  A dropped term, a wrong sign or index, a transposed operand or a wrong
constant in oracle/genga_kick_oracle.c fails at least one of these."""
import os
from fractions import Fraction

import mpmath as mp
import numpy as np
import pytest

import genga_inputs as gi
from tests import harness_integrator as hi

G = gi.G_AU_DAY_MSUN
U = 2.0 ** -53
HERE = os.path.dirname(os.path.abspath(__file__))


def _ulp_diff(a, b):
    return np.abs(a - b) / (np.spacing(np.abs(b)) + 1e-300)


# ---------------------------------------------------------------- P2: the changeover function K
def test_P2_K_golden_values(oracle_mod):
    """Values from tests/golden/changeover_values.txt (PAPER.md:70, :619, :642 + reading G1)."""
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "changeover_values.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 9
    for ys, ks, *_ in rows:
        y, k = Fraction(ys), Fraction(ks)
        got = oracle_mod.K_of_y(float(y))
        if k in (0, 1):
            assert got == float(k)                       # exactly 0 / 1 outside the band
        else:
            assert abs(got - float(k)) <= 2 * U * float(k)


def test_P2_K_band_edges_in_r(oracle_mod):
    rc = 0.037
    assert oracle_mod.K(0.05 * rc, rc) == 0.0            # below the inner radius 0.1 rc
    assert oracle_mod.K(0.0999 * rc, rc) == 0.0
    assert oracle_mod.K(1.0001 * rc, rc) == 1.0          # above rc
    assert oracle_mod.K(1.5 * rc, rc) == 1.0
    assert 0.0 < oracle_mod.K(0.11 * rc, rc) < 1e-3
    assert 0.999 < oracle_mod.K(0.99 * rc, rc) < 1.0
    assert abs(oracle_mod.K(0.55 * rc, rc) - 0.5) < 1e-15   # mid-band: y = 1/2


def test_P2_K_symmetry_monotone_C1(oracle_mod):
    ys = np.linspace(0.0, 1.0, 2001)
    k = np.array([oracle_mod.K_of_y(y) for y in ys])
    assert np.all(np.diff(k) >= 0.0) and k[0] == 0.0 and k[-1] == 1.0
    assert np.max(np.abs(k + k[::-1] - 1.0)) < 4 * U     # K(y) + K(1-y) = 1
    # continuity of K and K' at both bounds (north_star (b)); K' = 2y(1-y)/(2y^2-2y+1)^2
    h = 1e-6
    assert oracle_mod.K_of_y(h) < 2 * h * h              # K -> 0 like y^2: K and K' continuous at 0
    assert 1.0 - oracle_mod.K_of_y(1.0 - h) < 2 * h * h  # same at y = 1
    d_mid = (oracle_mod.K_of_y(0.5 + h) - oracle_mod.K_of_y(0.5 - h)) / (2 * h)
    assert abs(d_mid - 2.0) < 1e-8                       # K'(1/2) = 2
    # K'' jumps 0 -> 2 at y = 0 (C1 only; known, reported in DESIGN.md, not a failure)
    dd0 = (oracle_mod.K_of_y(2 * h) - 2 * oracle_mod.K_of_y(h) + oracle_mod.K_of_y(0.0)) / (h * h)
    assert abs(dd0 - 2.0) < 1e-4


# ---------------------------------------------------------------- P1: two-body closed form
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_P1_two_body_closed_form(oracle_mod, seed):
    u = gi.uniforms(seed, 0, 8)
    nvec = np.array([u[0] - 0.5, u[1] - 0.5, u[2] - 0.5]); nvec /= np.linalg.norm(nvec)
    D = 0.3 + u[3]
    x1 = np.array([1.0 + u[4], -0.5 + u[5], 0.1 * u[6]])
    pos = np.stack([x1, x1 + D * nvec], axis=1)
    m = np.array([3e-6, 7e-7])
    rc = np.full((1, 2), 1e-6)                            # far outside r_crit: K = 1
    r = oracle_mod.kick(pos, m, rc, 2, G=G)
    Dtrue = np.linalg.norm(pos[:, 1] - pos[:, 0]); n_true = (pos[:, 1] - pos[:, 0]) / Dtrue
    a1 = G * m[1] / Dtrue ** 2 * n_true                   # body 1 is pulled TOWARD body 2 (sign!)
    a2 = -G * m[0] / Dtrue ** 2 * n_true                  # and feels the OTHER body's mass (index!)
    assert np.all(_ulp_diff(r.acc[:, 0], a1) <= 4) and np.all(_ulp_diff(r.acc[:, 1], a2) <= 4)
    assert np.all(_ulp_diff(r.S[:, 0], np.abs(a1)) <= 4)
    assert r.count.tolist() == [0, 0] and not r.coincident


def test_P2_two_body_in_band(oracle_mod):
    m = np.array([1e-6, 2e-6]); rc = 0.04
    for frac, kexp in ((0.55, 0.5), (0.05, 0.0), (1.5, 1.0), (0.1 + 0.9 * 0.25, 0.1), (0.1 + 0.9 * 0.75, 0.9)):
        d = frac * rc
        pos = np.array([[1.0, 1.0 + d], [0.0, 0.0], [0.0, 0.0]])
        r = oracle_mod.kick(pos, m, np.array([[0.5 * rc, rc]]), 2, G=G)   # pair radius = max(...) = rc
        want = kexp * G * m[1] / d ** 2
        if kexp == 0.0:
            assert r.acc[0, 0] == 0.0 and r.acc[0, 1] == 0.0              # exactly zero deep inside
        else:
            assert abs(r.acc[0, 0] - want) <= 1e-13 * want
            assert abs(r.acc[0, 1] + kexp * G * m[0] / d ** 2) <= 1e-13 * want
        assert r.count.tolist() == ([1, 1] if frac < 1.0 else [0, 0])


# ---------------------------------------------------------------- P3: momentum
@pytest.mark.parametrize("cfg,n,level", [(0, None, 0), (2, 1500, 1), (3, 3000, 1), (3, 3000, 0), (1, 1000, 0)])
def test_P3_momentum(oracle_mod, cfg, n, level):
    k = gi.make_config(cfg, n=n, level=level)
    r = oracle_mod.kick(k.pos, k.mass, k.rcrit, k.n_massive, 0, level, k.G)
    mom = (k.mass * r.acc).sum(axis=1)
    scale = (k.mass * r.S).sum(axis=1)
    assert np.all(np.abs(mom) <= 8 * U * scale), (mom, scale)
    assert r.count.sum() % 2 == 0


def test_P3_momentum_tp_mode_massive_only(oracle_mod):
    k = gi.make_config(4, n=300, n_test=2000)
    r = oracle_mod.kick(k.pos, k.mass, k.rcrit, k.n_massive, k.n_test, 0, k.G)
    nm = k.n_massive
    mom = (k.mass[:nm] * r.acc[:, :nm]).sum(axis=1)
    assert np.all(np.abs(mom) <= 8 * U * (k.mass[:nm] * r.S[:, :nm]).sum(axis=1))


# ---------------------------------------------------------------- P4: Newtonian limit
def _newton_numpy(pos, mass, G_):
    """Independent Newtonian direct sum: float64 per pair, sequential long-double sum over j."""
    n = pos.shape[1]
    out = np.zeros((3, n))
    for i in range(n):
        d = pos - pos[:, i:i + 1]
        r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2]
        keep = np.arange(n) != i
        r = np.sqrt(r2[keep])
        s = G_ * mass[keep] * 1.0 / (r2[keep] * r)
        for c in range(3):
            out[c, i] = float(np.cumsum((s * d[c][keep]).astype(np.longdouble))[-1])
    return out


def test_P4_newtonian_limit_bit_for_bit(oracle_mod):
    k = gi.make_config(0, n=200)
    rc = np.full((1, k.n), 1e-30)
    r = oracle_mod.kick(k.pos, k.mass, rc, k.n, G=k.G)
    assert np.array_equal(r.acc, _newton_numpy(k.pos, k.mass, k.G))
    assert r.count.sum() == 0
    # and with the real r_crit the result differs only through pairs inside r_crit
    r2 = oracle_mod.kick(k.pos, k.mass, k.rcrit, k.n, G=k.G)
    same = r2.count == 0
    assert np.array_equal(r2.acc[:, same], r.acc[:, same])


# ---------------------------------------------------------------- P5-P7: level weights, eq. 62-63
def test_P5_partition_of_unity(oracle_mod):
    u = gi.uniforms(77, 0, 4000).reshape(-1, 4)
    for a, b, c, d in u:
        rc = np.sort(np.array([0.02 + 0.1 * a, 0.02 + 0.1 * b, 0.02 + 0.1 * c]))[::-1].copy()
        r = 0.25 * d
        for nlev in (1, 2, 3):
            tot = sum(oracle_mod.weight(r, rc, l) for l in range(nlev)) + oracle_mod.weight_bs(r, rc, nlev)
            assert abs(tot - 1.0) <= 4 * U


def test_eq62_eq63_literal(oracle_mod):
    """eq. 62 (one level) and eq. 63 (two levels, s = 2) typed out literally from PAPER.md:621-632."""
    rc = np.array([0.05, 0.025])
    for r in np.linspace(0.001, 0.06, 60):
        K0, K1 = oracle_mod.K(r, rc[0]), oracle_mod.K(r, rc[1])
        assert oracle_mod.weight(r, rc, 0) == K0                         # K_symplectic = K(r)
        assert oracle_mod.weight_bs(r, rc, 1) == 1.0 - K0                # K_BS = 1 - K(r)
        assert oracle_mod.weight(r, rc, 1) == (1.0 - K0) * K1            # (1 - K(dt)) K(dt/2)
        assert oracle_mod.weight_bs(r, rc, 2) == (1.0 - K0) * (1.0 - K1)


def test_P6_substep10_at_most_two_levels_active(oracle_mod):
    rc = np.array([0.05, 0.005, 0.0005])                 # velocity-dominated, s = 10
    for r in np.geomspace(1e-5, 0.1, 600):
        ks = [oracle_mod.K(r, c) for c in rc]
        assert sum(0.0 < kk < 1.0 for kk in ks) <= 1     # bands are disjoint
        w = [oracle_mod.weight(r, rc, l) for l in range(3)] + [oracle_mod.weight_bs(r, rc, 3)]
        assert sum(x != 0.0 for x in w) <= 2             # "no more than two levels are active"


def test_P7_level1_identical_rows(oracle_mod):
    rc = np.array([0.04, 0.04])
    ys = np.linspace(0.0, 1.0, 1001)
    w = np.array([oracle_mod.weight(0.1 * 0.04 + 0.9 * 0.04 * y, rc, 1) for y in ys])
    assert abs(w.max() - 0.25) < 1e-12 and abs(ys[w.argmax()] - 0.5) < 2e-3
    assert w[0] == 0.0 and w[-1] == 0.0


# ---------------------------------------------------------------- P8: symplectic 2nd order
def _three_body():
    m = np.array([3e-6, 1e-5]); m_star = 1.0
    q = np.array([[1.0, 0.0, 0.0], [0.0, 1.6, 0.05]]).T.copy()
    vh = np.array([[0.0, np.sqrt(G / 1.0), 0.0], [-np.sqrt(G / 1.6) * 0.98, 0.0, 0.0]]).T.copy()
    # heliocentric -> barycentric velocities (democratic coordinates)
    vsun = -(m * vh).sum(axis=1, keepdims=True) / (m_star + m.sum())
    return q, vh + vsun, m, m_star


def _run_energy_err(oracle_mod, dt, nsteps):
    q, v, m, m_star = _three_body()
    rc = np.full((1, 2), 1e-4)                           # K = 1 everywhere: G5 readings coincide
    kick = lambda qq: oracle_mod.kick(qq, m, rc, 2, G=G).acc
    e0 = hi.energy(q, v, m, m_star, G)
    errs = []
    for _ in range(nsteps):
        q, v = hi.leapfrog_step(q, v, m, m_star, G, dt, kick)
        errs.append(abs(hi.energy(q, v, m, m_star, G) - e0) / abs(e0))
    return np.array(errs)


def test_P8_energy_error_scales_as_dt2_no_drift(oracle_mod):
    T = 600.0
    e1 = _run_energy_err(oracle_mod, 4.0, int(T / 4.0)).max()
    e2 = _run_energy_err(oracle_mod, 2.0, int(T / 2.0)).max()
    e3 = _run_energy_err(oracle_mod, 1.0, int(T / 1.0)).max()
    assert 3.6 < e1 / e2 < 4.4 and 3.6 < e2 / e3 < 4.4, (e1, e2, e3)
    long = _run_energy_err(oracle_mod, 2.0, 10000)
    assert long[5000:].max() < 1.5 * long[:5000].max()   # bounded oscillation, no secular growth


# ---------------------------------------------------------------- P9: ring with exactly 8 partners
@pytest.mark.parametrize("n", [16, 17, 64, 128, 1000, 4096])
def test_P9_ring_eight_partners(oracle_mod, n):
    k = gi.make_ring(n)
    r = oracle_mod.kick(k.pos, k.mass, k.rcrit, n, G=k.G)
    assert np.all(r.count == 8)
    ps = oracle_mod.pair_set(r, n)
    assert ps.shape == (4 * n, 2) and np.all(ps[:, 0] < ps[:, 1])
    for q in (0, n // 2, n - 1):
        want = sorted(((q + s) % n) for s in (-4, -3, -2, -1, 1, 2, 3, 4))
        assert r.partners[q].tolist() == want


# ---------------------------------------------------------------- P10: brute force, other formulation
def _mp_reference(pos, mass, rcrit, level, G_, nm):
    """50-digit reference, formulated differently: one force per unordered pair, applied to both
    bodies with opposite signs (Newton's third law), weights from exact rational arithmetic on y."""
    mp.mp.dps = 50
    n = pos.shape[1]
    acc = [[mp.mpf(0)] * 3 for _ in range(n)]
    def Kmp(r, rc):
        y = (r - mp.mpf(rc) / 10) / (mp.mpf(9) * mp.mpf(rc) / 10)
        if y <= 0: return mp.mpf(0)
        if y >= 1: return mp.mpf(1)
        return y * y / (y * y + (1 - y) * (1 - y))
    for i in range(n):
        for j in range(i + 1, n):
            d = [mp.mpf(pos[c, j]) - mp.mpf(pos[c, i]) for c in range(3)]
            r = mp.sqrt(sum(x * x for x in d))
            W = mp.mpf(1)
            for kk in range(level):
                W *= 1 - Kmp(r, max(rcrit[kk, i], rcrit[kk, j]))
            W *= Kmp(r, max(rcrit[level, i], rcrit[level, j]))
            f = G_ * W / r ** 3
            for c in range(3):
                if j < nm: acc[i][c] += f * mp.mpf(mass[j]) * d[c]
                if i < nm: acc[j][c] -= f * mp.mpf(mass[i]) * d[c]
    return np.array([[float(acc[i][c]) for i in range(n)] for c in range(3)])


@pytest.mark.parametrize("level", [0, 1, 2])
def test_P10_bruteforce_mpmath(oracle_mod, level):
    n = 8
    u = gi.uniforms(500 + level, 0, 6 * n).reshape(6, n)
    pos = np.ascontiguousarray(1.0 + 0.05 * u[:3])                  # compact cloud: many pairs in band
    mass = 1e-7 * (1.0 + u[3])
    rc0 = 0.03 + 0.03 * u[4]
    rcrit = np.stack([rc0 / (1.6 ** kk) for kk in range(level + 1)])
    r = oracle_mod.kick(pos, mass, rcrit, n, level=level, G=G)
    ref = _mp_reference(pos, mass, rcrit, level, G, n)
    # Tolerance: binary64 evaluation of W has ABSOLUTE error ~u per factor (1 - K_k loses relative
    # accuracy as K_k -> 1, but the weight -> 0 there), so the error of a term is bounded by a few u
    # times the UNWEIGHTED term: scale with the Newtonian sum of |term|.
    newt = oracle_mod.kick(pos, mass, np.full((1, n), 1e-30), n, level=0, G=G)
    assert np.any((r.acc != 0)) and np.all(np.abs(r.acc - ref) <= 16 * U * newt.S + 1e-300)
    if level == 0:
        assert np.all(np.abs(r.acc - ref) <= 8 * U * r.S + 1e-300)
    # the in-band weights matter here: the Newtonian sum is far away
    assert np.max(np.abs(newt.acc - r.acc) / (np.abs(newt.acc) + 1e-300)) > 0.1


# ---------------------------------------------------------------- J(i), counts, borderline, overflow of maxp
def test_tp_mode_equals_massless_full_mode(oracle_mod):
    """sec. 8.1: test particles feel the massive bodies and not each other.  With massless particles
    the fully interactive sum gives the same accelerations bit for bit; only the lists differ."""
    k = gi.make_config(4, n=200, n_test=1500)
    tp = oracle_mod.kick(k.pos, k.mass, k.rcrit, k.n_massive, k.n_test, 0, k.G)
    full = oracle_mod.kick(k.pos, k.mass, k.rcrit, k.n, 0, 0, k.G)
    assert np.array_equal(tp.acc, full.acc)
    nm = k.n_massive
    for q in range(nm, k.n, 97):                                      # a test particle lists massive partners only
        assert np.all(tp.partners[q] < nm)
        assert tp.partners[q].tolist() == [j for j in full.partners[q].tolist() if j < nm]
    assert np.array_equal(tp.count[:nm], full.count[:nm])             # massive bodies list everyone
    # every tp->massive entry has its massive->tp mirror: list entries are consistent
    mirror = sum(int((tp.partners[q] >= nm).sum()) for q in range(nm))
    assert mirror == int(tp.count[nm:].sum())


def test_borderline_band_and_strict_threshold(oracle_mod):
    rc = 0.05
    m = np.array([1e-6, 1e-6])
    for eps, is_partner, is_border in ((-1e-13, True, True), (1e-13, False, True), (-1e-9, True, False), (1e-9, False, False)):
        pos = np.array([[0.0, rc * (1.0 + eps)], [0.0, 0.0], [0.0, 0.0]])
        r = oracle_mod.kick(pos, m, np.full((1, 2), rc), 2, G=G)
        assert (r.count[0] == 1) == is_partner and (len(r.border) > 0) == is_border
    # enc_factor widens the net without touching K (reading G4)
    pos = np.array([[0.0, 1.5 * rc], [0.0, 0.0], [0.0, 0.0]])
    a1 = oracle_mod.kick(pos, m, np.full((1, 2), rc), 2, G=G, enc_factor=1.0)
    a2 = oracle_mod.kick(pos, m, np.full((1, 2), rc), 2, G=G, enc_factor=2.0)
    assert a1.count.tolist() == [0, 0] and a2.count.tolist() == [1, 1] and np.array_equal(a1.acc, a2.acc)


def test_partner_list_regrows_and_counts_consistent(oracle_mod):
    k = gi.make_config(3, n=2000, level=0)
    r = oracle_mod.kick(k.pos, k.mass, k.rcrit * 6.0, k.n, G=k.G, maxp=2)   # force the second pass
    assert r.count.max() > 2 and all(len(p) == c for p, c in zip(r.partners, r.count))
    ps = oracle_mod.pair_set(r, k.n)
    assert 2 * len(ps) == r.count.sum()                                # sum_i count_i = 2 * total (TP 0)
    sub = oracle_mod.kick(k.pos, k.mass, k.rcrit * 6.0, k.n, G=k.G, rows=np.array([5, 77, 1999]))
    for q, i in enumerate((5, 77, 1999)):
        assert np.array_equal(sub.acc[:, q], r.acc[:, i]) and sub.partners[q].tolist() == r.partners[i].tolist()


def test_coincident_pair_flagged_not_nan(oracle_mod):
    pos = np.array([[1.0, 1.0, 2.0], [0.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    r = oracle_mod.kick(pos, np.full(3, 1e-6), np.full((1, 3), 1e-3), 3, G=G)
    assert r.coincident and np.all(np.isfinite(r.acc))


def test_threshold_is_strict_at_exact_equality(oracle_mod):
    """r2 == (f rc)^2 exactly (all values dyadic): NOT a partner, the test is strict (reading G4)."""
    pos = np.array([[0.0, 0.25], [0.0, 0.0], [0.0, 0.0]])
    m = np.array([1e-6, 1e-6])
    r = oracle_mod.kick(pos, m, np.full((1, 2), 0.25), 2, G=G)
    assert r.count.tolist() == [0, 0]
    r = oracle_mod.kick(pos, m, np.full((1, 2), 0.125), 2, G=G, enc_factor=2.0)
    assert r.count.tolist() == [0, 0]
    r = oracle_mod.kick(pos, m, np.full((1, 2), np.nextafter(0.25, 1.0)), 2, G=G)
    assert r.count.tolist() == [1, 1]


def test_semi_active_particles_with_mass_exert_no_force_on_this_path(oracle_mod):
    """sec. 8.1 + reading G10: on this path J(i) = massive bodies for every i, also when the test
    particles carry mass (their back-reaction on the massive bodies is SURVEY.md NEXT-3)."""
    pos = np.array([[1.0, 1.3, 1.1, 0.9], [0.0, 0.1, 0.4, -0.3], [0.0, 0.0, 0.02, 0.01]])
    m = np.array([1e-6, 2e-6, 5e-7, 5e-7])
    rc = np.full((1, 4), 1e-4)
    tp = oracle_mod.kick(pos, m, rc, 2, 2, 0, G)
    only = oracle_mod.kick(pos[:, :2].copy(), m[:2].copy(), rc[:, :2].copy(), 2, 0, 0, G)
    assert np.array_equal(tp.acc[:, :2], only.acc)                    # massive bodies ignore the particles
    for q in (2, 3):                                                  # particles feel exactly the two massive bodies
        want = sum(G * m[j] * (pos[:, j] - pos[:, q]) / np.linalg.norm(pos[:, j] - pos[:, q]) ** 3 for j in (0, 1))
        assert np.all(np.abs(tp.acc[:, q] - want) <= 8 * U * tp.S[:, q])


# ---------------------------------------------------------------- TP 2 (semi-active particles)
def _tp2_case(n_m=40, n_t=300, seed=3):
    ki = gi.make_config(4, n=n_m, n_test=n_t)
    u = gi.uniforms(seed, 0, n_t)
    ki.mass = ki.mass.copy()
    ki.mass[n_m:] = 1e-12 * (1.0 + u)                       # semi-active particles WITH mass
    return ki


def test_TP2_momentum_over_all_bodies(oracle_mod):
    """Every force term of Fig. 14's right panel has its reaction: sum over ALL bodies of m a = 0 (TP 1: it is not)."""
    ki = _tp2_case()
    r2 = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, G=ki.G, tp_mode=2)
    p = (ki.mass * r2.acc).sum(axis=1)
    assert np.all(np.abs(p) <= 8 * U * (ki.mass * r2.S).sum(axis=1))
    r1 = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, G=ki.G, tp_mode=1)
    p1 = (ki.mass * r1.acc).sum(axis=1)
    assert np.any(np.abs(p1) > 1e3 * U * (ki.mass * r1.S).sum(axis=1))
    assert np.array_equal(r1.count, r2.count)                # the encounter list does not depend on the mode


def test_TP2_is_the_full_interaction_minus_tp_tp(oracle_mod):
    """Massive bodies: exactly the fully interactive sum (TP 0) over all N.  Semi-active bodies: the TP 0 sum
    minus the sum over the other semi-active bodies (computed as a TP 0 run on that subset alone)."""
    ki = _tp2_case()
    nm, n = ki.n_massive, ki.n
    r2 = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, nm, ki.n_test, G=ki.G, tp_mode=2)
    full = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, n, 0, G=ki.G)
    assert np.array_equal(r2.acc[:, :nm], full.acc[:, :nm]) and np.array_equal(r2.S[:, :nm], full.S[:, :nm])
    tt = oracle_mod.kick(ki.pos[:, nm:], ki.mass[nm:], ki.rcrit[:, nm:], n - nm, 0, G=ki.G)
    want = full.acc[:, nm:] - tt.acc
    assert np.all(np.abs(r2.acc[:, nm:] - want) <= 4 * U * (full.S[:, nm:] + tt.S))
    # and TP 1 differs from TP 2 only on the massive bodies
    r1 = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, nm, ki.n_test, G=ki.G, tp_mode=1)
    assert np.array_equal(r1.acc[:, nm:], r2.acc[:, nm:]) and not np.array_equal(r1.acc[:, :nm], r2.acc[:, :nm])


# ---------------------------------------------------------------- KickS: the kick over a pair list (App. A)
def test_KickS_over_the_level0_list_is_the_all_pairs_level_kick(oracle_mod):
    """W_L = 0 for r >= rc0_ij (factor 1 - K_0 of eq. 63), so the level-L kick over the level-0 encounter list
    (every pair with r < rc0_ij) equals the all-pairs level-L kick, and its level-L pre-check gives the same list."""
    for cfg, n, kw in [(3, 4000, {}), (2, 3000, {}), (4, 300, dict(n_test=4000))]:
        ki = gi.make_config(cfg, n=n, level=2, **kw)
        top = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=0, G=ki.G, maxp=128)
        lst = oracle_mod.pair_set(top, ki.n_massive)
        assert len(lst) > 10
        for L in (1, 2):
            full = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=L, G=ki.G, maxp=128)
            ks = oracle_mod.kick_list(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, lst, level=L, G=ki.G)
            assert np.all(np.abs(ks.acc - full.acc) <= 4 * U * full.S) and np.all(np.abs(ks.S - full.S) <= 4 * U * full.S)
            assert np.array_equal(ks.count, full.count)
            want = {tuple(p) for p in oracle_mod.pair_set(full, ki.n_massive).tolist()}
            assert {tuple(p) for p in lst[ks.enc].tolist()} == want


def test_KickS_all_pairs_list_at_level0_and_closed_form(oracle_mod):
    ki = gi.make_config(0, n=60)
    every = np.array([(i, j) for i in range(60) for j in range(i + 1, 60)], dtype=np.int32)
    full = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, 60, 0, level=0, G=ki.G)
    ks = oracle_mod.kick_list(ki.pos, ki.mass, ki.rcrit, 60, 0, every, level=0, G=ki.G)
    assert np.all(np.abs(ks.acc - full.acc) <= 4 * U * full.S) and np.array_equal(ks.count, full.count)
    # two bodies in mid-band of K: a = (1/2) G m / r^2 each way, momentum exactly balanced in the terms
    rc, m = 0.03, np.array([2e-7, 5e-8])
    pos = np.array([[0.0, 0.55 * rc], [0.0, 0.0], [0.0, 0.0]])
    ks = oracle_mod.kick_list(pos, m, np.full((1, 2), rc), 2, 0, [[0, 1]], level=0, G=G)
    r = 0.55 * rc
    assert abs(ks.acc[0, 0] - 0.5 * G * m[1] / r ** 2) <= 8 * U * ks.S[0, 0]
    assert abs(ks.acc[0, 1] + 0.5 * G * m[0] / r ** 2) <= 8 * U * ks.S[0, 1]
    assert ks.enc.tolist() == [True] and ks.count.tolist() == [1, 1]


def test_KickS_test_particle_rules(oracle_mod):
    ki = gi.make_config(4, n=100, n_test=2000)
    ki.mass = ki.mass.copy(); ki.mass[100:] = 1e-12
    top = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, 100, 2000, level=0, G=ki.G)
    lst = oracle_mod.pair_set(top, 100)
    for mode in (1, 2):
        full = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, 100, 2000, level=0, G=ki.G, tp_mode=mode)
        ks = oracle_mod.kick_list(ki.pos, ki.mass, ki.rcrit, 100, 2000, lst, level=0, G=ki.G, tp_mode=mode)
        # level 0 over a partial list: only the listed pairs' terms -- compare with the all-pairs kick restricted to r < rc
        assert np.array_equal(ks.count, full.count)
        if mode == 2:
            p = (ki.mass * ks.acc).sum(axis=1)
            assert np.all(np.abs(p) <= 8 * U * (ki.mass * ks.S).sum(axis=1))
