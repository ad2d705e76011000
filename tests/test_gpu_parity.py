"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Acceptance (BASELINE.json north_star): |a_gpu - a_oracle| <= 1e-13 * sum_j |term_ij| per component;
the encounter pair list equal as a sorted set except pairs within 1e-12 (relative) of the
threshold, which are counted; per-body counts equal (same exception)."""
import numpy as np
import pytest

import genga_inputs as gi
from tests.gpu_harness import run_gpu, compare, sorted_pairs

pytestmark = pytest.mark.gpu
TOL = 1e-13


@pytest.fixture(params=[1, 2], ids=["caller_order", "sorted_order"], autouse=True)
def order_mode(request, monkeypatch):
    """Every test runs with both internal body orders (GENGA_KICK_ORDER_CALLER / _SORTED)."""
    import tests.gpu_harness as h
    orig = h.run_gpu
    monkeypatch.setattr(h, "run_gpu", lambda *a, **k: orig(*a, **{"order_mode": request.param, **k}))
    globals()["run_gpu"] = h.run_gpu
    yield request.param
    globals()["run_gpu"] = orig


def _full(ki, oracle_mod, level=None, **kw):
    level = ki.level if level is None else level
    gpu = run_gpu(ki, level=level, **kw)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=level, G=ki.G,
                          enc_factor=ki.enc_factor)
    assert not orc.coincident and gpu.status == 0
    d = compare(gpu, orc, ki.n_massive, tol=TOL)
    assert gpu.total == len(gpu.pairs)
    return gpu, orc, d


def test_config0_full(oracle_mod):
    ki = gi.make_config(0)
    gpu, orc, d = _full(ki, oracle_mod)
    assert gpu.total > 50                        # the recipe gives ~2e2 pairs
    assert int(gpu.counts.sum()) == 2 * gpu.total


@pytest.mark.parametrize("n", [1, 2, 3, 31, 33, 127, 129, 257, 1000, 2047, 2049, 5000])
def test_ragged_sizes_level0(oracle_mod, n):
    ki = gi.make_config(0, n=n)
    _full(ki, oracle_mod)


@pytest.mark.parametrize("level", [0, 1, 2])
def test_config2_giants_levels(oracle_mod, level):
    ki = gi.make_config(2, n=6000, level=2)
    gpu, orc, d = _full(ki, oracle_mod, level=level)
    assert gpu.total > 0


@pytest.mark.parametrize("level", [0, 1])
def test_config3_reduced(oracle_mod, level):
    ki = gi.make_config(3, n=9001, level=1)
    gpu, orc, d = _full(ki, oracle_mod, level=level)
    assert gpu.total > 0


def test_config1_single_kick(oracle_mod):
    ki = gi.make_config(1)
    _full(ki, oracle_mod)


@pytest.mark.parametrize("nm,nt", [(300, 5000), (2048, 20000), (1, 100), (257, 1)])
def test_config4_test_particles_reduced(oracle_mod, nm, nt):
    ki = gi.make_config(4, n=nm, n_test=nt)
    gpu, orc, d = _full(ki, oracle_mod)
    # test particles exert no force and do not meet each other
    assert all(p[0] < ki.n_massive for p in gpu.pairs.tolist())


def test_no_massive_bodies(oracle_mod):
    ki = gi.make_config(4, n=0, n_test=500)
    gpu = run_gpu(ki)
    assert gpu.total == 0 and not gpu.counts.any() and not gpu.acc.any()


@pytest.mark.parametrize("n", [16, 64, 1024, 4096])
def test_ring_eight_partners(oracle_mod, n):
    ki = gi.make_ring(n)
    gpu = run_gpu(ki)
    assert (gpu.counts == 8).all() and gpu.total == 4 * n


def test_close_pairs_and_band(oracle_mod):
    """Pairs all through the changeover band, incl. r < 0.1 rc (K = 0) and bodies 1e-9 AU apart."""
    ki = gi.make_config(0, n=1024)
    pos = ki.pos.copy()
    rng = np.random.RandomState(5)
    for q, frac in enumerate(np.concatenate([np.linspace(0.02, 1.2, 200), [1e-7, 1e-5, 0.0999, 0.1, 0.1001, 0.9999, 1.0, 1.0001]])):
        i, j = 2 * q, 2 * q + 1
        rc = max(ki.rcrit[0, i], ki.rcrit[0, j])
        u = rng.normal(size=3); u /= np.linalg.norm(u)
        pos[:, j] = pos[:, i] + frac * rc * u
    ki.pos = np.ascontiguousarray(pos)
    _full(ki, oracle_mod)


def test_levels_with_substeps_10(oracle_mod):
    ki = gi.make_disk(3000, 77, level=3, substeps=10, total_mass=5 * gi.M_EARTH)
    for level in range(4):
        _full(ki, oracle_mod, level=level)


def test_enc_factor(oracle_mod):
    ki = gi.make_config(0, n=3000)
    ki.enc_factor = 1.7
    gpu, orc, d = _full(ki, oracle_mod)
    ki.enc_factor = 0.5
    _full(ki, oracle_mod)


def test_bit_reproducible_and_vel_update(oracle_mod):
    ki = gi.make_config(3, n=5000, level=1)
    a = run_gpu(ki, level=0, with_vel=True)
    b = run_gpu(ki, level=0, with_vel=True)
    assert np.array_equal(a.acc, b.acc) and np.array_equal(a.counts, b.counts) and a.total == b.total
    assert np.array_equal(sorted_pairs(a.pairs), sorted_pairs(b.pairs))
    want = ki.vel + ki.dt * a.acc
    assert np.allclose(a.vel, want, rtol=0, atol=4e-16 * np.abs(want).max())
    assert np.max(np.abs(a.vel - want) / (np.abs(ki.vel) + np.abs(ki.dt * a.acc))) < 3e-16


def test_pair_capacity_overflow(oracle_mod):
    ki = gi.make_config(0)
    full = run_gpu(ki)
    small = run_gpu(ki, capacity=16)
    assert small.total == full.total and len(small.pairs) == 16
    allp = {tuple(p) for p in full.pairs.tolist()}
    assert all(tuple(p) in allp for p in small.pairs.tolist())
    zero = run_gpu(ki, capacity=0)
    assert zero.total == full.total and np.array_equal(zero.counts, full.counts)


def test_host_entry_point(oracle_mod):
    ki = gi.make_config(0, n=1500)
    h = run_gpu(ki, host=True, with_vel=True)
    d = run_gpu(ki, with_vel=True)
    assert np.array_equal(h.acc, d.acc) and np.array_equal(h.vel, d.vel)
    assert np.array_equal(sorted_pairs(h.pairs), sorted_pairs(d.pairs)) and np.array_equal(h.counts, d.counts)


def test_momentum(oracle_mod):
    ki = gi.make_config(1, n=4096)
    gpu = run_gpu(ki)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, level=0, G=ki.G)
    p = (ki.mass * gpu.acc).sum(axis=1)
    scale = (ki.mass * orc.S).sum(axis=1)
    assert np.all(np.abs(p) <= 1e-13 * scale)


def test_coincident_bodies_flagged():
    ki = gi.make_config(0, n=100)
    ki.pos[:, 7] = ki.pos[:, 3]
    gpu = run_gpu(ki)
    assert gpu.status & 1 and np.isfinite(gpu.acc).all()


def test_error_codes():
    import torch
    import paper_2201_10058_b200 as g
    with pytest.raises(g.GengaKickError) as e:
        g.GengaKick(0, 0)
    assert e.value.code == g.E_SIZE
    k = g.GengaKick(64, 0, max_level=0, pair_capacity=8)
    x = torch.zeros(3 * 64 + 1, dtype=torch.float64, device="cuda")
    m = torch.ones(64, dtype=torch.float64, device="cuda")
    acc = torch.zeros(3, 64, dtype=torch.float64, device="cuda")
    pr = torch.zeros(8, 2, dtype=torch.int32, device="cuda")
    npr = torch.zeros(65, dtype=torch.int32, device="cuda")
    with pytest.raises(g.GengaKickError) as e:
        k.kick(x[1:], None, m, m, 0, 1.0, acc, pr, npr)
    assert e.value.code == g.E_ALIGN
    with pytest.raises(g.GengaKickError) as e:
        k.kick(x, None, m, torch.ones(128, dtype=torch.float64, device="cuda"), 1, 1.0, acc, pr, npr)
    assert e.value.code == g.E_LEVEL
    with pytest.raises(g.GengaKickError) as e:
        k.kick(x, None, m, m, 0, 1.0, None, pr, npr)
    assert e.value.code == g.E_NULL
    # what the library cannot check on a bare pointer, the binding does before the call: side, dtype, layout, size
    for bad, exc in [(lambda: k.kick(x.cpu(), None, m, m, 0, 1.0, acc, pr, npr), ValueError),
                     (lambda: k.kick(x.float(), None, m, m, 0, 1.0, acc, pr, npr), TypeError),
                     (lambda: k.kick(x, None, m, m, 0, 1.0, acc.t(), pr, npr), ValueError),
                     (lambda: k.kick(x, None, m[:63], m, 0, 1.0, acc, pr, npr), ValueError),
                     (lambda: k.kick(x, None, m, m, 0, 1.0, acc, pr[:7], npr), ValueError),
                     (lambda: k.kick(x, None, m, m, 0, 1.0, acc, pr, npr[:64]), ValueError),
                     (lambda: k.kick(x, None, m, m, 0, 1.0, acc, pr.long(), npr), TypeError),
                     (lambda: k.kick_host(x, None, m, m, 0, 1.0, acc, pr, npr), ValueError)]:
        with pytest.raises(exc):
            bad()
    k.free()


def test_order_reuse_across_levels(oracle_mod):
    """genga_kick_set_order_reuse: the level-1 kick of a step keeps the internal order the level-0 kick sorted -- the
    same positions, so the same order as a fresh sort and the same bits; on MOVED positions a kept order is still
    correct (it only decides what the culling can clear)."""
    from paper_2201_10058_b200 import GengaKick
    ki = gi.make_config(3, n=9000, level=1)
    fresh = run_gpu(ki, level=1, order_mode=2)
    k = GengaKick(ki.n, 0, max_level=1, pair_capacity=1 << 20, G=ki.G, order_mode=2)
    run_gpu(ki, level=0, kick=k)
    k.set_order_reuse(True)
    kept = run_gpu(ki, level=1, kick=k)
    assert np.array_equal(kept.acc, fresh.acc) and np.array_equal(kept.counts, fresh.counts)
    assert np.array_equal(sorted_pairs(kept.pairs), sorted_pairs(fresh.pairs)) and kept.launches < 2 * fresh.launches
    moved = gi.make_config(3, n=9000, level=1)
    moved.pos = moved.pos + 0.05 * np.sin(7.0 * moved.pos[::-1])            # ~0.05 AU away from where the order was taken
    stale = run_gpu(moved, level=0, kick=k)
    orc = oracle_mod.kick(moved.pos, moved.mass, moved.rcrit, moved.n, 0, level=0, G=moved.G)
    assert stale.status == 0
    compare(stale, orc, moved.n, tol=TOL)
    k.free()


@pytest.mark.parametrize("tp_mode,n,n_test", [(1, 9000, 0), (1, 30000, 0), (1, 1500, 4500), (2, 1500, 4500)])
def test_list_reuse_across_levels(oracle_mod, tp_mode, n, n_test):
    """GENGA_KICK_REUSE_LIST: the level-1 and level-2 kicks of a step evaluate the near pairs the level-0 kick has listed
    (no neighbour search of their own): the same bits, counts and pair set as their own search, with and without test
    particles, below and above the size from which level 0 runs the symmetric loop.  If a body's filter radius at the
    level exceeds its level-0 one (here: row 1 of rcrit scaled up), the device check sends that kick to the all-pairs
    search; the results are still those of the oracle."""
    from paper_2201_10058_b200 import GengaKick
    make = lambda: gi.make_config(4, n=n, n_test=n_test, level=2) if n_test else gi.make_config(3, n=n, level=2)
    ki = make()
    if tp_mode == 2:
        _with_tp_masses(ki)
    kw = dict(max_level=2, pair_capacity=1 << 20, G=ki.G, enc_factor=ki.enc_factor, tp_mode=tp_mode)
    k = GengaKick(ki.n_massive, ki.n_test, **kw)
    run_gpu(ki, level=0, kick=k)
    k.set_order_reuse(2)
    for level in (1, 2):
        before = k.launch_count()
        kept = run_gpu(ki, level=level, kick=k)
        kept.launches -= before
        fresh = run_gpu(ki, level=level, tp_mode=tp_mode)
        assert kept.status == 0
        assert np.array_equal(kept.acc, fresh.acc) and np.array_equal(kept.counts, fresh.counts)
        assert np.array_equal(sorted_pairs(kept.pairs), sorted_pairs(fresh.pairs))
        assert kept.launches < fresh.launches
    grown = make()
    grown.mass = ki.mass
    grown.rcrit = grown.rcrit.copy()
    grown.rcrit[1, ::7] = 3.0 * grown.rcrit[0, ::7]                      # f rc1 > f rc0 for every seventh body
    run_gpu(grown, level=0, kick=k)
    wide = run_gpu(grown, level=1, kick=k)
    orc = oracle_mod.kick(grown.pos, grown.mass, grown.rcrit, grown.n_massive, grown.n_test, level=1, G=grown.G,
                          enc_factor=grown.enc_factor, tp_mode=tp_mode)
    assert wide.status == 0
    compare(wide, orc, grown.n_massive, tol=TOL)
    k.free()


def test_reuse_setting_is_validated_and_a_level_without_a_list_searches(oracle_mod):
    """genga_kick_set_order_reuse takes 0, 1 or 2; with GENGA_KICK_REUSE_LIST a level >= 1 kick that finds no level-0
    list at hand (the first call on the context; a level-1 kick in between has replaced the list) searches itself."""
    from paper_2201_10058_b200 import GengaKick, GengaKickError, E_SIZE
    ki = gi.make_config(3, n=5000, level=1)
    k = GengaKick(ki.n, 0, max_level=1, pair_capacity=1 << 18, G=ki.G)
    for bad in (-1, 3):
        with pytest.raises(GengaKickError) as e:
            k.set_order_reuse(bad)
        assert e.value.code == E_SIZE
    fresh = run_gpu(ki, level=1)
    k.set_order_reuse(2)
    first = run_gpu(ki, level=1, kick=k)                     # no level-0 kick yet on this context
    run_gpu(ki, level=0, kick=k)
    kept = run_gpu(ki, level=1, kick=k)                      # on the level-0 list
    again = run_gpu(ki, level=1, kick=k)                     # still on it (a kick on a kept list writes none)
    for got in (first, kept, again):
        assert got.status == 0 and np.array_equal(got.acc, fresh.acc) and np.array_equal(got.counts, fresh.counts)
        assert np.array_equal(sorted_pairs(got.pairs), sorted_pairs(fresh.pairs))
    k.free()


def test_internal_order_is_invisible(oracle_mod):
    """Caller's order, sorted order and auto give the same pair set and counts; accelerations agree
    to the rounding of a different summation order."""
    ki = gi.make_config(3, n=7000, level=1)
    for level in (0, 1):
        a = run_gpu(ki, level=level, order_mode=1)
        b = run_gpu(ki, level=level, order_mode=2)
        c = run_gpu(ki, level=level, order_mode=0)
        assert np.array_equal(sorted_pairs(a.pairs), sorted_pairs(b.pairs)) and np.array_equal(a.counts, b.counts)
        assert np.array_equal(b.acc, c.acc)                      # auto sorts at this size
        orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, level=level, G=ki.G)
        assert np.all(np.abs(a.acc - b.acc) <= 2e-13 * orc.S)


# ------------------------------------------------------------------ TP 2
def _with_tp_masses(ki, seed=11):
    u = gi.uniforms(seed, 0, ki.n_test)
    ki.mass = ki.mass.copy()
    ki.mass[ki.n_massive:] = 1e-11 * (0.5 + u)
    ki.mass[ki.n_massive::7] = 0.0                        # some stay massless
    return ki


@pytest.mark.parametrize("nm,nt,level", [(300, 5000, 0), (2048, 20000, 0), (1, 100, 0), (257, 1, 0), (700, 3000, 1),
                                         (5000, 300, 0)])
def test_tp2_semi_active_particles_act_on_massive_bodies(oracle_mod, nm, nt, level):
    import tests.gpu_harness as h
    ki = _with_tp_masses(gi.make_config(4, n=nm, n_test=nt, level=level))
    gpu = run_gpu(ki, level=level, tp_mode=2)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, nm, nt, level=level, G=ki.G, tp_mode=2)
    assert gpu.status == 0
    compare(gpu, orc, nm, tol=TOL)
    # momentum over ALL bodies (every term of Fig. 14's right panel has its reaction)
    p = (ki.mass * gpu.acc).sum(axis=1)
    assert np.all(np.abs(p) <= TOL * (ki.mass * orc.S).sum(axis=1))
    # TP 1 on the same input: the particles' accelerations are the same, the massive bodies' differ
    one = run_gpu(ki, level=level, tp_mode=1)
    assert np.array_equal(one.acc[:, nm:], gpu.acc[:, nm:])
    assert np.array_equal(sorted_pairs(one.pairs), sorted_pairs(gpu.pairs))


def test_candidate_list_overflow_is_complete(oracle_mod):
    """Everything inside everything's critical radius: 9e6 ordered candidates against a list of 2^20.  The excess is
    evaluated where it is found (slow path); the result is complete and the status word says the list overflowed."""
    import paper_2201_10058_b200 as g
    ki = gi.make_config(0, n=3000)
    ki.rcrit = np.full_like(ki.rcrit, 12.0)                  # AU: larger than the disk
    n = ki.n
    gpu = run_gpu(ki, capacity=1 << 23)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, n, 0, level=0, G=ki.G, maxp=n)
    assert gpu.status == g.STATUS_CAND_OVERFLOW
    assert gpu.total == n * (n - 1) // 2 and (gpu.counts == n - 1).all()
    gpu.status = 0
    compare(gpu, orc, n, tol=TOL)


def test_candidate_list_overflow_tp2_and_level1(oracle_mod):
    """The overflow fallback also covers the level >= 1 neighbour search and TP 2's transposed pass."""
    import paper_2201_10058_b200 as g
    ki = gi.make_config(3, n=2500, level=1)
    ki.rcrit = np.stack([np.full(ki.n, 12.0), np.full(ki.n, 6.0)])
    gpu = run_gpu(ki, level=1, capacity=1 << 22)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n, 0, level=1, G=ki.G, maxp=ki.n)
    assert gpu.status == g.STATUS_CAND_OVERFLOW
    gpu.status = 0
    compare(gpu, orc, ki.n, tol=TOL)
    kt = _with_tp_masses(gi.make_config(4, n=300, n_test=6000))
    kt.rcrit = np.full_like(kt.rcrit, 12.0)                   # 300 x 6000 x 2 + 300^2 ordered candidates > 2^20
    gpu = run_gpu(kt, level=0, capacity=1 << 22, tp_mode=2)
    orc = oracle_mod.kick(kt.pos, kt.mass, kt.rcrit, 300, 6000, level=0, G=kt.G, maxp=kt.n, tp_mode=2)
    assert gpu.status == g.STATUS_CAND_OVERFLOW
    gpu.status = 0
    compare(gpu, orc, 300, tol=TOL)
