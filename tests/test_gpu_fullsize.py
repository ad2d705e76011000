"""-m gpu: BASELINE.json's configs at their FULL sizes, in the launch configuration bench.py times
(internal order AUTO, pair capacity 2^20), against the CPU oracle under north_star's rule.

The oracle is a direct sum, so it finishes every full config on the GPU box's host cores in
seconds (N = 65,536: 4.3e9 pair evaluations per level): the comparison is element by element over
ALL bodies, not a sample.  Config 1 runs its 100 kicks with the harness drift between them."""
import numpy as np
import pytest

import genga_inputs as gi
from tests.gpu_harness import run_gpu, compare
from tests import harness_integrator as hi

pytestmark = pytest.mark.gpu
TOL = 1e-13
CAPACITY = 1 << 20


def _full(ki, oracle_mod, level):
    gpu = run_gpu(ki, level=level, capacity=CAPACITY, order_mode=0)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=level, G=ki.G,
                          enc_factor=ki.enc_factor, maxp=256)
    assert not orc.coincident and gpu.status == 0
    d = compare(gpu, orc, ki.n_massive, tol=TOL)
    assert gpu.total == len(gpu.pairs) <= CAPACITY
    # momentum (pin P3 on the GPU result): sum over the massive bodies, which only feel each other
    m = ki.mass[:ki.n_massive]
    p = (m * gpu.acc[:, :ki.n_massive]).sum(axis=1)
    scale = (m * orc.S[:, :ki.n_massive]).sum(axis=1)
    assert np.all(np.abs(p) <= TOL * scale)
    return gpu, orc, d


@pytest.mark.parametrize("level", [0, 1])
def test_config3_full(oracle_mod, level):
    """N = 65,536, the headline config; the paper's section 2.1 regime: O(10) partners per body."""
    ki = gi.make_config(3)
    assert ki.n == 65536
    gpu, orc, d = _full(ki, oracle_mod, level)
    if level == 0:
        assert 10.0 < gpu.counts.mean() < 25.0
        assert int(gpu.counts.sum()) == 2 * gpu.total


@pytest.mark.parametrize("level", [0, 1])
def test_config2_full(oracle_mod, level):
    """32,768 planetesimals + Jupiter + Saturn, higher-level changeover."""
    ki = gi.make_config(2)
    assert ki.n == 32770
    gpu, orc, d = _full(ki, oracle_mod, level)
    assert gpu.total > 1000


def test_config4_full(oracle_mod):
    """2048 massive + 1,048,576 semi-active test particles (rectangular kick)."""
    ki = gi.make_config(4)
    assert ki.n_massive == 2048 and ki.n_test == 1 << 20
    gpu, orc, d = _full(ki, oracle_mod, 0)
    pr = gpu.pairs
    assert (pr[:, 0] < ki.n_massive).all()                # no tp-tp pairs
    assert (pr[:, 1] >= ki.n_massive).sum() > 1000        # tp-massive pairs exist
    # a massive body counts its test-particle partners (reading G11)
    want = np.bincount(pr.ravel(), minlength=ki.n)
    assert np.array_equal(want, gpu.counts)


def test_config4_full_tp2(oracle_mod):
    """Config 4's shape with semi-active particles that HAVE mass (TP 2): the massive bodies also
    sum over the 1,048,576 particles (the transposed rectangular kick)."""
    ki = gi.make_config(4)
    u = gi.uniforms(77, 0, ki.n_test)
    ki.mass = ki.mass.copy()
    ki.mass[ki.n_massive:] = 1e-12 * (0.5 + u)
    gpu = run_gpu(ki, level=0, capacity=CAPACITY, order_mode=0, tp_mode=2)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=0, G=ki.G, maxp=256, tp_mode=2)
    assert gpu.status == 0
    compare(gpu, orc, ki.n_massive, tol=TOL)
    p = (ki.mass * gpu.acc).sum(axis=1)
    assert np.all(np.abs(p) <= TOL * (ki.mass * orc.S).sum(axis=1))


@pytest.mark.parametrize("nm,nt", [(16, 1048560), (600, 1 << 20)])
def test_tp2_last_iblock_reaches_past_the_massive_records(oracle_mod, nm, nt):
    """TP 2 where the transposed pass's i-block (512 records) does not divide the padded massive range (256 / 768
    records): the i-records beyond it are particles and must take no part -- particles never feel each other
    (sec. 8.1).  (16 massive bodies + N - 16 particles is the paper's own test-particle benchmark
    shape.)"""
    from paper_2201_10058_b200 import binding
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    p2 = binding.make_plan_tp2(nm, nt, sms)
    assert p2.m_pad % p2.i_block != 0, "the case this test is for: the last i-block spills past m_pad"
    ki = gi.make_config(4, n=nm, n_test=nt)
    u = gi.uniforms(78, 0, ki.n_test)
    ki.mass = ki.mass.copy()
    ki.mass[ki.n_massive:] = 1e-12 * (0.5 + u)
    gpu = run_gpu(ki, level=0, capacity=CAPACITY, order_mode=0, tp_mode=2)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=0, G=ki.G, maxp=256, tp_mode=2)
    assert gpu.status == 0
    compare(gpu, orc, ki.n_massive, tol=TOL)
    p = (ki.mass * gpu.acc).sum(axis=1)
    assert np.all(np.abs(p) <= TOL * (ki.mass * orc.S).sum(axis=1))


def _tp_masses(ki, seed):
    u = gi.uniforms(seed, 0, ki.n_test)
    ki.mass = ki.mass.copy()
    ki.mass[ki.n_massive:] = 1e-12 * (0.5 + u)
    return ki


@pytest.mark.parametrize("nm,nt,tp_mode,order_mode", [(24577, 0, 1, 0), (30001, 20000, 1, 0), (30001, 20000, 2, 0),
                                                      (26000, 0, 1, 1), (40000, 300, 2, 2)])
def test_symmetric_pass_ragged_sizes_and_particles(oracle_mod, nm, nt, tp_mode, order_mode):
    """The symmetric level-0 pass (every unordered massive pair once, from 24,576 massive bodies on) at sizes that are
    multiples of neither its 1536-record i-blocks nor its 256-record j-tiles, alone, beside the particles' one-sided
    rows (TP 1) and beside TP 2's transposed pass; caller's order, sorted order and auto."""
    from paper_2201_10058_b200 import binding
    import torch
    assert binding.make_plan_sym(nm, nt, torch.cuda.get_device_properties(0).multi_processor_count).n_ctas > 0
    ki = gi.make_config(3 if nt == 0 else 4, n=nm, n_test=nt if nt else None, level=0)
    if tp_mode == 2:
        ki = _tp_masses(ki, 79)
    gpu = run_gpu(ki, level=0, capacity=CAPACITY, order_mode=order_mode, tp_mode=tp_mode)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=0, G=ki.G, maxp=256, tp_mode=tp_mode)
    assert gpu.status == 0 and not orc.coincident
    d = compare(gpu, orc, ki.n_massive, tol=TOL)
    assert gpu.total == len(gpu.pairs) and gpu.total > 1000
    nmom = ki.n if tp_mode == 2 else ki.n_massive           # TP 2: every term has its reaction
    p = (ki.mass[:nmom] * gpu.acc[:, :nmom]).sum(axis=1)
    assert np.all(np.abs(p) <= TOL * (ki.mass[:nmom] * orc.S[:, :nmom]).sum(axis=1))
    print(f"nm={nm} nt={nt} tp={tp_mode} order={order_mode}: {gpu.total} pairs, max |da|/S = {d['max_err_over_S']:.2e}")


def test_symmetric_pass_candidate_list_overflow(oracle_mod):
    """More pairs inside critical radii than the candidate list holds (64 per body), with the symmetric pass as the
    far field: the fallback search repeats the pair loop's trip rule on the same bits, so the result is complete."""
    import paper_2201_10058_b200 as g
    ki = gi.make_config(3, n=24576, level=0)
    ki.rcrit = ki.rcrit * 4.0
    gpu = run_gpu(ki, level=0, capacity=1 << 23, order_mode=0)
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n, 0, level=0, G=ki.G, maxp=4096)
    assert gpu.status == g.STATUS_CAND_OVERFLOW and gpu.total > 64 * ki.n // 2
    gpu.status = 0
    compare(gpu, orc, ki.n, tol=TOL)


def test_symmetric_pass_edge_cases(oracle_mod):
    """The symmetric pass with a widened and a narrowed pre-check net (enc_factor), with a pair list too small for the
    pairs found (true total kept, rows clipped, never out of bounds), with coincident bodies (skipped and flagged, in a
    symmetric tile and in a diagonal one), with the level-1 kick on top (symmetric candidates of the neighbour search),
    and through the host entry point."""
    ki = gi.make_config(3, n=25000, level=1)
    for f in (1.6, 0.5):
        ki.enc_factor = f
        for level in (0, 1):
            gpu = run_gpu(ki, level=level, capacity=CAPACITY, order_mode=0)
            orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n, 0, level=level, G=ki.G, enc_factor=f, maxp=512)
            assert gpu.status == 0
            compare(gpu, orc, ki.n, tol=TOL)
    ki.enc_factor = 1.0
    full = run_gpu(ki, level=0, capacity=CAPACITY, order_mode=0)
    small = run_gpu(ki, level=0, capacity=100, order_mode=0)
    assert small.total == full.total > 100 and len(small.pairs) == 100 and np.array_equal(small.counts, full.counts)
    allp = {tuple(p) for p in full.pairs.tolist()}
    assert all(tuple(p) in allp for p in small.pairs.tolist()) and np.array_equal(small.acc, full.acc)
    host = run_gpu(ki, level=0, capacity=CAPACITY, order_mode=0, host=True)
    assert np.array_equal(host.acc, full.acc) and host.total == full.total
    ki.pos = ki.pos.copy()
    ki.pos[:, 20000] = ki.pos[:, 7]                          # far apart in the caller's order: a symmetric tile or a diagonal one,
    ki.pos[:, 8] = ki.pos[:, 9]                              # wherever the internal order puts them
    gpu = run_gpu(ki, level=0, capacity=CAPACITY, order_mode=0)
    assert gpu.status & 1 and np.isfinite(gpu.acc).all()
    orc = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n, 0, level=0, G=ki.G, maxp=512)
    assert orc.coincident
    gpu.status = 0
    compare(gpu, orc, ki.n, tol=TOL)


def test_symmetric_pass_is_bit_reproducible():
    ki = gi.make_config(3, n=33000, level=0)
    a = run_gpu(ki, level=0, capacity=CAPACITY, with_vel=True)
    b = run_gpu(ki, level=0, capacity=CAPACITY, with_vel=True)
    assert np.array_equal(a.acc, b.acc) and np.array_equal(a.counts, b.counts) and np.array_equal(a.vel, b.vel)
    assert np.array_equal(sorted(map(tuple, a.pairs.tolist())), sorted(map(tuple, b.pairs.tolist())))


def test_config1_hundred_kicks(oracle_mod):
    """N = 8192, 100 kicks separated by an oracle-matched heliocentric drift: both sides see the
    same state at every step (the harness advances it with the ORACLE's acceleration), the
    encounter list evolves, momentum is checked at every step."""
    ki = gi.make_config(1)
    assert ki.n == 8192
    from paper_2201_10058_b200 import GengaKick
    n, dt = ki.n, ki.dt
    kick = GengaKick(n, 0, max_level=0, pair_capacity=CAPACITY, G=ki.G, enc_factor=ki.enc_factor)
    q, v, mass = ki.pos.copy(), ki.vel.copy(), ki.mass
    seen = set()
    totals = []
    for step in range(100):
        a_sma = gi.semi_major_axis(q, v, ki.G)
        ki.pos, ki.vel = np.ascontiguousarray(q), np.ascontiguousarray(v)
        ki.rcrit = gi.rcrit_rows(a_sma, v, mass, dt, 2, 1)
        gpu = run_gpu(ki, level=0, capacity=CAPACITY, kick=kick)
        orc = oracle_mod.kick(q, mass, ki.rcrit, n, 0, level=0, G=ki.G, enc_factor=ki.enc_factor, maxp=64)
        assert gpu.status == 0
        compare(gpu, orc, n, tol=TOL)
        for acc in (gpu.acc, orc.acc):
            p = (mass * acc).sum(axis=1)
            assert np.all(np.abs(p) <= TOL * (mass * orc.S).sum(axis=1)), f"momentum at step {step}"
        totals.append(gpu.total)
        seen.add(frozenset(map(tuple, gpu.pairs.tolist())))
        # between kicks: v += dt a_oracle, then the heliocentric drift
        # HC(dt/2) FG(dt) HC(dt/2) of App. A
        v = v + dt * orc.acc
        q = hi.sun_drift(q, v, mass, 1.0, 0.5 * dt)
        q, v = hi.kepler_drift(q, v, ki.G * 1.0, dt)
        q = hi.sun_drift(q, v, mass, 1.0, 0.5 * dt)
    kick.free()
    assert len(seen) > 50, "the encounter list did not evolve"
    assert min(totals) > 1000
