"""-m gpu: genga_detect and genga_multilevel_step (include/genga_senc.h) through the C ABI against
oracle/genga_detect_oracle.c and oracle.step.multilevel_step.

Detection: the decision is an integer taken from floating point; both sides take it in IEEE binary64 without contraction
in the same order, so the encounter SET must be identical (no borderline allowance is needed; the oracle's 1e-12 band is
still honoured).  Multi-level step: bodies outside every encounter agree to rounding (<= 32 u), bodies inside to 1e-10
relative (their sub-step start states differ by the kick's rounding, which an encounter amplifies), the per-level
counts of candidates / encounter pairs / Bulirsch-Stoer groups exactly."""
import numpy as np
import pytest

import genga_inputs as gi
from tests.gpu_harness import sorted_pairs

pytestmark = pytest.mark.gpu
U = 2.0 ** -53
G = gi.G_AU_DAY_MSUN


def _dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a))
    return (t if dtype is None else t.to(dtype)).cuda()


def _gpu_detect(k, n, pos0, vel0, pos1, vel1, rc_row, h, pairs, cap, enc_factor=1.0, n_override=None):
    import torch
    d_in = torch.zeros(max(len(pairs), 2), 2, dtype=torch.int32, device="cuda")
    if len(pairs):
        d_in[:len(pairs)] = _dev(np.asarray(pairs, np.int32))
    d_n = torch.tensor([len(pairs) if n_override is None else n_override, 0, 0, 0], dtype=torch.int32, device="cuda")
    out = torch.full((max(cap, 1), 2), -7, dtype=torch.int32, device="cuda")
    npairs = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    k.detect(_dev(pos0), _dev(vel0), _dev(pos1), _dev(vel1), _dev(rc_row), h, d_in, d_n, len(pairs), out, npairs,
             enc_factor=enc_factor)
    torch.cuda.synchronize()
    c = npairs.cpu().numpy()
    return out.cpu().numpy()[:min(int(c[n]), cap)], c[:n], int(c[n])


def _compare_detect(got_pairs, got_count, got_total, want, cand):
    assert got_total == int(want.enc.sum()) or want.border.any()
    gs = {tuple(p) for p in got_pairs.tolist()}
    assert len(gs) == len(got_pairs) and all(a < b for a, b in gs)
    ws = {tuple(sorted(p)) for p in want.pairs.tolist()}
    border = {tuple(sorted(p)) for p in np.asarray(cand)[want.border].tolist()}
    assert (gs ^ ws) <= border, sorted(gs ^ ws)[:10]
    if not (gs ^ ws):
        assert np.array_equal(got_count, want.count)
    return len(gs ^ ws)


@pytest.mark.parametrize("cfg,n,f", [(0, 2048, 3.0), (1, 8192, 2.5), (3, 20000, 2.0)])
def test_detect_on_disks_against_oracle(oracle_mod, cfg, n, f):
    """Candidates from a widened pre-check (enc_factor f), states before / after the oracle's Kepler drift."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    ki = gi.make_config(cfg, n=n)
    q1, v1, _ = oracle_mod.step.fg(ki.pos, ki.vel, ki.G, ki.dt)
    wide = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n, 0, level=0, G=ki.G, enc_factor=f, maxp=512)
    cand = oracle_mod.pair_set(wide, ki.n)
    rng = np.random.default_rng(3)
    cand = cand[rng.permutation(len(cand))]
    flip = rng.random(len(cand)) < 0.5
    cand[flip] = cand[flip][:, ::-1]                                  # either orientation in the input
    want = oracle_mod.detect.detect(ki.pos, ki.vel, q1, v1, ki.rcrit[0], ki.dt, cand)
    assert 0 < want.enc.sum() < len(cand)
    k = GengaKick(ki.n, 0, G=ki.G, pair_capacity=1 << 20)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    gp, gc, gt = _gpu_detect(k, ki.n, ki.pos, ki.vel, q1, v1, ki.rcrit[0], ki.dt, cand, 1 << 20)
    assert _compare_detect(gp, gc, gt, want, cand) == 0 and k.status() == 0
    # enc_factor scales the radius
    want2 = oracle_mod.detect.detect(ki.pos, ki.vel, q1, v1, ki.rcrit[0], ki.dt, cand, enc_factor=0.5)
    gp, gc, gt = _gpu_detect(k, ki.n, ki.pos, ki.vel, q1, v1, ki.rcrit[0], ki.dt, cand, 1 << 20, enc_factor=0.5)
    assert _compare_detect(gp, gc, gt, want2, cand) == 0 and gt < int(want.enc.sum())
    # bit-reproducible counts; the device count of candidates is honoured (clipped to the rows passed)
    gp2, gc2, gt2 = _gpu_detect(k, ki.n, ki.pos, ki.vel, q1, v1, ki.rcrit[0], ki.dt, cand, 1 << 20, enc_factor=0.5,
                                n_override=len(cand) + 1000)
    assert gt2 == gt and np.array_equal(gc, gc2) and np.array_equal(sorted_pairs(gp), sorted_pairs(gp2))
    half = len(cand) // 2
    want3 = oracle_mod.detect.detect(ki.pos, ki.vel, q1, v1, ki.rcrit[0], ki.dt, cand[:half])
    gp, gc, gt = _gpu_detect(k, ki.n, ki.pos, ki.vel, q1, v1, ki.rcrit[0], ki.dt, cand, 1 << 20, n_override=half)
    assert _compare_detect(gp, gc, gt, want3, cand[:half]) == 0
    k.free()


def test_detect_flybys_capacity_bad_rows_and_errors(oracle_mod):
    """Straight-line fly-bys that are outside the radius at both ends and inside in between; capacity overflow counts
    but does not write; bad rows are ignored and reported; argument errors."""
    import torch
    from paper_2201_10058_b200 import GengaKick, binding as g
    rng = np.random.default_rng(11)
    npair, h = 3000, 2.0
    n = 2 * npair
    pos0 = rng.normal(size=(3, n)); vel = rng.normal(scale=0.3, size=(3, n))
    pos0[:, npair:] = pos0[:, :npair] + rng.normal(scale=0.4, size=(3, npair))
    pos1 = pos0 + h * vel
    pairs = np.stack([np.arange(npair), np.arange(npair) + npair], 1).astype(np.int32)
    rc = np.full(n, 0.3)
    want = oracle_mod.detect.detect(pos0, vel, pos1, vel, rc, h, pairs)
    d0 = ((pos0[:, pairs[:, 1]] - pos0[:, pairs[:, 0]]) ** 2).sum(0); d1 = ((pos1[:, pairs[:, 1]] - pos1[:, pairs[:, 0]]) ** 2).sum(0)
    assert (want.enc & (np.minimum(d0, d1) >= 0.09)).sum() > 20
    k = GengaKick(n, 0, G=1.0, pair_capacity=100)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    gp, gc, gt = _gpu_detect(k, n, pos0, vel, pos1, vel, rc, h, pairs, 100)
    assert gt == int(want.enc.sum()) > 100 and len(gp) == 100 and np.array_equal(gc, want.count)
    assert {tuple(p) for p in gp.tolist()} <= {tuple(p) for p in want.pairs.tolist()}
    bad = pairs.copy(); bad[5] = (7, 7); bad[9] = (-1, 3); bad[11] = (2, n)
    ok = np.ones(npair, bool); ok[[5, 9, 11]] = False
    want_b = oracle_mod.detect.detect(pos0, vel, pos1, vel, rc, h, pairs[ok])
    gp, gc, gt = _gpu_detect(k, n, pos0, vel, pos1, vel, rc, h, bad, 100)
    assert gt == int(want_b.enc.sum()) and np.array_equal(gc, want_b.count) and k.status() == g.STATUS_BAD_PAIR
    # empty list
    gp, gc, gt = _gpu_detect(k, n, pos0, vel, pos1, vel, rc, h, pairs[:0], 100)
    assert gt == 0 and not gc.any()
    x = torch.zeros(3, n, dtype=torch.float64, device="cuda"); i = torch.zeros(n + 4, dtype=torch.int32, device="cuda")
    L = g.lib()
    p = lambda t: None if t is None else t.data_ptr()
    assert L.genga_detect(k._ctx, None, p(x), p(x), p(x), p(x), 1.0, 1.0, p(i), p(i), 1, p(i), p(i)) == g.E_NULL
    assert L.genga_detect(k._ctx, p(x) + 8, p(x), p(x), p(x), p(x), 1.0, 1.0, p(i), p(i), 1, p(i), p(i)) == g.E_ALIGN
    assert L.genga_detect(k._ctx, p(x), p(x), p(x), p(x), p(x), 0.0, 1.0, p(i), p(i), 1, p(i), p(i)) == g.E_SIZE
    assert L.genga_detect(k._ctx, p(x), p(x), p(x), p(x), p(x), 1.0, 1.0, p(i), p(i), -1, p(i), p(i)) == g.E_SIZE
    k.free()


def _ml_buffers(n, cap, slevels):
    import torch
    return (torch.empty(3, n, dtype=torch.float64, device="cuda"), torch.empty(cap, 2, dtype=torch.int32, device="cuda"),
            torch.empty(n + 1, dtype=torch.int32, device="cuda"), torch.full((slevels, 4), -1, dtype=torch.int32, device="cuda"))


IN_ENC_SAME = 2.5e-13    # bodies inside encounters, both sides took the same Bulirsch-Stoer decisions (see _ml_check)


def _ml_check(ki, q, v, r, in_enc, gpu_totals=None, tol=1e-12, label=""):
    """Bodies outside every encounter: <= 32 u (the step's rounding).  Bodies inside: their Bulirsch-Stoer start states
    differ by the kicks' rounding (<= 32 u), which the encounter amplifies.  If the kernel's record of the step-size
    control (genga_bs_totals: accepted steps, halvings, force evaluations, groups) equals the oracle's, both sides did
    the same operations on inputs 32 u apart: bound IN_ENC_SAME = 2.5e-13 relative, ~100 x the largest difference measured
    on these disks (printed).  If the records differ, some error estimate fell within rounding of tol and the two sides
    are two valid answers of the scheme: bound 4 tol (accepted macro steps of the largest group ~ 1) x 1e3 for the
    amplification, and the flip is reported."""
    rr = np.sqrt((ki.pos ** 2).sum(0)); sp = np.sqrt((ki.vel ** 2).sum(0))
    sq, sv = rr + sp * ki.dt, sp + rr * np.sqrt(ki.G / rr ** 3)
    assert np.all(np.abs(q - r.pos)[:, ~in_enc] <= 32 * U * sq[~in_enc])
    assert np.all(np.abs(v - r.vel)[:, ~in_enc] <= 32 * U * sv[~in_enc])
    same = gpu_totals is None or tuple(gpu_totals) == tuple(r.bs_totals)
    bound = IN_ENC_SAME if same else 4e3 * tol
    worst = 0.0
    if in_enc.any():
        worst = max(np.max(np.abs(q - r.pos)[:, in_enc] / sq[in_enc]), np.max(np.abs(v - r.vel)[:, in_enc] / sv[in_enc]))
    print(f"{label}bodies in encounters: worst difference {worst:.2e} (bound {bound:.0e}); Bulirsch-Stoer record "
          f"(accepted, rejected, force evaluations, groups) kernel {gpu_totals} oracle {r.bs_totals}"
          + ("" if same else "  ** a step-size decision flipped **"))
    assert worst <= bound


@pytest.mark.parametrize("slevels,substeps,detect,f", [(1, 2, False, 1.0), (1, 2, True, 2.0), (2, 2, True, 1.0),
                                                       (2, 2, False, 1.0), (3, 2, True, 1.5), (2, 10, True, 1.0),
                                                       (4, 2, True, 1.0)])
def test_multilevel_step_against_oracle(oracle_mod, slevels, substeps, detect, f):
    import torch
    from paper_2201_10058_b200 import GengaKick
    ki = gi.make_config(1, n=4000)
    n = ki.n
    cap = 1 << 18
    k = GengaKick(n, 0, max_level=slevels - 1, G=ki.G, pair_capacity=cap, enc_factor=f)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    q, v, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    acc, pairs, npairs, stats = _ml_buffers(n, cap, slevels)
    k.multilevel_step(q, v, mass, 1.0, ki.dt, slevels, substeps, 1e-12, acc, pairs, npairs, stats, detect=detect)
    torch.cuda.synchronize()
    r = oracle_mod.step.multilevel_step(ki.pos, ki.vel, ki.mass, n, 0, 1.0, ki.G, ki.dt, slevels=slevels,
                                        substeps=substeps, tol=1e-12, enc_factor=f, detect=detect)
    assert k.status() == 0
    assert np.array_equal(stats.cpu().numpy(), r.stats), (stats.cpu().numpy(), r.stats)
    assert r.stats[0, 1] > 50 and r.stats[-1, 2] > 10
    c = npairs.cpu().numpy()
    want = oracle_mod.pair_set(r.first, n)
    assert np.array_equal(sorted_pairs(pairs.cpu().numpy()[:c[n]]), want)
    in_enc = r.first.count > 0
    _ml_check(ki, q.cpu().numpy(), v.cpu().numpy(), r, in_enc, gpu_totals=k.bs_totals())
    if slevels == 1 and not detect:
        # the same launch sequence as genga_hybrid_step: identical bits
        q2, v2 = _dev(ki.pos), _dev(ki.vel)
        i32 = lambda m: torch.empty(m, dtype=torch.int32, device="cuda")
        k.hybrid_step(q2, v2, mass, 1.0, ki.dt, 1e-12, acc, pairs, npairs, i32(n), i32(n), i32(n + 1), i32(4))
        torch.cuda.synchronize()
        assert torch.equal(q, q2) and torch.equal(v, v2)
    k.free()


def test_multilevel_step_repeats_bit_for_bit_and_in_a_cuda_graph():
    import torch
    from paper_2201_10058_b200 import GengaKick
    ki = gi.make_config(0, n=3000)
    n, cap = ki.n, 1 << 16
    k = GengaKick(n, 0, max_level=2, G=ki.G, pair_capacity=cap)
    stream = torch.cuda.Stream()
    out = []
    with torch.cuda.stream(stream):
        k.set_stream(stream.cuda_stream)
        mass = _dev(ki.mass)
        acc, pairs, npairs, stats = _ml_buffers(n, cap, 3)
        q, v = _dev(ki.pos), _dev(ki.vel)
        for rep in range(2):                                       # warm-up allocates the scratch
            q.copy_(_dev(ki.pos)); v.copy_(_dev(ki.vel))
            k.multilevel_step(q, v, mass, 1.0, ki.dt, 3, 2, 1e-12, acc, pairs, npairs, stats)
            stream.synchronize()
            out.append((q.clone(), v.clone(), stats.clone()))
        assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1])
        q.copy_(_dev(ki.pos)); v.copy_(_dev(ki.vel))
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            k.multilevel_step(q, v, mass, 1.0, ki.dt, 3, 2, 1e-12, acc, pairs, npairs, stats)
        q.copy_(_dev(ki.pos)); v.copy_(_dev(ki.vel))
        graph.replay()
        stream.synchronize()
        assert torch.equal(q, out[0][0]) and torch.equal(v, out[0][1]) and torch.equal(stats, out[0][2])
        assert int(stats[2, 2]) > 0
    assert k.status() == 0
    k.free()


def test_multilevel_step_keeps_the_energy_through_an_encounter():
    """The device integrator through the close encounter of tests/test_step_oracle_pins.py at 3 levels x 2 sub-steps."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    mass = np.array([3e-5, 3e-5])
    a = np.array([1.0, 1.02]); e = np.array([0.02, 0.03]); z = np.zeros(2)
    pos, vel = gi.elements_to_cartesian(a, e, z + 0.001, z, np.array([0.0, 0.6]), np.array([0.0, -0.57]), G)
    vel = vel - (mass * vel).sum(1, keepdims=True) / (1.0 + mass.sum())

    def energy(q, v):
        p = mass * v
        return (0.5 * (mass * (v * v).sum(0)).sum() + 0.5 * (p.sum(1) ** 2).sum() - (G * mass / np.sqrt((q * q).sum(0))).sum()
                - G * mass[0] * mass[1] / np.sqrt(((q[:, 0] - q[:, 1]) ** 2).sum()))

    e0 = energy(pos, vel)
    k = GengaKick(2, 0, max_level=2, G=G, pair_capacity=16)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    q, v, m = _dev(pos), _dev(vel), _dev(mass)
    acc, pairs, npairs, stats = _ml_buffers(2, 16, 3)
    worst, deep = 0.0, 0
    for _ in range(400):
        k.multilevel_step(q, v, m, 1.0, 2.0, 3, 2, 1e-13, acc, pairs, npairs, stats)
        deep += int(stats[2, 2])
        worst = max(worst, abs(energy(q.cpu().numpy(), v.cpu().numpy()) - e0) / abs(e0))
    # The pair stays a temporary binary for ~60 steps (chaotic: 1 ulp grows to 1e-6 AU) and passes within 5e-4 AU: at
    # such a passage a body's heliocentric speed can exceed the escape speed for a sub-step, FGS then reports it
    # (GENGA_KICK_STATUS_UNBOUND) and leaves it to the Bulirsch-Stoer phase, which integrates that body anyway.
    from paper_2201_10058_b200 import binding as g
    assert (k.status() & ~g.STATUS_UNBOUND) == 0 and deep > 3 and worst < 1e-5
    k.free()


def test_multilevel_step_reports_a_clipped_list():
    import torch
    from paper_2201_10058_b200 import GengaKick, binding as g
    ki = gi.make_config(0, n=3000)
    n, cap = ki.n, 64                                                # the disk has ~500 level-0 encounter pairs
    k = GengaKick(n, 0, max_level=1, G=ki.G, pair_capacity=cap)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    q, v, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    acc, pairs, npairs, stats = _ml_buffers(n, cap, 2)
    k.multilevel_step(q, v, mass, 1.0, ki.dt, 2, 2, 1e-12, acc, pairs, npairs, stats)
    torch.cuda.synchronize()
    assert int(npairs[n]) > cap and k.status() == g.STATUS_LIST_CLIPPED
    assert torch.isfinite(q).all() and torch.isfinite(v).all()
    k.free()


def test_multilevel_step_error_codes():
    import torch
    from paper_2201_10058_b200 import GengaKick, binding as g
    k = GengaKick(64, 0, max_level=1, G=1.0, pair_capacity=16)
    x = torch.ones(3, 64, dtype=torch.float64, device="cuda"); m = torch.ones(64, dtype=torch.float64, device="cuda")
    i = torch.zeros(80, dtype=torch.int32, device="cuda")
    L = g.lib()
    p = lambda t: t.data_ptr()

    def call(sl, ss, tol=1e-12, m_star=1.0, pos=p(x)):
        import ctypes as C
        cfg = g.GengaSencConfig(sl, ss, 1, 0, 3.0, 0.4, tol)
        return L.genga_multilevel_step(k._ctx, pos, p(x), p(m), m_star, 1.0, C.byref(cfg), None, p(i), p(i), None)

    assert call(0, 2) == g.E_SIZE and call(5, 2) == g.E_SIZE and call(2, 0) == g.E_SIZE and call(2, 2, tol=0.0) == g.E_SIZE
    assert call(2, 2, m_star=0.0) == g.E_SIZE and call(3, 2) == g.E_LEVEL and call(2, 2, pos=None) == g.E_NULL
    assert call(2, 2, pos=p(x) + 8) == g.E_ALIGN
    k.free()


def test_multilevel_step_full_size_config3(oracle_mod):
    """configs[3] at its full size (N = 65,536) in the configuration bench.py times: 2 levels x 10 sub-steps with
    detection, capacity 2^20 -- the regime of PAPER.md:78-82 where the level-0 pairs link half the disk into one group
    and the higher level dissolves it into ~4000 small groups per sub-step."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    ki = gi.make_config(3)
    n, cap = ki.n, 1 << 20
    assert n == 65536
    k = GengaKick(n, 0, max_level=1, G=ki.G, pair_capacity=cap)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    q, v, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    acc, pairs, npairs, stats = _ml_buffers(n, cap, 2)
    k.multilevel_step(q, v, mass, 1.0, ki.dt, 2, 10, 1e-12, acc, pairs, npairs, stats)
    torch.cuda.synchronize()
    assert k.status() == 0
    r = oracle_mod.step.multilevel_step(ki.pos, ki.vel, ki.mass, n, 0, 1.0, ki.G, ki.dt, slevels=2, substeps=10, tol=1e-12)
    gs = stats.cpu().numpy()
    assert r.stats[0, 1] > 400000 and r.stats[1, 2] > 30000
    # the per-level decisions (integers from floating point) may differ for a pair within rounding of a threshold: the
    # critical radii of the two sides differ by <= 7 u (tests/test_gpu_step.py); allow 2 in 1e5, report exact equality
    assert np.all(np.abs(gs - r.stats) <= np.maximum(2, 2e-5 * r.stats)), (gs.tolist(), r.stats.tolist())
    print("per-level statistics identical:", bool(np.array_equal(gs, r.stats)), gs.tolist())
    _ml_check(ki, q.cpu().numpy(), v.cpu().numpy(), r, r.first.count > 0, gpu_totals=k.bs_totals())
    k.free()


@pytest.mark.parametrize("tp_mode,slevels", [(1, 2), (2, 3)])
def test_multilevel_step_with_semi_active_particles(oracle_mod, tp_mode, slevels):
    """A reduced config 4 (massive bodies + semi-active particles, sec. 8.1) through the multi-level
    step: particles feel the massive bodies (TP 2: and act on them), never each other -- in the kicks of every level."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    ki = gi.make_config(4, n=400, n_test=6000)
    mass = ki.mass.copy()
    if tp_mode == 2:
        mass[ki.n_massive:] = 1e-12
    n, cap = ki.n, 1 << 16
    k = GengaKick(ki.n_massive, ki.n_test, max_level=slevels - 1, G=ki.G, pair_capacity=cap, tp_mode=tp_mode)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    q, v, m = _dev(ki.pos), _dev(ki.vel), _dev(mass)
    acc, pairs, npairs, stats = _ml_buffers(n, cap, slevels)
    k.multilevel_step(q, v, m, 1.0, ki.dt, slevels, 2, 1e-12, acc, pairs, npairs, stats)
    torch.cuda.synchronize()
    assert k.status() == 0
    r = _oracle_ml_tp(oracle_mod, ki, mass, slevels, tp_mode)
    assert np.array_equal(stats.cpu().numpy(), r.stats), (stats.cpu().numpy().tolist(), r.stats.tolist())
    assert r.stats[0, 1] > 20 and r.stats[-1, 2] > 5
    c = npairs.cpu().numpy()
    pr = pairs.cpu().numpy()[:c[n]]
    assert (pr[:, 0] < ki.n_massive).all()                              # no particle-particle pairs
    _ml_check(ki, q.cpu().numpy(), v.cpu().numpy(), r, r.first.count > 0, gpu_totals=k.bs_totals())
    k.free()


def _oracle_ml_tp(oracle_mod, ki, mass, slevels, tp_mode):
    return oracle_mod.step.multilevel_step(ki.pos, ki.vel, mass, ki.n_massive, ki.n_test, 1.0, ki.G, ki.dt,
                                           slevels=slevels, substeps=2, tol=1e-12, tp_mode=tp_mode)
