"""-m gpu: genga_bs (include/genga_bs.h) through the C ABI against oracle/genga_bs_oracle.c.

Both sides run the same Gragg-Bulirsch-Stoer scheme (reading G15) in IEEE binary64 without contraction.  The oracle adds
a body's pair terms in member order, for every group size; the kernel does the same for groups of up to 8 bodies (one
lane per body) and spreads the sum over eight lanes with a tree above that -- its choice, not the oracle's.  Hence:

  * groups of <= 8 bodies: same operations in the same order => the bar is EQUAL BITS (and equal step-size decisions);
  * larger groups: the force sums differ at rounding level.  As long as both sides take the same step-size decisions
    (accepted steps, halvings, force evaluations -- the kernel reports them per group, genga_bs_set_stats), the results
    differ by that rounding, amplified by the encounter; where an error estimate falls within rounding of tol the two
    sides may decide differently (a FLIP: counted and reported, the analogue of north_star's borderline pairs), and then
    they are two valid answers of the scheme.  Either way each side's local error per accepted macro step is <= tol
    (relative, per body, in position and in velocity: the scheme's own acceptance test), so
        |dq| / |q|,  |dv| / |v|   <=   C_TOL * tol * (accepted macro steps of the group)
    with C_TOL = 4 (2 sides x 2 for the error estimate being that of the previous column).  The measured worst ratio
    to that bound is printed, so the record shows the slack; without a flip it is 1e-7 .. 1e-1 (1 .. 3000 u).
  * a flipped group whose encounter amplifies perturbations (a bound, nearly radial passage takes thousands of macro
    steps) is compared under the same bound times the amplification A of the flow, MEASURED on the oracle: the
    relative change of its result under a relative perturbation of 2^-40 of the group's input positions, over 2^-40
    (at least 1).  A is printed with the flip; where A * bound exceeds 1 the group is chaotic at this tolerance, the
    two answers are both valid and nothing more can be asserted than that the kernel reports it took other decisions."""
import numpy as np
import pytest

import genga_inputs as gi

pytestmark = pytest.mark.gpu
U = 2.0 ** -53
G = gi.G_AU_DAY_MSUN
C_TOL = 4.0
SEQ_MAX = 8            # groups up to here are summed in member order by the kernel too (include/genga_bs.h)


def _dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a))
    return (t if dtype is None else t.to(dtype)).cuda()


def _gpu_bs(n, pos_in, vel_in, mass, rcrit, nlevels, dt, tol, members, offsets, pos, vel):
    """Returns (pos, vel, status, per-group rows (accepted, rejected, force evaluations, bodies))."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    k = GengaKick(n, 0, G=G, pair_capacity=8)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    ng = len(offsets) - 1
    d_mem = torch.zeros(max(n, 4), dtype=torch.int32, device="cuda"); d_mem[:len(members)] = _dev(np.asarray(members, np.int32))
    d_off = torch.zeros(n + 4, dtype=torch.int32, device="cuda"); d_off[:ng + 1] = _dev(np.asarray(offsets, np.int32))
    largest = int(np.diff(np.asarray(offsets)).max()) if ng else 0
    d_sum = torch.tensor([ng, len(members), largest, 0], dtype=torch.int32, device="cuda")
    gstats = torch.full((max(ng, 1), 4), -1, dtype=torch.int32, device="cuda")
    k.bs_set_stats(gstats, max(ng, 1))
    q, v = _dev(pos), _dev(vel)
    k.bs(_dev(pos_in), _dev(vel_in), _dev(mass), _dev(np.asarray(rcrit)[:nlevels]), nlevels, 1.0, dt, tol, d_mem, d_off,
         d_sum, q, v)
    torch.cuda.synchronize()
    st = k.status()
    tot = k.bs_totals()
    gs = gstats.cpu().numpy()[:ng]
    assert tot[3] == ng and tot[0] == gs[:, 0].sum() and tot[2] == gs[:, 2].sum()
    k.free()
    return q.cpu().numpy(), v.cpu().numpy(), st, gs


def _amplification(rerun, idx, qw, vw):
    """Sensitivity of the oracle's result for one group to its input: see the header."""
    delta = 2.0 ** -40
    qp, vp = rerun(idx, delta)
    nq = np.sqrt((qw[:, idx] ** 2).sum(0)); nv = np.sqrt((vw[:, idx] ** 2).sum(0))
    rel = max(np.max(np.sqrt(((qp - qw[:, idx]) ** 2).sum(0)) / nq), np.max(np.sqrt(((vp - vw[:, idx]) ** 2).sum(0)) / nv))
    return max(1.0, rel / delta)


def _check(q, v, qw, vw, members, offsets, gstats, ostats, tol, label="", rerun=None):
    """The rule of this file's header, group by group.  Returns (all bits equal, number of flipped groups).
    rerun(idx, delta) -> the oracle's (q, v) of the group with bodies idx from input positions scaled by 1 + delta *
    (a fixed +-1 pattern); needed only if a group flips."""
    members = np.asarray(members); offsets = np.asarray(offsets)
    flips, worst, worst_u, small, equal = 0, 0.0, 0.0, 0, True
    for g in range(len(offsets) - 1):
        idx = members[offsets[g]:offsets[g + 1]]
        want = (ostats[g].accepted, ostats[g].rejected, ostats[g].force_evaluations, len(idx))
        flip = tuple(int(x) for x in gstats[g]) != want
        flips += flip
        nq = np.sqrt((qw[:, idx] ** 2).sum(0)); nv = np.sqrt((vw[:, idx] ** 2).sum(0))
        rel = max(np.max(np.sqrt(((q[:, idx] - qw[:, idx]) ** 2).sum(0)) / nq),
                  np.max(np.sqrt(((v[:, idx] - vw[:, idx]) ** 2).sum(0)) / nv))
        same = np.array_equal(q[:, idx], qw[:, idx]) and np.array_equal(v[:, idx], vw[:, idx])
        equal &= bool(same)
        if len(idx) <= SEQ_MAX:
            small += 1
            assert same and not flip, f"group {g} of {len(idx)} bodies (member-order sum on both sides): bits differ"
            continue
        steps = max(int(gstats[g][0]), ostats[g].accepted)
        amp = 1.0
        if flip and rel > C_TOL * tol * steps and rerun is not None:
            amp = _amplification(rerun, idx, qw, vw)
            print(f"{label}group {g} ({len(idx)} bodies): flipped decision, kernel {tuple(int(x) for x in gstats[g][:3])} vs "
                  f"oracle {want[:3]}; difference {rel:.2e}; amplification of the flow {amp:.2e}; bound "
                  f"{min(1.0, amp * C_TOL * tol * steps):.2e}" + (" (chaotic at this tolerance)" if amp * C_TOL * tol * steps >= 1 else ""))
        if amp * C_TOL * tol * steps < 1.0:
            assert rel <= amp * C_TOL * tol * steps, (f"group {g} ({len(idx)} bodies, flip={flip}): {rel:.2e} > "
                                                      f"{amp:.1e} * {C_TOL} * tol * {steps} accepted steps")
        worst = max(worst, rel / (amp * C_TOL * tol * steps))
        if not flip:
            worst_u = max(worst_u, rel / U)
    ng = len(offsets) - 1
    print(f"{label}{ng} groups ({small} of <= {SEQ_MAX} bodies: bit-identical); larger groups: {flips} with a flipped "
          f"step-size decision, worst difference / (C_TOL tol steps) = {worst:.2e}, worst without a flip = {worst_u:.0f} u")
    return equal, flips


def test_groups_of_a_disk_kick_group_bs_chain(oracle_mod):
    """Config 1's shape: the pair list of the oracle's kick, grouped by the oracle, every group integrated on both
    sides from the pre-drift state; bodies in no group keep the (Kepler-drifted) state passed in."""
    ki = gi.make_config(1, n=6000)
    n = ki.n
    res = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, n, 0, level=0, G=ki.G)
    gr = oracle_mod.group.group(n, oracle_mod.pair_set(res, n))
    assert gr.n_groups > 100
    qf, vf, _ = oracle_mod.step.fg(ki.pos, ki.vel, ki.G, ki.dt)                     # what FG left in pos / vel
    qw, vw, stats, skipped = oracle_mod.bs.bs(ki.pos, ki.vel, ki.mass, ki.rcrit, gr.members, gr.offsets, G, 1.0, ki.dt,
                                              1e-12, qf, vf, nlevels=1)
    assert not skipped and not any(s.failed for s in stats)
    q, v, st, gs = _gpu_bs(n, ki.pos, ki.vel, ki.mass, ki.rcrit, 1, ki.dt, 1e-12, gr.members, gr.offsets, qf, vf)
    assert st == 0
    exact, _ = _check(q, v, qw, vw, gr.members, gr.offsets, gs, stats, 1e-12)
    untouched = gr.group_of < 0
    assert np.array_equal(q[:, untouched], qf[:, untouched]) and np.array_equal(v[:, untouched], vf[:, untouched])
    assert np.max(np.abs(q[:, ~untouched] - qf[:, ~untouched])) > 1e-12               # the encounters matter
    print("every group bit-identical to the oracle:", exact)


@pytest.mark.parametrize("nlevels,tol,dt", [(1, 1e-13, 6.0), (2, 1e-11, 6.0), (1, 1e-9, -3.0), (3, 1e-12, 0.75)])
def test_dense_groups_levels_tolerances(oracle_mod, nlevels, tol, dt):
    """A denser disk (larger groups, up to the 256-body limit), several levels / tolerances / a negative step."""
    ki = gi.make_disk(3000, 31, level=2, substeps=2, total_mass=20 * gi.M_EARTH, a_lo=0.9, a_hi=1.3)
    n = ki.n
    res = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, n, 0, level=0, G=ki.G, maxp=256)
    gr = oracle_mod.group.group(n, oracle_mod.pair_set(res, n))
    qw, vw, stats, skipped = oracle_mod.bs.bs(ki.pos, ki.vel, ki.mass, ki.rcrit, gr.members, gr.offsets, G, 1.0, dt, tol,
                                              ki.pos, ki.vel, nlevels=nlevels, max_group=None)
    q, v, st, gs = _gpu_bs(n, ki.pos, ki.vel, ki.mass, ki.rcrit, nlevels, dt, tol, gr.members, gr.offsets, ki.pos, ki.vel)
    assert st == 0 and not skipped
    assert gr.max_size > 20 and len(stats) > 50
    _check(q, v, qw, vw, gr.members, gr.offsets, gs, stats, tol)


def test_large_groups_whole_grid_regime(oracle_mod):
    """Groups above 256 bodies are integrated by the whole grid, one group at a time (the paper's BS-M regime with the
    sub-steps kept on the device): rings of 257 .. 3000 bodies, one group each, and a mix of small and large groups."""
    for m in (200, 257, 700, 1024, 3000):
        ki = gi.make_ring(m)
        qw, vw, stats, _ = oracle_mod.bs.bs(ki.pos, ki.vel, ki.mass, ki.rcrit, np.arange(m), [0, m], ki.G, 1.0, 6.0, 1e-12,
                                            ki.pos, ki.vel, max_group=None)
        q, v, st, gs = _gpu_bs(m, ki.pos, ki.vel, ki.mass, ki.rcrit, 1, 6.0, 1e-12, np.arange(m), [0, m], ki.pos, ki.vel)
        assert st == 0
        _check(q, v, qw, vw, np.arange(m), [0, m], gs, stats, 1e-12, label=f"ring of {m}: ")
    # three groups in one call: 300 (whole grid), 40 (one CTA), 500 (whole grid) bodies of one ring
    ki = gi.make_ring(840)
    members, offsets = np.arange(840), [0, 300, 340, 840]
    qw, vw, stats, _ = oracle_mod.bs.bs(ki.pos, ki.vel, ki.mass, ki.rcrit, members, offsets, ki.G, 1.0, -6.0, 1e-11, ki.pos,
                                        ki.vel, max_group=None)
    q, v, st, gs = _gpu_bs(840, ki.pos, ki.vel, ki.mass, ki.rcrit, 1, -6.0, 1e-11, members, offsets, ki.pos, ki.vel)
    assert st == 0
    _check(q, v, qw, vw, members, offsets, gs, stats, 1e-11)


def test_bs_error_codes_and_empty():
    import torch
    import paper_2201_10058_b200 as g
    k = g.GengaKick(64, 0, pair_capacity=8)
    x = torch.zeros(3, 64, dtype=torch.float64, device="cuda"); y = torch.zeros_like(x)
    m = torch.zeros(64, dtype=torch.float64, device="cuda")
    i = torch.zeros(80, dtype=torch.int32, device="cuda")
    for call, code in [(lambda: k.bs(x, x, m, m, 1, 1.0, 6.0, 1e-12, i, i, i, None, y), g.E_NULL),
                       (lambda: k.bs(x, x, m, m, 0, 1.0, 6.0, 1e-12, i, i, i, y, y), g.E_SIZE),
                       (lambda: k.bs(x, x, m, m, 1, 1.0, 6.0, 0.0, i, i, i, y, y), g.E_SIZE),
                       (lambda: k.bs(x, x, m, m, 1, 1.0, 6.0, 1e-12, i, i, i, x, y), g.E_SIZE),
                       (lambda: k.bs(x, x, m, m, 1, 1.0, 6.0, 1e-12, i[1:], i, i, y, y.clone()), g.E_ALIGN)]:
        with pytest.raises(g.GengaKickError) as e:
            call()
        assert e.value.code == code
    z = y.clone()
    k.bs(x, x, m, m, 1, 1.0, 6.0, 1e-12, i, i, i, y, z)              # no groups: nothing happens
    torch.cuda.synchronize()
    assert k.status() == 0 and not y.any()
    k.free()


def _hybrid_buffers(n, cap):
    import torch
    i32 = lambda m: torch.empty(m, dtype=torch.int32, device="cuda")
    return (torch.empty(3, n, dtype=torch.float64, device="cuda"), torch.empty(cap, 2, dtype=torch.int32, device="cuda"),
            i32(n + 1), i32(n), i32(n), i32(n + 1), i32(4))


def test_hybrid_step_against_oracle(oracle_mod):
    """genga_hybrid_step (kick, HC, FG, grouping, Bulirsch-Stoer, HC, kick on the device) against oracle.step.hybrid_step."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    ki = gi.make_config(1, n=5000)
    n = ki.n
    k = GengaKick(n, 0, G=ki.G, pair_capacity=1 << 18)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    q, v, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    acc, pairs, npairs, group_of, members, offsets, summary = _hybrid_buffers(n, 1 << 18)
    k.hybrid_step(q, v, mass, 1.0, ki.dt, 1e-12, acc, pairs, npairs, group_of, members, offsets, summary)
    torch.cuda.synchronize()
    r = oracle_mod.step.hybrid_step(ki.pos, ki.vel, ki.mass, n, 0, 1.0, ki.G, ki.dt, tol=1e-12)
    assert k.status() == 0 and not r.skipped and r.groups.n_groups > 50
    s = summary.cpu().numpy()
    assert s[0] == r.groups.n_groups and s[1] == r.groups.n_members and s[2] == r.groups.max_size
    assert np.array_equal(group_of.cpu().numpy(), r.groups.group_of)
    rr = np.sqrt((ki.pos ** 2).sum(0)); sp = np.sqrt((ki.vel ** 2).sum(0))
    sq, sv = rr + sp * ki.dt, sp + rr * np.sqrt(ki.G / rr ** 3)
    # the states entering Bulirsch-Stoer differ by the kick's and HC's rounding (<= 32 u), which an encounter
    # amplifies.  Same record of the step-size control on both sides (the usual case): same operations on inputs 32 u
    # apart, bound 2.5e-13 relative (~100 x the largest difference measured here, 1.8e-15; printed).  A different record: some
    # error estimate fell within rounding of tol, two valid answers of the scheme: 4 tol x 1e3 (amplification), reported.
    in_group = r.groups.group_of >= 0
    assert np.all(np.abs(q.cpu().numpy() - r.pos)[:, ~in_group] <= 32 * U * sq[~in_group])
    assert np.all(np.abs(v.cpu().numpy() - r.vel)[:, ~in_group] <= 32 * U * sv[~in_group])
    tot = k.bs_totals()
    same = tuple(tot) == tuple(r.bs_totals)
    bound = 2.5e-13 if same else 4e3 * 1e-12
    worst = max(np.max(np.abs(q.cpu().numpy() - r.pos)[:, in_group] / sq[in_group]),
                np.max(np.abs(v.cpu().numpy() - r.vel)[:, in_group] / sv[in_group]))
    print(f"hybrid step: bodies in groups: worst difference {worst:.2e} (bound {bound:.0e}); Bulirsch-Stoer record kernel {tot} "
          f"oracle {r.bs_totals}" + ("" if same else "  ** a step-size decision flipped **"))
    assert worst <= bound
    k.free()


def test_hybrid_step_keeps_the_energy_through_an_encounter():
    """The device integrator through the close encounter of tests/test_step_oracle_pins.py: energy error < 1e-5
    (the plain step loses 6e-3 there)."""
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
    k = GengaKick(2, 0, G=G, pair_capacity=16)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    q, v, m = _dev(pos), _dev(vel), _dev(mass)
    acc, pairs, npairs, group_of, members, offsets, summary = _hybrid_buffers(2, 16)
    worst, enc, dmin = 0.0, 0, 1e9
    for _ in range(400):
        k.hybrid_step(q, v, m, 1.0, 2.0, 1e-13, acc, pairs, npairs, group_of, members, offsets, summary)
        enc += int(summary[0])
        qq, vv = q.cpu().numpy(), v.cpu().numpy()
        dmin = min(dmin, np.sqrt(((qq[:, 0] - qq[:, 1]) ** 2).sum()))
        worst = max(worst, abs(energy(qq, vv) - e0) / abs(e0))
    assert k.status() == 0 and enc > 3 and dmin < 5e-3
    assert worst < 1e-5
    k.free()


@pytest.mark.parametrize("tp_mode", [1, 2])
def test_semi_active_particles_in_groups(oracle_mod, tp_mode):
    """Groups that mix massive bodies and semi-active particles WITH mass (sec. 8.1): particles feel
    the massive bodies, act on them only in TP 2 and never feel each other -- bit for bit against the oracle's rule."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    rng = np.random.default_rng(17)
    n_m, n_t = 40, 360
    n = n_m + n_t
    ki = gi.make_config(0, n=n)
    pos, vel = ki.pos.copy(), ki.vel.copy()
    # ten particles in a tight cloud around each of the first 36 massive bodies; one group per cloud
    members, offsets = [], [0]
    for g in range(36):
        idx = np.arange(n_m + 10 * g, n_m + 10 * g + 10)
        pos[:, idx] = pos[:, [g]] + rng.normal(scale=4e-3, size=(3, 10))
        vel[:, idx] = vel[:, [g]] + rng.normal(scale=3e-5, size=(3, 10))
        members += [g] + idx.tolist(); offsets.append(len(members))
    mass = np.full(n, 2e-6); mass[n_m:] = rng.uniform(1e-8, 1e-7, n_t)
    rc = np.full((2, n), 0.03); rc[1] = 0.012
    k = GengaKick(n_m, n_t, G=G, pair_capacity=8, tp_mode=tp_mode)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    d_mem = _dev(np.asarray(members + [0] * (n - len(members)), np.int32))
    d_off = torch.zeros(n + 4, dtype=torch.int32, device="cuda"); d_off[:len(offsets)] = _dev(np.asarray(offsets, np.int32))
    d_sum = torch.tensor([36, len(members), 11, 0], dtype=torch.int32, device="cuda")
    gstats = torch.full((36, 4), -1, dtype=torch.int32, device="cuda")
    k.bs_set_stats(gstats, 36)
    q, v = _dev(pos), _dev(vel)
    k.bs(_dev(pos), _dev(vel), _dev(mass), _dev(rc), 2, 1.0, 3.0, 1e-12, d_mem, d_off, d_sum, q, v)
    torch.cuda.synchronize()
    assert k.status() == 0
    k.free()
    qw, vw, stats, _ = oracle_mod.bs.bs(pos, vel, mass, rc, np.asarray(members), np.asarray(offsets), G, 1.0, 3.0, 1e-12,
                                        pos, vel, nlevels=2, n_massive=n_m, tp_mode=tp_mode)
    sign = np.where(rng.random(pos.shape) < 0.5, -1.0, 1.0)

    def rerun(idx, delta):
        qq, vv, _ = oracle_mod.bs.bs_group(pos[:, idx] * (1.0 + delta * sign[:, idx]), vel[:, idx], mass[idx], rc[:, idx], G, 1.0,
                                           3.0, 1e-12, is_tp=idx >= n_m, tp_mode=tp_mode)
        return qq, vv

    _check(q.cpu().numpy(), v.cpu().numpy(), qw, vw, members, offsets, gstats.cpu().numpy(), stats, 1e-12, rerun=rerun)
    # and the rule matters here: the fully interactive result is far away
    qf, vf, _, _ = oracle_mod.bs.bs(pos, vel, mass, rc, np.asarray(members), np.asarray(offsets), G, 1.0, 3.0, 1e-12,
                                    pos, vel, nlevels=2)
    assert np.abs(qf - qw).max() > 1e-9


@pytest.mark.parametrize("tp_mode,m", [(1, 300), (2, 300), (2, 2600)])
def test_semi_active_particles_in_a_large_group(oracle_mod, tp_mode, m):
    """The test-particle rules in the whole-grid regime (teams and the full grid), where they decide what a body's
    neighbour list holds: a ring in which every third body is massive and the others are semi-active particles with mass,
    one group; against the oracle's rule, and the rule matters (TP 1, TP 2 and the fully interactive result differ)."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    ring = gi.make_ring(m)
    n_m = m // 3
    order = np.concatenate([np.arange(0, 3 * n_m, 3), np.setdiff1d(np.arange(m), np.arange(0, 3 * n_m, 3))])
    pos, vel = np.ascontiguousarray(ring.pos[:, order]), np.ascontiguousarray(ring.vel[:, order])
    mass = np.full(m, 3e-7); mass[n_m:] = 1e-7 * (0.5 + gi.uniforms(23, 0, m - n_m))
    rc = np.ascontiguousarray(ring.rcrit[:1] * 1.5)
    members, offsets = np.arange(m), [0, m]
    k = GengaKick(n_m, m - n_m, G=G, pair_capacity=8, tp_mode=tp_mode)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    d_sum = torch.tensor([1, m, m, 0], dtype=torch.int32, device="cuda")
    d_off = torch.zeros(m + 4, dtype=torch.int32, device="cuda"); d_off[1] = m
    gstats = torch.full((1, 4), -1, dtype=torch.int32, device="cuda")
    k.bs_set_stats(gstats, 1)
    q, v = _dev(pos), _dev(vel)
    k.bs(_dev(pos), _dev(vel), _dev(mass), _dev(rc), 1, 1.0, 6.0, 1e-11, _dev(members.astype(np.int32)), d_off, d_sum, q, v)
    torch.cuda.synchronize()
    assert k.status() == 0
    k.free()
    qw, vw, stats, _ = oracle_mod.bs.bs(pos, vel, mass, rc, members, np.asarray(offsets), G, 1.0, 6.0, 1e-11, pos, vel,
                                        n_massive=n_m, tp_mode=tp_mode, max_group=None)
    _check(q.cpu().numpy(), v.cpu().numpy(), qw, vw, members, offsets, gstats.cpu().numpy(), stats, 1e-11)
    qo, vo, _, _ = oracle_mod.bs.bs(pos, vel, mass, rc, members, np.asarray(offsets), G, 1.0, 6.0, 1e-11, pos, vel,
                                    n_massive=n_m, tp_mode=3 - tp_mode, max_group=None)
    assert np.abs(qo - qw).max() > 1e-10


def test_dense_large_group_falls_back_to_all_pairs(oracle_mod):
    """A large group in which every body is inside every other's critical radius: its neighbour lists (n^2 entries) do
    not fit the team's share of the list scratch, the group is integrated over all pairs instead -- same result."""
    m = 2000
    ki = gi.make_ring(m)
    rc = np.full((1, m), 10.0)                                    # AU: K = 0, W_BS = 1 for every pair
    mass = np.full(m, 1e-10)
    qw, vw, stats, _ = oracle_mod.bs.bs(ki.pos, ki.vel, mass, rc, np.arange(m), [0, m], ki.G, 1.0, 1.0, 1e-10, ki.pos, ki.vel,
                                        max_group=None)
    q, v, st, gs = _gpu_bs(m, ki.pos, ki.vel, mass, rc, 1, 1.0, 1e-10, np.arange(m), [0, m], ki.pos, ki.vel)
    assert st == 0 and not stats[0].failed
    _check(q, v, qw, vw, np.arange(m), [0, m], gs, stats, 1e-10)


def test_giant_group_fewer_lanes_per_body(oracle_mod):
    """A group too large for eight lanes per body on the full grid (above 9472 bodies on a B200) is integrated with four
    lanes per body (two, one beyond 18,944 / 37,888), each lane holding more of the eight partial sums: the same tree."""
    m = 12500
    ki = gi.make_ring(m)
    qw, vw, stats, _ = oracle_mod.bs.bs(ki.pos, ki.vel, ki.mass, ki.rcrit, np.arange(m), [0, m], ki.G, 1.0, 2.0, 1e-9,
                                        ki.pos, ki.vel, max_group=None)
    q, v, st, gs = _gpu_bs(m, ki.pos, ki.vel, ki.mass, ki.rcrit, 1, 2.0, 1e-9, np.arange(m), [0, m], ki.pos, ki.vel)
    assert st == 0 and not stats[0].failed
    _check(q, v, qw, vw, np.arange(m), [0, m], gs, stats, 1e-9)
    assert np.abs(q - ki.pos).max() > 1e-3


@pytest.mark.parametrize("m", [20000, 40000])
def test_giant_rings_two_and_one_lanes_per_body(m):
    """Groups above 18,944 and above 37,888 bodies (two lanes, one lane per body: 128 and 256 bodies' lists pooled per CTA)
    are beyond what the oracle integrates in a test's time; a ring has a check of its own: its bodies are images of one
    another under rotation by 2 pi / m, so after the call they must still lie on one circle with one speed and the ring's
    spacing -- a list that lost or doubled an entry, a carry added to the wrong body or a body left out would break it.
    (Rounding differs from body to body: 1e-12.)  The same holds at 12,500 bodies, where the oracle agrees as well."""
    for n in (12500, m):
        ki = gi.make_ring(n)
        q, v, st, gs = _gpu_bs(n, ki.pos, ki.vel, ki.mass, ki.rcrit, 1, 2.0, 1e-9, np.arange(n), [0, n], ki.pos, ki.vel)
        assert st == 0 and gs[0][3] == n and gs[0][0] >= 1
        r, sp = np.linalg.norm(q, axis=0), np.linalg.norm(v, axis=0)
        assert np.ptp(r) <= 1e-12 * r.mean() and np.ptp(sp) <= 1e-12 * sp.mean()
        phi = np.unwrap(np.arctan2(q[1], q[0]))
        assert np.abs(np.diff(phi) - 2.0 * np.pi / n).max() <= 1e-12
        assert np.abs(q[2]).max() == 0.0 and np.abs(q - ki.pos).max() > 1e-3      # planar, and it moved
        if n == 12500:
            ref = (r.mean(), sp.mean())
        else:                                                  # rings of equal bodies with 8 partners each: nearly the same motion
            assert abs(r.mean() - ref[0]) < 1e-6 and abs(sp.mean() - ref[1]) < 1e-7


@pytest.mark.parametrize("size,count,dt,tol", [(40, 700, 3.0, 1e-10), (257, 258, 0.01, 1e-6), (600, 41, 0.5, 1e-8)])
def test_many_mid_size_groups_are_all_found(oracle_mod, size, count, dt, tol):
    """More groups of one regime than one batch of the device-side group scan holds (256): 700 groups of 40 bodies for
    the cluster regime (dealt round-robin to the clusters across batches), 258 groups of 257 bodies for the teams of 64
    CTAs of the whole-grid regime and 41 groups of 600 bodies for its teams of 256 CTAs (several groups at a time, each
    team with its own barrier and neighbour lists) -- arcs of one large ring, every group integrated."""
    m = size * count
    ki = gi.make_ring(m, partners=4)
    members = np.arange(m)
    offsets = np.arange(0, m + 1, size)
    qw, vw, stats, _ = oracle_mod.bs.bs(ki.pos, ki.vel, ki.mass, ki.rcrit, members, offsets, ki.G, 1.0, dt, tol,
                                        ki.pos, ki.vel, max_group=None)
    q, v, st, gs = _gpu_bs(m, ki.pos, ki.vel, ki.mass, ki.rcrit, 1, dt, tol, members, offsets, ki.pos, ki.vel)
    assert st == 0 and len(stats) == count
    _check(q, v, qw, vw, members, offsets, gs, stats, tol)
    # every group moved away from the state the arrays held before the call
    moved = np.abs(q - ki.pos).max(axis=0).reshape(count, size).max(axis=1)
    assert np.all(moved > 1e-6)
