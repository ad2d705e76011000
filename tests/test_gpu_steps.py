"""-m gpu: genga_steps (include/genga_senc.h) -- n consecutive steps with the closing kick of a step and the opening
kick of the next merged into one pass over the pairs -- against the oracle's n single steps (oracle.step.steps: the
repetition of the step IS the definition; the merge may only change the rounding of the far-field sums).

Bounds.  One step agrees with the oracle's step to 32 u (tests/test_gpu_step.py).  Over n free-running steps the two
trajectories drift apart by at most n x 32 u x the Kepler shear's amplification 1.5 n_K t (a relative error e in the
semi-major axis becomes a phase error 1.5 n_K t e; n_K t = mean motion x elapsed time at the disk's inner edge, at
least 1): the same derivation as test_twenty_steps_track_the_oracle.  Bodies inside close encounters: as
tests/test_gpu_senc.py (same Bulirsch-Stoer decisions => 2.5e-13 per step)."""
import numpy as np
import pytest

import genga_inputs as gi
from tests.gpu_harness import sorted_pairs

pytestmark = pytest.mark.gpu
U = 2.0 ** -53
G = gi.G_AU_DAY_MSUN


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _ctx(ki, max_level=0, capacity=1 << 20, **kw):
    import torch
    from paper_2201_10058_b200 import GengaKick
    k = GengaKick(ki.n_massive, ki.n_test, max_level=max_level, pair_capacity=capacity, G=ki.G, enc_factor=ki.enc_factor, **kw)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    return k


def _buffers(n, cap, slevels):
    import torch
    return (torch.empty(3, n, dtype=torch.float64, device="cuda"), torch.empty(cap, 2, dtype=torch.int32, device="cuda"),
            torch.empty(n + 1, dtype=torch.int32, device="cuda"),
            torch.zeros(max(slevels, 1), 4, dtype=torch.int32, device="cuda"))


def _scales(pos, vel, dt):
    r = np.sqrt((pos ** 2).sum(0)); sp = np.sqrt((vel ** 2).sum(0))
    return r + sp * dt, sp + r * np.sqrt(G / r ** 3)


def _bound_u(ki, n_steps):
    a_min = 0.5                                               # inner edge of every disk of genga_inputs
    nkt = np.sqrt(G / a_min ** 3) * n_steps * ki.dt
    return n_steps * 32 * max(1.0, 1.5 * nkt)


def test_one_step_is_genga_step_bit_for_bit():
    """n_steps = 1 has no kick to merge: the launch sequence of genga_step, the same bits."""
    ki = gi.make_config(1, n=3000)
    n = ki.n
    k = _ctx(ki, capacity=1 << 16)
    mass = _dev(ki.mass)
    acc, pairs, npairs, stats = _buffers(n, 1 << 16, 0)
    q1, v1 = _dev(ki.pos), _dev(ki.vel)
    k.step(q1, v1, mass, 1.0, ki.dt, None, acc, pairs, npairs)
    a1, p1 = acc.clone(), sorted_pairs(pairs.cpu().numpy()[:int(npairs[n])])
    q2, v2 = _dev(ki.pos), _dev(ki.vel)
    k.steps(q2, v2, mass, 1.0, ki.dt, 1, 0, 2, 1e-12, acc, pairs, npairs, None)
    import torch
    torch.cuda.synchronize()
    assert torch.equal(q1, q2) and torch.equal(v1, v2) and torch.equal(a1, acc)
    assert np.array_equal(p1, sorted_pairs(pairs.cpu().numpy()[:int(npairs[n])])) and k.status() == 0
    k.free()


@pytest.mark.parametrize("name,n,n_steps", [("cfg1", 3000, 5), ("cfg1", 8192, 3), ("cfg3_full", 65536, 3), ("cfg4_tp", 2048, 4)])
def test_merged_steps_without_encounter_branch(oracle_mod, name, n, n_steps):
    import torch
    ki = {"cfg1": lambda: gi.make_config(1, n=n), "cfg3_full": lambda: gi.make_config(3, level=0),
          "cfg4_tp": lambda: gi.make_config(4, n=2048, n_test=50000)}[name]()
    nn = ki.n
    k = _ctx(ki)
    mass = _dev(ki.mass)
    acc, pairs, npairs, stats = _buffers(nn, 1 << 20, 0)
    q, v = _dev(ki.pos), _dev(ki.vel)
    k.steps(q, v, mass, 1.0, ki.dt, n_steps, 0, 2, 1e-12, acc, pairs, npairs, None)
    torch.cuda.synchronize()
    assert k.status() == 0
    # the same steps one by one on the device: the merge only changes the rounding of the far-field sums
    qs, vs = _dev(ki.pos), _dev(ki.vel)
    acc2, pairs2, npairs2, _ = _buffers(nn, 1 << 20, 0)
    for _ in range(n_steps):
        k.step(qs, vs, mass, 1.0, ki.dt, None, acc2, pairs2, npairs2)
    torch.cuda.synchronize()
    rs = oracle_mod.step.steps(ki.pos, ki.vel, ki.mass, ki.n_massive, ki.n_test, 1.0, ki.G, ki.dt, n_steps)
    r = rs[-1]
    sq, sv = _scales(r.pos, r.vel, ki.dt)
    dq = np.max(np.abs(q.cpu().numpy() - r.pos) / sq) / U; dv = np.max(np.abs(v.cpu().numpy() - r.vel) / sv) / U
    sep_q = np.max(np.abs(q.cpu().numpy() - qs.cpu().numpy()) / sq) / U
    sep_v = np.max(np.abs(v.cpu().numpy() - vs.cpu().numpy()) / sv) / U
    bound = _bound_u(ki, n_steps)
    print(f"{name} N={nn}, {n_steps} merged steps: {dq:.1f} u (pos), {dv:.1f} u (vel) from the oracle's {n_steps} steps "
          f"(bound {bound:.0f} u); {sep_q:.1f} u / {sep_v:.1f} u from {n_steps} separate device steps")
    assert dq <= bound and dv <= bound and sep_q <= bound and sep_v <= bound
    # the candidates handed out are those of the LAST step's opening kick
    got = {tuple(p) for p in pairs.cpu().numpy()[:int(npairs[nn])].tolist()}
    want = {tuple(p) for p in oracle_mod.pair_set(r.first, ki.n_massive).tolist()}
    border = {tuple(sorted(p)) for p in r.first.border.tolist()}
    # (a pair within rounding of the threshold may differ: the two sides' states differ by the bound above)
    assert len(got ^ want) <= max(2, 1e-4 * len(want)) or (got ^ want) <= border, len(got ^ want)
    k.free()


@pytest.mark.parametrize("slevels,substeps,detect,n_steps", [(1, 2, False, 3), (2, 2, True, 3), (3, 2, True, 2)])
def test_merged_steps_with_encounters(oracle_mod, slevels, substeps, detect, n_steps):
    import torch
    ki = gi.make_config(1, n=4000)
    n, cap = ki.n, 1 << 18
    k = _ctx(ki, max_level=slevels - 1, capacity=cap)
    mass = _dev(ki.mass)
    acc, pairs, npairs, stats = _buffers(n, cap, slevels)
    q, v = _dev(ki.pos), _dev(ki.vel)
    k.steps(q, v, mass, 1.0, ki.dt, n_steps, slevels, substeps, 1e-12, acc, pairs, npairs, stats, detect=detect)
    torch.cuda.synchronize()
    assert k.status() == 0
    rs = oracle_mod.step.steps(ki.pos, ki.vel, ki.mass, n, 0, 1.0, ki.G, ki.dt, n_steps, slevels=slevels,
                               substeps=substeps, tol=1e-12, detect=detect)
    r = rs[-1]
    want_stats = sum(x.stats for x in rs)
    want_tot = tuple(sum(x.bs_totals[i] for x in rs) for i in range(4))
    got_stats, got_tot = stats.cpu().numpy(), tuple(k.bs_totals())
    same = np.array_equal(got_stats, want_stats) and got_tot == want_tot
    in_enc = np.zeros(n, bool)
    for x in rs:
        in_enc |= x.first.count > 0
    sq, sv = _scales(r.pos, r.vel, ki.dt)
    eq = np.abs(q.cpu().numpy() - r.pos) / sq; ev = np.abs(v.cpu().numpy() - r.vel) / sv
    out_u = max(eq[:, ~in_enc].max(), ev[:, ~in_enc].max()) / U
    ins = max(eq[:, in_enc].max(), ev[:, in_enc].max())
    bound = _bound_u(ki, n_steps)
    in_bound = (2.5e-13 if same else 4e-9) * n_steps * max(1.0, bound / (32 * n_steps))
    print(f"{slevels} levels x {substeps}, {n_steps} merged steps: outside encounters {out_u:.1f} u (bound {bound:.0f} u), "
          f"inside {ins:.2e} (bound {in_bound:.1e}); statistics and Bulirsch-Stoer record equal to the oracle's: {same} "
          f"{got_tot} / {want_tot}")
    assert out_u <= bound and ins <= in_bound
    assert np.all(np.abs(got_stats - want_stats) <= np.maximum(2, 1e-3 * want_stats))
    k.free()


def test_rcrit_jump_is_reported():
    """The merged kick builds its candidate list for critical radii up to 1 + 1/64 times those of the step that ends.
    Two heavy bodies (1e-2 solar masses, Hill-dominated critical radii) 0.7 AU apart and a 60-day step: the closing
    kick changes a semi-major axis, hence a Hill radius, by 2 % -- the next step's radius is outside that allowance and
    the status word says so (the caller repeats those steps with genga_step).  The disks above never raise it."""
    import torch
    import paper_2201_10058_b200 as g
    pos = np.array([[1.0, 1.0], [0.0, 0.7], [0.0, 0.0]])
    r = np.sqrt((pos ** 2).sum(0)); vc = np.sqrt(G / r)
    vel = np.stack([-pos[1] / r * vc, pos[0] / r * vc, np.zeros(2)])
    k = g.GengaKick(2, 0, max_level=0, pair_capacity=16, G=G)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    q, v = _dev(pos), _dev(vel)
    k.steps(q, v, _dev(np.array([1e-2, 1e-2])), 1.0, 60.0, 2, 0, 2, 1e-12, None, torch.empty(16, 2, dtype=torch.int32, device="cuda"),
            torch.empty(3, dtype=torch.int32, device="cuda"), None)
    torch.cuda.synchronize()
    assert k.status() & g.binding.STATUS_RCRIT_JUMP
    k.free()


def test_steps_error_codes_and_graph_capture():
    import torch
    import paper_2201_10058_b200 as g
    ki = gi.make_config(1, n=2000)
    n, cap = ki.n, 1 << 16
    k = _ctx(ki, max_level=1, capacity=cap)
    mass = _dev(ki.mass)
    acc, pairs, npairs, stats = _buffers(n, cap, 2)
    q, v = _dev(ki.pos), _dev(ki.vel)
    for call, code in [(lambda: k.steps(q, v, mass, 1.0, ki.dt, 0, 0, 2, 1e-12, acc, pairs, npairs, None), g.E_SIZE),
                       (lambda: k.steps(q, v, mass, 1.0, ki.dt, 2, 5, 2, 1e-12, acc, pairs, npairs, None), g.E_SIZE),
                       (lambda: k.steps(q, v, mass, 1.0, ki.dt, 2, 3, 2, 1e-12, acc, pairs, npairs, None), g.E_LEVEL),
                       (lambda: k.steps(q, v, mass, 0.0, ki.dt, 2, 0, 2, 1e-12, acc, pairs, npairs, None), g.E_SIZE),
                       (lambda: k.steps(q, None, mass, 1.0, ki.dt, 2, 0, 2, 1e-12, acc, pairs, npairs, None), g.E_NULL)]:
        with pytest.raises(g.GengaKickError) as e:
            call()
        assert e.value.code == code
    # plain launches, then the same call captured in a CUDA graph and replayed: same bits
    k.steps(q, v, mass, 1.0, ki.dt, 3, 2, 2, 1e-12, acc, pairs, npairs, stats)
    torch.cuda.synchronize()
    want_q, want_v, want_s = q.clone(), v.clone(), stats.clone()
    q.copy_(_dev(ki.pos)); v.copy_(_dev(ki.vel))
    gs = torch.cuda.Stream()
    torch.cuda.synchronize()
    k.set_stream(gs.cuda_stream)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=gs):
        k.steps(q, v, mass, 1.0, ki.dt, 3, 2, 2, 1e-12, acc, pairs, npairs, stats)
    q.copy_(_dev(ki.pos)); v.copy_(_dev(ki.vel))
    torch.cuda.synchronize()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(q, want_q) and torch.equal(v, want_v) and torch.equal(stats, want_s) and k.status() == 0
    k.free()
