"""-m gpu: the O(N) neighbours of the kick (include/genga_step.h: Rcrit, HC, FG, drift) and the composed
step of App. A through the C ABI, against oracle/genga_step_oracle.c (long double).

Tolerances, derived from the kernels' arithmetic (u = 2^-53):
  Rcrit  16 u relative: 1/a = 2/r - v^2/mu is a difference of terms ~2/a and ~1/a (<= 4 u), cbrt and the
         products add <= 3 u; measured <= 7 u.
  HC     |dq| <= 2 u |q| + (|dt| / m_star) 64 u sum_j |m_j v_j|: one rounding of the sum q + shift, the
         shift's own roundings, and the FP64 momentum sum (<= 4 sequential + 8 tree + <= 1024 CTA partials,
         far below 64 u sum|m v| for the disks here; measured: bit-identical to the long double result).
  FG     |dq| <= 32 u (|q| + |v| |dt|), |dv| <= 32 u (|v| + n |q|): dM = n dt carries <= 4 u, the Newton root
         ~2 u / (1 - e), f, g, fdot, gdot a few u each relative to 1, dt, n, 1; measured <= 3.3 u.
  step   the same bound as FG on the final state (the kicks contribute 1e-13 * sum|term| * dt/2, far
         below it); pair list of the first kick equal as a set outside the 1e-12 band.
"""
import numpy as np
import pytest

import genga_inputs as gi

pytestmark = pytest.mark.gpu
U = 2.0 ** -53
G = gi.G_AU_DAY_MSUN


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _ctx(ki, capacity=1 << 20):
    import torch
    from paper_2201_10058_b200 import GengaKick
    k = GengaKick(ki.n_massive, ki.n_test, max_level=0, pair_capacity=capacity, G=ki.G, enc_factor=ki.enc_factor)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    return k


def _scales(pos, vel, dt, mu=G):
    r = np.sqrt((pos ** 2).sum(0)); v = np.sqrt((vel ** 2).sum(0))
    n = np.sqrt(mu / r ** 3)
    return r + v * abs(dt), v + n * r


CASES = [("cfg0", lambda: gi.make_config(0)), ("cfg3_20k", lambda: gi.make_config(3, n=20000, level=1)),
         ("cfg2_giants", lambda: gi.make_config(2, n=5000)), ("cfg4_tp", lambda: gi.make_config(4, n=2048, n_test=50000)),
         ("n1", lambda: gi.make_config(0, n=1)), ("n257", lambda: gi.make_config(0, n=257)),
         ("n1025", lambda: gi.make_config(0, n=1025))]


@pytest.mark.parametrize("name,make", CASES, ids=[c[0] for c in CASES])
def test_rcrit_hc_fg_against_oracle(oracle_mod, name, make):
    import torch
    ost = oracle_mod.step
    ki = make()
    n = ki.n
    k = _ctx(ki)
    pos, vel, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    # Rcrit: three rows, s = 2
    rc = torch.full((3, n), float("nan"), dtype=torch.float64, device="cuda")
    k.rcrit(pos, vel, mass, 1.0, ki.dt, rc, substeps=2.0, nrows=3)
    want, bad = ost.rcrit(ki.pos, ki.vel, ki.mass, 1.0, ki.G, ki.dt, 2.0, 3)
    assert bad == 0 and np.all(np.abs(rc.cpu().numpy() - want) <= 16 * U * want)
    # HC
    for dt in (3.0, -1.5):
        q = pos.clone()
        k.hc(q, vel, mass, 1.0, dt)
        qw, P = ost.hc(ki.pos, ki.vel, ki.mass, 1.0, dt)
        bound = 2 * U * np.abs(ki.pos) + abs(dt) * 64 * U * np.abs(ki.mass * ki.vel).sum(1, keepdims=True)
        assert np.all(np.abs(q.cpu().numpy() - qw) <= bound)
    # FG
    for dt in (ki.dt, -0.37 * ki.dt, 40.0):
        q, v = pos.clone(), vel.clone()
        k.fg(q, v, 1.0, dt)
        qw, vw, bad = ost.fg(ki.pos, ki.vel, ki.G, dt)
        sq, sv = _scales(ki.pos, ki.vel, dt)
        assert bad == 0
        assert np.all(np.abs(q.cpu().numpy() - qw) <= 32 * U * sq) and np.all(np.abs(v.cpu().numpy() - vw) <= 32 * U * sv)
    assert k.status() == 0
    k.free()


def test_fg_eccentric_orbits_and_long_steps(oracle_mod):
    """e up to 0.95 and dt up to several periods: the bracketed Newton iteration must converge everywhere."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    n = 20000
    u = gi.uniforms(99, 0, 6 * n).reshape(6, n)
    a = 0.3 + 5.0 * u[0]; e = 0.95 * u[1]
    pos, vel = gi.elements_to_cartesian(a, e, 0.5 * u[2], 2 * np.pi * u[3], 2 * np.pi * u[4], 2 * np.pi * u[5], G)
    k = GengaKick(n, 0, G=G)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    for dt in (6.0, 365.25, -1000.0):
        q, v = _dev(pos), _dev(vel)
        k.fg(q, v, 1.0, dt)
        qw, vw, bad = oracle_mod.step.fg(pos, vel, G, dt)
        assert bad == 0
        # the conditioning grows with the number of revolutions (n dt) and with 1 / (1 - e): both sides solve the
        # same equation, the double-precision side carries u n dt / (1 - e)^2 of the mean anomaly's rounding
        nmot = np.sqrt(G / a ** 3)
        amp = 32 * (1.0 + nmot * abs(dt)) / (1.0 - e) ** 2
        sq, sv = _scales(pos, vel, 0.0)
        assert np.all(np.abs(q.cpu().numpy() - qw) <= amp * U * a * 2) and np.isfinite(q.cpu().numpy()).all()
        assert np.all(np.abs(v.cpu().numpy() - vw) <= amp * U * np.sqrt(G / a) / (1.0 - e))
    assert k.status() == 0
    k.free()


def test_hyperbolic_bodies_drift_and_rcrit_reports_them(oracle_mod):
    """Bodies above the escape speed follow their hyperbolic two-body orbit in FG (same bound as the elliptic ones);
    Rcrit has no Hill radius for them and says so."""
    import torch
    import paper_2201_10058_b200 as g
    ki = gi.make_config(0, n=300)
    ki.vel[:, 17] *= 3.0                                     # hyperbolic
    ki.vel[:, 40] *= -1.6
    ki.vel[:, 41] = 1.5 * ki.vel[:, 41] + 1.5 * np.sqrt(G / (ki.pos[:, 41] ** 2).sum()) * ki.pos[:, 41]     # outwards at 45 degrees
    k = _ctx(ki)
    for dt in (ki.dt, -50.0):
        q, v = _dev(ki.pos), _dev(ki.vel)
        k.fg(q, v, 1.0, dt)
        assert k.status() == 0
        qw, vw, bad = oracle_mod.step.fg(ki.pos, ki.vel, ki.G, dt)
        assert bad == 0 and np.abs(qw[:, 17] - ki.pos[:, 17]).max() > 0.1
        sq, sv = _scales(ki.pos, ki.vel, dt)
        assert np.all(np.abs(q.cpu().numpy() - qw) <= 32 * U * sq) and np.all(np.abs(v.cpu().numpy() - vw) <= 32 * U * sv)
    q, v = _dev(ki.pos), _dev(ki.vel)
    rc = torch.empty(1, ki.n, dtype=torch.float64, device="cuda")
    k.rcrit(_dev(ki.pos), _dev(ki.vel), _dev(ki.mass), 1.0, ki.dt, rc)
    want, bad = oracle_mod.step.rcrit(ki.pos, ki.vel, ki.mass, 1.0, ki.G, ki.dt)
    assert bad == 3 and np.all(np.abs(rc.cpu().numpy() - want) <= 16 * U * want)
    assert k.status() == g.STATUS_UNBOUND
    k.free()


def test_drift_equals_hc_fg_hc_bit_for_bit_and_is_reproducible():
    import torch
    for ki in (gi.make_config(1), gi.make_config(4, n=2048, n_test=300000)):
        k = _ctx(ki)
        mass = _dev(ki.mass)
        a_q, a_v = _dev(ki.pos), _dev(ki.vel)
        k.drift(a_q, a_v, mass, 1.0, ki.dt)
        b_q, b_v = _dev(ki.pos), _dev(ki.vel)
        k.hc(b_q, b_v, mass, 1.0, 0.5 * ki.dt); k.fg(b_q, b_v, 1.0, ki.dt); k.hc(b_q, b_v, mass, 1.0, 0.5 * ki.dt)
        c_q, c_v = _dev(ki.pos), _dev(ki.vel)
        k.drift(c_q, c_v, mass, 1.0, ki.dt)
        assert torch.equal(a_q, b_q) and torch.equal(a_v, b_v) and torch.equal(a_q, c_q) and torch.equal(a_v, c_v)
        k.free()


def _run_step(k, ki, q, v, mass, rrow, acc, pairs, npairs):
    import torch
    k.step(q, v, mass, 1.0, ki.dt, rrow, acc, pairs, npairs)
    torch.cuda.synchronize()
    total = int(npairs[ki.n].item())
    return {tuple(p) for p in pairs[:total].cpu().numpy().tolist()}, npairs[:ki.n].cpu().numpy()


@pytest.mark.parametrize("name,make", [("cfg0", lambda: gi.make_config(0)), ("cfg3_full", lambda: gi.make_config(3)),
                                       ("cfg4_tp", lambda: gi.make_config(4, n=2048, n_test=50000))],
                         ids=["cfg0", "cfg3_full", "cfg4_tp"])
def test_step_against_oracle(oracle_mod, name, make):
    import torch
    ki = make()
    n = ki.n
    k = _ctx(ki)
    q, v, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    rrow = torch.empty(n, dtype=torch.float64, device="cuda")
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    pairs = torch.empty(1 << 20, 2, dtype=torch.int32, device="cuda")
    npairs = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    got, counts = _run_step(k, ki, q, v, mass, rrow, acc, pairs, npairs)
    r = oracle_mod.step.step(ki.pos, ki.vel, ki.mass, ki.n_massive, ki.n_test, 1.0, ki.G, ki.dt)
    assert k.status() == 0 and r.unbound == 0
    assert np.all(np.abs(rrow.cpu().numpy() - r.rcrit[0]) <= 16 * U * r.rcrit[0])
    sq, sv = _scales(ki.pos, ki.vel, ki.dt)
    assert np.all(np.abs(q.cpu().numpy() - r.pos) <= 32 * U * sq)
    assert np.all(np.abs(v.cpu().numpy() - r.vel) <= 32 * U * sv)
    # candidates of the first kick: equal as a set outside the 1e-12 band (r_crit differs by <= 16 u)
    want = {tuple(p) for p in oracle_mod.pair_set(r.first, ki.n_massive).tolist()}
    border = {tuple(sorted(p)) for p in r.first.border.tolist()}
    assert (got ^ want) <= border and len(want) > 0
    if not (got ^ want):
        assert np.array_equal(counts, r.first.count)
    # the closing kick's acceleration under the kick's own rule (north_star: 1e-13 * sum|term|), like for like: the
    # oracle's kick of the positions and critical radii the DEVICE kicked (positions do not change in a kick, so
    # these are the step's final positions) -- no allowance for the <= 32 u by which the two states differ
    like = oracle_mod.kick(q.cpu().numpy(), ki.mass, rrow.cpu().numpy()[None, :], ki.n_massive, ki.n_test, level=0, G=ki.G,
                           enc_factor=ki.enc_factor, maxp=256)
    err = np.abs(acc.cpu().numpy() - like.acc)
    assert np.all(err <= 1e-13 * like.S)
    print(f"closing kick: max |da| / sum|term| = {np.max(err / np.maximum(like.S, 1e-300)):.2e} (bound 1e-13)")
    k.free()


def test_twenty_steps_track_the_oracle(oracle_mod):
    """The state after 20 device steps against 20 oracle steps (each side advancing its own state)."""
    import torch
    ki = gi.make_config(1, n=1500)
    n = ki.n
    k = _ctx(ki, capacity=1 << 16)
    q, v, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    pairs = torch.empty(1 << 16, 2, dtype=torch.int32, device="cuda")
    npairs = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    oq, ov = ki.pos.copy(), ki.vel.copy()
    worst = 0.0
    for _ in range(20):
        gq, gv = q.cpu().numpy(), v.cpu().numpy()                  # the device's state before this step
        k.step(q, v, mass, 1.0, ki.dt, None, acc, pairs, npairs)
        r = oracle_mod.step.step(oq, ov, ki.mass, n, 0, 1.0, ki.G, ki.dt)
        oq, ov = r.pos, r.vel
        # every single step like for like: the oracle's step from the device's own state, at the one-step bound (32 u)
        one = oracle_mod.step.step(gq, gv, ki.mass, n, 0, 1.0, ki.G, ki.dt)
        sq, sv = _scales(gq, gv, ki.dt)
        eq = np.max(np.abs(q.cpu().numpy() - one.pos) / sq) / U; ev = np.max(np.abs(v.cpu().numpy() - one.vel) / sv) / U
        assert eq <= 32 and ev <= 32
        worst = max(worst, eq, ev)
    torch.cuda.synchronize()
    sq, sv = _scales(oq, ov, ki.dt)
    # ... and the two free-running trajectories: 20 steps of <= 32 u each, amplified by the Kepler shear: a relative
    # error e in the semi-major axis turns into a phase error 1.5 n t e, n t <= 2 pi 120 d / (0.5^1.5 x 365.25 d) = 5.8
    # at the disk's inner edge (a = 0.5 AU): amplification <= 1.5 x 5.8 = 8.8
    dq = np.max(np.abs(q.cpu().numpy() - oq) / sq) / U; dv = np.max(np.abs(v.cpu().numpy() - ov) / sv) / U
    print(f"20 steps: worst single step {worst:.1f} u (bound 32 u); free-running difference {dq:.0f} u (pos), {dv:.0f} u (vel) "
          f"(bound 20 x 32 x 8.8 = 5632 u)")
    assert dq <= 20 * 32 * 8.8 and dv <= 20 * 32 * 8.8
    assert k.status() == 0
    k.free()


def test_step_error_codes():
    import torch
    import paper_2201_10058_b200 as g
    ki = gi.make_config(0, n=64)
    k = _ctx(ki, capacity=64)
    q, v, m = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    rc = torch.empty(64, dtype=torch.float64, device="cuda")
    for call, code in [(lambda: k.rcrit(q, v, m, 1.0, 6.0, None), g.E_NULL),
                       (lambda: k.rcrit(q, v, m, 1.0, 6.0, rc, nrows=0), g.E_SIZE),
                       (lambda: k.rcrit(q, v, m, 0.0, 6.0, rc), g.E_SIZE),
                       (lambda: k.hc(q, v, None, 1.0, 6.0), g.E_NULL),
                       (lambda: k.hc(q, v, m, -1.0, 6.0), g.E_SIZE),
                       (lambda: k.fg(q, None, 1.0, 6.0), g.E_NULL),
                       (lambda: k.fg(torch.zeros(3 * 64 + 1, dtype=torch.float64, device="cuda")[1:], v, 1.0, 6.0), g.E_ALIGN),
                       (lambda: k.drift(q, v, None, 1.0, 6.0), g.E_NULL),
                       (lambda: k.step(q, v, m, 1.0, 6.0, None, None, None, None), g.E_NULL)]:
        with pytest.raises(g.GengaKickError) as e:
            call()
        assert e.value.code == code
    k.free()


def test_rcritS_fgS_on_the_members_of_the_groups(oracle_mod):
    """RcritS / FGS (App. A): the device chain kick -> group -> rcrit_list / fg_list on `members`
    with no host round trip; listed bodies match the oracle's Rcrit / FG, the others are not touched."""
    import torch
    import paper_2201_10058_b200 as g
    ost = oracle_mod.step
    ki = gi.make_config(3, n=20000, level=1)
    n = ki.n
    k = _ctx(ki)
    pos, vel, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    pairs = torch.empty(1 << 20, 2, dtype=torch.int32, device="cuda")
    npairs = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    k.kick(pos, None, mass, _dev(ki.rcrit[:1]), 0, ki.dt, acc, pairs, npairs)
    i32 = lambda m: torch.empty(m, dtype=torch.int32, device="cuda")
    group_of, members, offsets, summary = i32(n), i32(n), i32(n + 1), i32(4)
    k.group(pairs, npairs[n:], 1 << 20, group_of, members, offsets, summary)
    rc = torch.full((2, n), -1.0, dtype=torch.float64, device="cuda")
    k.rcrit_list(pos, vel, mass, 1.0, 0.5 * ki.dt, members, summary[1:], n, rc, substeps=2.0, nrows=2)
    q, v = pos.clone(), vel.clone()
    k.fg_list(q, v, 1.0, 0.5 * ki.dt, members, summary[1:], n)
    torch.cuda.synchronize()
    assert k.status() == 0
    nm = int(summary[1])
    mem = members[:nm].cpu().numpy()
    assert 1000 < nm < n
    inlist = np.zeros(n, bool); inlist[mem] = True
    want_rc, _ = ost.rcrit(ki.pos, ki.vel, ki.mass, 1.0, ki.G, 0.5 * ki.dt, 2.0, 2)
    got_rc = rc.cpu().numpy()
    assert np.all(np.abs(got_rc[:, inlist] - want_rc[:, inlist]) <= 16 * U * want_rc[:, inlist])
    assert np.all(got_rc[:, ~inlist] == -1.0)
    qw, vw, _ = ost.fg(ki.pos, ki.vel, ki.G, 0.5 * ki.dt)
    sq, sv = _scales(ki.pos, ki.vel, 0.5 * ki.dt)
    gq, gv = q.cpu().numpy(), v.cpu().numpy()
    assert np.all(np.abs(gq[:, inlist] - qw[:, inlist]) <= 32 * U * sq[inlist])
    assert np.all(np.abs(gv[:, inlist] - vw[:, inlist]) <= 32 * U * sv[inlist])
    assert np.array_equal(gq[:, ~inlist], ki.pos[:, ~inlist]) and np.array_equal(gv[:, ~inlist], ki.vel[:, ~inlist])
    # the same bits as the all-bodies kernels on the listed bodies
    q2, v2 = pos.clone(), vel.clone()
    k.fg(q2, v2, 1.0, 0.5 * ki.dt)
    assert np.array_equal(q2.cpu().numpy()[:, inlist], gq[:, inlist])
    # a bad index is ignored and reported
    bad = torch.tensor([5, n + 3, -2, 7], dtype=torch.int32, device="cuda")
    cnt = torch.tensor([4, 0, 0, 0], dtype=torch.int32, device="cuda")
    k.fg_list(q, v, 1.0, 1.0, bad, cnt, 4)
    assert k.status() & 16
    k.free()


def test_step_can_be_captured_in_a_cuda_graph():
    """After one warm-up call (lazy scratch allocation) the library only enqueues kernels and async memsets on its
    stream: a caller may capture genga_step in a CUDA graph (launch-bound small-N loops) and gets the same bits."""
    import torch
    ki = gi.make_config(0, n=2048)
    n = ki.n
    k = _ctx(ki, capacity=1 << 16)
    q, v, mass = _dev(ki.pos), _dev(ki.vel), _dev(ki.mass)
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    pairs = torch.empty(1 << 16, 2, dtype=torch.int32, device="cuda")
    npairs = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    rrow = torch.empty(n, dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        k.set_stream(s.cuda_stream)
        k.step(q, v, mass, 1.0, ki.dt, rrow, acc, pairs, npairs)           # warm-up
        q.copy_(_dev(ki.pos)); v.copy_(_dev(ki.vel))
        for _ in range(5):
            k.step(q, v, mass, 1.0, ki.dt, rrow, acc, pairs, npairs)
        s.synchronize()
        qe, ve, ne = q.clone(), v.clone(), npairs.clone()
        q.copy_(_dev(ki.pos)); v.copy_(_dev(ki.vel))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            k.step(q, v, mass, 1.0, ki.dt, rrow, acc, pairs, npairs)
        q.copy_(_dev(ki.pos)); v.copy_(_dev(ki.vel))
        for _ in range(5):
            g.replay()
        s.synchronize()
    assert torch.equal(q, qe) and torch.equal(v, ve) and torch.equal(npairs, ne) and k.status() == 0
    k.free()
