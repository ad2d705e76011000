"""-m gpu: genga_kick_list (KickS, App. A) through the C ABI against oracle.kick_list, under
north_star's rule (|da| <= 1e-13 * sum|term|, pair sets equal outside the 1e-12 band), and against the all-pairs
kick of the same level."""
import numpy as np
import pytest

import genga_inputs as gi
from tests.gpu_harness import sorted_pairs

pytestmark = pytest.mark.gpu
TOL = 1e-13


def _dev(a, dt=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a))
    return (t if dt is None else t.to(dt)).cuda()


def _list_kick(ki, lst, level, tp_mode=1, with_vel=False, n_override=None, capacity=1 << 20):
    import torch
    from paper_2201_10058_b200 import GengaKick
    n = ki.n
    k = GengaKick(ki.n_massive, ki.n_test, max_level=level, pair_capacity=capacity, G=ki.G, enc_factor=ki.enc_factor,
                  tp_mode=tp_mode)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    pr = np.ascontiguousarray(np.asarray(lst, dtype=np.int32).reshape(-1, 2))
    d_in = _dev(pr) if pr.size else torch.zeros(4, 2, dtype=torch.int32, device="cuda")
    d_n = torch.tensor([len(pr) if n_override is None else n_override, 0, 0, 0], dtype=torch.int32, device="cuda")
    acc = torch.full((3, n), float("nan"), dtype=torch.float64, device="cuda")
    vel = _dev(ki.vel) if with_vel else None
    pairs = torch.full((capacity, 2), -7, dtype=torch.int32, device="cuda")
    npairs = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    k.kick_list(_dev(ki.pos), vel, _dev(ki.mass), _dev(ki.rcrit[:level + 1]), level, ki.dt, d_in, d_n, len(pr), acc,
                pairs, npairs)
    torch.cuda.synchronize()
    npn = npairs.cpu().numpy()
    out = dict(acc=acc.cpu().numpy(), counts=npn[:n], total=int(npn[n]), pairs=pairs.cpu().numpy()[:int(npn[n])],
               vel=None if vel is None else vel.cpu().numpy(), status=k.status(), launches=k.launch_count())
    k.free()
    return out


def _check(got, ks, lst):
    assert got["status"] == 0
    assert np.all(np.abs(got["acc"] - ks.acc) <= TOL * ks.S)
    want = {tuple(p) for p in np.asarray(lst)[ks.enc].tolist()}
    have = {tuple(p) for p in got["pairs"].tolist()}
    border = {tuple(p) for p in np.asarray(lst)[ks.border].tolist()}
    assert (have ^ want) <= border and len(have) == got["total"]
    if not (have ^ want):
        assert np.array_equal(got["counts"], ks.count)


@pytest.mark.parametrize("cfg,n,kw,levels", [(3, 9001, {}, (1, 2)), (2, 6000, {}, (1, 2)), (0, 2048, {}, (0, 1)),
                                             (4, 300, dict(n_test=5000), (0, 1))])
def test_list_kick_against_oracle_and_all_pairs_kick(oracle_mod, cfg, n, kw, levels):
    ki = gi.make_config(cfg, n=n, level=2, **kw)
    top = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=0, G=ki.G, maxp=128)
    lst = oracle_mod.pair_set(top, ki.n_massive)
    assert len(lst) > 10
    perm = np.argsort(gi.uniforms(5, 0, len(lst)))
    for L in levels:
        ks = oracle_mod.kick_list(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, lst, level=L, G=ki.G)
        got = _list_kick(ki, lst, L)
        _check(got, ks, lst)
        again = _list_kick(ki, lst[perm], L)                 # the order of the list does not change a bit
        assert np.array_equal(again["acc"], got["acc"]) and np.array_equal(again["counts"], got["counts"])
        assert np.array_equal(sorted_pairs(again["pairs"]), sorted_pairs(got["pairs"]))
        if L >= 1:                                           # W_L = 0 beyond rc0: equals the all-pairs level-L kick
            full = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=L, G=ki.G, maxp=128)
            assert np.all(np.abs(got["acc"] - full.acc) <= TOL * full.S)
            assert {tuple(p) for p in got["pairs"].tolist()} == {tuple(p) for p in oracle_mod.pair_set(full, ki.n_massive).tolist()}


def test_list_kick_full_size_config3(oracle_mod):
    """N = 65,536: the level-1 kick over the level-0 list (499,679 pairs) against the oracle, and the device chain
    genga_kick(level 0) -> genga_kick_list(level 1) with no host round trip against genga_kick(level 1)."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    ki = gi.make_config(3)
    n = ki.n
    k = GengaKick(n, 0, max_level=1, pair_capacity=1 << 20, G=ki.G)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    pos, mass, rc = _dev(ki.pos), _dev(ki.mass), _dev(ki.rcrit)
    acc0 = torch.empty(3, n, dtype=torch.float64, device="cuda")
    p0 = torch.empty(1 << 20, 2, dtype=torch.int32, device="cuda"); n0 = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    acc1 = torch.empty_like(acc0); p1 = torch.empty_like(p0); n1 = torch.empty_like(n0)
    acc2 = torch.empty_like(acc0); p2 = torch.empty_like(p0); n2 = torch.empty_like(n0)
    k.kick(pos, None, mass, rc, 0, ki.dt, acc0, p0, n0)
    k.kick_list(pos, None, mass, rc, 1, ki.dt, p0, n0[n:], 1 << 20, acc1, p1, n1)
    k.kick(pos, None, mass, rc, 1, ki.dt, acc2, p2, n2)
    torch.cuda.synchronize()
    assert k.status() == 0
    t1, t2 = int(n1[n]), int(n2[n])
    assert t1 == t2 and torch.equal(n1, n2)
    assert np.array_equal(sorted_pairs(p1[:t1].cpu().numpy()), sorted_pairs(p2[:t2].cpu().numpy()))
    full = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, n, 0, level=1, G=ki.G, maxp=256)
    assert np.all(np.abs(acc1.cpu().numpy() - full.acc) <= TOL * full.S)
    assert np.all(np.abs(acc2.cpu().numpy() - full.acc) <= TOL * full.S)
    k.free()


def test_list_kick_tp2_vel_update_and_edge_cases(oracle_mod):
    import paper_2201_10058_b200 as g
    ki = gi.make_config(4, n=200, n_test=3000)
    ki.mass = ki.mass.copy(); ki.mass[200:] = 1e-12
    top = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, 200, 3000, level=0, G=ki.G)
    lst = oracle_mod.pair_set(top, 200)
    for mode in (1, 2):
        ks = oracle_mod.kick_list(ki.pos, ki.mass, ki.rcrit, 200, 3000, lst, level=0, G=ki.G, tp_mode=mode)
        got = _list_kick(ki, lst, 0, tp_mode=mode, with_vel=True)
        _check(got, ks, lst)
        want_v = ki.vel + ki.dt * got["acc"]
        assert np.max(np.abs(got["vel"] - want_v) / (np.abs(ki.vel) + np.abs(ki.dt * got["acc"]) + 1e-300)) < 3e-16
    # empty list: zero acceleration, no pairs
    got = _list_kick(ki, np.zeros((0, 2), np.int32), 0)
    assert got["total"] == 0 and not got["acc"].any() and not got["counts"].any()
    # a count larger than the rows present is clipped; bad rows are ignored and reported
    got = _list_kick(ki, lst[:5], 0, n_override=1000)
    _check(got, oracle_mod.kick_list(ki.pos, ki.mass, ki.rcrit, 200, 3000, lst[:5], level=0, G=ki.G), lst[:5])
    bad = lst.copy(); bad[1] = (3, 3); bad[2] = (-4, 9)
    got = _list_kick(ki, bad, 0)
    assert got["status"] & g.STATUS_BAD_PAIR
    keep = np.ones(len(bad), bool); keep[[1, 2]] = False
    ks = oracle_mod.kick_list(ki.pos, ki.mass, ki.rcrit, 200, 3000, bad[keep], level=0, G=ki.G)
    assert np.all(np.abs(got["acc"] - ks.acc) <= TOL * ks.S)
