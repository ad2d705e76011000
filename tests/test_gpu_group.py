"""-m gpu: genga_group (include/genga_group.h) through the C ABI against oracle/genga_group_oracle.c.
Integer work: every output must be BIT-EXACT (the partition into connected components is unique and is
returned in a canonical form), whatever the order of the pair list."""
import numpy as np
import pytest

import genga_inputs as gi

pytestmark = pytest.mark.gpu


def _gpu_group(n, pairs, n_pairs=None, rows=None, kick=None):
    import torch
    from paper_2201_10058_b200 import GengaKick
    own = kick is None
    if own:
        kick = GengaKick(n, 0, G=1.0, pair_capacity=8)
        kick.set_stream(torch.cuda.current_stream().cuda_stream)
    pr = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
    rows = pr.shape[0] if rows is None else rows
    d_pairs = torch.from_numpy(pr).cuda() if pr.size else torch.zeros(4, 2, dtype=torch.int32, device="cuda")
    d_n = torch.tensor([pr.shape[0] if n_pairs is None else n_pairs, 0, 0, 0], dtype=torch.int32, device="cuda")
    group_of = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    members = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    offsets = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    summary = torch.full((4,), -7, dtype=torch.int32, device="cuda")
    kick.group(d_pairs, d_n, rows, group_of, members, offsets, summary)
    torch.cuda.synchronize()
    s = summary.cpu().numpy()
    out = dict(group_of=group_of.cpu().numpy(), members=members.cpu().numpy()[:s[1]], offsets=offsets.cpu().numpy()[:s[0] + 1],
               n_groups=int(s[0]), n_members=int(s[1]), max_size=int(s[2]), used=int(s[3]), status=kick.status())
    if own:
        kick.free()
    return out


def _same(got, want):
    assert got["n_groups"] == want.n_groups and got["n_members"] == want.n_members and got["max_size"] == want.max_size
    assert np.array_equal(got["group_of"], want.group_of)
    assert np.array_equal(got["members"], want.members)
    assert np.array_equal(got["offsets"], want.offsets)
    assert got["status"] == 0


def _random_pairs(n, m, seed):
    u = gi.uniforms(seed, 0, 2 * m)
    a = np.minimum((u[:m] * n).astype(np.int64), n - 1); b = np.minimum((u[m:] * n).astype(np.int64), n - 1)
    keep = a != b
    return np.stack([a[keep], b[keep]], axis=1).astype(np.int32)


@pytest.mark.parametrize("n,m,seed", [(2, 1, 1), (50, 20, 1), (1000, 400, 2), (1000, 3000, 3), (4097, 2000, 6),
                                      (100000, 60000, 4), (1 << 20, 400000, 5), (300000, 900000, 7)])
def test_random_graphs(oracle_mod, n, m, seed):
    pairs = _random_pairs(n, m, seed)
    want = oracle_mod.group.group(n, pairs)
    _same(_gpu_group(n, pairs), want)
    # the order of the list and the orientation of a pair do not matter
    perm = np.argsort(gi.uniforms(seed + 100, 0, len(pairs)))
    _same(_gpu_group(n, pairs[perm][:, ::-1]), want)


def test_known_shapes(oracle_mod):
    grp = oracle_mod.group.group
    n = 5000
    for pairs in ([[2 * k, 2 * k + 1] for k in range(n // 2)],                   # disjoint pairs
                  [[k + 1, k] for k in range(n - 1)],                             # one long chain (deep trees)
                  [[n - 1 - k, n - 2 - k] for k in range(n - 1)],                 # the same chain, worst order
                  [[0, k] for k in range(1, n)],                                  # star on the smallest body
                  [[n - 1, k] for k in range(n - 1)],                             # star on the largest body
                  [[1, 2], [2, 1], [1, 2], [7, 9]],                               # duplicates
                  np.zeros((0, 2), dtype=np.int32)):                              # empty list
        _same(_gpu_group(n, pairs), grp(n, pairs))


def test_ring_is_one_group(oracle_mod):
    """Fig. 7: pair list from the KICK on the device, then grouped on the device."""
    import torch
    from paper_2201_10058_b200 import GengaKick
    for n in (16, 1024, 4096):
        ki = gi.make_ring(n)
        k = GengaKick(n, 0, pair_capacity=1 << 16, G=ki.G)
        k.set_stream(torch.cuda.current_stream().cuda_stream)
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
        pairs = torch.empty(1 << 16, 2, dtype=torch.int32, device="cuda")
        npairs = torch.empty(n + 1, dtype=torch.int32, device="cuda")
        k.kick(dev(ki.pos), None, dev(ki.mass), dev(ki.rcrit), 0, ki.dt, acc, pairs, npairs)
        group_of = torch.empty(n, dtype=torch.int32, device="cuda"); members = torch.empty(n, dtype=torch.int32, device="cuda")
        offsets = torch.empty(n + 1, dtype=torch.int32, device="cuda"); summary = torch.empty(4, dtype=torch.int32, device="cuda")
        k.group(pairs, npairs[n:], 1 << 16, group_of, members, offsets, summary)      # no host round trip in between
        torch.cuda.synchronize()
        assert summary.cpu().tolist() == [1, n, n, 4 * n]
        assert (group_of == 0).all() and torch.equal(members, torch.arange(n, dtype=torch.int32, device="cuda"))
        k.free()


@pytest.mark.parametrize("cfg,level", [(0, 0), (1, 0), (3, 0), (3, 1), (4, 0)])
def test_disk_pair_lists_full_size(oracle_mod, cfg, level):
    """The pair lists of BASELINE.json's configs at full size (from the oracle's kick), grouped on both sides."""
    ki = gi.make_config(cfg)
    res = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=level, G=ki.G, maxp=256)
    pairs = oracle_mod.pair_set(res, ki.n_massive)
    want = oracle_mod.group.group(ki.n, pairs)
    got = _gpu_group(ki.n, pairs)
    _same(got, want)
    if cfg == 3 and level == 0:
        assert want.max_size > 1000          # at high N the pairs link into very large groups


def test_clipped_count_bad_rows_and_errors(oracle_mod):
    import torch
    import paper_2201_10058_b200 as g
    n = 1000
    pairs = _random_pairs(n, 500, 9)
    # the true total exceeds the rows present (pair-list overflow of genga_kick): clipped to pair_rows
    got = _gpu_group(n, pairs[:200], n_pairs=len(pairs), rows=200)
    _same(got, oracle_mod.group.group(n, pairs[:200]))
    assert got["used"] == 200
    bad = pairs.copy(); bad[7] = (3, n + 5); bad[9] = (-1, 4)
    got = _gpu_group(n, bad)
    assert got["status"] & g.STATUS_BAD_PAIR
    keep = np.ones(len(bad), bool); keep[[7, 9]] = False
    want = oracle_mod.group.group(n, bad[keep])
    assert np.array_equal(got["group_of"], want.group_of) and np.array_equal(got["members"], want.members)
    k = g.GengaKick(64, 0, pair_capacity=8)
    t = torch.zeros(80, dtype=torch.int32, device="cuda")
    with pytest.raises(g.GengaKickError) as e:
        k.group(t, None, 4, t, t, t, t)
    assert e.value.code == g.E_NULL
    with pytest.raises(g.GengaKickError) as e:
        k.group(t, t, -1, t, t, t, t)
    assert e.value.code == g.E_SIZE
    with pytest.raises(g.GengaKickError) as e:
        k.group(t, t, 4, t[1:], t, t, t)
    assert e.value.code == g.E_ALIGN
    k.free()
