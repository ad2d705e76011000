"""Pins of oracle/genga_group_oracle.c (close-encounter groups = connected components of the pair graph,
PAPER.md:78, :563) against a library routine and cases with a known answer.  CPU only."""
import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

import genga_inputs as gi


@pytest.fixture(scope="module")
def grp(oracle_mod):
    return oracle_mod.group.group


def _check_canonical(n, pairs, g):
    """The canonical form itself: names are the smallest member, members sorted by (group, body), offsets consistent."""
    pairs = np.asarray(pairs).reshape(-1, 2)
    touched = np.zeros(n, bool); touched[pairs.ravel()] = True
    assert np.array_equal(g.group_of >= 0, touched)
    assert g.n_members == touched.sum() == len(g.members) and g.offsets[0] == 0 and g.offsets[-1] == g.n_members
    assert len(g.offsets) == g.n_groups + 1
    sizes = np.diff(g.offsets)
    assert (sizes >= 2).all() and (sizes.max() if len(sizes) else 0) == g.max_size
    names = []
    for a, b in zip(g.offsets[:-1], g.offsets[1:]):
        m = g.members[a:b]
        assert (np.diff(m) > 0).all() and (g.group_of[m] == m[0]).all()
        names.append(m[0])
    assert (np.diff(names) > 0).all()
    assert (g.group_of[pairs[:, 0]] == g.group_of[pairs[:, 1]]).all()          # an edge never crosses groups


@pytest.mark.parametrize("n,m,seed", [(50, 20, 1), (1000, 400, 2), (1000, 3000, 3), (20000, 15000, 4), (5000, 2500, 5)])
def test_against_scipy_connected_components(grp, n, m, seed):
    u = gi.uniforms(seed, 0, 2 * m)
    a = np.minimum((u[:m] * n).astype(np.int64), n - 1); b = np.minimum((u[m:] * n).astype(np.int64), n - 1)
    keep = a != b
    pairs = np.stack([a[keep], b[keep]], axis=1)
    g = grp(n, pairs)
    _check_canonical(n, pairs, g)
    ncomp, lab = connected_components(coo_matrix((np.ones(len(pairs)), (pairs[:, 0], pairs[:, 1])), shape=(n, n)), directed=False)
    # same partition: two touched bodies share a scipy label iff they share a group name
    t = np.nonzero(g.group_of >= 0)[0]
    first = {}
    for i in t:
        first.setdefault(lab[i], i)                  # scipy label -> its smallest touched body (ascending visit)
    assert all(g.group_of[i] == first[lab[i]] for i in t)
    assert g.n_groups == len(first)


def test_ring_is_one_group(grp, oracle_mod):
    """Fig. 7: every body in an encounter with 8 neighbours -> all N in a single group."""
    for n in (16, 64, 1000):
        ki = gi.make_ring(n)
        res = oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, n, 0, level=0, G=ki.G)
        pairs = oracle_mod.pair_set(res, n)
        assert len(pairs) == 4 * n
        g = grp(n, pairs)
        assert g.n_groups == 1 and g.max_size == n and (g.group_of == 0).all() and np.array_equal(g.members, np.arange(n))


def test_known_shapes(grp):
    n = 12
    g = grp(n, [[2 * k, 2 * k + 1] for k in range(6)])                    # disjoint pairs
    assert g.n_groups == 6 and g.max_size == 2 and np.array_equal(g.offsets, np.arange(0, 13, 2))
    g = grp(n, [[k + 1, k] for k in range(3, 9)])                          # a chain 3-4-...-9, pairs reversed
    assert g.n_groups == 1 and np.array_equal(g.members, np.arange(3, 10)) and (g.group_of[3:10] == 3).all()
    assert (g.group_of[:3] == -1).all() and (g.group_of[10:] == -1).all()
    g = grp(n, [[7, k] for k in (0, 11, 5)] + [[1, 2], [2, 1], [1, 2]])    # a star + a duplicated pair
    assert g.n_groups == 2 and np.array_equal(g.members, [0, 5, 7, 11, 1, 2]) and np.array_equal(g.offsets, [0, 4, 6])
    g = grp(n, np.zeros((0, 2), dtype=np.int32))                           # empty list
    assert g.n_groups == 0 and g.n_members == 0 and (g.group_of == -1).all() and np.array_equal(g.offsets, [0])


def test_disk_groups_are_plausible(grp, oracle_mod):
    """Config 0: ~2e2 pairs -> mostly groups of two; a dense disk at N = 20,000 links large groups."""
    ki = gi.make_config(0)
    pairs = oracle_mod.pair_set(oracle_mod.kick(ki.pos, ki.mass, ki.rcrit, ki.n, 0, level=0, G=ki.G), ki.n)
    g = grp(ki.n, pairs)
    _check_canonical(ki.n, pairs, g)
    assert g.n_groups > 50 and np.median(np.diff(g.offsets)) == 2
