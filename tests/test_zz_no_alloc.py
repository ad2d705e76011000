"""genga_kick_list_static (include/genga_kick_static.h): the list kick with its scratch in a static device array of the
library -- no context, no allocation -- against genga_kick_list on a context (the existing path) on the same inputs.

Collected last on purpose (pytest -x: a failure here must not hide another test).  The static
array is shared by every call and keeps the last call's contents, so the checks run on several calls in a row, of
different sizes, in one process; each is also compared with the oracle under north_star's rule."""
import numpy as np
import pytest

import genga_inputs as gi
from tests.gpu_harness import sorted_pairs

TOL = 1e-13


def test_static_entry_point_is_declared_and_exported():
    import os
    import re
    import paper_2201_10058_b200 as g
    from paper_2201_10058_b200 import binding
    header = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include",
                               "genga_kick_static.h")).read()
    declared = set(re.findall(r"\bint\s+(genga_\w+)\s*\(", header))
    assert declared == set(binding.STATIC_EXPORTS)
    assert all(hasattr(g.lib(), name) for name in declared)
    assert int(re.search(r"#define GENGA_KICK_STATIC_MAX_BODIES (\d+)", header).group(1)) == binding.STATIC_MAX_BODIES
    assert "static scratch" in g.strerror(binding.E_STATIC_MAX)


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _inputs(ki, lst, level, capacity):
    import torch
    n = ki.n
    pr = np.ascontiguousarray(np.asarray(lst, dtype=np.int32).reshape(-1, 2))
    return dict(pos=_dev(ki.pos), mass=_dev(ki.mass), rcrit=_dev(ki.rcrit[:level + 1]), d_in=_dev(pr),
                d_n=torch.tensor([len(pr), 0, 0, 0], dtype=torch.int32, device="cuda"), rows=len(pr),
                acc=torch.full((3, n), float("nan"), dtype=torch.float64, device="cuda"), vel=_dev(ki.vel),
                pairs=torch.full((capacity, 2), -7, dtype=torch.int32, device="cuda"),
                npairs=torch.full((n + 1,), -7, dtype=torch.int32, device="cuda"))


def _result(t, n, status):
    import torch
    torch.cuda.synchronize()
    npn = t["npairs"].cpu().numpy()
    return dict(acc=t["acc"].cpu().numpy(), vel=t["vel"].cpu().numpy(), counts=npn[:n].copy(), total=int(npn[n]),
                pairs=t["pairs"].cpu().numpy()[:int(npn[n])].copy(), status=status)


def _context_path(ki, lst, level, tp_mode, capacity=1 << 18):
    import torch
    from paper_2201_10058_b200 import GengaKick
    t = _inputs(ki, lst, level, capacity)
    k = GengaKick(ki.n_massive, ki.n_test, max_level=level, pair_capacity=capacity, G=ki.G, enc_factor=ki.enc_factor,
                  tp_mode=tp_mode)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    k.kick_list(t["pos"], t["vel"], t["mass"], t["rcrit"], level, ki.dt, t["d_in"], t["d_n"], t["rows"], t["acc"],
                t["pairs"], t["npairs"])
    out = _result(t, ki.n, k.status())
    k.free()
    return out


def _static_path(ki, lst, level, tp_mode, capacity=1 << 18):
    import torch
    from paper_2201_10058_b200.binding import kick_list_static
    t = _inputs(ki, lst, level, capacity)
    status = torch.full((4,), -7, dtype=torch.int32, device="cuda")
    kick_list_static(t["pos"], t["vel"], t["mass"], t["rcrit"], ki.n_massive, ki.n_test, level, ki.dt, t["d_in"], t["d_n"],
                     t["rows"], t["acc"], t["pairs"], t["npairs"], status, G=ki.G, enc_factor=ki.enc_factor,
                     tp_mode=tp_mode, cuda_stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return _result(t, ki.n, int(status[0].item()))


def _same(a, b):
    assert a["status"] == b["status"] == 0
    assert np.array_equal(a["acc"], b["acc"]) and np.array_equal(a["vel"], b["vel"])
    assert np.array_equal(a["counts"], b["counts"]) and a["total"] == b["total"]
    assert np.array_equal(sorted_pairs(a["pairs"]), sorted_pairs(b["pairs"]))


@pytest.mark.gpu
def test_static_list_kick_equals_the_context_path_on_calls_in_a_row(oracle_mod):
    """Four calls in a row on the one static array -- a disk of 9001 bodies at levels 1 and 2, then a SMALLER system
    with semi-active particles (TP 2: what the larger call left behind it must not leak in), then the first again --
    each equal to genga_kick_list on a fresh context bit for bit (same kernels, fixed-point sums), hence within the
    1e-13 * sum|term| of north_star too, which is checked against the oracle."""
    big = gi.make_config(3, n=9001, level=2)
    top = oracle_mod.kick(big.pos, big.mass, big.rcrit, big.n_massive, big.n_test, level=0, G=big.G, maxp=128)
    lst_big = oracle_mod.pair_set(top, big.n_massive)
    small = gi.make_config(4, n=300, n_test=5000, level=1)
    small.mass = small.mass.copy()
    small.mass[small.n_massive:] = 1e-11 * (0.5 + gi.uniforms(11, 0, small.n_test))
    top = oracle_mod.kick(small.pos, small.mass, small.rcrit, small.n_massive, small.n_test, level=0, G=small.G, maxp=128,
                          tp_mode=2)
    lst_small = oracle_mod.pair_set(top, small.n_massive)
    assert len(lst_big) > 1000 and len(lst_small) > 10
    first = None
    for ki, lst, level, tp_mode in ((big, lst_big, 1, 1), (big, lst_big, 2, 1), (small, lst_small, 1, 2),
                                    (big, lst_big, 1, 1)):
        got = _static_path(ki, lst, level, tp_mode)
        _same(got, _context_path(ki, lst, level, tp_mode))
        ks = oracle_mod.kick_list(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, lst, level=level, G=ki.G,
                                  tp_mode=tp_mode)
        assert np.all(np.abs(got["acc"] - ks.acc) <= TOL * ks.S)
        assert np.all(np.abs(got["vel"] - (ki.vel + ki.dt * ks.acc)) <= TOL * ki.dt * ks.S + 4e-16 * (np.abs(ki.vel) + ki.dt * np.abs(ks.acc)))
        want = {tuple(p) for p in np.asarray(lst)[ks.enc].tolist()}
        border = {tuple(p) for p in np.asarray(lst)[ks.border].tolist()}
        assert ({tuple(p) for p in got["pairs"].tolist()} ^ want) <= border
        if first is None:
            first = got
    _same(got, first)                                        # the fourth call repeats the first


@pytest.mark.gpu
def test_static_list_kick_refuses_what_the_array_cannot_hold():
    """N beyond GENGA_KICK_STATIC_MAX_BODIES: a clear error before anything is launched; the status word and the
    outputs stay as they were.  N at the maximum (configs[3]'s size) runs."""
    import torch
    from paper_2201_10058_b200 import GengaKickError, binding
    n = binding.STATIC_MAX_BODIES + 1
    z = lambda *s: torch.zeros(*s, dtype=torch.float64, device="cuda")
    ints = lambda *s: torch.full(s, -7, dtype=torch.int32, device="cuda")
    acc, npairs, status = torch.full((3, n), 5.0, dtype=torch.float64, device="cuda"), ints(n + 1), ints(4)
    with pytest.raises(GengaKickError) as e:
        binding.kick_list_static(z(3, n), None, z(n), z(1, n), n, 0, 0, 1.0, ints(4, 2), ints(4), 0, acc, None, npairs, status)
    assert e.value.code == binding.E_STATIC_MAX and "GENGA_KICK_STATIC_MAX_BODIES" in str(e.value)
    torch.cuda.synchronize()
    assert int(status[0]) == -7 and float(acc.min()) == 5.0 and int(npairs[0]) == -7
    n = binding.STATIC_MAX_BODIES                            # an empty list at the largest size: a = 0, no pairs
    acc, npairs, status = torch.full((3, n), 5.0, dtype=torch.float64, device="cuda"), ints(n + 1), ints(4)
    zero = torch.zeros(4, dtype=torch.int32, device="cuda")
    binding.kick_list_static(z(3, n), None, z(n), z(1, n) + 1.0, n, 0, 0, 1.0, ints(4, 2), zero, 4, acc, None, npairs, status)
    torch.cuda.synchronize()
    assert int(status[0]) == 0 and float(acc.abs().max()) == 0.0 and int(npairs.abs().max()) == 0
    # ... and a list that reaches the last bodies, i.e. the last accumulators of the array: equal to the context path
    ki = gi.make_config(3)
    assert ki.n == n
    lst = np.array([(n - 1 - k, n - 2 - k) for k in range(40)] + [(0, n - 1), (n - 1, 31), (17, 32768)], dtype=np.int32)
    got = _static_path(ki, lst, 0, 1)
    _same(got, _context_path(ki, lst, 0, 1))
    assert np.all(got["acc"][:, n - 1] != 0.0) and np.count_nonzero(got["acc"][0]) == 45
