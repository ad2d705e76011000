"""Small runs of the synchronisation-heavy kernels for compute-sanitizer (one tool per gpurun call; the summaries are
kept in profiles/sanitizer_r02.md).  Not a pytest module: run as

    compute-sanitizer --tool racecheck python -m tests.sanitizer_cases <case> [...]

Cases: kick_sym   the symmetric level-0 pair loop (mbarrier ring, hand-over counters in shared memory), N = 24,576
       kick       the one-sided pair loop + the level-1 neighbour search + exact path, N = 6000 and 300 + 4000 particles
       bs_cluster Bulirsch-Stoer groups of 33 .. 256 bodies on thread-block clusters (distributed shared memory)
       bs_team    groups of 300 .. 700 bodies on teams of the cooperative grid (team barriers, neighbour lists)
       bs_grid    one group of 2500 bodies on the whole grid
       kick_tp_full  configs[4] at full size (2048 + 1,048,576 particles): the one-sided pair loop at its large-N shape (profiler runs)
       steps      three merged steps of the multi-level scheme (2 levels x 2 sub-steps), N = 3000
       multilevel_2x2  one multi-level step of configs[3] at full size, 2 levels x 2 sub-steps: one Bulirsch-Stoer group of
                  16,823 bodies on the whole grid, four lanes per body (profiler runs)
Each case checks its status word and prints one line."""
import sys

import numpy as np
import torch

import genga_inputs as gi
from paper_2201_10058_b200 import GengaKick

dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _kick(ki, level, tp_mode=1):
    n = ki.n
    k = GengaKick(ki.n_massive, ki.n_test, max_level=level, pair_capacity=1 << 18, G=ki.G, tp_mode=tp_mode)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    pairs = torch.empty(1 << 18, 2, dtype=torch.int32, device="cuda")
    npairs = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    args = (dev(ki.pos), dev(ki.vel), dev(ki.mass), dev(ki.rcrit[:level + 1]), level, 3.0, acc, pairs, npairs)
    for _ in range(2):                                          # (the second call is the warm one a profiler looks at)
        k.kick(*args)
    torch.cuda.synchronize()
    st, tot = k.status(), int(npairs[n])
    k.free()
    assert st == 0 and np.isfinite(acc.cpu().numpy()).all()
    return tot


def _bs_ring(sizes):
    m = sum(sizes)
    ki = gi.make_ring(m, partners=4)
    k = GengaKick(m, 0, G=ki.G, pair_capacity=8)
    k.set_stream(torch.cuda.current_stream().cuda_stream)
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    d_off = torch.zeros(m + 4, dtype=torch.int32, device="cuda"); d_off[:len(off)] = dev(off)
    d_sum = torch.tensor([len(sizes), m, max(sizes), 0], dtype=torch.int32, device="cuda")
    q, v = dev(ki.pos), dev(ki.vel)
    k.bs(dev(ki.pos), dev(ki.vel), dev(ki.mass), dev(ki.rcrit[:1]), 1, 1.0, 0.5, 1e-8,
         torch.arange(max(m, 4), dtype=torch.int32, device="cuda"), d_off, d_sum, q, v)
    torch.cuda.synchronize()
    st, tot = k.status(), k.bs_totals()
    k.free()
    assert st == 0 and tot[3] == len(sizes)
    return tot


def main(cases):
    for c in cases:
        if c == "kick_sym":
            out = _kick(gi.make_config(3, n=24576, level=0), 0)
        elif c == "kick":
            out = (_kick(gi.make_config(1, n=6000), 0), _kick(gi.make_config(3, n=6000, level=1), 1),
                   _kick(gi.make_config(4, n=300, n_test=4000), 0, tp_mode=2))
        elif c == "kick_tp_full":
            out = _kick(gi.make_config(4), 0)
        elif c == "bs_cluster":
            out = _bs_ring([40, 256, 100, 33])
        elif c == "bs_team":
            out = _bs_ring([300, 700, 512, 513])
        elif c == "bs_grid":
            out = _bs_ring([2500])
        elif c == "steps":
            ki = gi.make_config(1, n=3000)
            n = ki.n
            k = GengaKick(n, 0, max_level=1, pair_capacity=1 << 16, G=ki.G)
            k.set_stream(torch.cuda.current_stream().cuda_stream)
            q, v = dev(ki.pos), dev(ki.vel)
            stats = torch.zeros(2, 4, dtype=torch.int32, device="cuda")
            k.steps(q, v, dev(ki.mass), 1.0, ki.dt, 3, 2, 2, 1e-10, None, torch.empty(1 << 16, 2, dtype=torch.int32, device="cuda"),
                    torch.empty(n + 1, dtype=torch.int32, device="cuda"), stats)
            torch.cuda.synchronize()
            assert k.status() == 0
            out = stats.cpu().tolist()
            k.free()
        elif c == "multilevel_2x2":
            ki = gi.make_config(3)
            n = ki.n
            k = GengaKick(n, 0, max_level=1, pair_capacity=1 << 20, G=ki.G)
            k.set_stream(torch.cuda.current_stream().cuda_stream)
            q, v = dev(ki.pos), dev(ki.vel)
            stats = torch.zeros(2, 4, dtype=torch.int32, device="cuda")
            k.multilevel_step(q, v, dev(ki.mass), 1.0, ki.dt, 2, 2, 1e-12, torch.empty(3, n, dtype=torch.float64, device="cuda"),
                              torch.empty(1 << 20, 2, dtype=torch.int32, device="cuda"),
                              torch.empty(n + 1, dtype=torch.int32, device="cuda"), stats)
            torch.cuda.synchronize()
            assert k.status() == 0
            out = (stats.cpu().tolist(), k.bs_totals())
            k.free()
        else:
            raise SystemExit(f"unknown case {c}")
        print(f"sanitizer case {c}: ok {out}", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or ["kick_sym", "kick", "bs_cluster", "bs_team", "bs_grid", "steps"])
