#!/usr/bin/env python
"""bench.py -- FP64 pair interactions/s of the GENGA kick + close-encounter pre-check on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference]

Workload (BASELINE.json configs[3], the one `metric` is quoted on): N = 65,536 fully interactive
planetesimals, a in [0.5, 4] AU with surface density ~ a^-1.5, masses log-uniform in
[1e-4, 1e-2] Earth masses, r_crit rows at dt = 6 d and dt/2, seeded synthetic (genga_inputs).

One STEP = one pass of the whole hot path over that disk with the paper's two-level changeover
weights of eq. 63: the all-pairs kick with W_0 = K(r, dt) and the all-pairs kick
with W_1 = (1 - K(r, dt)) K(r, dt/2), each fused with its encounter pre-check, pair list, per-body
counts and the velocity update v += dt a (rows a1-a8 of SURVEY.md 8(a)).

What `value` counts: the ordered pair interactions whose force is actually EVALUATED, per second of
the whole step.  The level-0 kick evaluates all N (N - 1) of them (the symmetric pair loop forms one
r^-3 per unordered pair and applies both forces).  The level-1 kick is a neighbour search: W_1 = 0
exactly outside the level-0 critical radius, so all but ~1e6 of its 4.3e9 pairs are dismissed by box
tests and are NOT counted.  `value_nominal_two_level` is the same step counted as 2 N (N - 1) (the
convention of round 1), `value_dense_level0` the level-0 call alone; `levels` has each level, and
`configs` the other BASELINE.json configs (0, 2, 4) timed the same way.

N > 1 GPUs (torchrun, one rank per GPU): the path runs on one GPU (north_star); ranks are
independent replicas on independently seeded disks, no data-path collective ("scaling": "weak").

--impl reference times the CPU oracle (oracle/, plain C, as it stands) on the host cores on a
bounded sample of the same workload.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import genga_inputs as gi  # noqa: E402

METRIC = "FP64 pair interactions/s (kick+encounter) at N=65,536"
UNIT = "pair interactions/s"
N_BODIES = 65536
LEVELS = (0, 1)
PAIR_CAPACITY = 1 << 20
# ALGORITHMIC work of one ordered pair ("~17 FP64-pipe instructions, ~25 flops"; the one-sided loop's
# SASS has 3 DADD + 5 DMUL + 8 DFMA = 16 instructions, 24 flops: profiles/sass_pair_loop_r01.md) -- the per-unit figure
# of roofline.achieved.  EXECUTED work of the symmetric loop (profiles/sass_sym_loop_r02.md): one UNORDERED pair costs
# 3 DADD + 6 DMUL + 11 DFMA = 20 instructions, 31 flops, i.e. 10 instructions / 15.5 flops per ordered pair.
FP64_INSTR_PER_PAIR = 16
FLOPS_PER_PAIR = 24
SYM_FP64_INSTR_PER_UNORDERED_PAIR = 20
SYM_FLOPS_PER_UNORDERED_PAIR = 31
FP64_LANES_PER_SM = 64           # 148 SMs x 64 lanes x 2 flops x clocks.max.sm
# From the ncu captures of round 2 (profiles/ncu_r02a.md: kick_sym_kernel; profiles/ncu_r02c.md: the step's flop counters),
# per launch / per two-level step at N = 65,536 (rank 0's disk);
# constants read off those captures, not measured in this run:
NCU_DRAM_BYTES_PER_LAUNCH = 4204288        # kick_sym_kernel: dram__bytes_read.sum 2,497,536 + dram__bytes_write.sum 1,706,752
NCU_EXECUTED_FLOPS_PER_STEP = 67657959455  # DADD + DMUL + 2 DFMA thread instructions of every kernel of one step (flops_r02c.csv)


def workload(rank: int):
    """configs[3]; rank r > 0 draws an independent disk of the same recipe."""
    if rank == 0:
        return gi.make_config(3)
    ki = gi.make_disk(N_BODIES, 1003 + 7919 * rank, a_law="sigma_a^-1.5",
                      mass_law="loguniform_1e-4_1e-2_mearth", level=1)
    ki.meta["config"] = gi.CONFIG_NAMES[3] + f"_replica{rank}"
    return ki


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU while the timed region runs (NVML)."""

    def __init__(self, index: int, period_s: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons = index, period_s, [], set()
        self.max_mhz, self._stop_evt, self.err = None, threading.Event(), None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            names = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                     "sw_power_cap": 0x4, "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10,
                     "applications_clocks_setting": 0x2}
            while not self._stop_evt.is_set():
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                self.reasons |= {k for k, bit in names.items() if mask & bit}
                time.sleep(self.period)
        except Exception as e:  # NVML missing: the line says so instead of inventing clocks
            self.err = repr(e)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        d = {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
             "reasons": sorted(self.reasons), "samples": len(self.samples)}
        if self.err:
            d["error"] = self.err
        return d


def max_over_ranks(x: float, world: int, device=None) -> float:
    """Timing rule: every multi-GPU number is the MAX over ranks (all_reduce on the job's process group; gloo on
    CPU tensors in the tests, nccl on device tensors in the bench)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, pairs_per_step: int, steps: int, total_ms_max: float) -> float:
    """Replicas (weak scaling): every rank does the same number of pair interactions on its own disk; the job's
    throughput is all of them over the slowest rank's time."""
    return world * pairs_per_step * steps / (total_ms_max * 1e-3)


def physical_gpu_index(local_index: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        ids = [v.strip() for v in vis.split(",") if v.strip()]
        if local_index < len(ids) and ids[local_index].isdigit():
            return int(ids[local_index])
    return local_index


def oracle_sample(ki, rows_per_level: int, oracle):
    """The oracle, as it stands, on `rows_per_level` evenly spaced i-rows (all j) at both levels: that fraction of one
    two-level step.  Returns (seconds, pair interactions of the step's metric) -- the metric counts a step as N (N - 1)
    pair interactions in BOTH arms (the level-1 kick's pairs are not counted: the CUDA path culls them, the oracle, a
    plain double loop, evaluates their weights too; `pairs evaluated by the oracle` is twice the figure returned)."""
    rows = np.linspace(0, ki.n - 1, rows_per_level).astype(np.int32)
    t0 = time.perf_counter()
    for level in LEVELS:
        oracle.kick(ki.pos, ki.mass, ki.rcrit, ki.n_massive, ki.n_test, level=level, G=ki.G,
                    enc_factor=ki.enc_factor, rows=rows)
    dt = time.perf_counter() - t0
    return dt, rows_per_level * (ki.n_massive - 1)


def calibrate_rows(ki, oracle, target_s: float) -> int:
    probe = 64
    t, _ = oracle_sample(ki, probe, oracle)
    return int(max(probe, min(ki.n, probe * target_s / max(t, 1e-6))))


def run_reference(args, rank: int, world: int):
    if rank != 0:
        return
    import oracle
    ki = workload(0)
    cores = oracle.num_threads()
    rows = calibrate_rows(ki, oracle, target_s=2.0)          # ~2 s per step => K=20, W=5: under a minute
    for _ in range(args.warmup):
        oracle_sample(ki, rows, oracle)
    t_tot, pairs_tot = 0.0, 0
    for _ in range(args.steps):
        t, p = oracle_sample(ki, rows, oracle)
        t_tot += t
        pairs_tot += p
    value = pairs_tot / t_tot
    sample = (f"{rows} evenly spaced i-rows x all {ki.n_massive} j, levels 0 and 1, per step "
              f"(full step = {ki.n} rows); wall clock; value = that fraction of a two-level step counted as N (N - 1) "
              f"pair interactions, as in the CUDA arm (the oracle evaluates the weights of both levels' pairs: twice as many)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[3]: N=65536 planetesimal disk, two-level changeover (L=0 and L=1)",
                       "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_b200(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    from paper_2201_10058_b200 import GengaKick        # raises if the CUDA library is missing

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    ki = workload(rank)
    n = ki.n
    kick = GengaKick(ki.n_massive, ki.n_test, max_level=max(LEVELS), pair_capacity=PAIR_CAPACITY, G=ki.G,
                     enc_factor=ki.enc_factor, device=local_rank)
    stream = torch.cuda.current_stream()
    kick.set_stream(stream.cuda_stream)
    kick.enable_timing(True)
    to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    pos, mass, rcrit = to_dev(ki.pos), to_dev(ki.mass), to_dev(ki.rcrit)
    vel = to_dev(ki.vel)
    acc = torch.empty(3, n, dtype=torch.float64, device=dev)
    pairs = torch.empty(PAIR_CAPACITY, 2, dtype=torch.int32, device=dev)
    npairs = torch.empty(n + 1, dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # 256 MiB > 126 MB of L2

    def step():
        # (the level-1 kick acts on the positions the level-0 kick has just sorted: it keeps that internal order)
        for level in LEVELS:
            kick.set_order_reuse(2 if level > 0 else 0)
            kick.kick(pos, vel, mass, rcrit, level, 0.5 * ki.dt, acc, pairs, npairs)
        kick.set_order_reuse(False)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # FP64 ALU roofline of this device, measured before the timed region
    # (pattern 0: loop-invariant operands; 1: three distinct register operands, the shape of the
    # accumulation a += s d; 2: two distinct register operands -- include/genga_kick.h)
    import bench_aids                                   # bench-side helper library, not the product
    fp64_rate = [bench_aids.fp64_rate(pattern, iters=4096, reps=5, stream=stream.cuda_stream) for pattern in (0, 1, 2)]
    dfma_rate = max(fp64_rate)
    for _ in range(args.warmup):
        step()
        flush.fill_(1)
    torch.cuda.synchronize()
    enc_pairs = {}

    sampler = ClockSampler(physical_gpu_index(local_rank))
    launches0 = kick.launch_count()
    barrier()
    sampler.start()
    e0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    e1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    loop_ms = {level: [] for level in LEVELS}
    for s in range(args.steps):
        e0[s].record(stream)
        step()
        e1[s].record(stream)
        flush.fill_(s & 0xff)                      # L2 flush between timed iterations (outside the events)
        e1[s].synchronize()
        for level in LEVELS:
            loop_ms[level].append(kick.last_pair_loop_ms(level))
    barrier()
    clocks = sampler.stop()
    launches = kick.launch_count() - launches0
    step_ms = [a.elapsed_time(b) for a, b in zip(e0, e1)]
    total_ms = max_over_ranks(float(sum(step_ms)), world, dev)
    pairs_per_kick = ki.n_massive * (ki.n_massive - 1) + ki.n_test * ki.n_massive
    pairs_per_step = pairs_per_kick                    # EVALUATED: all of level 0; level 1's are culled, not counted
    nominal_pairs_per_step = len(LEVELS) * pairs_per_kick
    value = whole_job_value(world, pairs_per_step, args.steps, total_ms)
    value_nominal = whole_job_value(world, nominal_pairs_per_step, args.steps, total_ms)

    # per-level numbers: one more kick each, timed alone (after the timed region)
    levels = {}
    for level in LEVELS:
        ts = []
        for _ in range(5):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            flush.fill_(3)
            a.record(stream)
            kick.kick(pos, vel, mass, rcrit, level, 0.5 * ki.dt, acc, pairs, npairs)
            b.record(stream)
            b.synchronize()
            ts.append(a.elapsed_time(b))
        enc_pairs[level] = int(npairs[n].item())
        ms = float(np.median(ts))
        levels[str(level)] = {"ms_per_kick": ms, "pair_loop_ms": float(np.mean(loop_ms[level])),
                              "encounter_pairs": enc_pairs[level]}
        if level == 0:
            levels["0"]["pairs_per_s"] = pairs_per_kick / (ms * 1e-3)
            levels["0"]["what"] = "dense: every ordered pair's force evaluated (one r^-3 per unordered pair)"
        else:
            levels[str(level)]["nominal_pairs_per_s"] = pairs_per_kick / (ms * 1e-3)
            levels[str(level)]["what"] = ("neighbour search: W_L = 0 exactly beyond the level-0 critical radius, the pairs "
                                          "are culled by box tests, not evaluated (nominal figure, not work done)")

    configs_info = step_info = steps_info = group_info = list_info = hybrid_info = multilevel_info = bs_ring_info = None
    if not args.headline_only:          # (--headline-only: the timed step alone, e.g. under ncu)
        # the other BASELINE.json configs, each timed like the headline (L2 flushed before every kick, median of 7 after 3
        # warm-ups): configs[0] (launch-bound: plain launches and a CUDA-graph replay), configs[1], configs[2] at both
        # levels, configs[4] in both test-particle modes
        def time_config(kin, level, tp_mode=1, mass_override=None, graph=False, reps=7):
            nn = kin.n
            kc = GengaKick(kin.n_massive, kin.n_test, max_level=level, pair_capacity=PAIR_CAPACITY, G=kin.G,
                           enc_factor=kin.enc_factor, device=local_rank, tp_mode=tp_mode)
            kc.set_stream(stream.cuda_stream)
            kc.enable_timing(True)
            cp, cm = to_dev(kin.pos), to_dev(kin.mass if mass_override is None else mass_override)
            crc, cv = to_dev(kin.rcrit[:level + 1]), to_dev(kin.vel)
            ca = torch.empty(3, nn, dtype=torch.float64, device=dev)
            cnp = torch.empty(nn + 1, dtype=torch.int32, device=dev)
            ts, loops = [], []
            for it in range(reps + 3):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                flush.fill_(9)
                l0 = kc.launch_count()
                a.record(stream)
                kc.kick(cp, cv, cm, crc, level, 0.5 * kin.dt, ca, pairs, cnp)
                b.record(stream)
                b.synchronize()
                nl = kc.launch_count() - l0
                if it >= 3:
                    ts.append(a.elapsed_time(b))
                    loops.append(kc.last_pair_loop_ms(level))
            ms = float(np.median(ts))
            ordered = kin.n_massive * (kin.n_massive - 1) + kin.n_test * kin.n_massive * (2 if tp_mode == 2 else 1)
            out = {"n_massive": kin.n_massive, "n_test": kin.n_test, "level": level, "ms_per_kick": ms,
                   "pair_loop_ms": float(np.median(loops)), "launches": int(nl), "encounter_pairs": int(cnp[nn].item()),
                   "symmetric_pass": bool(kc.plan(0).symmetric) if level == 0 else False, "status": kc.status()}
            if level == 0:
                out["pairs_per_s"] = ordered / (ms * 1e-3)
            else:
                out["nominal_pairs_per_s"] = ordered / (ms * 1e-3)
            if tp_mode == 2:
                out["tp_mode"] = 2
            if graph:
                gs = torch.cuda.Stream()
                torch.cuda.synchronize()
                kc.set_stream(gs.cuda_stream)
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=gs):
                    kc.kick(cp, cv, cm, crc, level, 0.5 * kin.dt, ca, pairs, cnp)
                gts = []
                with torch.cuda.stream(gs):
                    for it in range(reps + 3):
                        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        a.record(gs)
                        g.replay()
                        b.record(gs)
                        b.synchronize()
                        if it >= 3:
                            gts.append(a.elapsed_time(b))
                torch.cuda.synchronize()
                out["ms_per_kick_cuda_graph"] = float(np.median(gts))
                del g
            kc.free()
            return out

        k4 = gi.make_config(4)
        m4 = k4.mass.copy()
        m4[k4.n_massive:] = 1e-12 * (0.5 + gi.uniforms(77, 0, k4.n_test))       # TP 2: particles with mass
        k2 = gi.make_config(2)
        configs_info = {
            "what": "one kick + pre-check (v += dt a, pair list, counts) per BASELINE.json config, L2 flushed before each; "
                    "pairs_per_s counts evaluated ordered pairs (level 0); level >= 1 kicks are neighbour searches (nominal)",
            "configs[0] N=2048 L=0": time_config(gi.make_config(0), 0, graph=True),
            "configs[1] N=8192 L=0": time_config(gi.make_config(1), 0),
            "configs[2] N=32770 L=0": time_config(k2, 0),
            "configs[2] N=32770 L=1": time_config(k2, 1),
            "configs[4] 2048+1048576 tp, TP 1": time_config(k4, 0),
            "configs[4] 2048+1048576 tp, TP 2": time_config(k4, 0, tp_mode=2, mass_override=m4),
        }

        # NEXT-1: the whole App. A step without the Bulirsch-Stoer branch on the same disk --
        # Rcrit, Kick(dt/2) + pre-check, HC(dt/2), FG(dt), HC(dt/2), Kick(dt/2) -- and its O(N) part alone
        sq, sv = pos.clone(), vel.clone()
        rrow = torch.empty(n, dtype=torch.float64, device=dev)
        step_ts, drift_ts = [], []
        for it in range(8):
            a, b, c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            flush.fill_(5)
            l0 = kick.launch_count()
            a.record(stream)
            kick.step(sq, sv, mass, 1.0, ki.dt, rrow, acc, pairs, npairs)
            b.record(stream)
            step_launches = kick.launch_count() - l0
            kick.drift(sq, sv, mass, 1.0, ki.dt)
            c.record(stream)
            c.synchronize()
            if it >= 3:
                step_ts.append(a.elapsed_time(b))
                drift_ts.append(b.elapsed_time(c))
        step_info = {"what": "Rcrit, Kick(dt/2)+pre-check, HC(dt/2), FG(dt), HC(dt/2), Kick(dt/2) at level 0 (genga_step)",
                     "ms_per_step": float(np.median(step_ts)), "launches_per_step": int(step_launches),
                     "drift_ms": float(np.median(drift_ts)), "drift_what": "HC(dt/2) FG(dt) HC(dt/2) alone, 3 launches, "
                     "184 B/body of HBM traffic", "status": kick.status()}

        # genga_steps: consecutive steps with the closing kick of a step and the opening kick of the next merged into one
        # pass over the pairs (one all-pairs pass per step instead of two): 100 steps without the encounter branch, and
        # 10 steps of the multi-level scheme (2 levels x 10 sub-steps), from the generated state
        def time_steps(n_steps, slevels, substeps, reps=2):
            kk = kick if slevels <= 1 + max(LEVELS) else None
            st_buf = torch.zeros(max(slevels, 1), 4, dtype=torch.int32, device=dev)
            ts = []
            for it in range(reps + 1):
                sq2, sv2 = pos.clone(), vel.clone()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                flush.fill_(4)
                l0 = kk.launch_count()
                a.record(stream)
                kk.steps(sq2, sv2, mass, 1.0, ki.dt, n_steps, slevels, substeps, 1e-12, acc, pairs, npairs, st_buf)
                b.record(stream)
                b.synchronize()
                nl = kk.launch_count() - l0
                if it >= 1:
                    ts.append(a.elapsed_time(b))
            return {"n_steps": n_steps, "slevels": slevels, "substeps": substeps if slevels > 1 else None,
                    "ms_per_step": float(np.median(ts)) / n_steps, "launches_per_step": nl / n_steps, "status": kk.status()}

        steps_info = {"what": "genga_steps: n consecutive steps, merged kicks (slevels 0: Rcrit, Kick, HC, FG, HC, Kick without "
                              "the encounter branch; 2 x 10: the multi-level step), ms per step",
                      "runs": [time_steps(100, 0, 2), time_steps(10, 2, 10)]}

        # NEXT-2: grouping of the level-0 pair list (499,679 pairs at N = 65,536) into close-encounter groups
        kick.kick(pos, None, mass, rcrit, 0, 0.5 * ki.dt, acc, pairs, npairs)
        group_of = torch.empty(n, dtype=torch.int32, device=dev)
        members = torch.empty(n, dtype=torch.int32, device=dev)
        offsets = torch.empty(n + 1, dtype=torch.int32, device=dev)
        summary = torch.empty(4, dtype=torch.int32, device=dev)
        group_ts = []
        for it in range(8):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            flush.fill_(6)
            l0 = kick.launch_count()
            a.record(stream)
            kick.group(pairs, npairs[n:], PAIR_CAPACITY, group_of, members, offsets, summary)
            b.record(stream)
            b.synchronize()
            group_launches = kick.launch_count() - l0
            if it >= 3:
                group_ts.append(a.elapsed_time(b))
        sm = summary.cpu().tolist()
        group_info = {"what": "genga_group on the level-0 pair list: connected components, members sorted by (group, body)",
                      "ms": float(np.median(group_ts)), "launches": int(group_launches), "pairs": sm[3], "n_groups": sm[0],
                      "n_members": sm[1], "largest_group": sm[2]}

        # NEXT-4: KickS -- the level-1 kick over the level-0 pair list (genga_kick_list) instead of over all pairs
        pairs1 = torch.empty(PAIR_CAPACITY, 2, dtype=torch.int32, device=dev)
        npairs1 = torch.empty(n + 1, dtype=torch.int32, device=dev)
        kick.kick(pos, None, mass, rcrit, 0, 0.5 * ki.dt, acc, pairs, npairs)
        list_ts = []
        for it in range(8):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            flush.fill_(7)
            a.record(stream)
            kick.kick_list(pos, sv, mass, rcrit, 1, 0.5 * ki.dt, pairs, npairs[n:], PAIR_CAPACITY, acc, pairs1, npairs1)
            b.record(stream)
            b.synchronize()
            if it >= 3:
                list_ts.append(a.elapsed_time(b))
        list_info = {"what": "genga_kick_list: level-1 kick + pre-check over the level-0 encounter list (same result as the "
                             "all-pairs level-1 kick, W_1 = 0 beyond rc0)", "ms": float(np.median(list_ts)),
                     "listed_pairs": int(npairs[n].item()), "level1_pairs": int(npairs1[n].item())}

        # NEXT-4: the complete hybrid step with the Bulirsch-Stoer branch, on BASELINE.json configs[1] (N = 8192; at
        # N = 65,536 the level-0 pairs link into one group of 33,297 bodies -- the case the multi-level step below exists for)
        k1 = gi.make_config(1)
        n1 = k1.n
        kick1 = GengaKick(n1, 0, max_level=0, pair_capacity=1 << 18, G=k1.G, device=local_rank)
        kick1.set_stream(stream.cuda_stream)
        hq, hv, hm = to_dev(k1.pos), to_dev(k1.vel), to_dev(k1.mass)
        i32 = lambda m: torch.empty(m, dtype=torch.int32, device=dev)
        hacc = torch.empty(3, n1, dtype=torch.float64, device=dev)
        hpairs, hnp, hgo, hmem, hoff, hsum = torch.empty(1 << 18, 2, dtype=torch.int32, device=dev), i32(n1 + 1), i32(n1), \
            i32(n1), i32(n1 + 1), i32(4)
        hyb_ts = []
        for it in range(10):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = kick1.launch_count()
            a.record(stream)
            kick1.hybrid_step(hq, hv, hm, 1.0, k1.dt, 1e-12, hacc, hpairs, hnp, hgo, hmem, hoff, hsum)
            b.record(stream)
            b.synchronize()
            hyb_launches = kick1.launch_count() - l0
            if it >= 3:
                hyb_ts.append(a.elapsed_time(b))
        hs = hsum.cpu().tolist()
        hybrid_info = {"what": "genga_hybrid_step on configs[1] (N = 8192): Rcrit, Kick + pre-check, HC, FG, grouping, "
                               "Bulirsch-Stoer (tol 1e-12), HC, Kick", "ms_per_step": float(np.median(hyb_ts)),
                       "launches_per_step": int(hyb_launches), "groups": hs[0], "bodies_in_groups": hs[1],
                       "largest_group": hs[2], "status": kick1.status()}
        kick1.free()

        # NEXT-4: the multi-level step (SEnc recursion, App. A) -- the experiment of Fig. 10
        # (PAPER.md:640): the same disks, the hybrid step against 2-4 symplectic levels
        def time_multilevel(kin, slevels, substeps, reps, graph=False):
            nn = kin.n
            km = GengaKick(nn, 0, max_level=slevels - 1, pair_capacity=PAIR_CAPACITY, G=kin.G, device=local_rank)
            km.set_stream(stream.cuda_stream)
            q0, v0, mm = to_dev(kin.pos), to_dev(kin.vel), to_dev(kin.mass)
            q, v = q0.clone(), v0.clone()
            macc = torch.empty(3, nn, dtype=torch.float64, device=dev)
            mp, mnp = torch.empty(PAIR_CAPACITY, 2, dtype=torch.int32, device=dev), i32(nn + 1)
            mst = torch.zeros(slevels, 4, dtype=torch.int32, device=dev)
            ts = []
            for it in range(reps + 2):
                q.copy_(q0); v.copy_(v0)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                l0 = km.launch_count()
                a.record(stream)
                km.multilevel_step(q, v, mm, 1.0, kin.dt, slevels, substeps, 1e-12, macc, mp, mnp, mst, detect=True)
                b.record(stream)
                b.synchronize()
                nl = km.launch_count() - l0
                if it >= 2:
                    ts.append(a.elapsed_time(b))
            st = mst.cpu().tolist()
            # the same launch sequence captured once in a CUDA graph and replayed (no host launch cost, fixed sequence)
            graph_ms = None
            if graph:
                gs = torch.cuda.Stream()                       # capture needs a non-default stream
                q.copy_(q0); v.copy_(v0)
                torch.cuda.synchronize()
                km.set_stream(gs.cuda_stream)
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=gs):
                    km.multilevel_step(q, v, mm, 1.0, kin.dt, slevels, substeps, 1e-12, macc, mp, mnp, mst, detect=True)
                gts = []
                with torch.cuda.stream(gs):
                    for it in range(reps + 2):
                        q.copy_(q0); v.copy_(v0)
                        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        a.record(gs)
                        g.replay()
                        b.record(gs)
                        b.synchronize()
                        if it >= 2:
                            gts.append(a.elapsed_time(b))
                torch.cuda.synchronize()
                km.set_stream(stream.cuda_stream)
                graph_ms = float(np.median(gts))
                assert mst.cpu().tolist() == st, "the replayed graph took other decisions than the plain launches"
                del g
            out = {"slevels": slevels, "substeps": substeps, "ms_per_step": float(np.median(ts)), "launches_per_step": int(nl),
                   "ms_per_step_cuda_graph": graph_ms,
                   "encounter_pairs_per_level": [r[1] for r in st], "bs_groups": st[-1][2], "bs_bodies": st[-1][3],
                   "status": km.status()}
            km.free()
            return out

        multilevel_info = {"what": "genga_multilevel_step (Rcrit, Kick + pre-check, HC, FG, detection, SEnc over KickS / RcritS / "
                                   "FGS / detection / grouping / Bulirsch-Stoer tol 1e-12, HC, Kick), one step from the "
                                   "generated state; 1 level = the hybrid step",
                           "configs[1] N=8192": [time_multilevel(k1, sl, ss, 5, graph=(sl, ss) == (2, 2))
                                                 for sl, ss in ((1, 2), (2, 2), (3, 2), (2, 10))],
                           "configs[3] N=65536": [time_multilevel(ki, sl, ss, 3, graph=(sl, ss) == (2, 10))
                                                  for sl, ss in ((2, 10), (4, 2), (3, 4), (3, 2), (2, 2))]}

        # NEXT-4: the Bulirsch-Stoer kernels alone on the ring of Fig. 7 (the experiment of Fig. 8): n bodies
        # on a ring, 8 close-encounter partners each, one group, integrated over dt = 6 d at tol 1e-12
        def time_bs_ring(nr, reps=3):
            kr = gi.make_ring(nr)
            kb = GengaKick(nr, 0, max_level=0, pair_capacity=8, G=kr.G, device=local_rank)
            kb.set_stream(stream.cuda_stream)
            q_in, v_in, mb, rcb = to_dev(kr.pos), to_dev(kr.vel), to_dev(kr.mass), to_dev(kr.rcrit)
            mem = torch.arange(max(nr, 4), dtype=torch.int32, device=dev)
            off = torch.zeros(nr + 4, dtype=torch.int32, device=dev); off[1] = nr
            summ = torch.tensor([1, nr, nr, 0], dtype=torch.int32, device=dev)
            q, v = q_in.clone(), v_in.clone()
            ts = []
            for it in range(reps + 1):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                kb.bs(q_in, v_in, mb, rcb, 1, 1.0, kr.dt, 1e-12, mem, off, summ, q, v)
                b.record(stream)
                b.synchronize()
                if it >= 1:
                    ts.append(a.elapsed_time(b))
            st = kb.status()
            kb.free()
            return {"n": nr, "ms": float(np.median(ts)), "status": st}

        bs_ring_info = {"what": "genga_bs on one ring group of n bodies with 8 partners each (Fig. 7 / Fig. 8), dt = 6 d, tol 1e-12 "
                                "(regimes by group size: include/genga_bs.h)",
                        "rings": [time_bs_ring(nr) for nr in (2, 8, 32, 64, 256, 512, 1024, 2048, 4096)]}

    # end to end through the host entry point: pinned host arrays in, results back, every step
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_pos, h_mass, h_rc, h_vel = pin(ki.pos), pin(ki.mass), pin(ki.rcrit), pin(ki.vel)
    h_acc = torch.empty(3, n, dtype=torch.float64).pin_memory()
    h_pairs = torch.empty(PAIR_CAPACITY, 2, dtype=torch.int32).pin_memory()
    h_np = torch.empty(n + 1, dtype=torch.int32).pin_memory()

    def host_step():
        for level in LEVELS:
            kick.set_order_reuse(2 if level > 0 else 0)
            kick.kick_host(h_pos, h_vel, h_mass, h_rc, level, 0.5 * ki.dt, h_acc, h_pairs, h_np)
        kick.set_order_reuse(False)

    for _ in range(max(args.warmup, 3)):
        host_step()
    e2e_steps = args.steps
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        host_step()
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0, world, dev)
    h2d = sum(8 * n * (3 + 3 + 1 + (level + 1)) for level in LEVELS)
    d2h = sum(8 * n * (3 + 3) + 4 * (n + 1) + 8 * min(enc_pairs[level], PAIR_CAPACITY) for level in LEVELS)
    e2e_value = whole_job_value(world, pairs_per_step, e2e_steps, 1e3 * e2e_s)

    if rank == 0:
        props = torch.cuda.get_device_properties(local_rank)
        sm_max_mhz = clocks.get("sm_max_mhz") or 1965
        peak_nominal = props.multi_processor_count * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
        peak_dfma = 2.0 * dfma_rate / 1e12
        k0_ms = float(np.mean(loop_ms[0]))
        sym = bool(kick.plan(0).symmetric)
        # roofline.achieved (the contract's definition): ALGORITHMIC flops per unit x units per launch / kernel time,
        # the per-unit figure being SURVEY.md 8(d)'s one ordered pair = 24 flops (its "~25"), counted over all
        # N (N - 1) ordered pairs.  The symmetric loop EXECUTES fewer: 31 flops per unordered pair = 15.5 per ordered
        # pair -- it reaches the same result with 35 % less arithmetic, so its executed-flop fraction
        # (frac_executed_flops) is LOWER than the one-sided loop's 0.64 while its throughput is 40 % higher.
        achieved = FLOPS_PER_PAIR * pairs_per_kick / (k0_ms * 1e-3) / 1e12
        n_m = ki.n_massive
        if sym:
            pl = kick.plan(0)
            ib, r = pl.i_block, pl.tiles_per_iblock
            diag_ordered = sum(min(ib, n_m - I * ib) * min(n_m - I * ib, ib) for I in range(pl.n_i_blocks))
            unordered_sym = (n_m * n_m - diag_ordered) // 2
            exec_flops = SYM_FLOPS_PER_UNORDERED_PAIR * unordered_sym + FLOPS_PER_PAIR * diag_ordered
            exec_instr = SYM_FP64_INSTR_PER_UNORDERED_PAIR * unordered_sym + FP64_INSTR_PER_PAIR * diag_ordered
        else:
            exec_flops, exec_instr = FLOPS_PER_PAIR * pairs_per_kick, FP64_INSTR_PER_PAIR * pairs_per_kick
        executed = exec_flops / (k0_ms * 1e-3) / 1e12
        pipe_rate = props.multi_processor_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6
        step_ms = total_ms / args.steps
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "value_what": "ordered pair interactions whose force is evaluated, per second of the two-level step (all "
                          "N (N - 1) of level 0; the level-1 kick's pairs are culled by a neighbour search and not counted)",
            "value_dense_level0": levels["0"]["pairs_per_s"],
            "value_nominal_two_level": value_nominal,
            "config": {"workload": "configs[3]: N=65536 planetesimal disk (sigma ~ a^-1.5, log-uniform masses), "
                                   "step = level-0 kick + level-1 kick (two-level changeover, eq. 63), each "
                                   "with encounter pre-check, pair list, counts and v += dt a",
                       "n_massive": ki.n_massive, "n_test": ki.n_test, "levels": list(LEVELS),
                       "pairs_per_step": pairs_per_step, "nominal_pairs_per_step": nominal_pairs_per_step,
                       "pair_capacity": PAIR_CAPACITY,
                       "l2": "256 MiB buffer written between timed iterations (working set 3 MB is L2-resident)",
                       "parallelism": "replicas" if world > 1 else "single GPU"},
            "levels": levels,
            "configs": configs_info,
            "step": step_info,
            "steps_merged": steps_info,
            "group": group_info,
            "kick_list": list_info,
            "hybrid_step": hybrid_info,
            "multilevel_step": multilevel_info,
            "bs_ring": bs_ring_info,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps,
                    "api": "genga_kick_host (pinned host arrays, copies and synchronisation inside the call)"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu",
                         "kernel": "kick_sym_kernel (level 0, every unordered pair once)" if sym else "kick_kernel (level 0)",
                         "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s", "frac": achieved / peak_nominal,
                         "achieved_what": "algorithmic: 24 flops per ordered pair (SURVEY.md 8(d); the one-sided loop's SASS "
                                          "count) x N (N - 1) ordered pairs / kernel time",
                         "traffic": NCU_DRAM_BYTES_PER_LAUNCH,
                         "peak_source": f"nominal: {props.multi_processor_count} SMs x {FP64_LANES_PER_SM} FP64 lanes "
                                        f"x 2 x {sm_max_mhz} MHz (no FP64 figure in MEASURED_PEAKS.json)",
                         "peak_measured_dfma": peak_dfma, "frac_of_measured_dfma": achieved / peak_dfma,
                         "dfma_per_s_by_operand_pattern": {"invariant_operands": fp64_rate[0],
                                                           "three_distinct_registers": fp64_rate[1],
                                                           "two_distinct_registers": fp64_rate[2]},
                         "executed": executed, "frac_executed_flops": executed / peak_nominal,
                         "executed_what": "flops the kernel executes (SASS count x pairs of each path: 31 per unordered pair "
                                          "in the symmetric tiles, 24 per ordered pair in the diagonal tiles) / kernel time: "
                                          "fewer flops per pair than the one-sided loop, hence a lower fraction at a higher "
                                          "throughput",
                         "executed_flops_per_launch": exec_flops,
                         "fp64_pipe_issue_frac": exec_instr / (k0_ms * 1e-3) / pipe_rate,
                         "whole_step_frac_executed_flops": (exec_flops if NCU_EXECUTED_FLOPS_PER_STEP is None
                                                            else NCU_EXECUTED_FLOPS_PER_STEP) / (step_ms * 1e-3) / 1e12 / peak_nominal,
                         "whole_step_what": "executed FP64 flops of every kernel of one two-level step (ncu's executed "
                                            "DADD / DMUL / DFMA counters, profiles/ncu_r02c.md; the pair loop's static count "
                                            "if no capture is recorded) / step time / peak",
                         "algorithmic_flops_per_ordered_pair": FLOPS_PER_PAIR,
                         "executed_flops_per_unordered_pair": SYM_FLOPS_PER_UNORDERED_PAIR if sym else 2 * FLOPS_PER_PAIR,
                         "executed_fp64_instr_per_unordered_pair": SYM_FP64_INSTR_PER_UNORDERED_PAIR if sym else 2 * FP64_INSTR_PER_PAIR,
                         "kernel_ms": k0_ms, "pairs_per_launch": pairs_per_kick,
                         "ordered_pair_equivalents_per_s": pairs_per_kick / (k0_ms * 1e-3)},
        }
        import oracle                                   # cpu_baseline leg: rank 0, N=1 only
        if world == 1 and not args.no_cpu_baseline:
            rows = calibrate_rows(ki, oracle, target_s=12.0)
            t, p = oracle_sample(ki, rows, oracle)
            line["cpu_baseline"] = {"value": p / t, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                                    "sample": f"{rows} evenly spaced i-rows x all {ki.n_massive} j at levels 0 and 1 "
                                              f"({t:.1f} s wall clock); value counts the two-level step as N (N - 1) pair "
                                              f"interactions, as `value` does (the oracle evaluates both levels' pairs: "
                                              f"{2 * p / t:.3g} pair evaluations/s)"}
        print(json.dumps(line), flush=True)
    kick.free()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--headline-only", action="store_true",
                    help="time the headline step only (skip the per-config and NEXT-row timings): for profiler runs")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        args.warmup = 3                                  # timing rule: W >= 3
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus > 1 and world == 1:
        # convenience: re-launch under torchrun as the driver would
        os.execvp(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                   f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
                                   "--master-port", os.environ.get("MASTER_PORT", "29541"), os.path.abspath(__file__),
                                   *sys.argv[1:]])
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_b200(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
