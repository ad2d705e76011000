"""-m "not gpu": the N > 1 path of bench.py on CPU -- world_size 2, gloo, 127.0.0.1.  The path does not shard
(north_star: "everything runs on one GPU"): ranks are independent replicas on independently seeded disks, there is
no data-path collective; what the ranks share is the barrier, the max-over-ranks timing and rank 0's JSON line.
Also: `--impl reference` under torchrun runs on rank 0 only."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
WORKER = r'''
import json, os, sys
sys.path.insert(0, {root!r})
import numpy as np
import torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=world)
ki = bench.workload(rank)
ms = 10.0 + 5.0 * rank                                   # rank 1 is the slow one
worst = bench.max_over_ranks(ms, world)
value = bench.whole_job_value(world, 1000, 2, worst)
dist.barrier()
print(json.dumps(dict(rank=rank, n=ki.n, levels=int(ki.rcrit.shape[0]), x0=float(ki.pos[0, 0]), m0=float(ki.mass[0]),
                      config=ki.meta["config"], worst=worst, value=value)))
dist.destroy_process_group()
'''


def _spawn(script, world, port, extra_env=None):
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="1", **(extra_env or {}))
        procs.append(subprocess.Popen([sys.executable, "-c", script], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    return [o for o, _ in outs]


def test_replicas_max_over_ranks_and_independent_disks():
    outs = _spawn(WORKER.format(root=ROOT, port=29617), 2, 29617)
    r = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda d: d["rank"])
    assert [d["rank"] for d in r] == [0, 1]
    assert r[0]["n"] == r[1]["n"] == 65536 and r[0]["levels"] == r[1]["levels"] == 2       # same recipe ...
    assert r[0]["x0"] != r[1]["x0"] and r[0]["m0"] != r[1]["m0"]                            # ... different seeds
    assert "replica1" in r[1]["config"]
    assert r[0]["worst"] == r[1]["worst"] == 15.0                                           # the slow rank's time, on both
    want = 2 * 1000 * 2 / 15e-3
    assert r[0]["value"] == r[1]["value"] == pytest.approx(want, rel=1e-15)


def test_reference_arm_runs_on_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 prints the line, rank 1 exits 0 without work."""
    outs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT="29618")
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps",
                            "1", "--warmup", "0"], env=env, capture_output=True, text=True, cwd=ROOT, timeout=600)
        assert p.returncode == 0, p.stderr[-2000:]
        outs.append(p.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["unit"] == "pair interactions/s" and line["higher_is_better"] is True
