"""Host logic of bench.py's N > 1 path (replicas) on CPU: two gloo ranks agree on the maximum over ranks,
the whole-job value counts the particles of all ranks, every rank gets its own problem of the same shape, and the reference
arm runs on rank 0 only."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
rank, local_rank, world = bench.dist_env()
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["MASTER_PORT"], rank=rank, world_size=world)
# rank r "measured" 100 steps in (130 + 20 r) ms and one end-to-end step in (1.7 + 0.5 r) ms
out = bench.aggregate_over_ranks(130.0 + 20.0 * rank, 1.7 + 0.5 * rank, 1000000, 100, world, "cpu")
pos, q, c = bench.make_workload("cfg1_cube4096_f64", rank)
dist.barrier()
print("RESULT " + json.dumps(dict(rank=rank, world=world, out=out, seed=c["seed"], shape=list(pos.shape), first=float(pos[0, 0]))), flush=True)
dist.destroy_process_group()
""" % ROOT


def test_two_gloo_ranks_take_the_max_and_sum_the_work(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = 29500 + os.getpid() % 2000
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    res = {}
    for pr in procs:
        so, se = pr.communicate(timeout=240)
        assert pr.returncode == 0, se[-2000:]
        line = [l for l in so.splitlines() if l.startswith("RESULT ")][0]
        d = json.loads(line[7:])
        res[d["rank"]] = d
    assert set(res) == {0, 1}
    for r in (0, 1):
        ms_per_step, value, e2e_ms, e2e_value = res[r]["out"]
        assert abs(ms_per_step - 1.5) < 1e-12          # max(130, 150) ms / 100 steps
        assert abs(value - 2 * 1e6 / 1.5 / 1e3) < 1e-9  # particles of BOTH ranks over the slower rank's time
        assert abs(e2e_ms - 2.2) < 1e-12 and abs(e2e_value - 2 * 1e6 / 2.2 / 1e3) < 1e-9
    assert res[0]["shape"] == res[1]["shape"] == [4096, 3]
    assert res[1]["seed"] == res[0]["seed"] + 1000 and res[0]["first"] != res[1]["first"]  # independent replicas


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    ms, val, e2e_ms, e2e_val = bench.aggregate_over_ranks(129.4, 1.7, 1000000, 100, 1, "cpu")
    assert abs(ms - 1.294) < 1e-12 and abs(val - 1e6 / 1.294 / 1e3) < 1e-9 and abs(e2e_val - 1e6 / 1.7 / 1e3) < 1e-9


def test_reference_arm_runs_on_rank_0_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
