"""N > 1 plumbing of bench.py on CPU: world_size-2 gloo processes (no GPU, no data-path collective:
trajectories are independent units, only the timing max and the unit sum cross ranks)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
sys.path.insert(0, os.environ["LM_ROOT"])
import numpy as np
import torch
import bench
from oracle import lm_oracle as orc
from paper_2309_09102_b200 import workloads as wl

rank, world = bench.dist_init("gloo")
assert world == 2 and rank == int(os.environ["RANK"])
bench.dist_barrier()
# each rank "measures" a different time and processes its own units
ms, units = bench.dist_max_sum(10.0 + 5.0 * rank, 1000.0 * (rank + 1), torch.device("cpu"))
ch = wl.panda_chain()
w = bench.make_workload("C2", lambda q: orc.fk(ch, q), 2, 16, rank)
o = orc.lm_run(ch, orc.Params(tol=w.tol), w.target_pos.astype(float), w.target_quat.astype(float),
               w.seeds.astype(float), w.max_iters)
_, executed_all = bench.dist_max_sum(0.0, float(o.executed), torch.device("cpu"))
bench.dist_barrier()
print(json.dumps({"rank": rank, "ms": ms, "units": units, "seed0": float(w.seeds[0, 0]),
                  "executed": int(o.executed), "executed_all": executed_all,
                  "converged": bool(np.all(o.status & 1))}))
'''


def _spawn(rank, port, code):
    env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
               MASTER_PORT=str(port), LM_ROOT=ROOT, OMP_NUM_THREADS="2")
    return subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                            text=True, cwd=ROOT)


@pytest.mark.timeout(300)
def test_two_rank_gloo_reduction_and_sharding():
    port = 29600 + os.getpid() % 300
    procs = [_spawn(r, port, WORKER) for r in range(2)]
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=280)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    # time = MAX over ranks, units = SUM over ranks, identical on both ranks
    assert outs[0]["ms"] == outs[1]["ms"] == 15.0
    assert outs[0]["units"] == outs[1]["units"] == 3000.0
    # weak scaling: every rank draws its own batch of the same shape
    assert outs[0]["seed0"] != outs[1]["seed0"]
    assert outs[0]["executed_all"] == outs[1]["executed_all"] == outs[0]["executed"] + outs[1]["executed"]
    assert outs[0]["converged"] and outs[1]["converged"]


def test_reference_arm_runs_on_rank0_only():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
           "--ref-traj", "2", "--gpus", "2"]
    env1 = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r1 = subprocess.run(cmd, env=env1, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=120)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    env0 = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="2")
    r0 = subprocess.run(cmd, env=env0, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=120)
    assert r0.returncode == 0, r0.stderr[-1000:]
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "waypoint_lm_iterations_per_sec"
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["higher_is_better"] is True and line["config"]["workload"].startswith("C4")


def test_shard_seeds_are_rank_specific():
    import bench
    assert bench.rank_seed_offset(0) == 0 and bench.rank_seed_offset(3) == 3000


@pytest.mark.timeout(300)
def test_bench_starts_its_own_ranks():
    """`python bench.py --gpus 2` with no launcher around it starts two ranks itself (torch.distributed.run, 127.0.0.1):
    the self-test leg runs the bench's cross-rank reductions over gloo and rank 0's line says n_gpus = 2.  Without the
    self-test flag, on a box with fewer GPUs than requested, it fails loudly instead of running one rank."""
    bench = os.path.join(ROOT, "bench.py")
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    env["OMP_NUM_THREADS"] = "1"
    r = subprocess.run([sys.executable, bench, "--gpus", "2", "--dist-selftest"], env=env, stdout=subprocess.PIPE,
                       stderr=subprocess.PIPE, text=True, timeout=280, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1                                          # rank 0 alone prints
    assert lines[0]["n_gpus"] == 2 and lines[0]["ms_max"] == 2.0 and lines[0]["units_sum"] == 2.0
    import torch
    if torch.cuda.device_count() < 2:
        r = subprocess.run([sys.executable, bench, "--gpus", "2", "--steps", "1"], env=env, stdout=subprocess.PIPE,
                           stderr=subprocess.PIPE, text=True, timeout=120, cwd=ROOT)
        assert r.returncode != 0 and "2 GPUs requested" in r.stderr and r.stdout.strip() == ""
