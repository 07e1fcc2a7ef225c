"""N > 1 path of bench.py on CPU (gloo, world size 2). The method does not shard (north_star: one GPU, no
collectives; DESIGN.md section 9 "replicas only"), so the whole multi-rank logic is: barrier, MAX of the
device-timed milliseconds over the ranks, value = all ranks' updates / that time, and a reference arm that
runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
sys.path.insert(0, os.environ["MPC_ROOT"])
import torch
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
dist.barrier()
ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow one
ms = bench.max_over_ranks(dist, ms_local, torch.device("cpu"))
val = bench.whole_job_rate(world, 1000, 4, ms)
dist.barrier()
print(json.dumps({"rank": rank, "ms": ms, "value": val}), flush=True)
dist.destroy_process_group()
'''


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch(code_or_args, extra_env=None):
    env = dict(os.environ, MPC_ROOT=ROOT, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(free_port()), WORLD_SIZE="2")
    env.update(extra_env or {})
    procs = []
    for r in range(2):
        e = dict(env, RANK=str(r), LOCAL_RANK=str(r))
        procs.append(subprocess.Popen([sys.executable] + code_or_args, env=e, cwd=ROOT, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=600) for p in procs]
    for p, (o, err) in zip(procs, outs):
        assert p.returncode == 0, err[-2000:]
    return [o for o, _ in outs]


def test_max_over_ranks_and_whole_job_rate_gloo_world2():
    outs = launch(["-c", WORKER])
    res = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda d: d["rank"])
    for d in res:
        assert d["ms"] == pytest.approx(15.0)                       # the MAX over ranks, on every rank
        assert d["value"] == pytest.approx(2 * 1000 * 4 / 15e-3)    # both replicas' updates over that time


def test_reference_arm_runs_on_rank0_only_world2():
    # bench.py --impl reference under a 2-rank launch: rank 0 times the oracle and prints the line, rank 1 exits 0
    # without work (no process group is needed for that: the ranks never talk)
    args = [os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
            "--workload", "cfg1"]
    outs = launch(args)
    lines = [[l for l in o.splitlines() if l.startswith("{")] for o in outs]
    assert len(lines[0]) == 1 and lines[1] == []
    d = json.loads(lines[0][0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
