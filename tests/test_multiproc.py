"""N > 1 plumbing of bench.py on CPU (gloo, world size 2): replicas only -- every rank owns its own
ensembles with rank-specific seeds, there is no data-path collective; only the barrier, the
max-over-ranks time and the sum of moves cross ranks."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["PT_ROOT"])
import numpy as np
import bench
from paper_1107_3490_b200 import synth
rank, world, local = bench.dist_setup(2, backend="gloo")
assert world == 2 and rank == int(os.environ["RANK"])
bench.dist_barrier(world)
inp = synth.make_inputs(1, rank=rank)
mine = list(synth.shard_ensembles(5, world, rank))
t = bench.dist_max(1.0 + rank, world)          # slowest rank decides
moves = bench.dist_sum(float(inp.workload.chains * inp.workload.N * 10), world)
print(json.dumps({"rank": rank, "tmax": t, "moves": moves, "seed0": int(inp.seeds[0]), "mine": mine,
                  "x0": float(inp.conformations[0, 0, 1, 0])}), flush=True)
import torch.distributed as dist
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(code_or_args, world=2, extra_env=None):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), PT_ROOT=str(ROOT), OMP_NUM_THREADS="1")
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable, *code_or_args], env=env, cwd=str(ROOT),
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


def test_two_ranks_gloo_timing_and_sharding():
    outs = _spawn(["-c", WORKER])
    rows = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda d: d["rank"])
    assert [d["rank"] for d in rows] == [0, 1]
    assert rows[0]["tmax"] == rows[1]["tmax"] == 2.0                 # max over ranks
    assert rows[0]["moves"] == rows[1]["moves"] == 2 * 8 * 13 * 10   # whole-job aggregate
    assert rows[0]["seed0"] != rows[1]["seed0"] and rows[0]["x0"] != rows[1]["x0"]   # independent replicas
    assert rows[0]["mine"] + rows[1]["mine"] == list(range(5))       # ensembles partitioned, none shared


def test_reference_arm_runs_on_rank0_only():
    outs = _spawn(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                   "--config", "1", "--sweeps", "50"])
    lines = [o.strip() for o in outs]
    assert lines[1] == ""                                            # rank 1 exits 0 without work
    d = json.loads(lines[0].splitlines()[-1])
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["unit"] == "moves/s"
