"""N > 1 host logic on CPU: two processes, gloo backend, rendezvous on 127.0.0.1.

The path shards as independent replicas, so what must be right across ranks is: distinct seeds per
rank, the max-over-ranks of the timed region, the whole-job rate, and that only rank 0 of the
reference arm prints.  No GPU and no CUDA library call is involved.
"""
import json
import os
import pathlib
import socket
import subprocess
import sys

import pytest

from paper_2501_09308_b200 import replicas

ROOT = pathlib.Path(__file__).resolve().parents[1]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["XRDVI_ROOT"])
import torch.distributed as dist
from paper_2501_09308_b200 import replicas
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
seeds = replicas.replica_seeds(rank)
t_local = 2.0 + 0.5 * rank                       # rank 1 is the slow one
t_max = replicas.max_over_ranks(t_local, dist, "cpu")
dist.barrier()
rate = replicas.whole_job_rate(1000.0, world, t_max)
print(json.dumps({"rank": rank, "world": world, "seeds": seeds, "t_max": t_max, "rate": rate}), flush=True)
dist.destroy_process_group()
"""


def test_two_rank_gloo_replica_logic(tmp_path):
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), XRDVI_ROOT=str(ROOT))
        procs.append(subprocess.Popen([sys.executable, "-c", _WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda o: o["rank"])
    assert [o["world"] for o in outs] == [2, 2]
    assert outs[0]["seeds"] != outs[1]["seeds"]                    # replicas are different restarts
    assert outs[0]["seeds"] == {"state_seed": 0, "restart_offset": 0, "draw_seed": 1}   # rank 0 = the single-GPU run
    assert outs[1]["seeds"]["restart_offset"] == 1                 # rank 1 starts from restart 1's jittered state
    assert outs[0]["t_max"] == outs[1]["t_max"] == 2.5             # max over ranks, on every rank
    assert outs[0]["rate"] == pytest.approx(2 * 1000.0 / 2.5)      # all ranks' units / slowest time


def test_single_process_helpers():
    assert replicas.max_over_ranks(1.25) == 1.25
    assert replicas.whole_job_rate(10.0, 4, 2.0) == 20.0
    with pytest.raises(ValueError):
        replicas.whole_job_rate(1.0, 0, 1.0)
    with pytest.raises(ValueError):
        replicas.replica_seeds(-1)


def test_reference_arm_non_zero_rank_prints_nothing():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "1", "--config", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_rank0_line():
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="1")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "2", "--warmup", "1",
                        "--config", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["value"] == line["value"] and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["unit"] == "pair-evals/s" and line["higher_is_better"] is True
