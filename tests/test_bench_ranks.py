"""Multi-process plumbing of bench.py on CPU (gloo, world_size 2): the path does not shard, so N ranks are N
independent reconstructions and the only cross-rank operations are the barrier and the
max-over-ranks of the device time.  No GPU and no compute here."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update({"RANK": str(rank), "WORLD_SIZE": str(world), "LOCAL_RANK": str(rank),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.rank_env() == (rank, world, rank)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")     # the slowest rank's time is the job's
    seed = bench.rank_seed(1234, rank)
    dist.barrier()
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms": ms, "seed": seed, "value": bench.aggregate_value(4, world, ms)}, f)
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_value_world2(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    got = [json.load(open(tmp_path / f"r{r}.json")) for r in range(world)]
    assert got[0]["ms"] == got[1]["ms"] == 15.0
    assert got[0]["seed"] != got[1]["seed"]                      # independent noise realisations
    assert got[0]["value"] == pytest.approx(2 * 4 / 15e-3)      # units of all ranks / slowest rank's time


def test_single_process_helpers_are_no_ops():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.aggregate_value(10, 1, 2000.0) == 5.0


def test_reference_arm_under_two_ranks_prints_one_line():
    """`--impl reference` under torchrun: rank 0 alone runs the oracle and prints the JSON line."""
    port = _free_port()
    outs = []
    for rank in (1, 0):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--steps", "1", "--warmup", "0", "--workload", "config1"],
                           env=env, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    assert outs[0] == ""
    line = json.loads(outs[1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["gpu_launches"] == 0 and line["vs_baseline"] is None
