"""N > 1 host logic on CPU (gloo, world_size 2): the path does not shard (replicas only), so
the only cross-rank step of bench.py is the max-over-ranks of the device-timed milliseconds and the whole-job value
computed from it; the reference arm must run on rank 0 alone."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
    mx = bench.max_over_ranks(ms, world, torch.device("cpu"))
    val = bench.job_value(1_000_000, 3, world, mx)
    dist.barrier()
    dist.destroy_process_group()
    with open(out + f".{rank}", "w") as f:
        json.dump({"max": mx, "value": val}, f)


def test_max_over_ranks_and_job_value_gloo(tmp_path):
    import socket
    with socket.socket() as sk:                 # a free port for the rendezvous on 127.0.0.1
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    world = 2
    out = str(tmp_path / "r")
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    res = [json.load(open(out + f".{r}")) for r in range(world)]
    for r in res:
        assert r["max"] == 15.0                                  # every rank sees the slowest replica's time
        assert abs(r["value"] - 2 * 1_000_000 * 3 / 15e-3 / 1e6) < 1e-9   # both replicas' points over that time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5, 1, torch.device("cpu")) == 7.5


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--workload", "cfg1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
