"""Host logic of the N > 1 bench path on CPU: world_size 2, `gloo` backend (no GPU needed).

The hot path does not shard (replicas only, no data-path collective), so what runs under
torchrun is: every rank times its own replica, the reported time is the MAX over ranks, `value` is the
whole-job aggregate, rank 0 alone prints, and `--impl reference` does its work on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [5.0, 8.0][rank]                                     # rank 1 is the slow replica
    got = bench.max_over_ranks(ms, dist, device="cpu")
    dist.barrier()
    with open(f"{out}.{rank}", "w") as f:
        json.dump({"max_ms": got, "value": bench.whole_job_value(world, 1000, got)}, f)
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    import torch.multiprocessing as mp

    port, out = _free_port(), str(tmp_path / "r")
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    for rank in (0, 1):
        r = json.load(open(f"{out}.{rank}"))
        assert r["max_ms"] == 8.0                              # every rank sees the slowest replica's time
        assert r["value"] == pytest.approx(2 * 1000 / 8e-3)    # units of all ranks / max time


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25, None) == 3.25
    assert bench.whole_job_value(1, 99_488_250, 5.0) == pytest.approx(99_488_250 / 5e-3)


def test_reference_arm_nonzero_rank_exits_without_work():
    """Under torchrun only rank 0 runs the oracle and prints; the other ranks exit 0 silently."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
