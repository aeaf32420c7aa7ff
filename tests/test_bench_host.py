"""Host-side logic of bench.py's N > 1 arm (replicas only) on CPU: world-size-2 gloo."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times = [0.010 * (rank + 1), 0.020 * (world - rank)]          # rank-dependent device times
    mx = bench.max_over_ranks(times, "cpu")
    dist.barrier()
    if rank == 0:
        torch.save({"mx": mx, "rate": bench.whole_job_rate(world, 4096, 10, mx[0])}, out)
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_world2(tmp_path):
    out = str(tmp_path / "r.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    r = torch.load(out)
    assert r["mx"] == pytest.approx([0.020, 0.040])
    assert r["rate"] == pytest.approx(2 * 4096 * 10 / 0.020)


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert bench.whole_job_rate(1, 64, 3, 0.5) == 64 * 3 / 0.5


def test_reference_arm_nonzero_rank_exits_without_work(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    class A: config = 1; steps = 1; warmup = 0; gpus = 2
    assert bench.run_reference(A()) is None
