"""Multi-GPU path = replicas only: no data-path collective, only the max-over-ranks timing.
World-size-2 gloo test of that aggregation on CPU (the driver's N>1 launch uses the same code with nccl)."""
import os
import socket
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank: int, world: int, port: int, q):
    import torch.distributed as dist

    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" (r + 1) * 10 ms for 1e6 updates
    value, ms = bench.job_throughput(1.0e6, 10.0 * (rank + 1), world, device="cpu")
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, value, ms))


def test_replicas_aggregate_max_over_ranks():
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms in out:
        assert ms == pytest.approx(20.0)                  # the slowest rank
        assert value == pytest.approx(2.0e6 / 20.0e-3)    # both ranks' updates over that time


def test_single_rank_is_identity():
    import bench

    value, ms = bench.job_throughput(5.0e5, 4.0, 1, device="cpu")
    assert ms == 4.0 and value == pytest.approx(5.0e5 / 4.0e-3)
