"""Multi-GPU path = independent replicas (the path does not shard by contract).  The only
cross-rank logic is bench.py's aggregation (time = max over ranks, units = sum over ranks); it is covered
here with world_size 2 on the gloo backend, on CPU."""
from __future__ import annotations

import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank), UF_DIST_BACKEND="gloo")
    import torch.distributed as dist
    import bench
    r, w, local = bench.dist_setup(world)
    assert (r, w, local) == (rank, world, rank)
    bench.barrier()
    # rank r "measured" (r + 1) * 10 ms and processed (r + 1) * 1.5 units
    t, u = bench.aggregate_over_ranks(10.0 * (rank + 1), 1.5 * (rank + 1))
    q.put((rank, t, u))
    bench.barrier()
    dist.destroy_process_group()


def test_aggregate_over_ranks_world2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, u in res:
        assert t == pytest.approx(20.0) and u == pytest.approx(4.5), (rank, t, u)


def test_aggregate_single_process_is_identity():
    import bench
    assert bench.aggregate_over_ranks(3.25, 7.0) == (3.25, 7.0)
