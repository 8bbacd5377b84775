"""The N>1 path of bench.py (replicas: one lattice per rank, max-over-ranks timing,
whole-job aggregate) exercised with world_size 2 on the gloo backend, CPU only."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as tmp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 100.0 + 50.0 * rank                       # rank 1 is the slow replica
    ms = bench.max_over_ranks(ms_local, world)
    dist.barrier()
    val = bench.aggregate_gsups(1 << 20, 10, world, ms)
    out.put((rank, ms, val))
    dist.destroy_process_group()


def test_two_rank_replicas_max_time_and_aggregate():
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    ctx = tmp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 150.0                                 # the max over ranks, on every rank
        assert val == pytest.approx((1 << 20) * 10 * 2 / 0.150 / 1e9)


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(12.5, 1) == 12.5
    assert bench.aggregate_gsups(1000, 4, 1, 2.0) == pytest.approx(1000 * 4 / 2e-3 / 1e9)
