"""Slab decomposition, host logic on the CPU.

The decomposition argument -- a time step moves information by exactly 4 sites per direction,
so a slab with 4 valid ghost layers evolved with its own periodic wrap has exact owned layers --
holds for any implementation of the step.  Here the slabs are evolved by the oracle and the ghost
layers travel through paper_1907_12834_b200.slab.exchange_halos on the gloo backend
(world_size 2 and 3, one process per slab): partition, ring wiring, message order (with two
ranks both neighbours are the same peer) and the all-reduce are the code the GPU path uses;
tests/test_gpu_parity.py runs the same decomposition on the CUDA kernels."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as tmp

from conftest import ROOT
from paper_1907_12834_b200 import inputs
from paper_1907_12834_b200.slab import GHOST, SlabLayout, exchange_halos


def test_layout_partitions_the_slow_axis():
    lay = SlabLayout(2, (40, 50), 3)
    assert lay.counts == [17, 17, 16] and lay.starts == [0, 17, 34]
    assert lay.local_dims(2) == (40, 16 + 2 * GHOST) and lay.layer_sites() == 40 and lay.axis == -2
    assert [lay.neighbours(r) for r in range(3)] == [(2, 1), (0, 2), (1, 0)]
    assert SlabLayout(1, (119,), 2).local_dims(0) == (60 + 2 * GHOST,)
    assert SlabLayout(3, (8, 6, 20), 2).local_dims(1) == (8, 6, 10 + 2 * GHOST)
    assert SlabLayout(3, (8, 6, 20), 2).layer_sites() == 48
    with pytest.raises(ValueError):
        SlabLayout(2, (40, 10), 3)           # slabs of 3 layers cannot feed 4 ghost layers
    with pytest.raises(ValueError):
        SlabLayout(2, (40,), 1)


@pytest.mark.parametrize("ndim,dims,world", [(1, (37,), 3), (2, (5, 23), 2), (3, (3, 4, 17), 4)])
def test_cut_owned_assemble_roundtrip(ndim, dims, world):
    lay = SlabLayout(ndim, dims, world)
    lat = (1, dims[0]) if ndim == 1 else tuple(reversed(dims))
    f = np.arange(10 * int(np.prod(lat))).reshape((5, 2) + lat)
    parts = []
    for r in range(world):
        loc = lay.cut(r, f)
        assert loc.shape[lay.axis] == lay.counts[r] + 2 * GHOST
        # ghost layers are the periodic neighbours' layers
        lo = np.take(loc, np.arange(GHOST), axis=lay.axis)
        want = np.take(f, (lay.starts[r] - GHOST + np.arange(GHOST)) % dims[-1], axis=lay.axis)
        assert np.array_equal(lo, want)
        parts.append(lay.owned(r, loc))
    assert np.array_equal(lay.assemble(parts), f)


def test_single_slab_exchange_is_the_periodic_wrap():
    e_lo, e_hi = torch.arange(6.0), torch.arange(6.0) + 10
    g_lo, g_hi = torch.zeros(6), torch.zeros(6)
    exchange_halos(e_lo, e_hi, g_lo, g_hi, 0, 1)
    assert torch.equal(g_lo, e_hi) and torch.equal(g_hi, e_lo)


# ---- world_size 2 / 3 on gloo: oracle-evolved slabs with real halo exchange -------------------
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _layers(a, lay, first, count):
    idx = [slice(None)] * a.ndim
    idx[lay.axis] = slice(first, first + count)
    return idx


def _worker(rank, world, port, ndim, dims, order, steps, out):
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle.qlga_oracle import Oracle
    orc = Oracle("double")
    c = (1.0, 0.3, -0.1)
    q0 = inputs.random_spinor_state(dims if ndim > 1 else (dims[0], 1), seed=11, amplitude=0.05)
    lay = SlabLayout(ndim, dims, world)
    loc = lay.cut(rank, q0)
    n = loc.shape[lay.axis]
    for _ in range(steps):
        loc = orc.step(loc, ndim, c, order, 1)                         # periodic wrap of the extended slab
        e_lo = torch.from_numpy(np.ascontiguousarray(loc[tuple(_layers(loc, lay, GHOST, GHOST))]))
        e_hi = torch.from_numpy(np.ascontiguousarray(loc[tuple(_layers(loc, lay, n - 2 * GHOST, GHOST))]))
        g_lo, g_hi = torch.empty_like(e_lo), torch.empty_like(e_hi)
        exchange_halos(e_lo, e_hi, g_lo, g_hi, rank, world)
        loc[tuple(_layers(loc, lay, 0, GHOST))] = g_lo.numpy()
        loc[tuple(_layers(loc, lay, n - GHOST, GHOST))] = g_hi.numpy()
    own = np.ascontiguousarray(lay.owned(rank, loc))
    t = torch.tensor([float(np.sum(np.abs(own) ** 2))], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    out.put((rank, own, float(t[0])))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("ndim,dims,world,order", [(2, (12, 21), 2, 1), (2, (10, 26), 3, 0), (1, (29,), 2, 1)])
def test_oracle_slabs_with_gloo_exchange_reproduce_the_global_step(oracle, ndim, dims, world, order):
    steps = 3
    ctx = tmp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, ndim, dims, order, steps, out))
             for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=180) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    q0 = inputs.random_spinor_state(dims if ndim > 1 else (dims[0], 1), seed=11, amplitude=0.05)
    ref = oracle.step(q0, ndim, (1.0, 0.3, -0.1), order, steps)
    lay = SlabLayout(ndim, dims, world)
    got = lay.assemble([r[1] for r in res])
    # the oracle is translation covariant bit for bit, so the slabs reproduce it exactly
    assert np.array_equal(got, ref)
    for _, _, total in res:
        assert total == pytest.approx(float(np.sum(np.abs(ref) ** 2)), rel=1e-13)


def test_three_ghost_layers_are_not_enough(oracle):
    # the domain of dependence of one step is exactly 4 sites: with 3 ghost layers the slab differs
    dims, c = (8, 24), (1.0, 0.3, -0.1)
    q0 = inputs.random_spinor_state(dims, seed=5, amplitude=0.05)
    ref = oracle.step(q0, 2, c, 1, 1)
    for ghost, ok in ((4, True), (3, False)):
        lay = SlabLayout(2, dims, 2, ghost=ghost)
        parts = [lay.owned(r, oracle.step(lay.cut(r, q0), 2, c, 1, 1)) for r in range(2)]
        assert np.array_equal(lay.assemble(parts), ref) == ok
