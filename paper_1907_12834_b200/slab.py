"""Slab-decomposed QLGA time step: one lattice over several GPUs.

The paper only says its code "naturally scales with the number of GPUs".
Decomposition used here (include/qlga.h, "Slab decomposition"): the lattice is cut along its
slowest axis (x in 1D, y in 2D, z in 3D) into `world` slabs, one per GPU / process.  A slab is
an ordinary library context on the extended lattice

    [GHOST ghost layers | owned layers | GHOST ghost layers]

One time step (eq. 108 / 112) moves information by exactly 4 sites per direction -- four
kinetic factors of radius 1, the interaction is site-local -- so with GHOST = 4 valid ghost
layers before the step the owned layers are exact after it, whatever the periodic wrap of the
extended slab wrote into its own ghost layers.  After every step each slab sends its lowest and
highest GHOST owned layers to its two ring neighbours, which overwrite their ghost layers: one
exchange of 2 x 4 x 160 B per site of a layer per step in fp64 (5.2 MB per side at Nx = 8192),
a few microseconds on NVLink against a 40 ms step, so the exchange is not overlapped with the
pass kernels and no fused compute + transfer kernel is written for it.
Every step of the arithmetic still runs in the library's kernels; this module holds the host
logic (partition, neighbour ring, exchange order) and the transport (torch.distributed P2P:
NCCL for CUDA tensors, gloo in the CPU tests; a device copy when both slabs are in one process).
"""
from __future__ import annotations

import numpy as np

GHOST = 4     # sites per direction that one time step moves information (see module docstring)


class SlabLayout:
    """Host-side partition of the slowest lattice axis into `world` contiguous slabs.

    dims = (Nx,), (Nx, Ny) or (Nx, Ny, Nz); arrays carry the lattice as their last axes
    [..., Ny, Nx] (1D: [..., 1, Nx]) or [..., Nz, Ny, Nx], so the slab axis is array axis
    -ndim.  Slab r owns layers [start_r, start_r + count_r); the remainder of an uneven
    division goes to the first slabs."""

    def __init__(self, ndim, dims, world, ghost=GHOST):
        self.ndim, self.world, self.ghost = int(ndim), int(world), int(ghost)
        self.dims = tuple(int(v) for v in dims)[:self.ndim]
        if len(self.dims) != self.ndim or self.ndim not in (1, 2, 3) or self.world < 1:
            raise ValueError("SlabLayout: bad ndim / dims / world")
        self.extent = self.dims[-1]
        base, rem = divmod(self.extent, self.world)
        self.counts = [base + (1 if r < rem else 0) for r in range(self.world)]
        self.starts = [sum(self.counts[:r]) for r in range(self.world)]
        if min(self.counts) < self.ghost:
            raise ValueError(f"SlabLayout: a slab of {min(self.counts)} layers is thinner than the "
                             f"{self.ghost} layers it must send to a neighbour")
        self.axis = -self.ndim

    def neighbours(self, rank):
        """(down, up): the ranks owning the layers below / above this slab (periodic ring)."""
        return (rank - 1) % self.world, (rank + 1) % self.world

    def local_dims(self, rank):
        """Lattice dims of the slab's library context (owned + 2 * ghost layers)."""
        return self.dims[:-1] + (self.counts[rank] + 2 * self.ghost,)

    def layer_sites(self):
        return int(np.prod(self.dims[:-1])) if self.ndim > 1 else 1

    def extended_layers(self, rank):
        """Global layer index of every layer of the extended slab (periodic)."""
        n = self.counts[rank] + 2 * self.ghost
        return (self.starts[rank] - self.ghost + np.arange(n)) % self.extent

    def cut(self, rank, field):
        """The extended slab (ghost layers filled from the periodic global field)."""
        return np.ascontiguousarray(np.take(field, self.extended_layers(rank), axis=self.axis))

    def owned(self, rank, local):
        """The owned layers of an extended-slab array."""
        idx = [slice(None)] * local.ndim
        idx[self.axis] = slice(self.ghost, self.ghost + self.counts[rank])
        return local[tuple(idx)]

    def assemble(self, parts):
        """Global array from the owned parts of all slabs, in rank order."""
        return np.concatenate(parts, axis=self.axis)


def exchange_halos(edge_lo, edge_hi, ghost_lo, ghost_hi, rank, world, group=None):
    """Ring exchange of one step: ghost_lo <- the down neighbour's edge_hi, ghost_hi <- the up
    neighbour's edge_lo.  The tensors may live on a GPU (NCCL, i.e. NVLink / NVSwitch P2P) or on
    the host (gloo).  The two messages of a pair of ranks are posted in the same order on both
    sides (to-up first) and tagged, so they also match when up == down (world == 2)."""
    if world == 1:
        ghost_lo.copy_(edge_hi)
        ghost_hi.copy_(edge_lo)
        return
    import torch.distributed as dist
    down, up = (rank - 1) % world, (rank + 1) % world
    ops = [dist.P2POp(dist.isend, edge_hi, up, group, 0),
           dist.P2POp(dist.isend, edge_lo, down, group, 1),
           dist.P2POp(dist.irecv, ghost_lo, down, group, 0),
           dist.P2POp(dist.irecv, ghost_hi, up, group, 1)]
    for work in dist.batch_isend_irecv(ops):
        work.wait()


class SlabQlga:
    """One slab of a lattice of global dims `dims`, on one GPU.  With transport="dist" (default
    when torch.distributed is initialised) the ring neighbours are the other ranks of `group`;
    SlabGroup drives several slabs of one process instead."""

    def __init__(self, ndim, dims, couplings, order="interleaved", precision="f64", rank=None, world=None,
                 device=None, group=None, keep_previous=False):
        import torch
        from . import qlga
        if rank is None or world is None:
            import torch.distributed as dist
            rank, world = dist.get_rank(group), dist.get_world_size(group)
        self.torch, self.group = torch, group
        self.rank, self.world = int(rank), int(world)
        self.layout = SlabLayout(ndim, dims, self.world)
        if device is None:
            device = f"cuda:{torch.cuda.current_device()}"
        self.sim = qlga.Qlga(ndim, self.layout.local_dims(self.rank), couplings, order=order,
                             precision=precision, device=device, keep_previous=keep_previous)
        self.sim.slab_configure(GHOST)
        n = 10 * GHOST * self.layout.layer_sites() * 2                   # reals per packed edge
        self.edge_lo, self.edge_hi, self.ghost_lo, self.ghost_hi = (
            torch.empty(n, dtype=self.sim.rdtype, device=self.sim.device) for _ in range(4))

    def close(self):
        self.sim.close()

    # -- state: global arrays are cut here; ghost layers come out of the periodic global field --
    def set_state_q(self, q_global):
        self.sim.set_state_q(self.layout.cut(self.rank, np.asarray(q_global)))

    def set_state_psi(self, psi_global):
        self.sim.set_state_psi(self.layout.cut(self.rank, np.asarray(psi_global)))

    def get_state_q(self):
        """The owned layers of q, [5][2][...owned...]."""
        return np.ascontiguousarray(self.layout.owned(self.rank, self.sim.get_state_q()))

    def get_state_psi(self):
        return np.ascontiguousarray(self.layout.owned(self.rank, self.sim.get_state_psi()))

    # -- one time step = the library's step on the extended slab, then the ghost refresh --------
    def pack_edges(self):
        self.sim.slab_edge_get(0, self.edge_lo)
        self.sim.slab_edge_get(1, self.edge_hi)

    def unpack_ghosts(self, ghost_lo=None, ghost_hi=None):
        self.sim.slab_ghost_set(0, self.ghost_lo if ghost_lo is None else ghost_lo)
        self.sim.slab_ghost_set(1, self.ghost_hi if ghost_hi is None else ghost_hi)

    def exchange(self):
        # the library packs and unpacks on the context's stream; the P2P operations must be issued on that
        # same stream, else NCCL's send / recv is not ordered against qlga_slab_edge_get / qlga_slab_ghost_set
        with self.torch.cuda.stream(self.sim.stream):
            self.pack_edges()
            exchange_halos(self.edge_lo, self.edge_hi, self.ghost_lo, self.ghost_hi, self.rank, self.world,
                           self.group)
            self.unpack_ghosts()

    def step(self, n=1):
        for _ in range(int(n)):
            self.sim.step(1)
            self.exchange()

    # -- diagnostics ------------------------------------------------------------------------
    def observables(self):
        """Lattice sums over the whole lattice: the owned-layer sums of every slab added up
        (all-reduce of 17 doubles), then the derived record."""
        sums = self.sim.observable_sums()
        if self.world > 1:
            import torch.distributed as dist
            on_gpu = dist.get_backend(self.group) == "nccl"
            t = self.torch.from_numpy(sums.copy())
            t = t.to(self.sim.device) if on_gpu else t
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
            sums = t.cpu().numpy()
        return self.sim.observables_from_sums(sums)

    def vorticity(self):
        """omega of the owned rows (2D): the stencil reaches one row into the ghost layers."""
        return np.ascontiguousarray(self.layout.owned(self.rank, self.sim.vorticity()))

    def vortices(self, max_out=65536):
        """(records, count) of the plaquettes anchored in the owned rows, y in global coordinates."""
        rec, _ = self.sim.vortices(max_out)
        lo, cnt = GHOST, self.layout.counts[self.rank]
        rec = rec[(rec[:, 2] >= lo) & (rec[:, 2] < lo + cnt)].copy()
        rec[:, 2] += self.layout.starts[self.rank] - GHOST
        return rec, len(rec)


class SlabGroup:
    """All `nslabs` slabs of a lattice in one process on one GPU, stepped one after the other and
    exchanged by device copies: the decomposition without the transport.  This is what the
    single-GPU parity tests run (no kernel ever waits on another one)."""

    def __init__(self, ndim, dims, couplings, order="interleaved", precision="f64", nslabs=2,
                 device="cuda:0", keep_previous=False):
        self.layout = SlabLayout(ndim, dims, nslabs)
        self.slabs = [SlabQlga(ndim, dims, couplings, order, precision, rank=r, world=nslabs, device=device,
                               keep_previous=keep_previous) for r in range(nslabs)]

    def close(self):
        for s in self.slabs:
            s.close()

    def set_state_q(self, q_global):
        for s in self.slabs:
            s.set_state_q(q_global)

    def step(self, n=1):
        R = len(self.slabs)
        for _ in range(int(n)):
            for s in self.slabs:
                s.sim.step(1)
            for s in self.slabs:
                s.pack_edges()
            for r, s in enumerate(self.slabs):
                s.unpack_ghosts(self.slabs[(r - 1) % R].edge_hi, self.slabs[(r + 1) % R].edge_lo)

    def get_state_q(self):
        return self.layout.assemble([s.get_state_q() for s in self.slabs])

    def observables(self):
        sums = sum(s.sim.observable_sums() for s in self.slabs)
        return self.slabs[0].sim.observables_from_sums(sums)

    def vorticity(self):
        return self.layout.assemble([s.vorticity() for s in self.slabs])

    def vortices(self, max_out=65536):
        recs = [s.vortices(max_out)[0] for s in self.slabs]
        rec = np.concatenate(recs, axis=0)
        return rec, len(rec)
