"""NEXT-2 host side: one mesh over several MeshBlockPacks / GPUs (ghost exchange at every
Runge-Kutta stage).

The block lattice is cut into slabs along z, one pack (one process, one GPU) per slab. The data plane is in the
kernels: the thread that updates a cell writes the cell's ghost images into whichever pack holds them -- its own or a
z-neighbour's, whose buffers are mapped into this process (CUDA IPC; NVLink peer stores on a multi-GPU node). This
module only does the plumbing around that: the partition map, the exchange of buffer handles, the barrier between
stages, the 8-double all-reduce of the constraint norms. No arithmetic of the method lives here.

Two drivers over the same C ABI calls (z4c_set_partition / z4c_set_neighbor / z4c_stage / z4c_constraints_raw):
  SlabSet          all slabs in ONE process on one device and one stream (the stream order is the barrier): how the
                   partitioned data path is checked bit for bit against the unpartitioned pack on a single GPU;
  DistributedSlab  one slab per torch.distributed rank (launch with torchrun, one rank per GPU): neighbours' buffers
                   are opened through CUDA IPC, the barrier is a stream-ordered all-reduce (NCCL) or, on the gloo
                   backend, a device synchronise + host barrier.
"""
from __future__ import annotations

from dataclasses import replace
from typing import List, Optional, Tuple

import numpy as np

from . import z4c as Z


def slab_partition(nbz_global: int, nranks: int) -> List[Tuple[int, int]]:
    """[(bz0, nbz)] per rank: contiguous, balanced (the first nbz_global % nranks slabs are one block thicker)."""
    if nranks < 1 or nbz_global < nranks:
        raise ValueError("every rank needs at least one layer of blocks along z")
    base, extra = divmod(nbz_global, nranks)
    out, z = [], 0
    for r in range(nranks):
        t = base + (1 if r < extra else 0)
        out.append((z, t))
        z += t
    return out


def slab_neighbours(rank: int, nranks: int, bc: int) -> Tuple[Optional[int], Optional[int]]:
    """(rank below, rank above) across the slab's z-faces; None at an outflow boundary or when the mesh has one slab."""
    if nranks == 1:
        return None, None
    lo, hi = rank - 1, rank + 1
    if bc == 0:
        return lo % nranks, hi % nranks
    return (lo if lo >= 0 else None), (hi if hi < nranks else None)


def slab_params(p, rank: int, nranks: int):
    """Parameters of rank's slab: same lattice in x and y, nbz blocks along z, lower corner moved up."""
    bz0, nbz = slab_partition(p.nb[2], nranks)[rank]
    xmin = (p.xmin[0], p.xmin[1], p.xmin[2] + bz0 * p.n * p.dx)
    return replace(p, nb=(p.nb[0], p.nb[1], nbz), xmin=xmin)


def slab_interior(u: np.ndarray, p, rank: int, nranks: int) -> np.ndarray:
    """The slab's part of a global interior array [F][Nz][Ny][Nx]."""
    bz0, nbz = slab_partition(p.nb[2], nranks)[rank]
    return np.ascontiguousarray(u[:, bz0 * p.n:(bz0 + nbz) * p.n])


def combine_raw_norms(raw_sum_max: np.ndarray, ncells_global: int) -> np.ndarray:
    """From the element-wise SUM (even entries) / MAX (odd entries) over slabs of z4c_constraints_raw to
    {H_rms, H_max, M_rms, M_max, Theta_rms, Theta_max, Z_rms, Z_max} of the whole mesh."""
    out = np.array(raw_sum_max, dtype=np.float64)
    out[0::2] = np.sqrt(out[0::2] / float(ncells_global))
    return out


class SlabSet:
    """All slabs of a partitioned mesh in one process, on one device and one stream."""

    def __init__(self, p, nranks: int, device: str = "cuda:0"):
        self.p, self.nranks = p, nranks
        self.parts = slab_partition(p.nb[2], nranks)
        self.slabs: List[Z.Z4c] = []
        for r in range(nranks):
            self.slabs.append(Z.Z4c(slab_params(p, r, nranks), device=device,
                                    stream=self.slabs[0].stream if self.slabs else None))
        for r, s in enumerate(self.slabs):
            s.set_partition(p.nb[2], self.parts[r][0])
        for r, s in enumerate(self.slabs):
            for side, nb in enumerate(slab_neighbours(r, nranks, p.bc)):
                if nb is not None:
                    o = self.slabs[nb]
                    s.set_neighbor(side, o.state.data_ptr(), o.state2_ptr(), *self.parts[nb])

    def set_fused(self, mode: int):
        for s in self.slabs:
            s.set_fused(mode)

    def set_initial_data(self, u: np.ndarray):
        for r, s in enumerate(self.slabs):
            s.set_initial_data(slab_interior(u, self.p, r, self.nranks))
        for s in self.slabs:                 # one stream: every interior is final before any ghost is pulled
            s.fill_ghosts()

    def step(self, nsteps: int = 1):
        one_kernel = self.slabs[0].effective_mode()[1] == 2
        for _ in range(nsteps):
            for stage in (1, 2, 3, 4):
                if one_kernel:               # two state buffers: one barrier per stage (here: the stream order)
                    for s in self.slabs:
                        s.stage(stage)
                else:                        # state updated in place: no slab may push before every slab has read
                    for s in self.slabs:
                        s.stage_rhs(stage)
                    for s in self.slabs:
                        s.stage_update(stage)

    def sync(self):
        for s in self.slabs:
            s.sync()

    def get_interior(self) -> np.ndarray:
        return np.concatenate([s.get_interior() for s in self.slabs], axis=1)

    def constraints(self) -> np.ndarray:
        raw = np.stack([s.constraints_raw() for s in self.slabs])
        red = raw.sum(axis=0)
        red[1::2] = raw[:, 1::2].max(axis=0)
        return combine_raw_norms(red, self.p.ncells)

    def close(self):
        for s in self.slabs:
            s.close()


class DistributedSlab:
    """This rank's slab of a mesh partitioned over torch.distributed ranks (one per GPU; torchrun)."""

    def __init__(self, p, device: str, group=None):
        import torch
        import torch.distributed as dist
        from torch.multiprocessing.reductions import reduce_tensor
        self.torch, self.dist, self.group = torch, dist, group
        self.p = p
        self.rank, self.nranks = dist.get_rank(group), dist.get_world_size(group)
        self.parts = slab_partition(p.nb[2], self.nranks)
        self.sim = Z.Z4c(slab_params(p, self.rank, self.nranks), device=device)
        self.sim.set_partition(p.nb[2], self.parts[self.rank][0])
        self.on_nccl = dist.get_backend(group) == "nccl"
        self._token = torch.zeros(1, device=device)
        # hand every rank the IPC handles of my two buffers; open my neighbours'
        mine = (reduce_tensor(self.sim.state), reduce_tensor(self.sim.work),
                self.sim.state2_ptr() - self.sim.work.data_ptr())
        everyone = [None] * self.nranks
        dist.all_gather_object(everyone, mine, group=group)
        self._peer_tensors = []
        for side, nb in enumerate(slab_neighbours(self.rank, self.nranks, p.bc)):
            if nb is None or nb == self.rank:
                continue
            (f_state, a_state), (f_work, a_work), off2 = everyone[nb]
            st, wk = f_state(*a_state), f_work(*a_work)        # tensors aliasing the neighbour's memory
            self._peer_tensors += [st, wk]
            self.sim.enable_peer(st.device.index)              # another GPU: let this GPU's kernels store into it
            self.sim.set_neighbor(side, st.data_ptr(), wk.data_ptr() + off2, *self.parts[nb])
        self.barrier()

    @property
    def stream(self):
        return self.sim.stream

    def sync(self):
        self.sim.sync()

    def launch_count(self) -> int:
        return self.sim.launch_count()

    def barrier(self):
        """Every slab has finished what it enqueued so far before any slab runs what comes next."""
        torch, dist = self.torch, self.dist
        if self.on_nccl:
            with torch.cuda.stream(self.sim.stream):           # stream-ordered: no host synchronisation
                dist.all_reduce(self._token, group=self.group)
        else:
            torch.cuda.synchronize(self.sim.device)
            dist.barrier(group=self.group)

    def set_initial_data(self, u_slab: np.ndarray):
        self.sim.set_initial_data(u_slab)
        self.barrier()
        self.sim.fill_ghosts()
        self.barrier()

    def step(self, nsteps: int = 1):
        one_kernel = self.sim.effective_mode()[1] == 2
        for _ in range(nsteps):
            for stage in (1, 2, 3, 4):
                if one_kernel:
                    self.sim.stage(stage)
                    self.barrier()
                else:
                    self.sim.stage_rhs(stage)
                    self.barrier()
                    self.sim.stage_update(stage)
                    self.barrier()

    def constraints(self) -> np.ndarray:
        torch, dist = self.torch, self.dist
        raw = torch.from_numpy(self.sim.constraints_raw())
        dev = self.sim.device if self.on_nccl else "cpu"
        sums, maxs = raw[0::2].clone().to(dev), raw[1::2].clone().to(dev)    # contiguous: collectives ignore strides
        dist.all_reduce(sums, op=dist.ReduceOp.SUM, group=self.group)
        dist.all_reduce(maxs, op=dist.ReduceOp.MAX, group=self.group)
        red = np.empty(8)
        red[0::2], red[1::2] = sums.cpu().numpy(), maxs.cpu().numpy()
        return combine_raw_norms(red, self.p.ncells)

    def close(self):
        self.barrier()
        self._peer_tensors.clear()
        self.sim.close()
