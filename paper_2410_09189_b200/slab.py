"""Grid-slab sharding of the RT-TDDFT step over ranks (one process per GPU) -- plumbing only.

The paper's own decomposition: the real-space grid is cut into slabs of x-planes, each rank holds
all N orbitals on its slab.  The two grid contractions are local to a slab -- a5 gives rho on the slab, a1 gives a
partial sum of dH over the slab ("partial sums ... followed by a reduction", L424) -- while the N x N propagator
(a2-a4) and the O(Ng) Poisson / xc stages (a7, a8) are replicated.  Per Hamiltonian update there are exactly two
exchange steps, both SUM all-reduces of library-owned device buffers (include/rt_tddft.h, rt_slab_*):

    xchg_rho [Ng + 8]   rho on the whole grid (every rank writes its slab, zeros elsewhere -- so the sum is an
                        all-gather that also works for slabs of different sizes and gives bit-identical copies on
                        every rank) followed by the partial dipole / charge sums
    xchg_H   [N * ldn]  partial H1 (the rank owning plane 0 adds diag(eps))

Past the crossover where the replicated N^3 work limits the speed-up ("once N exceeds a few
thousands") the N x N products of a2-a4 are sharded too: every rank owns a block of rows of each product
(`shard_propagator=True`), and three all-gathers of row blocks per Hamiltonian update (Y = X^2; C and S; P1) replace
the replicated GEMMs.  With `H_thrs > 0` the paper's dynamic loop on H (Alg. 1 lines 12-13, 24-26) runs on the sharded
system: the error norm is a max over replicated, bit-identical matrices, so every rank takes the same decision (made
inside the library: rt_slab_more_updates) without an extra collective.

All arithmetic runs in the CUDA library; this module only orders the phases and calls torch.distributed (NCCL over
NVLink/NVSwitch on GPUs).  `SlabStepper` is written against a small backend interface so that the host logic can be
covered on CPU (gloo, world_size 2) with a backend assembled from other pieces in tests/.
"""
from __future__ import annotations

import numpy as np


def slab_partition(nx: int, world: int):
    """Contiguous x-plane ranges [(x0, n), ...], sizes differing by at most one; needs 1 <= world <= nx."""
    if not (1 <= world <= nx):
        raise ValueError(f"cannot cut {nx} x-planes into {world} slabs")
    base, extra = divmod(nx, world)
    out, x0 = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((x0, n))
        x0 += n
    return out


class _DevicePointer:
    """Exposes a raw device allocation through __cuda_array_interface__ so torch can wrap it without a copy."""

    def __init__(self, ptr: int, count: int):
        self.__cuda_array_interface__ = {"shape": (int(count),), "typestr": "<f8", "data": (int(ptr), False),
                                         "version": 2, "strides": None}


def device_view(ptr: int, count: int, device: int):
    import torch
    return torch.as_tensor(_DevicePointer(ptr, count), device=torch.device("cuda", device))


class DistComm:
    """SUM all-reduce through torch.distributed (NCCL on GPUs, gloo in the CPU tests)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group

    def all_reduce_sum(self, t):
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)

    def all_gather_blocks(self, t, block: int):
        """In place: rank r's block t[r*block:(r+1)*block] is sent to every rank (t holds world * block elements or more)."""
        world, rank = self.dist.get_world_size(self.group), self.dist.get_rank(self.group)
        out = t[: world * block]
        mine = out[rank * block:(rank + 1) * block]
        if t.is_cuda:
            self.dist.all_gather_into_tensor(out, mine, group=self.group)      # NCCL, in place
        else:
            parts = [out[r * block:(r + 1) * block] if r != rank else mine.clone() for r in range(world)]
            self.dist.all_gather(parts, mine.clone(), group=self.group)        # gloo: views of `out` receive the blocks


class CudaSlabBackend:
    """One rt_handle created with a slab; the exchange buffers as torch views of the library's device memory."""

    def __init__(self, shape, h, phi_slab, eps, occ, dt, slab, device=0, stream=None, **kw):
        from . import binding as B
        self.B = B
        self.sim = B.RTTDDFT(shape, h, phi_slab, eps, occ, dt, slab=slab, device=device, stream=stream, **kw)
        b = B.rt_slab_get_buffers(self.sim.handle)
        self.xchg_rho = device_view(b.xchg_rho, b.xchg_rho_count, device)
        self.xchg_H = device_view(b.xchg_H, b.xchg_H_count, device)
        self.slab_offset, self.slab_count = int(b.slab_offset), int(b.slab_count)
        s = B.rt_slab_get_shard(self.sim.handle)
        self.prop_shards, self.shard_block = int(s.prop_shards), int(s.block_count)
        # matrices to all-gather after RT_SLAB_PROP_A / _B / _C (include/rt_tddft.h)
        self.gather = {}
        if self.prop_shards > 1:
            view = lambda p: device_view(p, s.total_count, device)
            self.gather = {SlabStepper.PROP_A: [view(s.Y)], SlabStepper.PROP_B: [view(s.C), view(s.S)],
                           SlabStepper.PROP_C: [view(s.P1re), view(s.P1im)]}

    def phase(self, phase: int, it: int = 0):
        self.B.rt_slab_phase(self.sim.handle, phase, it)

    def more_updates(self) -> bool:
        return self.B.rt_slab_more_updates(self.sim.handle)

    def set_field(self, E):
        self.sim.set_field(E)

    def dipole(self):
        return self.sim.dipole()

    def density(self):
        return self.sim.density()

    def close(self):
        self.sim.close()


class SlabStepper:
    """Runs Algorithm 1 lines 10-28 on one rank of a slab-sharded system: phases of the backend interleaved with the
    two all-reduces.  Every rank must call the same methods in the same order."""

    INIT, PROPAGATE, POTENTIAL, SHIFT, PROP_A, PROP_B, PROP_C, PROP_D, CHECK = range(9)   # include/rt_tddft.h RT_SLAB_*

    def __init__(self, backend, comm, n_hupdates: int = 2):
        """n_hupdates is kept for callers of round 1; the number of updates per step is decided by the backend
        (rt_slab_more_updates: fixed count or the H_thrs loop)."""
        self.backend, self.comm, self.m = backend, comm, int(n_hupdates)
        # rt_create left the local rho0 slab and the partial H(t = 0) in the exchange buffers
        comm.all_reduce_sum(backend.xchg_rho)
        comm.all_reduce_sum(backend.xchg_H)
        backend.phase(self.INIT, 0)
        self.exchanges = 2
        self.updates = 0

    def _propagate(self, it):
        b, c = self.backend, self.comm
        if getattr(b, "prop_shards", 1) > 1:                 # row-sharded N x N propagator: three gathers
            for ph in (self.PROP_A, self.PROP_B, self.PROP_C):
                b.phase(ph, it)
                for t in b.gather[ph]:
                    c.all_gather_blocks(t, b.shard_block)
                    self.exchanges += 1
            b.phase(self.PROP_D, it)                         # Hermitian P1, a5 (+ a6 partial sums) on the slab
        else:
            b.phase(self.PROPAGATE, it)                      # a2-a5 (+ a6 partial sums) on the slab

    def step(self, nsteps: int = 1):
        b, c = self.backend, self.comm
        for _ in range(int(nsteps)):
            it = 0
            while True:
                self._propagate(it)
                c.all_reduce_sum(b.xchg_rho)         # exchange 1: rho of the whole grid + dipole / charge sums
                b.phase(self.POTENTIAL, it)          # a7, a8 on the whole grid, a1 over the slab
                c.all_reduce_sum(b.xchg_H)           # exchange 2: H1 = sum of the partial projections
                self.exchanges += 2
                b.phase(self.CHECK, it)              # Alg. 1 lines 12-13, 24: the library decides on another update
                it += 1
                self.updates += 1
                if not b.more_updates():
                    break
            b.phase(self.SHIFT, 0)                   # line 28

    def set_field(self, E):
        self.backend.set_field(E)

    def dipole(self) -> np.ndarray:
        return self.backend.dipole()

    def density(self) -> np.ndarray:
        return self.backend.density()

    def close(self):
        self.backend.close()
