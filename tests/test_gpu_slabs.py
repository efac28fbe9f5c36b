"""GPU parity of the grid-slab mode (include/rt_tddft.h rt_slab_*, paper_2410_09189_b200/slab.py) on ONE GPU.

Every "rank" is a slab handle on cuda:0 driven by its own SlabStepper in a host thread; the all-reduce is a host-side
rendezvous (threading.Barrier) that sums the ranks' exchange buffers with torch ops -- no kernel waits on another
kernel, the ranks' launches simply interleave on the device.  What is checked: slab offsets of the density / dipole
kernels, the partial projection (+ diag(eps) on one rank only), the replicated Poisson / xc stages and the phase
protocol, against the UNSHARDED oracle at the 1e-9 gate, with slabs of unequal size and an odd-sized slab (cp.async
kernels on one rank, TMA kernels on the other)."""
import threading

import numpy as np
import pytest

from oracle import rt_oracle as O
from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy, strong_kick

pytestmark = pytest.mark.gpu

TOL = 1e-9


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2410_09189_b200.build import build
    build()
    from paper_2410_09189_b200 import binding
    return binding


class ThreadComm:
    """SUM all-reduce among `world` host threads that share one GPU."""

    def __init__(self, world):
        import torch
        self.torch, self.world = torch, world
        self.slots = [None] * world
        self.barrier = threading.Barrier(world)
        self.local = threading.local()

    def bind(self, rank):
        self.local.rank = rank

    def all_reduce_sum(self, t):
        self.torch.cuda.synchronize()
        self.slots[self.local.rank] = t
        self.barrier.wait()
        if self.local.rank == 0:
            total = self.slots[0].clone()
            for other in self.slots[1:]:
                total += other
            for s in self.slots:
                s.copy_(total)
            self.torch.cuda.synchronize()
        self.barrier.wait()

    def all_gather_blocks(self, t, block):
        """Rank r's block of its own buffer goes to every rank's buffer (what all_gather_into_tensor does in place)."""
        self.torch.cuda.synchronize()
        self.slots[self.local.rank] = t
        self.barrier.wait()
        if self.local.rank == 0:
            for r, src in enumerate(self.slots):
                for q, dst in enumerate(self.slots):
                    if q != r:
                        dst[r * block:(r + 1) * block].copy_(src[r * block:(r + 1) * block])
            self.torch.cuda.synchronize()
        self.barrier.wait()


def run_sharded(B, w, world, nsteps, laser=False, shard_propagator=False, **kw):
    import torch
    from paper_2410_09189_b200.slab import CudaSlabBackend, SlabStepper, slab_partition
    Phi, eps, occ = make_inputs_numpy(w)
    nyz = w.shape[1] * w.shape[2]
    parts = slab_partition(w.shape[0], world)
    comm = ThreadComm(world)
    results, errors = [None] * world, []

    def rank_main(rank):
        try:
            torch.cuda.set_device(0)
            comm.bind(rank)
            x0, nxl = parts[rank]
            phi_slab = torch.from_numpy(np.ascontiguousarray(Phi[:, x0 * nyz:(x0 + nxl) * nyz])).cuda()
            E0 = w.kick if not laser else w.E_of_t(0.0)
            extra = dict(prop_shard=(rank, world)) if shard_propagator else {}
            backend = CudaSlabBackend(w.shape, w.h, phi_slab, eps, occ, w.dt, (x0, nxl), device=0, E0=E0,
                                      n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles, **extra, **kw)
            sim = SlabStepper(backend, comm, n_hupdates=w.n_hupdates)
            mus = [sim.dipole()]
            for n in range(nsteps):
                if laser:
                    sim.set_field(w.E_of_t((n + 1) * w.dt))
                sim.step(1)
                mus.append(sim.dipole())
            results[rank] = (np.array(mus), sim.density(), backend.sim.pmatrix(), backend.sim.hmatrix(), backend.sim.time,
                             sim.updates, backend.sim.convergence())
            sim.close()
        except BaseException as e:          # noqa: BLE001 -- re-raised in the main thread
            errors.append(e)
            comm.barrier.abort()

    threads = [threading.Thread(target=rank_main, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    if errors:
        raise errors[0]
    return (Phi, eps, occ), results


def oracle_series(w, Phi, eps, occ, nsteps, laser=False):
    E0 = w.kick if not laser else w.E_of_t(0.0)
    cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=E0, n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles)
    mus = [cpu.dipole()]
    for n in range(nsteps):
        if laser:
            cpu.set_field(w.E_of_t((n + 1) * w.dt))
        cpu.step(1)
        mus.append(cpu.dipole())
    return cpu, np.array(mus)


@pytest.mark.parametrize("name,world,nsteps", [("tiny", 2, 10), ("ragged", 3, 8), ("odd", 2, 8), ("tiny", 1, 4)])
def test_slabs_match_unsharded_oracle(B, name, world, nsteps):
    w = strong_kick(WORKLOADS[name], 0.1)
    (Phi, eps, occ), res = run_sharded(B, w, world, nsteps)
    cpu, mu_ref = oracle_series(w, Phi, eps, occ, nsteps)
    assert np.max(np.abs(mu_ref - mu_ref[0])) > 1e-6
    for mus, rho, P, H, t, *_ in res:
        assert np.max(np.abs(mus - mu_ref)) / np.max(np.abs(mu_ref)) < TOL
        assert np.max(np.abs(rho - cpu.density())) / np.max(np.abs(cpu.density())) < TOL
        assert np.max(np.abs(P - cpu.P0)) < 1e-10
        assert np.max(np.abs(H - cpu.H0)) < 1e-10
        assert abs(t - cpu.t) < 1e-12
    for other in res[1:]:                   # replicated state is bit-identical on every rank
        assert np.array_equal(other[1], res[0][1]) and np.array_equal(other[3], res[0][3])


def test_slabs_small_molecule_and_laser(B):
    """64^3 x 128 orbitals in 4 slabs (tile multigrid kernels on the replicated grid), then the laser field path."""
    w = strong_kick(WORKLOADS["small"], 0.1)
    (Phi, eps, occ), res = run_sharded(B, w, 4, 3)
    cpu, mu_ref = oracle_series(w, Phi, eps, occ, 3)
    for mus, rho, *_ in res:
        assert np.max(np.abs(mus - mu_ref)) / np.max(np.abs(mu_ref)) < TOL
        assert np.max(np.abs(rho - cpu.density())) / np.max(np.abs(cpu.density())) < TOL
    import dataclasses
    wl = dataclasses.replace(WORKLOADS["ragged"], kick=(0.0, 0.0, 0.0),
                             laser={"E0": 0.05, "omega": 0.3, "tau": 1.0, "t0": 0.6, "axis": 1})
    (Phi, eps, occ), res = run_sharded(B, wl, 2, 8, laser=True)
    cpu, mu_ref = oracle_series(wl, Phi, eps, occ, 8, laser=True)
    for mus, rho, *_ in res:
        assert np.max(np.abs(mus - mu_ref)) / np.max(np.abs(mu_ref)) < TOL


def test_slab_handle_rejects_whole_grid_entry_points(B):
    w = WORKLOADS["tiny"]
    Phi, eps, occ = make_inputs_numpy(w)
    nyz = w.shape[1] * w.shape[2]
    sim = B.RTTDDFT(w.shape, w.h, np.ascontiguousarray(Phi[:, : 12 * nyz]), eps, occ, w.dt, slab=(0, 12))
    with pytest.raises(B.RTError):
        sim.step(1)
    with pytest.raises(B.RTError):
        B.rt_slab_phase(sim.handle, B.RT_SLAB_PROPAGATE, 0)          # RT_SLAB_INIT has not run
    with pytest.raises(B.RTError):
        B.rt_op_vxc(sim.handle, np.ones(w.ngrid), np.empty(w.ngrid))
    sim.close()
    with pytest.raises(B.RTError):
        B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, slab=(20, 8))   # past the end of the grid
    whole = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt)
    with pytest.raises(B.RTError):
        B.rt_slab_get_buffers(whole.handle)
    whole.close()


@pytest.mark.parametrize("name,world,nsteps", [("24k_twin", 2, 2), ("24k_twin", 3, 1), ("nano_twin", 2, 3), ("tiny", 2, 6)])
def test_row_sharded_propagator_matches_unsharded_oracle(B, name, world, nsteps):
    """NEXT(2) second half: the N x N products of a2-a4 computed by row blocks, one block per rank, with
    the three all-gathers of the protocol.  24k_twin: N = 1,625 runs the TMA stream-K GEMM on 13 tile rows (7 + 6, or
    5 + 5 + 3 -- unequal blocks and a ragged last tile); nano_twin: N = 300 on the 32 x 32-tile cp.async kernels
    (3 tile rows: 2 + 1); tiny: ONE tile row, so rank 1 owns nothing and only receives."""
    w = strong_kick(WORKLOADS[name], 0.05)
    (Phi, eps, occ), res = run_sharded(B, w, world, nsteps, shard_propagator=True)
    cpu, mu_ref = oracle_series(w, Phi, eps, occ, nsteps)
    assert np.max(np.abs(mu_ref - mu_ref[0])) > 1e-7
    for mus, rho, P, H, t, *_ in res:
        assert np.max(np.abs(mus - mu_ref)) / np.max(np.abs(mu_ref)) < TOL
        assert np.max(np.abs(rho - cpu.density())) / np.max(np.abs(cpu.density())) < TOL
        assert np.max(np.abs(P - cpu.P0)) < 1e-10 and np.max(np.abs(H - cpu.H0)) < 1e-10
        assert np.array_equal(P, P.conj().T)                    # made exactly Hermitian after the gather
    for other in res[1:]:                                       # every element is computed once: bit-identical copies
        assert np.array_equal(other[2], res[0][2]) and np.array_equal(other[1], res[0][1])


def test_dynamic_hamiltonian_loop_on_slabs(B):
    """Alg. 1 lines 12-13, 24-26 (H_thrs) on a sharded system (round 1 refused H_thrs > 0 on slab handles): every rank
    takes the same number of updates as the oracle's own dynamic loop, with and without the sharded propagator."""
    w = strong_kick(WORKLOADS["ragged"], 0.05)
    Phi, eps, occ = make_inputs_numpy(w)
    nsteps = 4
    cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=w.kick, n_vcycles=w.n_vcycles, H_thrs=1e-7, max_hupdates=12)
    counts, mu_ref = [], [cpu.dipole()]
    for _ in range(nsteps):
        cpu.step(1)
        counts.append(cpu.last_hupdates)
        mu_ref.append(cpu.dipole())
    mu_ref = np.array(mu_ref)
    assert max(counts) > 2 and min(counts) >= 1
    for sharded in (False, True):
        _, res = run_sharded(B, w, 2, nsteps, shard_propagator=sharded, H_thrs=1e-7, max_hupdates=12)
        for mus, rho, P, H, t, updates, conv in res:
            assert updates == sum(counts)
            assert conv["hupdates"] == counts[-1] and abs(conv["H_err"] - cpu.last_H_err) < 1e-11
            assert np.max(np.abs(mus - mu_ref)) / np.max(np.abs(mu_ref)) < TOL
            assert np.max(np.abs(rho - cpu.density())) / np.max(np.abs(cpu.density())) < TOL
