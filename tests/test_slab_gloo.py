"""N > 1 path on CPU: the grid-slab driver (paper_2410_09189_b200/slab.py) under a real world_size-2 gloo group.

The CUDA library cannot run here, so the ranks use a backend assembled from the ORACLE's pieces (test infrastructure)
that follows the same exchange protocol as include/rt_tddft.h rt_slab_* : local rho slab + partial sums in xchg_rho,
partial H (diag(eps) on the rank that owns plane 0) in xchg_H, SUM all-reduces in between.  What is checked is the
host logic: the partition, the order of phases and collectives in SlabStepper, and that the protocol reproduces the
unsharded oracle (dipole series and density) -- including slabs of different sizes."""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_partition():
    sys.path.insert(0, ROOT)
    from paper_2410_09189_b200.slab import slab_partition
    assert slab_partition(24, 1) == [(0, 24)]
    assert slab_partition(20, 3) == [(0, 7), (7, 7), (14, 6)]
    assert slab_partition(9, 2) == [(0, 5), (5, 4)]
    for nx in (5, 24, 104, 128):
        for world in (1, 2, 3, 4, 5):
            p = slab_partition(nx, world)
            assert p[0][0] == 0 and sum(n for _, n in p) == nx
            assert all(p[i][0] + p[i][1] == p[i + 1][0] for i in range(world - 1))
            assert max(n for _, n in p) - min(n for _, n in p) <= 1
    with pytest.raises(ValueError):
        slab_partition(4, 5)
    with pytest.raises(ValueError):
        slab_partition(4, 0)


class OracleSlabBackend:
    """The rt_slab_* protocol with the oracle's functions on a slab of Phi (CPU, torch float64 exchange buffers)."""

    def __init__(self, O, shape, h, Phi_slab, eps, occ, dt, slab, E0, n_vcycles, n_hupdates=2, H_thrs=0.0,
                 max_hupdates=20, shard=None):
        """shard = (rank, world): the N x N propagation is done by row blocks with the three all-gathers of the
        RT_SLAB_PROP_A..D protocol (blocks of ceil(N / world) rows, padded buffers)."""
        import torch
        self.m, self.H_thrs, self.max_hup, self.more, self.last_H_err = n_hupdates, H_thrs, max_hupdates, False, 0.0
        self.O, self.shape, self.h, self.dt, self.n_vc = O, tuple(shape), h, dt, n_vcycles
        self.Phi, self.eps, self.occ = Phi_slab, eps, occ
        self.N = len(eps)
        self.Ng = shape[0] * shape[1] * shape[2]
        self.x0, self.nxl = slab
        nyz = shape[1] * shape[2]
        self.lo, self.hi = self.x0 * nyz, (self.x0 + self.nxl) * nyz
        self.dVol = h ** 3
        self.xchg_rho = torch.zeros(self.Ng + 8, dtype=torch.float64)
        self.xchg_H = torch.zeros(self.N * self.N, dtype=torch.float64)
        self.coords = [O.field_potential(shape, h, e) for e in np.eye(3)]      # x, y, z of every grid point
        self.P0 = np.diag(occ).astype(np.complex128)
        self.E_next = np.zeros(3)
        self.VH = np.zeros(self.Ng)
        self.t = 0.0
        self._put_rho(O.density(self.Phi, np.diag(occ)), None)
        self._put_H(O.field_potential(shape, h, np.asarray(E0, float)))
        self.prop_shards = 1
        if shard:
            self.rank, self.prop_shards = shard
            self.rows = -(-self.N // self.prop_shards)
            self.shard_block = self.rows * self.N
            self.r0, self.r1 = min(self.N, self.rank * self.rows), min(self.N, (self.rank + 1) * self.rows)
            bufs = {k: torch.zeros(self.prop_shards * self.shard_block, dtype=torch.float64) for k in "YCSRI"}
            self.buf = bufs
            self.gather = {4: [bufs["Y"]], 5: [bufs["C"], bufs["S"]], 6: [bufs["R"], bufs["I"]]}

    def _mat(self, key):
        return self.buf[key].numpy()[: self.N * self.N].reshape(self.N, self.N)

    def more_updates(self):
        return self.more

    def _put_rho(self, rho_slab, rho0):
        r = self.xchg_rho.numpy()
        r[:] = 0.0
        r[self.lo:self.hi] = rho_slab
        s = [rho_slab.sum()] + [(c[self.lo:self.hi] * rho_slab).sum() for c in self.coords]
        s.append((rho_slab - rho0[self.lo:self.hi]).sum() if rho0 is not None else rho_slab.sum())
        r[self.Ng:self.Ng + 5] = s

    def _put_H(self, w_full):
        H = self.O.project(self.Phi, w_full[self.lo:self.hi], self.dVol)
        if self.x0 == 0:
            H = H + np.diag(self.eps)
        self.xchg_H.numpy()[:] = H.reshape(-1)

    def phase(self, phase, it=0):
        O = self.O
        rho_buf, H_buf = self.xchg_rho.numpy(), self.xchg_H.numpy().reshape(self.N, self.N)
        if phase == 0:                                             # RT_SLAB_INIT
            self.rho0 = rho_buf[:self.Ng].copy()
            self.vxc0 = O.vxc_lda(self.rho0)
            self.H0, self.Hm1, self.H1 = H_buf.copy(), H_buf.copy(), H_buf.copy()
            rho_buf[self.Ng + 4] = 0.0
        elif phase == 1:                                           # RT_SLAB_PROPAGATE
            if it == 0:
                self.H1 = 2.0 * self.H0 - self.Hm1
            else:
                self.H1 = H_buf.copy()
            self.P1 = O.propagate_eigh(0.5 * (self.H0 + self.H1), self.P0, self.dt)
            self._put_rho(O.density(self.Phi, self.P1.real), self.rho0)
        elif phase == 2:                                           # RT_SLAB_POTENTIAL
            rho = rho_buf[:self.Ng].copy()
            assert abs(rho_buf[self.Ng + 4] - (rho - self.rho0).sum()) < 1e-9
            self.VH = O.hartree_mg(self.VH, rho - self.rho0, self.shape, self.h, self.n_vc)
            dv = self.VH + O.vxc_lda(rho) - self.vxc0 + O.field_potential(self.shape, self.h, self.E_next)
            self._put_H(dv)
        elif phase == 4:                                           # RT_SLAB_PROP_A: line 11 / 14, Y = X^2 on own rows
            self.H1 = 2.0 * self.H0 - self.Hm1 if it == 0 else H_buf.copy()
            self.X = self.dt * 0.5 * (self.H0 + self.H1)
            for k in "YCSRI":
                self.buf[k].zero_()
            self._mat("Y")[self.r0:self.r1] = (self.X @ self.X)[self.r0:self.r1]
        elif phase == 5:                                           # RT_SLAB_PROP_B: U = C - i S on own rows
            assert np.allclose(self._mat("Y"), self.X @ self.X, rtol=0, atol=1e-13)      # the gather delivered all blocks
            U = O.propagator_eigh(self.X / self.dt, self.dt)
            self._mat("C")[self.r0:self.r1] = U.real[self.r0:self.r1]
            self._mat("S")[self.r0:self.r1] = -U.imag[self.r0:self.r1]
        elif phase == 6:                                           # RT_SLAB_PROP_C: P1 = U P0 U^+ on own rows
            U = self._mat("C") - 1j * self._mat("S")
            P1 = (U[self.r0:self.r1] @ self.P0) @ U.conj().T
            self._mat("R")[self.r0:self.r1] = P1.real
            self._mat("I")[self.r0:self.r1] = P1.imag
        elif phase == 7:                                           # RT_SLAB_PROP_D: Hermitian P1, density of the slab
            R, I = self._mat("R"), self._mat("I")
            self.P1 = (np.triu(R) + np.triu(R, 1).T) + 1j * (np.triu(I, 1) - np.triu(I, 1).T)
            self._put_rho(O.density(self.Phi, self.P1.real), self.rho0)
        elif phase == 8:                                           # RT_SLAB_CHECK (after the all-reduce of H)
            if self.H_thrs > 0:
                self.last_H_err = float(np.max(np.abs(H_buf - self.H1)))
                self.more = self.last_H_err > self.H_thrs and it + 1 < self.max_hup
            else:
                self.more = it + 1 < self.m
        elif phase == 3:                                           # RT_SLAB_SHIFT
            self.Hm1, self.H0, self.P0 = self.H0, H_buf.copy(), self.P1
            self.t += self.dt
        else:
            raise ValueError(phase)

    def set_field(self, E):
        self.E_next = np.asarray(E, float)

    def dipole(self):
        return self.dVol * self.xchg_rho.numpy()[self.Ng + 1:self.Ng + 4].copy()

    def density(self):
        return self.xchg_rho.numpy()[:self.Ng].copy()

    def close(self):
        pass


def _worker(rank, world, port, q, name, nsteps, shard=False, H_thrs=0.0):
    import torch.distributed as dist
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port), OMP_NUM_THREADS="2")
    sys.path.insert(0, ROOT)
    from oracle import rt_oracle as O
    from paper_2410_09189_b200.slab import DistComm, SlabStepper, slab_partition
    from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy, strong_kick
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = strong_kick(WORKLOADS[name], 0.05)
    Phi, eps, occ = make_inputs_numpy(w)
    x0, nxl = slab_partition(w.shape[0], world)[rank]
    nyz = w.shape[1] * w.shape[2]
    backend = OracleSlabBackend(O, w.shape, w.h, Phi[:, x0 * nyz:(x0 + nxl) * nyz].copy(), eps, occ, w.dt, (x0, nxl),
                                w.kick, w.n_vcycles, n_hupdates=w.n_hupdates, H_thrs=H_thrs, max_hupdates=12,
                                shard=(rank, world) if shard else None)
    sim = SlabStepper(backend, DistComm(), n_hupdates=w.n_hupdates)
    mus = [sim.dipole()]
    for _ in range(nsteps):
        sim.step(1)
        mus.append(sim.dipole())
    q.put((rank, np.array(mus), sim.density(), sim.exchanges, backend.t, sim.updates))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("name,world", [("tiny", 2), ("odd", 2)])
def test_slab_stepper_world2_gloo_matches_unsharded_oracle(name, world):
    sys.path.insert(0, ROOT)
    from oracle import rt_oracle as O
    from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy, strong_kick
    nsteps = 3
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000 + (7 if name == "odd" else 0)
    procs = [ctx.Process(target=_worker, args=(r, world, port, q, name, nsteps)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = strong_kick(WORKLOADS[name], 0.05)
    Phi, eps, occ = make_inputs_numpy(w)
    ref = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=w.kick, n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles)
    mu_ref = [ref.dipole()]
    for _ in range(nsteps):
        ref.step(1)
        mu_ref.append(ref.dipole())
    mu_ref = np.array(mu_ref)
    assert np.max(np.abs(mu_ref - mu_ref[0])) > 1e-6                       # the kick did something
    for rank, mus, rho, nex, t, _ in out:
        assert np.max(np.abs(mus - mu_ref)) < 1e-11 * np.max(np.abs(mu_ref))
        assert np.max(np.abs(rho - ref.density())) < 1e-11 * np.max(np.abs(ref.density()))
        assert nex == 2 + 2 * w.n_hupdates * nsteps                        # two exchanges per Hamiltonian update
        assert abs(t - ref.t) < 1e-12
    # every rank ends with bit-identical replicated data (the sum of disjoint slabs is exact)
    assert np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][1], out[1][1])


def _spawn(world, name, nsteps, **kw):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000 + 11 * len(kw) + (3 if kw.get("shard") else 0)
    procs = [ctx.Process(target=_worker, args=(r, world, port, q, name, nsteps), kwargs=kw) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    return out


def test_sharded_propagator_protocol_world2_gloo():
    """RT_SLAB_PROP_A..D: row blocks of the N x N propagation + three all-gathers (5 buffers) per Hamiltonian update,
    under a real gloo group, against the UNSHARDED oracle.  N = 37 on 2 ranks: blocks of 19 and 18 rows (padded)."""
    sys.path.insert(0, ROOT)
    from oracle import rt_oracle as O
    from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy, strong_kick
    nsteps = 3
    out = _spawn(2, "ragged", nsteps, shard=True)
    w = strong_kick(WORKLOADS["ragged"], 0.05)
    Phi, eps, occ = make_inputs_numpy(w)
    ref = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=w.kick, n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles)
    mu_ref = [ref.dipole()]
    for _ in range(nsteps):
        ref.step(1)
        mu_ref.append(ref.dipole())
    mu_ref = np.array(mu_ref)
    for rank, mus, rho, nex, t, updates in out:
        assert np.max(np.abs(mus - mu_ref)) < 1e-11 * np.max(np.abs(mu_ref))
        assert np.max(np.abs(rho - ref.density())) < 1e-11 * np.max(np.abs(ref.density()))
        assert updates == w.n_hupdates * nsteps
        assert nex == 2 + (2 + 5) * w.n_hupdates * nsteps           # 2 all-reduces + 5 gathered matrices per update
    assert np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][1], out[1][1])


def test_dynamic_h_loop_world2_gloo():
    """H_thrs > 0 on a sharded system: the stepper asks the backend after every update whether Alg. 1 wants another one;
    both ranks must take the oracle's own number of updates."""
    sys.path.insert(0, ROOT)
    from oracle import rt_oracle as O
    from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy, strong_kick
    nsteps = 3
    out = _spawn(2, "tiny", nsteps, H_thrs=1e-7)
    w = strong_kick(WORKLOADS["tiny"], 0.05)
    Phi, eps, occ = make_inputs_numpy(w)
    ref = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=w.kick, n_vcycles=w.n_vcycles, H_thrs=1e-7, max_hupdates=12)
    total = 0
    for _ in range(nsteps):
        ref.step(1)
        total += ref.last_hupdates
    assert total > 2 * nsteps
    for rank, mus, rho, nex, t, updates in out:
        assert updates == total
        assert np.max(np.abs(mus[-1] - ref.dipole())) < 1e-11 * np.max(np.abs(ref.dipole()))
