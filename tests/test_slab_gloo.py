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

    def __init__(self, O, shape, h, Phi_slab, eps, occ, dt, slab, E0, n_vcycles):
        import torch
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


def _worker(rank, world, port, q, name, nsteps):
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
                                w.kick, w.n_vcycles)
    sim = SlabStepper(backend, DistComm(), n_hupdates=w.n_hupdates)
    mus = [sim.dipole()]
    for _ in range(nsteps):
        sim.step(1)
        mus.append(sim.dipole())
    q.put((rank, np.array(mus), sim.density(), sim.exchanges, backend.t))
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
    for rank, mus, rho, nex, t in out:
        assert np.max(np.abs(mus - mu_ref)) < 1e-11 * np.max(np.abs(mu_ref))
        assert np.max(np.abs(rho - ref.density())) < 1e-11 * np.max(np.abs(ref.density()))
        assert nex == 2 + 2 * w.n_hupdates * nsteps                        # two exchanges per Hamiltonian update
        assert abs(t - ref.t) < 1e-12
    # every rank ends with bit-identical replicated data (the sum of disjoint slabs is exact)
    assert np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][1], out[1][1])
