"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (device-resident Phi borrowed
with RT_PHI_DEVICE, TMA kernels, CUDA graph), on sampled outputs the oracle can compute one by one.

A full oracle run is out of reach at these sizes (Phi = 40 GB / 117 GB), so one time step is checked stage by stage
against oracle pieces, each fed with the GPU's own intermediate of the stage before:

    a3/a4  P1 = U P0 U^+           full matrix against oracle.propagate_eigh (nano) / invariants (24k)
    a5     rho                     at sampled grid points against oracle.density on the gathered Phi columns
    a6     dipole, charge          against oracle.dipole of the GPU density (O(Ng))
    a7     V_H                     full grid against oracle.hartree_mg (O(Ng))
    a8     dV                      (inside a1's check) oracle.vxc_lda, full grid
    a1     H1                      a sampled block of rows/columns against oracle.project on those orbitals

With n_hupdates = 1 the first step has Hbar = H0 exactly (H-1 = H0), so every stage's input is
available through the diagnostic getters.  Tolerance: 1e-9 relative (north_star), tighter where the arithmetic allows.
"""
import dataclasses

import numpy as np
import pytest

from oracle import rt_oracle as O
from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_device

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2410_09189_b200.build import build
    build()
    from paper_2410_09189_b200 import binding
    return binding


def relmax(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def require_memory(name, w):
    """A B200 (>= 170 GB) must be able to hold every config: too little free memory there is a failure (something else
    is resident, or a leak), not a reason to drop the two largest configs silently.  Smaller devices skip."""
    import torch
    free, total = torch.cuda.mem_get_info()
    need = w.norb * w.ngrid * 8 * 1.02 + 20 * w.norb * w.norb * 8
    if free < need:
        msg = f"{name}: needs {need / 1e9:.0f} GB of device memory, {free / 1e9:.0f} of {total / 1e9:.0f} GB free"
        if total >= 170e9:
            pytest.fail(msg)
        pytest.skip(msg)


def check_one_step(B, name, kick, full_propagator):
    import torch
    w = dataclasses.replace(WORKLOADS[name], kick=kick, n_hupdates=1)
    require_memory(name, w)
    phi, eps, occ, ortho = make_inputs_device(w, device="cuda:0")
    assert ortho < 1e-12
    N, Ng = w.norb, w.ngrid
    rng = np.random.default_rng(4242)
    sim = B.RTTDDFT(w.shape, w.h, phi, eps, occ, w.dt, E0=w.kick, n_hupdates=1, n_vcycles=w.n_vcycles)
    info = sim.info()
    assert info["tma"] and info["graph"]

    # sampled orbitals (block of H) and grid points (rho); include first/last rows, tile edges and the ragged tail
    rows = np.unique(np.concatenate([[0, 1, 127, 128, N - 129, N - 2, N - 1], rng.integers(0, N, 17)]))
    pts = np.unique(np.concatenate([[0, 1, 127, 128, Ng - 129, Ng - 1], rng.integers(0, Ng, 1500)]))
    phi_rows = phi[torch.as_tensor(rows, device="cuda")].cpu().numpy()              # [nr][Ng]
    phi_cols = phi[:, torch.as_tensor(pts, device="cuda")].cpu().numpy()            # [N][npts]

    # t = 0: H0 = diag(eps) + Proj(E0 . r) on the sampled block; rho0 at the sampled points
    H0 = sim.hmatrix()
    ref = np.diag(eps)[np.ix_(rows, rows)] + O.project(phi_rows, O.field_potential(w.shape, w.h, np.array(w.kick)), w.dvol)
    assert np.max(np.abs(H0[np.ix_(rows, rows)] - ref)) < 1e-12
    rho0 = sim.density().copy()
    assert relmax(rho0[pts], O.density(phi_cols, np.diag(occ))) < 1e-12

    sim.step(1)
    P1 = sim.pmatrix()
    rho = sim.density()
    vh = B.rt_get_vhartree(sim.handle, np.empty(Ng))
    H1 = sim.hmatrix()

    # a3/a4: Hbar = H0 on the first step with m = 1
    P0 = np.diag(occ).astype(np.complex128)
    if full_propagator:
        assert np.max(np.abs(P1 - O.propagate_eigh(H0, P0, w.dt))) < 1e-11
    Pt = torch.from_numpy(P1).cuda()
    assert float((Pt - Pt.conj().T).abs().max()) == 0.0                               # exactly Hermitian
    assert abs(float(torch.trace(Pt).real) - occ.sum()) < 1e-9 * occ.sum()
    assert float((Pt @ Pt - 2 * Pt).abs().max()) < 1e-10                              # idempotent: P^2 = 2P
    del Pt
    if not full_propagator:
        # the paper's own commutator series (Eq. 39: dP^(k) = (-i dt/k)[Hbar, dP^(k-1)]) summed to
        # convergence with the library GEMM on the device -- a host eigendecomposition of 13,000^2 takes too long
        Ht = torch.from_numpy(H0).cuda().to(torch.complex128)
        dP = torch.from_numpy(P0).cuda()
        acc = dP.clone()
        for k in range(1, 60):
            dP = (-1j * w.dt / k) * (Ht @ dP - dP @ Ht)
            acc += dP
            if float(dP.abs().max()) < 1e-15:
                break
        assert k < 59
        assert float((acc - torch.from_numpy(P1).cuda()).abs().max()) < 1e-11
        del Ht, dP, acc
        torch.cuda.empty_cache()

    # a5, a6
    assert relmax(rho[pts], O.density(phi_cols, P1.real)) < 1e-11
    mu = sim.dipole()
    mu_ref = O.dipole(rho, w.shape, w.h)
    scale = w.dvol * np.sum(np.abs(rho)) * max(w.shape) * w.h
    assert np.max(np.abs(mu - mu_ref)) < 1e-13 * scale
    q = B.rt_get_charge(sim.handle)
    assert abs(q[0] - occ.sum()) < 1e-9 * occ.sum() and abs(q[1]) < 1e-9 * occ.sum()

    # a7 (full grid, warm start 0) and a8 + a1 on the sampled block
    vh_ref = O.hartree_mg(np.zeros(Ng), rho - rho0, w.shape, w.h, w.n_vcycles)
    assert np.max(np.abs(vh - vh_ref)) < 1e-11 * max(np.max(np.abs(vh_ref)), 1e-30) + 1e-16
    dv = vh + O.vxc_lda(rho) - O.vxc_lda(rho0)                                        # E(t_1) = 0 (delta kick)
    ref = np.diag(eps)[np.ix_(rows, rows)] + O.project(phi_rows, dv, w.dvol)
    got = H1[np.ix_(rows, rows)]
    assert np.max(np.abs(got - ref)) < 1e-12 * max(1.0, np.max(np.abs(ref)))
    assert np.array_equal(H1, H1.T)
    # the step did something
    assert np.max(np.abs(rho - rho0)) > 0 and np.max(np.abs(P1 - P0)) > 1e-8
    sim.close()
    del phi
    torch.cuda.empty_cache()


def test_nano_full_size_one_step(B):
    """nano: 128^3 grid, 2,400 orbitals (Phi = 40.3 GB), strong kick so that every stage carries signal."""
    check_one_step(B, "nano", (0.05, 0.0, 0.0), full_propagator=True)


def test_24k_full_size_one_step(B):
    """24,000-electron scale: 104^3 grid, 13,000 orbitals (Phi = 117 GB).  The 13,000^2 propagator is checked through
    its invariants (Hermitian, trace, idempotent) and against a restatement of the paper's commutator series (Eq. 39)
    written out in this test with the library GEMM on the device.  That restatement is NOT oracle/ code (the oracle's
    propagate_eigh / propagate_commutator on 13,000^2 complex matrices would take tens of minutes on the host): it is
    an independent second implementation of the same equation; the oracle itself checks this kernel in full at
    N = 2,400 (nano tests) and N = 1,625 (24k_twin)."""
    check_one_step(B, "24k", (0.05, 0.0, 0.0), full_propagator=False)


def test_nano_full_size_second_step_with_two_updates(B):
    """nano at full size with the configuration bench.py times (m = 2): the SECOND time step, where H-1 != H0 so that
    Alg. 1 line 11 extrapolates, and both Hamiltonian updates of the step.  The chain of the step is replayed from the
    checkpoint taken after step 1 with oracle pieces for everything the host can do in seconds (line 11, line 14, the
    exact-diagonalisation propagator at N = 2,400, the full-grid multigrid and xc) and the library's own per-stage entry
    points for the two grid contractions, each of which is checked against the oracle on sampled outputs (a block of
    H1, 1,500 grid points of rho).  The end of the chain must equal the state the real rt_step produced."""
    import torch
    w = dataclasses.replace(WORKLOADS["nano"], kick=(0.05, 0.0, 0.0))
    require_memory("nano", w)
    phi, eps, occ, ortho = make_inputs_device(w, device="cuda:0")
    N, Ng = w.norb, w.ngrid
    sim = B.RTTDDFT(w.shape, w.h, phi, eps, occ, w.dt, E0=w.kick, n_hupdates=2, n_vcycles=w.n_vcycles)
    assert sim.info()["tma"] and sim.info()["graph"]
    rho0 = sim.density().copy()
    vxc0 = O.vxc_lda(rho0)
    rng = np.random.default_rng(99)
    rows = np.unique(np.concatenate([[0, 127, 128, N - 1], rng.integers(0, N, 12)]))
    pts = np.unique(np.concatenate([[0, 127, 128, Ng - 1], rng.integers(0, Ng, 1500)]))
    phi_rows = phi[torch.as_tensor(rows, device="cuda")].cpu().numpy()
    phi_cols = phi[:, torch.as_tensor(pts, device="cuda")].cpu().numpy()

    def unpack(buf):
        d = buf[64:].view(np.float64)
        n2 = N * N
        P = d[:n2].reshape(N, N) + 1j * d[n2:2 * n2].reshape(N, N)
        return P, d[2 * n2:3 * n2].reshape(N, N), d[3 * n2:4 * n2].reshape(N, N), d[4 * n2:4 * n2 + Ng], d[4 * n2 + Ng:4 * n2 + 2 * Ng]

    sim.step(1)
    P0, H0, Hm1, VH, _ = (x.copy() for x in unpack(sim.get_state()))
    assert np.max(np.abs(H0 - Hm1)) > 1e-6                      # the kick is gone: H0 != H-1, line 11 does something
    sim.step(1)
    P2, H2, Hm2, VH2, rho2 = unpack(sim.get_state())
    mu2 = sim.dipole()

    H1 = 2.0 * H0 - Hm1                                          # Alg. 1 line 11
    for it in range(2):
        Hbar = 0.5 * (H0 + H1)                                   # line 14
        P1 = O.propagate_eigh(Hbar, P0, w.dt)                    # Eq. 15, exact diagonalisation
        rho, _ = B.rt_op_density(sim.handle, np.ascontiguousarray(P1.real), np.empty(Ng))
        assert relmax(rho[pts], O.density(phi_cols, P1.real)) < 1e-11
        VH = O.hartree_mg(VH, rho - rho0, w.shape, w.h, w.n_vcycles)
        dv = VH + O.vxc_lda(rho) - vxc0                          # E(t_2) = 0
        dH = B.rt_op_project(sim.handle, dv, np.empty((N, N)))
        assert np.max(np.abs(dH[np.ix_(rows, rows)] - O.project(phi_rows, dv, w.dvol))) < 1e-12
        H1 = np.diag(eps) + dH                                   # line 25
    assert np.max(np.abs(P2 - P1)) < 1e-10
    assert np.max(np.abs(H2 - H1)) < 1e-10 and np.array_equal(Hm2, H0)          # line 28
    assert relmax(rho2, rho) < 1e-10
    assert np.max(np.abs(VH2 - VH)) < 1e-10 * max(np.max(np.abs(VH)), 1e-30) + 1e-15
    assert np.max(np.abs(mu2 - O.dipole(rho, w.shape, w.h))) < 1e-9 * np.max(np.abs(mu2))
    sim.close()
    del phi
    torch.cuda.empty_cache()
