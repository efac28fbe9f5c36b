"""GPU parity of the closer-to-paper propagation: second Magnus term Omega_2 = dt^2/12 [H0, H1]
(Eq. 13) and density-matrix propagation in a NON-orthogonal basis (Eq. 33-38), both run
through the paper's series in its "one multiply + transpose" form (L434-L438), against the oracle's same modes."""
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


def run_pair(gpu, cpu, nsteps):
    mg, mc = [gpu.dipole()], [cpu.dipole()]
    for _ in range(nsteps):
        gpu.step(1)
        cpu.step(1)
        mg.append(gpu.dipole())
        mc.append(cpu.dipole())
        conv = gpu.convergence()
        k = cpu.last_orders[-1]
        assert abs(conv["orders"] - k) <= 1                      # the deciding norm may sit at the threshold
    mg, mc = np.array(mg), np.array(mc)
    assert np.max(np.abs(mc - mc[0])) > 1e-7
    assert np.max(np.abs(mg - mc)) / np.max(np.abs(mc)) < TOL
    assert np.max(np.abs(gpu.density() - cpu.density())) / np.max(np.abs(cpu.density())) < TOL
    assert np.max(np.abs(gpu.pmatrix() - cpu.P0)) < 1e-9
    assert np.max(np.abs(gpu.hmatrix() - cpu.H0)) < 1e-9


@pytest.mark.parametrize("name,nsteps,tma", [("tiny", 8, True), ("ragged", 6, True), ("ragged", 4, False), ("nano_twin", 2, True),
                                             ("24k_twin", 1, True)])
def test_second_magnus_term(B, name, nsteps, tma):
    """magnus_order = 2 against the oracle's series with the same Omega and dP_thrs; 24k_twin (N = 1,625) takes the
    TMA stream-K GEMM through its plain (non-symmetric) tile list, nano_twin the 32 x 32-tile kernels."""
    w = strong_kick(WORKLOADS[name], 0.05)
    Phi, eps, occ = make_inputs_numpy(w)
    kw = dict(dt=w.dt, E0=w.kick, n_hupdates=2, n_vcycles=w.n_vcycles, propagator="commutator", dP_thrs=1e-12)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, magnus=2, tma=tma, **kw)
    cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, magnus=2, **kw)
    run_pair(gpu, cpu, nsteps)
    P = gpu.pmatrix()
    assert np.array_equal(P, P.conj().T)                         # the transpose-add form keeps P exactly Hermitian
    assert abs(np.trace(P).real - occ.sum()) < 1e-10
    gpu.close()
    if name == "tiny":
        # the term is there: the trajectory differs from the first-order one by more than the parity tolerance
        g1 = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, magnus=1, **kw)
        g1.step(nsteps)
        assert np.max(np.abs(g1.pmatrix() - cpu.P0)) > 1e-8
        g1.close()


def nonorthogonal_inputs(w, Phi, eps, occ, seed, strength=0.15):
    rng = np.random.default_rng(seed)
    N = len(eps)
    A = np.eye(N) + strength * rng.standard_normal((N, N)) / np.sqrt(N / 16.0)
    Ai = np.linalg.inv(A)
    return A, np.ascontiguousarray(A @ Phi), A @ np.diag(eps) @ A.T, Ai.T @ np.diag(occ) @ Ai


@pytest.mark.parametrize("name,nsteps,magnus", [("tiny", 8, 1), ("tiny", 5, 2), ("ragged", 5, 1), ("nano_twin", 2, 2)])
def test_nonorthogonal_basis(B, name, nsteps, magnus):
    """Phi_n = A Phi: S = A A^T != 1, ground state handed over as matrices (rt_create_general).  The overlap and its
    Newton-Schulz inverse against the oracle's, the trajectory against the oracle's Eq. 37-38 series in the same basis,
    and -- basis invariance -- against the ORTHONORMAL oracle run."""
    w = strong_kick(WORKLOADS[name], 0.05)
    Phi, eps, occ = make_inputs_numpy(w)
    A, Phi_n, Hks_n, P0_n = nonorthogonal_inputs(w, Phi, eps, occ, 31)
    kw = dict(dt=w.dt, E0=w.kick, n_hupdates=2, n_vcycles=w.n_vcycles, propagator="commutator", dP_thrs=1e-12,
              magnus=magnus, Hks=Hks_n, P0=P0_n, nonorthogonal=True)
    gpu = B.RTTDDFT(w.shape, w.h, Phi_n, eps, None, **kw)
    cpu = O.RTOracle(w.shape, w.h, Phi_n, eps, occ, **kw)
    S, Si = gpu.overlap()
    assert np.max(np.abs(S - cpu.S)) < 1e-12 and np.max(np.abs(S - np.eye(w.norb))) > 0.05
    assert np.max(np.abs(Si - cpu.Sinv)) < 1e-11 * np.max(np.abs(cpu.Sinv))
    assert np.max(np.abs(S @ Si - np.eye(w.norb))) < 1e-12
    run_pair(gpu, cpu, nsteps)
    assert abs(np.trace(gpu.pmatrix() @ S).real - occ.sum()) < 1e-9          # Tr[P S] = N_e (L267)
    ref = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=w.kick, n_hupdates=2, n_vcycles=w.n_vcycles, magnus=magnus)
    ref.step(nsteps)                                                         # exact exponential, orthonormal basis
    assert np.max(np.abs(gpu.dipole() - ref.dipole())) / np.max(np.abs(ref.dipole())) < 1e-8
    assert np.max(np.abs(gpu.density() - ref.density())) / np.max(np.abs(ref.density())) < 1e-8
    assert abs(gpu.energy() - cpu.energy()) < 1e-10 * abs(cpu.energy())      # tr(H_KS P) + grid terms
    gpu.close()


def test_general_mode_argument_checks(B):
    w = WORKLOADS["tiny"]
    Phi, eps, occ = make_inputs_numpy(w)
    with pytest.raises(B.RTError) as ei:
        B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, magnus=2)                 # Taylor mode takes Omega_1 only
    assert ei.value.code == B.RT_EINVAL
    with pytest.raises(B.RTError):
        B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, nonorthogonal=True, propagator="commutator")    # no matrices
    with pytest.raises(B.RTError):
        B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, magnus=3, propagator="commutator")
    # linearly dependent functions: the overlap cannot be inverted
    bad = Phi.copy()
    bad[1] = bad[0]
    with pytest.raises(B.RTError):
        B.RTTDDFT(w.shape, w.h, bad, eps, None, w.dt, propagator="commutator", nonorthogonal=True, Hks=np.diag(eps),
                  P0=np.diag(occ))
    # rt_create_general in an orthonormal basis with diagonal matrices is rt_create
    a = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=(0.05, 0, 0), propagator="commutator")
    b = B.RTTDDFT(w.shape, w.h, Phi, eps, None, w.dt, E0=(0.05, 0, 0), propagator="commutator", Hks=np.diag(eps),
                  P0=np.diag(occ))
    a.step(3)
    b.step(3)
    assert np.array_equal(a.dipole(), b.dipole())
    a.close()
    b.close()


# ------------------------------------------------------------------ PBE and the fourth-order grid operators
@pytest.mark.parametrize("name", ["tiny", "ragged", "small", "odd"])
@pytest.mark.parametrize("order", [2, 4])
def test_stage_vxc_pbe(B, name, order):
    """rt_op_vxc with xc_functional = PBE against oracle.vxc_pbe (gradient pass + divergence pass), on the real rho0 of
    the workload and on a rough positive field spanning five decades (large reduced gradients)."""
    w = WORKLOADS[name]
    Phi, eps, occ = make_inputs_numpy(w)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, xc_functional="pbe", fd_order=order)
    rng = np.random.default_rng(51)
    rho0 = O.density(Phi, np.diag(occ))
    rough = np.exp(rng.uniform(np.log(1e-5), np.log(1.0), w.ngrid))
    for rho in (rho0, rough):
        out = B.rt_op_vxc(gpu.handle, rho, np.empty(w.ngrid))
        ref = O.vxc_pbe(rho, w.shape, w.h, order)
        assert np.max(np.abs(out - ref)) < 1e-11 * np.max(np.abs(ref))
    gpu.close()


@pytest.mark.parametrize("name", ["tiny", "ragged", "small"])
def test_stage_hartree_fourth_order(B, name):
    """rt_op_hartree with fd_order = 4: r = f - A4 u, one 7-point V-cycle on (0, r), u += d, per cycle -- against
    oracle.hartree_mg(order = 4); converged, it reaches the FFT solution of the 13-point operator."""
    w = WORKLOADS[name]
    Phi, eps, occ = make_inputs_numpy(w)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, n_vcycles=w.n_vcycles, fd_order=4)
    rng = np.random.default_rng(52)
    drho = rng.standard_normal(w.ngrid)
    v0 = rng.standard_normal(w.ngrid) * 0.1
    for ncyc in (0, 1, w.n_vcycles):
        vh = B.rt_op_hartree(gpu.handle, v0.copy(), drho, ncyc)
        ref = O.hartree_mg(v0.copy(), drho, w.shape, w.h, ncyc, order=4)
        assert np.max(np.abs(vh - ref)) < 1e-12 * max(1.0, np.max(np.abs(ref)))
    vh = B.rt_op_hartree(gpu.handle, np.zeros(w.ngrid), drho, 18)
    exact = O.spectral_solve_order((4 * np.pi * (drho - drho.mean())).reshape(w.shape), w.h, 4).reshape(-1)
    assert np.max(np.abs(vh - exact)) / np.max(np.abs(exact)) < 1e-8
    gpu.close()


@pytest.mark.parametrize("name,nsteps,xc,order", [("tiny", 20, "pbe", 2), ("tiny", 20, "pbe", 4), ("tiny", 10, "lda", 4),
                                                  ("ragged", 8, "pbe", 4), ("small", 4, "pbe", 4), ("odd", 8, "pbe", 4)])
def test_step_parity_pbe_and_fourth_order(B, name, nsteps, xc, order):
    """The whole time step (Taylor propagator) with the paper's functional and high-order grid operators, 1e-9 gate."""
    w = strong_kick(WORKLOADS[name], 0.1)
    Phi, eps, occ = make_inputs_numpy(w)
    kw = dict(dt=w.dt, E0=w.kick, n_hupdates=2, n_vcycles=w.n_vcycles, xc_functional=xc, fd_order=order)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, **kw)
    cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, **kw)
    mg, mc = [gpu.dipole()], [cpu.dipole()]
    assert abs(gpu.energy() - cpu.energy()) < 1e-11 * abs(cpu.energy())
    for _ in range(nsteps):
        gpu.step(1)
        cpu.step(1)
        mg.append(gpu.dipole())
        mc.append(cpu.dipole())
    mg, mc = np.array(mg), np.array(mc)
    assert np.max(np.abs(mc - mc[0])) > 1e-5
    assert np.max(np.abs(mg - mc)) / np.max(np.abs(mc)) < TOL
    assert np.max(np.abs(gpu.density() - cpu.density())) / np.max(np.abs(cpu.density())) < TOL
    assert np.max(np.abs(gpu.pmatrix() - cpu.P0)) < 1e-9
    assert abs(gpu.energy() - cpu.energy()) < 1e-10 * abs(cpu.energy())
    gpu.close()


def test_everything_the_paper_ran_together(B):
    """PBE + fourth-order operators + second Magnus term + the paper's series with its dynamic dP_thrs / H_thrs loops."""
    w = strong_kick(WORKLOADS["ragged"], 0.05)
    Phi, eps, occ = make_inputs_numpy(w)
    kw = dict(dt=w.dt, E0=w.kick, n_vcycles=w.n_vcycles, xc_functional="pbe", fd_order=4, magnus=2, propagator="commutator",
              dP_thrs=1e-12, H_thrs=1e-8, max_hupdates=12)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, **kw)
    cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, **kw)
    for _ in range(5):
        gpu.step(1)
        cpu.step(1)
        conv = gpu.convergence()
        assert conv["hupdates"] == cpu.last_hupdates or abs(cpu.last_H_err / 1e-8 - 1) < 1e-3
        assert np.max(np.abs(gpu.dipole() - cpu.dipole())) / np.max(np.abs(cpu.dipole())) < TOL
    assert np.max(np.abs(gpu.density() - cpu.density())) / np.max(np.abs(cpu.density())) < TOL
    gpu.close()
