"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on identical seeded inputs.

Tolerance (BASELINE.json north_star): 1e-9 relative, FP64 -- err_mu = max|mu_gpu - mu_cpu| / max|mu_cpu| over the
whole series and err_rho = |rho_gpu - rho_cpu|_inf / |rho_cpu|_inf.  Per-stage tests use tighter, stage-specific
bounds derived from the contraction length.
"""
import dataclasses

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


_cache = {}


def inputs(name):
    if name not in _cache:
        w = WORKLOADS[name]
        _cache[name] = (w,) + make_inputs_numpy(w)
    return _cache[name]


def make_pair(B, w, Phi, eps, occ, **kw):
    args = dict(dt=w.dt, E0=w.kick if not w.laser else w.E_of_t(0.0), n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles)
    args.update(kw)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, **args)
    cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, **args)
    return gpu, cpu


def relmax(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


# ------------------------------------------------------------------ per-stage parity

@pytest.mark.parametrize("name", ["tiny", "ragged", "small"])
def test_stage_project(B, name):
    w, Phi, eps, occ = inputs(name)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt)
    rng = np.random.default_rng(11)
    for v in (np.full(w.ngrid, 0.7), rng.standard_normal(w.ngrid)):
        H = B.rt_op_project(gpu.handle, v, np.empty((w.norb, w.norb)))
        ref = O.project(Phi, v, w.dvol)
        assert np.max(np.abs(H - ref)) < 1e-12 * max(1.0, np.max(np.abs(ref)))
        assert np.array_equal(H, H.T)
    gpu.close()


@pytest.mark.parametrize("name", ["tiny", "ragged", "small"])
def test_stage_density_and_dipole(B, name):
    w, Phi, eps, occ = inputs(name)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt)
    rng = np.random.default_rng(12)
    A = rng.standard_normal((w.norb, w.norb))
    A = A + A.T
    for S in (np.diag(occ), A):
        rho, sums = B.rt_op_density(gpu.handle, np.ascontiguousarray(S), np.empty(w.ngrid))
        ref = O.density(Phi, S)
        assert relmax(rho, ref) < 1e-12
        mu_ref = O.dipole(ref, w.shape, w.h)
        scale = w.dvol * np.sum(np.abs(ref)) * max(w.shape) * w.h
        assert np.max(np.abs(w.dvol * sums[1:4] - mu_ref)) < 1e-13 * scale
        assert abs(sums[0] - ref.sum()) < 1e-12 * np.sum(np.abs(ref))
    gpu.close()


@pytest.mark.parametrize("name", ["tiny", "ragged", "small"])
def test_stage_propagate(B, name):
    w, Phi, eps, occ = inputs(name)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt)
    rng = np.random.default_rng(13)
    N = w.norb
    A = rng.standard_normal((N, N)) * 0.02
    Hbar = np.diag(eps) + 0.5 * (A + A.T)
    Cc = rng.standard_normal((N, w.nocc)) + 1j * rng.standard_normal((N, w.nocc))
    Q, _ = np.linalg.qr(Cc)
    P0 = 2.0 * Q @ Q.conj().T
    P1r, P1i = B.rt_op_propagate(gpu.handle, np.ascontiguousarray(Hbar), np.ascontiguousarray(P0.real),
                                 np.ascontiguousarray(P0.imag), np.empty((N, N)), np.empty((N, N)))
    ref = O.propagate_eigh(Hbar, P0, w.dt)
    P1 = P1r + 1j * P1i
    assert np.max(np.abs(P1 - ref)) < 2e-13
    assert abs(np.trace(P1).real - 2 * w.nocc) < 1e-11
    assert np.max(np.abs(P1 @ P1 - 2 * P1)) < 1e-11
    gpu.close()


@pytest.mark.parametrize("name", ["tiny", "ragged", "small"])
def test_stage_hartree(B, name):
    w, Phi, eps, occ = inputs(name)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, n_vcycles=w.n_vcycles)
    rng = np.random.default_rng(14)
    drho = rng.standard_normal(w.ngrid)
    v0 = rng.standard_normal(w.ngrid) * 0.1
    for ncyc in (0, 1, w.n_vcycles):
        vh = B.rt_op_hartree(gpu.handle, v0.copy(), drho, ncyc)
        ref = O.hartree_mg(v0.copy(), drho, w.shape, w.h, ncyc)
        assert np.max(np.abs(vh - ref)) < 1e-12 * max(1.0, np.max(np.abs(ref)))
    # converged cycles reach the spectral solution of the same stencil
    vh = B.rt_op_hartree(gpu.handle, np.zeros(w.ngrid), drho, 16)
    exact = O.spectral_solve((4 * np.pi * (drho - drho.mean())).reshape(w.shape), w.h).reshape(-1)
    assert relmax(vh, exact) < 1e-8
    gpu.close()


def test_stage_vxc(B):
    w, Phi, eps, occ = inputs("tiny")
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt)
    rng = np.random.default_rng(15)
    rho = np.exp(rng.uniform(np.log(1e-8), np.log(50.0), w.ngrid))
    rho[:6] = [0.0, 1e-31, 1e-30, O.RHO_RS1, np.nextafter(O.RHO_RS1, 1), np.nextafter(O.RHO_RS1, 0)]
    out = B.rt_op_vxc(gpu.handle, rho, np.empty(w.ngrid))
    ref = O.vxc_lda(rho)
    assert np.max(np.abs(out - ref) / np.maximum(1e-300, np.maximum(np.abs(ref), 1e-3))) < 1e-13
    assert out[0] == 0.0 and out[1] == 0.0
    gpu.close()


# ------------------------------------------------------------------ whole-step parity

def run_series(gpu, cpu, w, nsteps, laser=False):
    mu_g, mu_c = [gpu.dipole()], [cpu.dipole()]
    for n in range(nsteps):
        if laser:
            E = w.E_of_t((n + 1) * w.dt)
            gpu.set_field(E)
            cpu.set_field(E)
        gpu.step(1)
        cpu.step(1)
        mu_g.append(gpu.dipole())
        mu_c.append(cpu.dipole())
    return np.array(mu_g), np.array(mu_c)


def check_run(B, gpu, cpu, w, nsteps, laser=False):
    mu_g, mu_c = run_series(gpu, cpu, w, nsteps, laser)
    err_mu = np.max(np.abs(mu_g - mu_c)) / np.max(np.abs(mu_c))
    rho_g, rho_c = gpu.density(), cpu.density()
    err_rho = relmax(rho_g, rho_c)
    P_g = gpu.pmatrix()
    err_P = np.max(np.abs(P_g - cpu.P0))
    assert err_mu < TOL, f"dipole series {err_mu:.3e}"
    assert err_rho < TOL, f"density {err_rho:.3e}"
    assert err_P < 1e-9, f"P {err_P:.3e}"
    assert abs(gpu.time - cpu.t) < 1e-12
    # the run must not be vacuous: something moved
    assert np.max(np.abs(mu_c - mu_c[0])) > 0
    q = B.rt_get_charge(gpu.handle)
    assert abs(q[0] - cpu.occ.sum()) < 1e-9 and abs(q[1]) < 1e-9
    return err_mu, err_rho


@pytest.mark.parametrize("name,nsteps", [("tiny", 50), ("ragged", 20), ("small", 12)])
def test_step_parity_weak_kick(B, name, nsteps):
    w, Phi, eps, occ = inputs(name)
    gpu, cpu = make_pair(B, w, Phi, eps, occ)
    check_run(B, gpu, cpu, w, nsteps)
    gpu.close()


@pytest.mark.parametrize("name,nsteps", [("tiny", 50), ("ragged", 20), ("small", 8)])
def test_step_parity_strong_kick(B, name, nsteps):
    w, Phi, eps, occ = inputs(name)
    ws = strong_kick(w, 0.1)
    gpu, cpu = make_pair(B, ws, Phi, eps, occ)
    mu0 = cpu.dipole().copy()
    check_run(B, gpu, cpu, ws, nsteps)
    assert np.max(np.abs(cpu.dipole() - mu0)) > 1e-5          # induced signal is well above rounding
    gpu.close()


def test_step_parity_scaled_twins(B):
    """Scaled-down twins of the two configs too large for a full oracle run: identical structure
    (random orthonormal orbitals, eps range, occupation ratio, dt, V-cycles, kick), end to end against the oracle.
    nano_twin: 64^3 x 300 orbitals (3 j-tiles, ragged); 24k_twin: 52^3 x 1,625 orbitals (13 j-tiles, 52 -> 26 -> 13)."""
    w, Phi, eps, occ = inputs("nano_twin")
    gpu, cpu = make_pair(B, w, Phi, eps, occ)
    check_run(B, gpu, cpu, w, 6)
    gpu.close()
    _cache.pop("nano_twin")
    w, Phi, eps, occ = inputs("24k_twin")
    ws = strong_kick(w, 0.05)
    gpu, cpu = make_pair(B, ws, Phi, eps, occ)
    assert gpu.info()["mg_levels"] == 3 and gpu.info()["coarsest"] == (13, 13, 13)
    check_run(B, gpu, cpu, ws, 2)
    gpu.close()
    _cache.pop("24k_twin")


def test_step_parity_mid_laser(B):
    """`mid` config as BASELINE.json states it: 96^3 grid, 512 Gaussian-sum orbitals, Gaussian-envelope laser along z
    driven through rt_set_field every step (first 3 of its 500 steps; the oracle needs ~10 s per step)."""
    w, Phi, eps, occ = inputs("mid")
    gpu, cpu = make_pair(B, w, Phi, eps, occ)
    check_run(B, gpu, cpu, w, 3, laser=True)
    gpu.close()
    _cache.pop("mid")


def test_step_parity_laser_set_field(B):
    """rt_set_field path: Gaussian-envelope laser along z (the `mid` config's driver) on the tiny system."""
    w, Phi, eps, occ = inputs("tiny")
    wl = dataclasses.replace(w, kick=(0, 0, 0), laser={"E0": 5e-2, "omega": 0.3, "tau": 2.0, "t0": 2.0, "axis": 2})
    gpu, cpu = make_pair(B, wl, Phi, eps, occ)
    check_run(B, gpu, cpu, wl, 30, laser=True)
    gpu.close()


def test_flags_no_hartree_no_xc_and_no_graph(B):
    w, Phi, eps, occ = inputs("tiny")
    ws = strong_kick(w, 0.05)
    for kw in (dict(hartree=False), dict(xc=False), dict(hartree=False, xc=False)):
        gpu, cpu = make_pair(B, ws, Phi, eps, occ, **kw)
        check_run(B, gpu, cpu, ws, 10)
        gpu.close()
    # graph replay and direct launches give bit-identical results
    g1 = B.RTTDDFT(ws.shape, ws.h, Phi, eps, occ, ws.dt, E0=ws.kick, n_vcycles=2, graph=True)
    g2 = B.RTTDDFT(ws.shape, ws.h, Phi, eps, occ, ws.dt, E0=ws.kick, n_vcycles=2, graph=False)
    g1.step(7)
    g2.step(7)
    assert np.array_equal(g1.dipole(), g2.dipole()) and np.array_equal(g1.density(), g2.density())
    assert g1.info()["graph"] and not g2.info()["graph"]
    g1.close()
    g2.close()


def test_m_and_vcycle_variants(B):
    w, Phi, eps, occ = inputs("tiny")
    ws = strong_kick(w, 0.1)
    for kw in (dict(n_hupdates=1, n_vcycles=1), dict(n_hupdates=3, n_vcycles=4), dict(n_vcycles=0),
               dict(nu_pre=1, nu_post=3), dict(nu_pre=3, nu_post=1, jacobi_omega=0.8)):
        okw = dict(kw)
        if "jacobi_omega" in okw:
            okw["omega"] = okw.pop("jacobi_omega")
        args = dict(dt=ws.dt, E0=ws.kick, n_hupdates=2, n_vcycles=2)
        gpu = B.RTTDDFT(ws.shape, ws.h, Phi, eps, occ, **{**args, **kw})
        cpu = O.RTOracle(ws.shape, ws.h, Phi, eps, occ, **{**args, **okw})
        check_run(B, gpu, cpu, ws, 8)
        gpu.close()


def test_device_phi_borrowed_and_device_outputs(B):
    import torch
    w, Phi, eps, occ = inputs("tiny")
    ws = strong_kick(w, 0.1)
    phi_d = torch.from_numpy(Phi).cuda()
    before = phi_d.clone()
    gpu = B.RTTDDFT(ws.shape, ws.h, phi_d, eps, occ, ws.dt, E0=ws.kick, n_vcycles=2)
    cpu = O.RTOracle(ws.shape, ws.h, Phi, eps, occ, dt=ws.dt, E0=ws.kick, n_vcycles=2)
    gpu.step(5)
    cpu.step(5)
    rho_d = torch.empty(w.ngrid, dtype=torch.float64, device="cuda")
    B.rt_get_density(gpu.handle, rho_d)
    assert relmax(rho_d.cpu().numpy(), cpu.density()) < TOL
    assert torch.equal(phi_d, before)                       # borrowed, never written
    gpu.close()


def test_cp_async_fallback_paths(B):
    """RT_NO_TMA forces the cp.async DMMA kernels; an odd Ng selects them automatically (and has one MG level)."""
    w, Phi, eps, occ = inputs("tiny")
    ws = strong_kick(w, 0.1)
    gpu = B.RTTDDFT(ws.shape, ws.h, Phi, eps, occ, ws.dt, E0=ws.kick, n_vcycles=ws.n_vcycles, tma=False)
    cpu = O.RTOracle(ws.shape, ws.h, Phi, eps, occ, dt=ws.dt, E0=ws.kick, n_vcycles=ws.n_vcycles)
    assert not gpu.info()["tma"]
    check_run(B, gpu, cpu, ws, 10)
    gpu.close()
    w, Phi, eps, occ = inputs("odd")
    gpu, cpu = make_pair(B, w, Phi, eps, occ)
    assert not gpu.info()["tma"] and gpu.info()["mg_levels"] == 1
    check_run(B, gpu, cpu, w, 20)
    gpu.close()
    # and the default path on an even grid does use TMA
    w, Phi, eps, occ = inputs("tiny")
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt)
    assert gpu.info()["tma"]
    gpu.close()


def test_zero_steps_and_initial_state(B):
    w, Phi, eps, occ = inputs("tiny")
    gpu, cpu = make_pair(B, w, Phi, eps, occ)
    gpu.step(0)
    assert gpu.time == 0.0
    assert relmax(gpu.density(), cpu.rho0) < 1e-13
    assert np.max(np.abs(gpu.dipole() - cpu.dipole())) < 1e-13
    assert np.max(np.abs(gpu.hmatrix() - cpu.H0)) < 1e-13
    assert np.array_equal(gpu.pmatrix(), np.diag(occ).astype(complex))
    info = gpu.info()
    assert info["mg_levels"] == 4 and info["coarsest"] == (3, 3, 3) and info["launches_per_step"] > 0
    gpu.close()


def test_energy_diagnostic_matches_oracle_and_is_conserved(B):
    """rt_get_energy against the oracle's energy() along a strong-kick trajectory, then conservation on the GPU over a
    run far longer than the oracle could follow in a test (Figs. 3-4: "no observable energy drift")."""
    w = strong_kick(WORKLOADS["tiny"], 0.1)
    Phi, eps, occ = inputs("tiny")[1:]
    gpu, cpu = make_pair(B, w, Phi, eps, occ, n_vcycles=6)
    assert abs(gpu.energy() - cpu.energy()) < 1e-11 * abs(cpu.energy())
    for _ in range(6):
        gpu.step(1)
        cpu.step(1)
        assert abs(gpu.energy() - cpu.energy()) < 1e-11 * abs(cpu.energy())
    e1 = gpu.energy()
    assert abs(e1 - np.sum(eps * occ)) > 1e-6                    # the kick deposited energy (3e-6 Ha)
    worst = 0.0
    for _ in range(20):
        gpu.step(100)
        worst = max(worst, abs(gpu.energy() - e1))
    assert worst < 2e-9, worst                                   # 2,000 steps, m = 2, 6 V-cycles per solve
    gpu.close()


def test_checkpoint_resume_is_bit_identical(B):
    """rt_get_state / rt_set_state: a run restored into a fresh handle continues exactly like the uninterrupted one."""
    w = strong_kick(WORKLOADS["ragged"], 0.1)
    Phi, eps, occ = inputs("ragged")[1:]
    kw = dict(E0=w.kick, n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles, history=16)
    a = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, **kw)
    a.step(4)
    state = a.get_state()
    a.step(5)
    b = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, **kw)
    b.set_state(state)
    assert abs(b.time - 4 * w.dt) < 1e-12
    assert np.array_equal(b.dipole_series(4, 1)[0], a.dipole_series(4, 1)[0])
    b.step(5)
    assert np.array_equal(a.dipole(), b.dipole()) and np.array_equal(a.density(), b.density())
    assert np.array_equal(a.pmatrix(), b.pmatrix()) and np.array_equal(a.hmatrix(), b.hmatrix())
    assert np.array_equal(a.vhartree(), b.vhartree()) and a.time == b.time
    assert np.array_equal(a.dipole_series(5, 5), b.dipole_series(5, 5))
    # a buffer from a different system is refused and leaves the handle usable
    w2 = WORKLOADS["tiny"]
    Phi2, eps2, occ2 = inputs("tiny")[1:]
    c = B.RTTDDFT(w2.shape, w2.h, Phi2, eps2, occ2, w2.dt)
    with pytest.raises(B.RTError):
        B._check(c.handle, B._lib.rt_set_state(c.handle, state.ctypes.data))
    c.step(1)
    for s in (a, b, c):
        s.close()


@pytest.mark.parametrize("norb", [130, 200, 225, 300, 384, 400])
def test_projection_and_density_tile_classes(B, norb):
    """Orbital counts that exercise every tile class of the a1 plan (full / narrow last column / diagonal; norb = 200 has
    no full tile at all, 225 has a last column of 97 > 96 columns, 384 no ragged tile) and the masked diagonal blocks of
    a5, against the oracle's plain contractions."""
    shape, h = (16, 12, 20), 0.4
    ng = shape[0] * shape[1] * shape[2]
    rng = np.random.default_rng(100 + norb)
    Phi = rng.standard_normal((norb, ng)) / np.sqrt(ng * h ** 3)
    eps = np.sort(rng.uniform(-1.0, 0.5, norb))
    occ = np.zeros(norb)
    occ[: norb // 2] = 2.0
    gpu = B.RTTDDFT(shape, h, Phi, eps, occ, 0.1)
    v = rng.standard_normal(ng)
    H = B.rt_op_project(gpu.handle, v, np.empty((norb, norb)))
    ref = O.project(Phi, v, h ** 3)
    assert np.max(np.abs(H - ref)) < 1e-12 * np.max(np.abs(ref))
    assert np.array_equal(H, H.T)
    S = rng.standard_normal((norb, norb))
    S = S + S.T
    rho = B.rt_op_density(gpu.handle, S, np.empty(ng))
    rho = rho[0] if isinstance(rho, tuple) else rho
    ref = O.density(Phi, S)
    assert np.max(np.abs(rho - ref)) < 1e-12 * np.max(np.abs(ref))
    gpu.close()
