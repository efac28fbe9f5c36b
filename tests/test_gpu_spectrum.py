"""GPU parity of the delta-kick driver pieces: the on-device dipole history, the
rt_spectrum kernel and three polarisations propagated together on three streams -- against the oracle."""
import numpy as np
import pytest

from oracle import rt_oracle as O
from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy, strong_kick

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2410_09189_b200.build import build
    build()
    from paper_2410_09189_b200 import binding
    return binding


def test_spectrum_kernel_matches_oracle(B):
    import torch
    rng = np.random.default_rng(31)
    for nt, nw in ((2, 5), (33, 1), (1000, 77), (4097, 130)):
        mu = rng.standard_normal((3, nt)) * 1e-3 + rng.standard_normal((3, 1))
        omega = np.sort(rng.uniform(0.0, 2.0, nw))
        for kappa in ((1e-4, 1e-4, 1e-4), (0.0, 2e-4, 0.0), (1e-4, 0.0, -3e-4)):
            ref = O.dipole_strength(mu, 0.2, 0.1, kappa, 0.01, omega)
            S = B.rt_spectrum(mu, 0.2, 0.1, kappa, 0.01, omega)
            assert np.max(np.abs(S - ref)) <= 1e-12 * max(np.max(np.abs(ref)), 1e-300)
    # device-resident inputs and output
    mu_d, om_d = torch.from_numpy(mu).cuda(), torch.from_numpy(omega).cuda()
    out_d = torch.zeros(len(omega), dtype=torch.float64, device="cuda")
    B.rt_spectrum(mu_d, 0.2, 0.1, (1e-4, 1e-4, 1e-4), 0.01, om_d, out=out_d)
    ref = O.dipole_strength(mu, 0.2, 0.1, (1e-4,) * 3, 0.01, omega)
    assert np.max(np.abs(out_d.cpu().numpy() - ref)) <= 1e-12 * np.max(np.abs(ref))
    with pytest.raises(B.RTError):
        B.rt_spectrum(mu, 0.2, 0.1, (0.0, 0.0, 0.0), 0.01, omega)


@pytest.mark.parametrize("graph", [True, False])
def test_dipole_history_matches_per_step_reads_and_oracle(B, graph):
    w = strong_kick(WORKLOADS["tiny"], 0.1)
    Phi, eps, occ = make_inputs_numpy(w)
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=w.kick, n_vcycles=w.n_vcycles, history=8, graph=graph)
    cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=w.kick, n_vcycles=w.n_vcycles)
    mus = [cpu.dipole()]
    assert np.array_equal(gpu.dipole_series(0, 1)[0, :3], gpu.dipole())
    gpu.step(5)                                   # five steps enqueued back to back, no read in between
    for _ in range(5):
        cpu.step(1)
        mus.append(cpu.dipole())
    series = gpu.dipole_series(0, 6)
    assert np.max(np.abs(series[:, :3] - np.array(mus))) < 1e-9 * np.max(np.abs(mus))
    assert np.max(np.abs(series[:, 3] - 2 * w.nocc)) < 1e-9
    assert np.array_equal(series[5, :3], gpu.dipole())
    gpu.step(7)                                   # 13 levels recorded, the ring keeps the last 8
    for _ in range(7):
        cpu.step(1)
        mus.append(cpu.dipole())
    tail = gpu.dipole_series(5, 8)
    assert np.max(np.abs(tail[:, :3] - np.array(mus[5:]))) < 1e-9 * np.max(np.abs(mus))
    with pytest.raises(B.RTError):
        gpu.dipole_series(4, 2)                   # level 4 has been overwritten
    with pytest.raises(B.RTError):
        gpu.dipole_series(12, 2)                  # level 13 does not exist yet
    gpu.close()
    plain = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt)
    with pytest.raises(B.RTError):
        plain.dipole_series(0, 1)
    plain.close()


def test_three_kicks_together_match_three_oracle_runs(B):
    import torch
    from paper_2410_09189_b200.spectrum import KickTriple
    w = WORKLOADS["ragged"]
    Phi, eps, occ = make_inputs_numpy(w)
    kick, nsteps = 0.02, 12
    phi_d = torch.from_numpy(Phi).cuda()
    trio = KickTriple(w.shape, w.h, phi_d, eps, occ, w.dt, kick=kick, n_vcycles=w.n_vcycles, max_steps=nsteps)
    trio.step(nsteps, chunk=5)
    mu = trio.dipoles()
    ref = np.zeros_like(mu)
    for q in range(3):
        cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=tuple(kick * np.eye(3)[q]), n_vcycles=w.n_vcycles)
        ref[q, 0] = cpu.dipole()[q]
        for n in range(nsteps):
            cpu.step(1)
            ref[q, n + 1] = cpu.dipole()[q]
    assert np.max(np.abs(ref - ref[:, :1])) > 1e-6
    assert np.max(np.abs(mu - ref)) < 1e-9 * np.max(np.abs(ref))
    omega = np.linspace(0.05, 1.5, 40)
    S = trio.spectrum(omega, 0.05)
    S_ref = O.dipole_strength(ref, w.dt, 0.5 * w.dt, (0.5 * kick * w.dt,) * 3, 0.05, omega)
    # the induced dipole is ~1e-3 of the total, so 1e-9 on mu is ~1e-6 on the transform of (mu - mu(0))
    assert np.max(np.abs(S - S_ref)) < 1e-5 * np.max(np.abs(S_ref))
    trio.close()


def test_three_kicks_share_the_gpu_with_the_stream_k_gemm(B):
    """N = 1,625 runs the stream-K N x N GEMM, whose CTAs wait on one another through flags.  Three handles on three
    streams keep all of them in flight at once: the ticket-ordered ranges must make that safe (no deadlock) and the
    results must be bit-identical to the same three runs done one after the other."""
    import torch
    from paper_2410_09189_b200.spectrum import KickTriple
    w = WORKLOADS["24k_twin"]
    Phi, eps, occ = make_inputs_numpy(w)
    phi_d = torch.from_numpy(Phi).cuda()
    kick, nsteps = 0.02, 3
    trio = KickTriple(w.shape, w.h, phi_d, eps, occ, w.dt, kick=kick, n_vcycles=w.n_vcycles, max_steps=nsteps)
    trio.step(nsteps, chunk=1)
    mu = trio.dipoles()
    trio.close()
    for q in range(3):
        one = B.RTTDDFT(w.shape, w.h, phi_d, eps, occ, w.dt, E0=tuple(kick * np.eye(3)[q]), n_vcycles=w.n_vcycles,
                        history=nsteps + 1)
        one.step(nsteps)
        assert np.array_equal(one.dipole_series(0, nsteps + 1)[:, q], mu[q])
        one.close()
    assert np.max(np.abs(mu - mu[:, :1])) > 1e-9
