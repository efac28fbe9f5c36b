"""Boundary behaviour of the C ABI on a GPU (include/rt_tddft.h): error paths and the contracts the round-1 review
found unenforced.  No oracle arithmetic is needed except where a result is compared."""
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


@pytest.fixture(scope="module")
def tiny():
    w = strong_kick(WORKLOADS["tiny"], 0.1)
    return (w,) + make_inputs_numpy(w)


def test_history_restarts_at_the_restored_level(B, tiny):
    """rt_set_state: the dipole history restarts at the restored time level -- older levels were never recorded in
    this handle and must be refused, not returned as zeros or garbage."""
    w, Phi, eps, occ = tiny
    kw = dict(E0=w.kick, n_vcycles=w.n_vcycles, history=16)
    a = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, **kw)
    a.step(4)
    state = a.get_state()
    b = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, **kw)
    assert np.all(b.dipole_series(0, 1)[0, :3] == b.dipole())
    b.set_state(state)
    for first, n in ((0, 5), (3, 2), (0, 1)):
        with pytest.raises(B.RTError) as ei:
            b.dipole_series(first, n)
        assert ei.value.code == B.RT_EINVAL
    assert np.array_equal(b.dipole_series(4, 1), a.dipole_series(4, 1))
    b.step(3)
    a.step(3)
    assert np.array_equal(b.dipole_series(4, 4), a.dipole_series(4, 4))
    with pytest.raises(B.RTError):
        b.dipole_series(3, 3)
    a.close()
    b.close()


def test_set_field_reads_its_argument_before_returning(B, tiny):
    """rt_set_field from page-locked host memory that is overwritten right after the call (no synchronisation in
    between): the step must see the value that was in the buffer AT the call."""
    import torch
    w, Phi, eps, occ = tiny
    Es = [(0.0, 0.0, 0.02), (0.01, -0.02, 0.0), (0.0, 0.03, 0.01), (0.0, 0.0, 0.0)]
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=(0, 0, 0), n_vcycles=w.n_vcycles, history=8)
    cpu = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=(0, 0, 0), n_vcycles=w.n_vcycles)
    e_host = torch.zeros(3, dtype=torch.float64).pin_memory()
    mus = [cpu.dipole()]
    for E in Es:
        e_host[0], e_host[1], e_host[2] = E
        B._check(gpu.handle, B._lib.rt_set_field(gpu.handle, e_host.data_ptr()))
        e_host.fill_(123.0)                       # poison: a late asynchronous read would pick this up
        gpu.step(1)
        cpu.set_field(E)
        cpu.step(1)
        mus.append(cpu.dipole())
    got = gpu.dipole_series(0, len(Es) + 1)[:, :3]
    assert np.max(np.abs(got - np.array(mus))) < 1e-9 * np.max(np.abs(mus))
    gpu.close()


def test_set_field_beyond_the_series_bound_is_refused(B, tiny):
    """The Taylor degree is fixed at rt_create from the spectral bound with E0 (DESIGN R8): a later field far outside
    that bound must not silently run with a truncated series."""
    w, Phi, eps, occ = tiny
    gpu = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=(0, 0, 0))
    gpu.set_field((0.0, 0.05, 0.0))               # well inside the 0.5 Ha margin
    with pytest.raises(B.RTError) as ei:
        gpu.set_field((50.0, 0.0, 0.0))
    assert ei.value.code == B.RT_EINVAL
    with pytest.raises(B.RTError):
        gpu.set_field((float("nan"), 0.0, 0.0))
    gpu.step(1)                                    # the handle stays usable, the accepted field is still in force
    gpu.close()
    # an explicit order is the caller's responsibility: accepted
    g2 = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=(0, 0, 0), exp_order=31)
    g2.set_field((5.0, 0.0, 0.0))
    g2.close()
    # commutator mode has the same guard on kmax
    g3 = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=(0, 0, 0), propagator="commutator")
    with pytest.raises(B.RTError):
        g3.set_field((50.0, 0.0, 0.0))
    g3.close()


def test_non_finite_values_are_reported_not_declared_converged(B, tiny):
    """A NaN in the state (bad input) must not read as `converged`: fmax-style reductions drop NaN, the library's do
    not.  Dynamic H loop: rt_step returns RT_ENUMERIC; fixed-count commutator mode: rt_get_convergence does."""
    w, Phi, eps, occ = tiny
    bad = eps.copy()
    bad[3] = float("inf")                          # H0 = diag(eps) + ... is then non-finite
    g = B.RTTDDFT(w.shape, w.h, Phi, np.where(np.isfinite(bad), bad, 1e300), occ, w.dt, E0=w.kick,
                  propagator="commutator", H_thrs=1e-7, max_order=20)
    with pytest.raises(B.RTError) as ei:
        g.step(1)
    assert ei.value.code == B.RT_ENUMERIC
    g.close()
    # a series cut off far above dP_thrs is reported too
    g = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=w.kick, propagator="commutator", max_order=2, dP_thrs=1e-14)
    g.step(1)
    with pytest.raises(B.RTError) as ei:
        g.convergence()
    assert ei.value.code == B.RT_ENUMERIC
    g.close()
    g = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=w.kick, propagator="commutator")
    g.step(1)
    c = g.convergence()
    assert 3 < c["orders"] < 40 and c["dP_err"] <= 1e-10
    g.close()


def test_op_propagate_reuses_its_scratch(B, tiny):
    """rt_op_propagate allocates its five N x N scratch matrices once per handle (round 1: cudaMalloc/cudaFree per call)."""
    import torch
    w, Phi, eps, occ = tiny
    g = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt)
    N = w.norb
    H = np.diag(eps)
    P0 = np.diag(occ).astype(complex)
    out = [np.empty((N, N)), np.empty((N, N))]
    B.rt_op_propagate(g.handle, H, np.ascontiguousarray(P0.real), np.ascontiguousarray(P0.imag), *out)
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(20):
        B.rt_op_propagate(g.handle, H, np.ascontiguousarray(P0.real), np.ascontiguousarray(P0.imag), *out)
    assert torch.cuda.mem_get_info()[0] == free0
    assert np.max(np.abs(out[0] - np.diag(occ))) < 1e-14 and np.max(np.abs(out[1])) < 1e-14
    g.close()


def test_spectrum_kick_forms_the_impulse_inside_the_library(B):
    rng = np.random.default_rng(5)
    mu = rng.standard_normal((3, 300)) * 1e-3
    omega = np.linspace(0.1, 1.0, 17)
    dt, E = 0.2, (1e-3, 0.0, 2e-3)
    S = B.rt_spectrum_kick(mu, dt, E, 0.02, omega)
    ref = O.dipole_strength(mu, dt, 0.5 * dt, tuple(0.5 * e * dt for e in E), 0.02, omega)
    assert np.max(np.abs(S - ref)) < 1e-12 * np.max(np.abs(ref))


@pytest.mark.parametrize("N,propagator", [(2400, "taylor"), (5000, "taylor"), (5000, "commutator")])
def test_propagator_is_bit_reproducible_and_accurate(B, N, propagator):
    """The stream-K N x N GEMMs fix their summation order by (N, #SMs) alone: the same propagation, run four times through
    rt_op_propagate, must give the same bits (a round-2 epilogue variant that batched the read-modify-writes of the series
    accumulators failed exactly this at N >= 5,000 while staying within 1e-9 of the right answer), and the right answer:
    U P0 U^dagger with U = exp(-i dt H) from torch.linalg.matrix_exp in complex128 -- a library routine, not oracle/
    (its eigendecomposition of 5,000^2 would take minutes on the host), hence kept apart from the parity tests."""
    import torch
    Ng = 16 ** 3
    gen = torch.Generator(device="cuda").manual_seed(1234 + N)
    phi = torch.randn(N, Ng, dtype=torch.float64, device="cuda", generator=gen) * 0.1     # only sizes the handle
    rng = np.random.default_rng(N)
    eps = np.sort(rng.uniform(-0.5, 0.3, N))
    occ = np.zeros(N)
    occ[: (5 * N) // 6] = 2.0
    # "commutator": the paper's series (Eq. 39), whose GEMMs accumulate P1 += dP^(k) in their epilogues (batched
    # read-modify-writes); it stops at max|dP^(k)| <= 1e-10, so its distance to the exact result is a few 1e-10
    sim = B.RTTDDFT((16, 16, 16), 0.4, phi, eps, occ, 0.2, E0=(0.05, 0.0, 0.0), n_hupdates=1, n_vcycles=1,
                    propagator=propagator)
    tol = 1e-11 if propagator == "taylor" else 2e-9
    assert sim.info()["tma"]
    A = torch.randn(N, N, dtype=torch.float64, device="cuda", generator=gen) * 2e-3
    H = torch.diag(torch.from_numpy(eps).cuda()) + 0.5 * (A + A.T)
    Hh = H.cpu().numpy()
    P0r, P0i = np.diag(occ), np.zeros((N, N))
    outs = []
    for _ in range(4):
        P1r, P1i = np.empty((N, N)), np.empty((N, N))
        B.rt_op_propagate(sim.handle, Hh, P0r, P0i, P1r, P1i)
        outs.append((P1r, P1i))
    for P1r, P1i in outs[1:]:
        assert np.array_equal(P1r, outs[0][0]) and np.array_equal(P1i, outs[0][1])
    U = torch.linalg.matrix_exp((-0.2j) * H.to(torch.complex128))
    Pref = (U * torch.from_numpy(occ).cuda().to(torch.complex128)[None, :]) @ U.conj().T
    P1 = torch.from_numpy(outs[0][0]).cuda() + 1j * torch.from_numpy(outs[0][1]).cuda()
    assert float((P1 - Pref).abs().max()) < tol
    assert float((P1 @ P1 - 2 * P1).abs().max()) < 4 * tol
    sim.close()


def test_paced_kernels_give_the_same_bits_alone_and_beside_another_handle(B):
    """Large systems run the projection and the density with persistent CTAs kept in lock-step by producer pacing
    (gemm_tma.cu).  Pacing only delays TMA issue, so it must not change a bit of the result -- neither from run to run
    (a held-back producer makes the consumer warps poll their barriers: this test is what exposed the divergent-warp race
    fixed by mbar_wait_warp) nor when the peers a CTA waits for are not resident because a second
    handle on another stream holds SMs (bounded waits, then the CTA runs free).  N = 4,096 on a 48 x 48 x 40 grid is the
    smallest shape on which both kernels pace."""
    import threading
    import torch
    N, shape, h, dt = 4096, (48, 48, 40), 0.4, 0.1
    Ng = shape[0] * shape[1] * shape[2]
    gen = torch.Generator(device="cuda").manual_seed(77)
    phi = torch.randn(N, Ng, dtype=torch.float64, device="cuda", generator=gen)
    phi *= 1.0 / (phi.norm(dim=1, keepdim=True) * (h ** 3) ** 0.5)           # normalised, not orthogonal: sizes only
    torch.cuda.synchronize()                  # the handles below run on their own streams
    rng = np.random.default_rng(5)
    eps = np.sort(rng.uniform(-0.5, 0.3, N))
    occ = np.zeros(N)
    occ[: N // 2] = 2.0
    kw = dict(E0=(1e-3, 0.0, 0.0), n_hupdates=2, n_vcycles=2)

    def run(stream, out, key):
        with torch.cuda.stream(stream):
            sim = B.RTTDDFT(shape, h, phi, eps, occ, dt, stream=stream.cuda_stream, **kw)
            info = sim.info()
            sim.step(2)
            out[key] = (sim.density().copy(), sim.hmatrix().copy(), info)
            sim.close()

    res = {}
    run(torch.cuda.Stream(), res, "alone")
    assert res["alone"][2]["paced_projection"] and res["alone"][2]["paced_density"]
    run(torch.cuda.Stream(), res, "again")
    assert np.array_equal(res["again"][0], res["alone"][0]) and np.array_equal(res["again"][1], res["alone"][1])
    threads = [threading.Thread(target=run, args=(torch.cuda.Stream(), res, k)) for k in ("a", "b")]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    for k in ("a", "b"):
        assert np.array_equal(res[k][0], res["alone"][0]) and np.array_equal(res[k][1], res["alone"][1])
    assert np.all(np.isfinite(res["alone"][0])) and np.array_equal(res["alone"][1], res["alone"][1].T)
