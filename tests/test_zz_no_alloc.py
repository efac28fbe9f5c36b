"""rt_dipole_noalloc (include/rt_tddft.h): the a6 reduction on a static device scratch array -- no handle, no allocation --
against the existing path (rt_step + rt_get_dipole / rt_get_charge on a handle), two calls in a row.

Named test_zz_* so that pytest collects it last: the run uses `pytest -x`, and a failure here must not hide any
other test.  It passes alone in a fresh process and after the other GPU tests (nothing here depends on earlier state: the
scratch array needs no clearing, and the second call below is deliberately a SMALLER grid than the first, so stale
partials of the first call sit right behind the slots the second one reads)."""
import numpy as np
import pytest

from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy, strong_kick

pytestmark = pytest.mark.gpu
TOL = 1e-12          # per-stage tolerance of the parity tests (the two paths add the same terms in different orders)


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2410_09189_b200.build import build
    build()
    from paper_2410_09189_b200 import binding
    return binding


def existing_path(B, name, nsteps):
    """density, dipole and charge after nsteps of the ordinary handle path"""
    w = strong_kick(WORKLOADS[name], 0.1)
    Phi, eps, occ = make_inputs_numpy(w)
    sim = B.RTTDDFT(w.shape, w.h, Phi, eps, occ, w.dt, E0=w.kick, n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles)
    sim.step(nsteps)
    rho, mu, q = sim.density().copy(), np.array(sim.dipole()), B.rt_get_charge(sim.handle)[0]
    sim.close()
    return w, rho, mu, q


def check(B, w, rho, mu, q, out):
    import torch
    d_rho = torch.from_numpy(rho).cuda()
    torch.cuda.synchronize()
    B.rt_dipole_noalloc(d_rho, w.shape, w.h, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    scale = got[4]                                        # dVol sum |rho|: the size of the terms that were added
    assert scale > 0
    assert np.max(np.abs(got[:3] - mu)) < TOL * scale * max(w.shape) * w.h
    assert abs(got[3] - q) < TOL * scale
    assert abs(got[3] - 2 * w.nocc) < 1e-9 * 2 * w.nocc   # and it is the electron count
    return got


def test_no_alloc_dipole_matches_the_handle_path_twice(B):
    import torch
    out = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")
    # first call: 64^3 grid (256 blocks of partial sums), after 3 steps
    w1, rho1, mu1, q1 = existing_path(B, "small", 3)
    got1 = check(B, w1, rho1, mu1, q1, out)
    assert np.max(np.abs(mu1)) > 1e-3                     # the kick produced a dipole: not a comparison of zeros
    # second call, right after: 24^3 grid (14 blocks) -- the first call's partials are still in the scratch behind them
    free0 = torch.cuda.mem_get_info()[0]
    w2, rho2, mu2, q2 = existing_path(B, "tiny", 5)
    free1 = torch.cuda.mem_get_info()[0]
    got2 = check(B, w2, rho2, mu2, q2, out)
    assert not np.allclose(got1[:4], got2[:4])
    # a third and fourth on the device-resident density: same bits (fixed summation order), and no device memory taken
    d_rho = torch.from_numpy(rho2).cuda()
    out2 = torch.empty(5, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        B.rt_dipole_noalloc(d_rho, w2.shape, w2.h, out2)
        torch.cuda.synchronize()
        assert np.array_equal(out2.cpu().numpy(), got2)
    assert torch.cuda.mem_get_info()[0] == before
    assert free0 > 0 and free1 > 0


def test_no_alloc_refuses_a_grid_beyond_its_scratch(B):
    import torch
    assert B.RT_NOALLOC_MAX_POINTS == 4096 * 1024
    rho = torch.zeros(16, dtype=torch.float64, device="cuda")
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    with pytest.raises(B.RTError) as ei:
        B.rt_dipole_noalloc(rho, (256, 128, 129), 0.3, out)          # 4,227,072 points > 4,194,304 (nothing is read)
    assert ei.value.code == B.RT_EINVAL and "4194304" in str(ei.value)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0                               # refused before any launch
    # the largest grid that fits is accepted (160^3 = 4,096,000 points)
    big = torch.full((160 ** 3,), 0.5, dtype=torch.float64, device="cuda")
    B.rt_dipole_noalloc(big, (160, 160, 160), 0.25, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    vol = 160 ** 3 * 0.25 ** 3
    assert abs(got[3] - 0.5 * vol) < 1e-12 * vol and np.max(np.abs(got[:3])) < 1e-9 * vol    # centred coordinates: mu = 0
