"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: it only draws random orbitals, orthonormalises them (library QR / Cholesky), draws
eigenvalues and evaluates the external-field envelope E(t).  It stands in for RMG ground states
(benzene / C60 / chlorophyll / Ag nanorods), which cannot be regenerated here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    shape: tuple          # (nx, ny, nz), z fastest
    h: float              # grid spacing, bohr
    norb: int             # N = N_occ + N_virt
    nocc: int             # doubly occupied orbitals
    eps_range: tuple      # eigenvalues sorted uniform[lo, hi] Ha
    dt: float
    nsteps: int
    n_vcycles: int
    seed: int
    kick: tuple = (0.0, 0.0, 0.0)        # E(t=0) (delta-kick, end-point sampled)
    laser: dict = field(default_factory=dict)   # {"E0","omega","tau","t0","axis"} Gaussian-envelope laser
    orbitals: str = "random"             # "random" | "gaussians"
    n_hupdates: int = 2

    @property
    def ngrid(self) -> int:
        return self.shape[0] * self.shape[1] * self.shape[2]

    @property
    def dvol(self) -> float:
        return self.h ** 3

    def E_of_t(self, t: float):
        """Field at time t.  delta-kick: E(0) = kick, 0 afterwards; laser: E0 exp(-(t-t0)^2/2tau^2) sin(omega t)."""
        if self.laser:
            L = self.laser
            amp = L["E0"] * math.exp(-((t - L["t0"]) ** 2) / (2.0 * L["tau"] ** 2)) * math.sin(L["omega"] * t)
            e = [0.0, 0.0, 0.0]
            e[L["axis"]] = amp
            return tuple(e)
        return tuple(self.kick) if t == 0.0 else (0.0, 0.0, 0.0)


WORKLOADS = {
    "tiny": Workload("tiny", (24, 24, 24), 0.35, 16, 8, (-0.8, 0.2), 0.2, 50, 2, 1001, kick=(1e-3, 0, 0)),
    "small": Workload("small", (64, 64, 64), 0.30, 128, 64, (-1.0, 0.5), 0.1, 1000, 3, 1002, kick=(1e-3, 0, 0)),
    "mid": Workload("mid", (96, 96, 96), 0.30, 512, 256, (-1.0, 0.5), 0.1, 500, 3, 1003,
                    laser={"E0": 5e-3, "omega": 0.1, "tau": 50.0, "t0": 25.0, "axis": 2}, orbitals="gaussians"),
    "nano": Workload("nano", (128, 128, 128), 0.35, 2400, 2000, (-0.5, 0.3), 0.2, 200, 3, 1004, kick=(1e-4, 0, 0)),
    "24k": Workload("24k", (104, 104, 104), 0.40, 13000, 12000, (-0.5, 0.3), 0.2, 20, 3, 1005, kick=(1e-4, 0, 0)),
    # scaled-down twins of identical structure, small enough for a full oracle run
    "nano_twin": Workload("nano_twin", (64, 64, 64), 0.35, 300, 250, (-0.5, 0.3), 0.2, 200, 3, 2004, kick=(1e-4, 0, 0)),
    "24k_twin": Workload("24k_twin", (52, 52, 52), 0.40, 1625, 1500, (-0.5, 0.3), 0.2, 20, 3, 2005, kick=(1e-4, 0, 0)),
    # ragged: odd orbital count, non-cubic grid with three different multigrid depths/coarsest sizes
    "ragged": Workload("ragged", (20, 12, 28), 0.33, 37, 11, (-0.9, 0.4), 0.15, 20, 2, 3001, kick=(2e-3, 1e-3, -1e-3)),
    # odd everything: Ng = 315 is odd (TMA cannot describe Phi -> cp.async kernels), a single multigrid level
    "odd": Workload("odd", (9, 5, 7), 0.4, 10, 3, (-0.7, 0.3), 0.2, 20, 2, 3002, kick=(0.05, -0.02, 0.03)),
}


def strong_kick(w: Workload, amp: float = 0.1) -> Workload:
    """Strong-kick twin of a delta-kick workload (induced/total ~ 4e-4, so the 1e-9 gate sees physics)."""
    k = [0.0, 0.0, 0.0]
    ax = int(np.argmax(np.abs(w.kick))) if any(w.kick) else 0
    k[ax] = amp
    return replace(w, name=w.name + "_strong", kick=tuple(k), laser={})


def eigenvalues_occ(w: Workload):
    rng = np.random.default_rng(w.seed + 7)
    eps = np.sort(rng.uniform(w.eps_range[0], w.eps_range[1], w.norb))
    occ = np.zeros(w.norb)
    occ[: w.nocc] = 2.0
    return eps, occ


def _raw_orbitals_numpy(w: Workload) -> np.ndarray:
    """Un-orthonormalised [Ng][N] columns."""
    rng = np.random.default_rng(w.seed)
    if w.orbitals == "random":
        return rng.standard_normal((w.ngrid, w.norb))
    # sums of 4 Gaussians (sigma = 1.5 bohr) on random centres, minimum-image distance (separable)
    sigma, ng = 1.5, 4
    nx, ny, nz = w.shape
    L = np.array(w.shape, dtype=np.float64) * w.h
    A = np.zeros((w.ngrid, w.norb))
    ax = [np.arange(n) * w.h for n in w.shape]
    for i in range(w.norb):
        acc = np.zeros(w.shape)
        for _g in range(ng):
            c = rng.uniform(0.0, 1.0, 3) * L
            wt = rng.standard_normal()
            g1 = []
            for d in range(3):
                dx = ax[d] - c[d]
                dx -= L[d] * np.round(dx / L[d])
                g1.append(np.exp(-0.5 * (dx / sigma) ** 2))
            acc += wt * g1[0][:, None, None] * g1[1][None, :, None] * g1[2][None, None, :]
        # a little white noise keeps the 512 localised functions well-conditioned before QR
        A[:, i] = acc.reshape(-1) + 1e-3 * rng.standard_normal(w.ngrid)
    return A


def make_inputs_numpy(w: Workload):
    """Phi [N][Ng] float64 with dV sum_r phi_i phi_j = delta_ij (Householder QR, diag R > 0), eps, occ."""
    A = _raw_orbitals_numpy(w)
    Q, R = np.linalg.qr(A)
    Q *= np.sign(np.diag(R))[None, :]
    Phi = np.ascontiguousarray(Q.T) / math.sqrt(w.dvol)
    eps, occ = eigenvalues_occ(w)
    return Phi, eps, occ


def phi_slab_sample(w: Workload, npts: int) -> np.ndarray:
    """[N][npts] slab of orbital values for the bounded CPU-baseline sample of the configs whose Phi only exists on the
    device: the generator's raw seeded draw N(0, 1/(Ng dV)) for those points, before orthonormalisation (which changes
    it by O(sqrt(N/Ng)); the oracle's run time does not depend on the values)."""
    rng = np.random.default_rng(w.seed)
    return rng.standard_normal((w.norb, int(npts))) / math.sqrt(w.ngrid * w.dvol)


def make_inputs_device(w: Workload, device="cuda", tile: int = 16384, passes: int = 2):
    """Large configs: Phi generated and orthonormalised in place on the device (no second copy).

    torch Philox normal with the workload seed, then Cholesky-QR `passes` times:
    G = dV Phi Phi^T (tiled library matmul), L = chol(G), Phi <- L^-1 Phi per grid tile.
    Returns (Phi torch tensor [N][Ng] on device, eps ndarray, occ ndarray, max|dV Phi Phi^T - I|)."""
    import torch
    N, Ng = w.norb, w.ngrid
    gen = torch.Generator(device=device)
    gen.manual_seed(w.seed)
    Phi = torch.empty((N, Ng), dtype=torch.float64, device=device)
    rows = max(1, (1 << 27) // Ng)
    for r0 in range(0, N, rows):
        r1 = min(N, r0 + rows)
        Phi[r0:r1].normal_(generator=gen)
    Phi.mul_(1.0 / math.sqrt(Ng * w.dvol))

    def gram():
        G = torch.zeros((N, N), dtype=torch.float64, device=device)
        for c0 in range(0, Ng, tile):
            blk = Phi[:, c0:c0 + tile]
            G.addmm_(blk, blk.T, alpha=w.dvol)
        return G

    for _ in range(passes):
        G = gram()
        Lc = torch.linalg.cholesky(G)
        del G
        for c0 in range(0, Ng, tile):
            blk = Phi[:, c0:c0 + tile]
            blk.copy_(torch.linalg.solve_triangular(Lc, blk, upper=False))
        del Lc
    G = gram()
    G.diagonal().sub_(1.0)
    err = float(G.abs().max())
    del G
    eps, occ = eigenvalues_occ(w)
    return Phi, eps, occ, err


def make_inputs_device_slab(w: Workload, slab, rank: int, all_reduce_sum, device="cuda", tile: int = 16384,
                            passes: int = 2):
    """Grid-slab version of make_inputs_device: this rank generates and keeps only the x-planes `slab = (x0, n)` of
    Phi ([N][n*ny*nz]); the Gram matrix of the Cholesky-QR passes is summed over ranks with `all_reduce_sum(tensor)`
    (in place), so every rank applies the same L^-1 to its slab.  Philox stream: seed + 1009 * rank."""
    import torch
    N = w.norb
    ngl = slab[1] * w.shape[1] * w.shape[2]
    gen = torch.Generator(device=device)
    gen.manual_seed(w.seed + 1009 * rank)
    Phi = torch.empty((N, ngl), dtype=torch.float64, device=device)
    rows = max(1, (1 << 27) // ngl)
    for r0 in range(0, N, rows):
        Phi[r0:min(N, r0 + rows)].normal_(generator=gen)
    Phi.mul_(1.0 / math.sqrt(w.ngrid * w.dvol))

    def gram():
        G = torch.zeros((N, N), dtype=torch.float64, device=device)
        for c0 in range(0, ngl, tile):
            blk = Phi[:, c0:c0 + tile]
            G.addmm_(blk, blk.T, alpha=w.dvol)
        all_reduce_sum(G)
        return G

    for _ in range(passes):
        G = gram()
        Lc = torch.linalg.cholesky(G)
        del G
        for c0 in range(0, ngl, tile):
            blk = Phi[:, c0:c0 + tile]
            blk.copy_(torch.linalg.solve_triangular(Lc, blk, upper=False))
        del Lc
    G = gram()
    G.diagonal().sub_(1.0)
    err = float(G.abs().max())
    del G
    eps, occ = eigenvalues_occ(w)
    return Phi, eps, occ, err
