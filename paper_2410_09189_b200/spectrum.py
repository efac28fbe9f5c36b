"""Photoabsorption spectrum from three delta-kick runs -- argument marshalling around the C ABI.

"Photoabsorption spectra are calculated as a sum of Fourier transforms of mu_x(t), mu_y(t) and mu_z(t) obtained from
three independent simulations with the kick perturbation potential polarized along x, y, and z".
`KickTriple` propagates the three polarisations TOGETHER: three rt_handles that borrow the SAME device-resident Phi
(it is read-only, so no copy: 40 / 117 GB stay single), each on its own CUDA stream, with the dipole history kept on
the device (rt_config.history), so that the host enqueues whole batches of steps without a synchronisation and the
three step graphs overlap on the GPU -- which is what pays at the small configs, where one system cannot fill 148 SMs
(SURVEY NEXT(3)).  The spectrum itself is the library's `rt_spectrum` kernel (DESIGN R16)."""
from __future__ import annotations

import numpy as np

from . import binding as B


class KickTriple:
    def __init__(self, shape, h, phi, eps, occ, dt, kick=1e-3, axes=(0, 1, 2), device=0, max_steps=4096, **kw):
        """phi: CUDA torch tensor [N][Ng] (borrowed by every handle).  kick: field strength E of the end-point sampled
        delta-kick (DESIGN R5): delivered impulse kappa = E dt / 2 at the effective time dt / 2."""
        import torch
        if not (hasattr(phi, "is_cuda") and phi.is_cuda):
            raise ValueError("KickTriple borrows a device-resident Phi: pass a CUDA tensor")
        self.torch, self.device = torch, int(device)
        self.dt, self.kick, self.axes = float(dt), float(kick), tuple(int(a) for a in axes)
        self.streams = [torch.cuda.Stream(device=self.device) for _ in self.axes]
        self.sims = []
        for ax, st in zip(self.axes, self.streams):
            E0 = [0.0, 0.0, 0.0]
            E0[ax] = self.kick
            with torch.cuda.stream(st):
                self.sims.append(B.RTTDDFT(shape, h, phi, eps, occ, dt, E0=tuple(E0), device=self.device,
                                           stream=st.cuda_stream, history=int(max_steps) + 1, **kw))
        self.nsteps = 0

    def step(self, n=1, chunk=16):
        """Enqueue n steps of every polarisation, interleaved in chunks so that the three streams stay fed."""
        done = 0
        while done < n:
            k = min(chunk, n - done)
            for sim in self.sims:
                sim.step(k)
            done += k
        self.nsteps += n

    def dipoles(self) -> np.ndarray:
        """mu[3][nsteps + 1]: row q = component axes[q] of the dipole of the run kicked along axes[q] (rows of unused
        axes stay zero).  One stream synchronisation per run."""
        mu = np.zeros((3, self.nsteps + 1))
        for ax, sim in zip(self.axes, self.sims):
            mu[ax] = sim.dipole_series(0, self.nsteps + 1)[:, ax]
        return mu

    def kick_field(self):
        """E_kick[q] = field strength of the run kicked along q (0 for axes that were not run)."""
        e = [0.0, 0.0, 0.0]
        for ax in self.axes:
            e[ax] = self.kick
        return e

    def spectrum(self, omega, gamma):
        """Dipole strength function S(omega) with exponential damping gamma (a.u.); the delivered impulse and the
        effective kick time of the end-point sampled kick are formed inside the library (rt_spectrum_kick)."""
        return B.rt_spectrum_kick(self.dipoles(), self.dt, self.kick_field(), gamma, omega, device=self.device)

    def synchronize(self):
        for st in self.streams:
            st.synchronize()

    def close(self):
        for sim in self.sims:
            sim.close()
        self.sims = []
