#!/usr/bin/env python
"""Mutation check of the oracle's pins (not collected by pytest; run by hand: `python tests/oracle_mutations.py`).

For every entry below, a copy of oracle/rt_oracle.py with ONE plausible mistake (a dropped term, a wrong sign or
index, a transposed operand) is put in a scratch tree next to the unmodified tests and
`pytest tests/test_oracle_pins.py -x` must FAIL on it.  The table in DESIGN.md section 3 is this script's output.
Calls only oracle/ and tests/ (CPU).
"""
import os
import shutil
import subprocess
import sys
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# (oracle function / Algorithm 1 line, text in rt_oracle.py, replacement)
MUTATIONS = [
    ("step: Alg.1 line 11 predictor", "H1 = 2.0 * self.H0 - self.Hm1", "H1 = self.H0"),
    ("step: Alg.1 line 11 sign", "H1 = 2.0 * self.H0 - self.Hm1", "H1 = 2.0 * self.H0 + self.Hm1"),
    ("step: line 14 midpoint", "Hbar = 0.5 * (self.H0 + H1)", "Hbar = H1"),
    ("step: line 28 shift order", "self.Hm1, self.H0, self.P0 = self.H0, H1, P1", "self.Hm1, self.H0, self.P0 = H1, H1, P1"),
    ("delta_v: E(t_{n+1}).x term", "dv = field_potential(self.shape, self.h, self.E_next)", "dv = 0.0 * field_potential(self.shape, self.h, self.E_next)"),
    ("delta_v: - vxc0", "dv = dv + self._vxc(rho) - self.vxc0", "dv = dv + self._vxc(rho)"),
    ("delta_v: + V_H", "dv = dv + self.VH", "dv = dv - self.VH"),
    ("set_field: stored value", "self.E_next = np.asarray(E, dtype=np.float64).copy()", "self.E_next = 0.5 * np.asarray(E, dtype=np.float64).copy()"),
    ("__init__: H0 holds V(t_0)", "self.H0 = self.Hks + project(", "self.H0 = self.Hks + 0.0 * project("),
    ("field_potential: axis order", "v = E[0] * x[:, None, None] + E[1] * y[None, :, None] + E[2] * z[None, None, :]", "v = E[0] * x[:, None, None] + E[2] * y[None, :, None] + E[1] * z[None, None, :]"),
    ("axis_coords: centring", "- 0.5 * (n - 1)) * h", "- 0.5 * n) * h"),
    ("project: dVol", "return dVol * ((Phi * v[None, :]) @ Phi.T)", "return ((Phi * v[None, :]) @ Phi.T)"),
    ("density: Re P transposed operand", "return np.sum((ReP @ Phi) * Phi, axis=0)", "return np.sum((np.triu(ReP) @ Phi) * Phi, axis=0)"),
    ("dipole: axis", "np.sum(axis_coords(ny, h)[None, :, None] * r3)", "np.sum(axis_coords(ny, h)[None, None, :] * r3)"),
    ("propagator_eigh: sign of i", "np.exp(-1j * w * dt)", "np.exp(+1j * w * dt)"),
    ("propagate_eigh: U P U^+", "return U @ P0 @ U.conj().T", "return U.conj().T @ P0 @ U"),
    ("propagate_commutator: 1/k", "dP = (-1j * dt / k) * (Hbar @ dP - dP @ Hbar)", "dP = (-1j * dt) * (Hbar @ dP - dP @ Hbar)"),
    ("vxc_lda: exchange prefactor", "vx = -np.cbrt(3.0 * r / np.pi)", "vx = -np.cbrt(3.0 * r / (4.0 * np.pi))"),
    ("vxc_lda: 7/6 beta1", "(7.0 / 6.0) * PZ_BETA1", "(7.0 / 3.0) * PZ_BETA1"),
    ("vxc_lda: high-density branch", "((2.0 * PZ_D - PZ_C) / 3.0) * rs[hi]", "((2.0 * PZ_D + PZ_C) / 3.0) * rs[hi]"),
    ("apply_A: sign/diagonal", "return (6.0 * u - nb) / (h * h)", "return (4.0 * u - nb) / (h * h)"),
    ("jacobi_sweep: omega", "return (1.0 - omega) * u + (omega / 6.0) * (h * h * f + nb)", "return (1.0 - omega) * u + (omega / 6.0) * (h * f + nb)"),
    ("restrict: weights", "r = 0.25 * np.roll(r, 1, ax) + 0.5 * r + 0.25 * np.roll(r, -1, ax)", "r = 0.5 * np.roll(r, 1, ax) + 0.5 * r"),
    ("prolong: odd points", "f[tuple(od)] = 0.5 * (e + np.roll(e, -1, ax))", "f[tuple(od)] = e"),
    ("vcycle: V(2,2) -> V(2,1)", "for _ in range(nu2):", "for _ in range(nu2 - 1):"),
    ("vcycle: coarse h", "ec = vcycle(np.zeros_like(fc), fc, 2.0 * h, nu1, nu2, omega)", "ec = vcycle(np.zeros_like(fc), fc, h, nu1, nu2, omega)"),
    ("hartree_mg: 4 pi", "f = 4.0 * np.pi * (drho - np.mean(drho))", "f = 2.0 * np.pi * (drho - np.mean(drho))"),
    ("spectral_solve: zero mode", "uh[0, 0, 0] = 0.0", "uh[0, 0, 0] = fh[0, 0, 0]"),
    ("energy: Hartree 1/2", "e += 0.5 * self.dVol * float(np.sum(drho * self.VH))", "e += self.dVol * float(np.sum(drho * self.VH))"),
    ("magnus_omega: sign of Omega_2 (Eq. 13)", "Om = Om + (dt * dt / 12.0) * (H0 @ H1 - H1 @ H0)", "Om = Om - (dt * dt / 12.0) * (H0 @ H1 - H1 @ H0)"),
    ("magnus_omega: 1/12", "Om = Om + (dt * dt / 12.0) * (H0 @ H1 - H1 @ H0)", "Om = Om + (dt * dt / 6.0) * (H0 @ H1 - H1 @ H0)"),
    ("magnus_omega: S^-1 side (Eq. 36)", "H0, H1 = Sinv @ H0, Sinv @ H1", "H0, H1 = H0 @ Sinv, H1 @ Sinv"),
    ("propagate_omega_series: Omega^dagger", "dP = (Om @ dP + dP @ Om.conj().T) / k", "dP = (Om @ dP + dP @ Om.T) / k"),
    ("propagate_exact_general: back-transform", "P1 = Li.T @ P1 @ Li", "P1 = Li @ P1 @ Li.T"),
    ("pbe_exc: kappa", "PBE_KAPPA = 0.804", "PBE_KAPPA = 0.84"),
    ("pbe_exc: d s^2/d n", "dex_dn = -Cx * n13 * ((4.0 / 3.0) * F - (8.0 / 3.0) * p * dF)", "dex_dn = -Cx * n13 * ((4.0 / 3.0) * F - (4.0 / 3.0) * p * dF)"),
    ("pbe_exc: t^2 prefactor", "du_ds = pi / (16.0 * (3.0 * pi * pi) ** (1.0 / 3.0) * n13 ** 7)", "du_ds = pi / (8.0 * (3.0 * pi * pi) ** (1.0 / 3.0) * n13 ** 7)"),
    ("pbe_exc: dA/d eps", "dA_deps = A * A * ex1 / PBE_BETA", "dA_deps = A * ex1 / PBE_BETA"),
    ("pw92: beta_3", "PW92_B1, PW92_B2, PW92_B3, PW92_B4 = 7.5957, 3.5876, 1.6382, 0.49294", "PW92_B1, PW92_B2, PW92_B3, PW92_B4 = 7.5957, 3.5876, 1.3682, 0.49294"),
    ("vxc_pbe: divergence sign", "v = v - grad_fd(2.0 * ds * g[ax], h, order)[ax]", "v = v + grad_fd(2.0 * ds * g[ax], h, order)[ax]"),
    ("vxc_pbe: factor 2", "v = v - grad_fd(2.0 * ds * g[ax], h, order)[ax]", "v = v - grad_fd(ds * g[ax], h, order)[ax]"),
    ("FD_GRAD: fourth-order weights", "FD_GRAD = {2: (0.5,), 4: (2.0 / 3.0, -1.0 / 12.0)}", "FD_GRAD = {2: (0.5,), 4: (2.0 / 3.0, 1.0 / 12.0)}"),
    ("FD_LAPL: fourth-order weights", "4: (-5.0 / 2.0, (4.0 / 3.0, -1.0 / 12.0))", "4: (-5.0 / 2.0, (4.0 / 3.0, -1.0 / 6.0))"),
    ("hartree_mg order 4: residual operator", "r = f - apply_A_order(u, h, order)", "r = f - apply_A(u, h)"),
    ("dipole_strength: sign", "S[iw] = -(2.0 * w / (len(used) * np.pi)) * acc", "S[iw] = (2.0 * w / (len(used) * np.pi)) * acc"),
    ("delta_v: V_H warm start (R6)", "self.VH = hartree_mg(self.VH, rho - self.rho0", "self.VH = hartree_mg(np.zeros_like(self.VH), rho - self.rho0"),
]

# readings that no pin can see would be listed here so that the output says so explicitly (none since round 2)
EXPECTED_SURVIVORS = []


def run(label, old, new):
    with tempfile.TemporaryDirectory() as tmp:
        for d in ("oracle", "tests", "paper_2410_09189_b200"):
            shutil.copytree(os.path.join(ROOT, d), os.path.join(tmp, d),
                            ignore=shutil.ignore_patterns("*.so", "build", "__pycache__", "csrc"))
        path = os.path.join(tmp, "oracle", "rt_oracle.py")
        src = open(path).read()
        assert src.count(old) >= 1, f"mutation target not found: {label}"
        open(path, "w").write(src.replace(old, new, 1))
        r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_oracle_pins.py", "-x", "-q", "-p", "no:cacheprovider"],
                           cwd=tmp, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        failed = [l.split("::")[1].split(" ")[0] for l in r.stdout.splitlines() if l.startswith("FAILED")]
        return r.returncode != 0, failed


def main():
    bad = 0
    print("| oracle part | mutation | caught by |\n|---|---|---|")
    for label, old, new in MUTATIONS:
        caught, failed = run(label, old, new)
        print(f"| {label} | `{old[:60]}` -> `{new[:60]}` | {failed[0] if caught else '**SURVIVES**'} |", flush=True)
        bad += not caught
    for label, old, new in EXPECTED_SURVIVORS:
        caught, failed = run(label, old, new)
        print(f"| {label} | `{old[:60]}` -> `{new[:60]}` | {failed[0] if caught else 'survives (declared: parity unpinned)'} |", flush=True)
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
