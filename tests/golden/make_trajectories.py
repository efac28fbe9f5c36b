#!/usr/bin/env python
"""Writes the full-length oracle trajectories that tests/test_gpu_trajectories.py compares the CUDA path with.

    python tests/golden/make_trajectories.py small_weak|small_strong|mid_laser|tiny_weak [--snapshot-every K]

Calls ONLY oracle/rt_oracle.py and the seeded input generator (paper_2410_09189_b200/workloads.py, which holds none of
the method's arithmetic).  Nothing here touches the CUDA path.  A full-length oracle run of `small` (1000 steps) takes
minutes and of `mid` (500 laser steps) hours on the host cores -- too long to repeat inside the GPU test budget, which is
why the oracle's output is stored ("tiny, small, mid: full-length oracle run, full parity").

File format (text): header lines starting with '#', then one line per time level n = 0..nsteps:
    n  mu_x  mu_y  mu_z            (%.17e: round-trip exact)
then a block "rho <index> <value>" for NPTS seeded sample points of the final density, and "rhomax <value>".

`--snapshot-every K`: every K steps the levels written so far plus the density block AT THAT LEVEL are published as a
complete, self-consistent trajectory file (atomic replace), so that an hours-long run of `mid` leaves a usable, shorter
golden file behind whenever it is interrupted; the last snapshot is the full-length file.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

NPTS = 512
CASES = {
    # name: (workload, strong-kick amplitude or None, steps)
    "tiny_weak": ("tiny", None, 50),
    "small_weak": ("small", None, 1000),
    "small_strong": ("small", 0.1, 1000),
    "mid_laser": ("mid", None, 500),
}


def sample_points(ngrid, seed=777):
    return np.sort(np.random.default_rng(seed).choice(ngrid, size=NPTS, replace=False))


def publish(part, out, o, w):
    """levels written so far + the density block of the oracle's CURRENT state -> `out` (atomic)."""
    rho = o.density()
    tmp = out + ".tmp"
    with open(part) as src, open(tmp, "w") as f:
        f.write(src.read())
        for r in sample_points(w.ngrid):
            f.write("rho %d %.17e\n" % (r, rho[r]))
        f.write("rhomax %.17e\n" % np.max(np.abs(rho)))
        f.write("trP %.17e\n" % np.trace(o.P0).real)
    os.replace(tmp, out)


def main():
    name = sys.argv[1]
    every = int(sys.argv[sys.argv.index("--snapshot-every") + 1]) if "--snapshot-every" in sys.argv else 0
    from oracle import rt_oracle as O
    from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy, strong_kick
    wname, amp, nsteps = CASES[name]
    w = WORKLOADS[wname]
    if amp is not None:
        w = strong_kick(w, amp)
    Phi, eps, occ = make_inputs_numpy(w)
    E0 = w.kick if not w.laser else w.E_of_t(0.0)
    o = O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=E0, n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"trajectory_{name}.txt")
    part = out + ".part"
    t0 = time.time()
    with open(part, "w") as f:
        f.write(f"# oracle/rt_oracle.py RTOracle trajectory, case {name}: workload {w.name}, grid {w.shape}, h {w.h}, "
                f"norb {w.norb}, nocc {w.nocc}, dt {w.dt}, E0 {tuple(E0)}, m {w.n_hupdates}, n_vc {w.n_vcycles}, "
                f"laser {w.laser}\n")
        f.write("# written by tests/golden/make_trajectories.py (calls only oracle/ and the seeded input generator)\n")
        f.write(f"# columns: n mu_x mu_y mu_z ; then {NPTS} sampled points of the final density (seed 777)\n")
        mu = o.dipole()
        f.write("0 %.17e %.17e %.17e\n" % tuple(mu))
        for n in range(nsteps):
            if w.laser:
                o.set_field(w.E_of_t((n + 1) * w.dt))
            o.step(1)
            mu = o.dipole()
            f.write("%d %.17e %.17e %.17e\n" % ((n + 1,) + tuple(mu)))
            f.flush()
            if (n + 1) % 10 == 0:
                print(f"{name}: step {n + 1}/{nsteps}, {time.time() - t0:.0f} s", flush=True)
            if every and (n + 1) % every == 0 and n + 1 < nsteps:
                publish(part, out, o, w)
    publish(part, out, o, w)
    os.remove(part)


if __name__ == "__main__":
    main()
