#!/usr/bin/env python
"""bench.py -- RT-TDDFT steps/s on B200 (arXiv 2410.09189 time step), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config nano|24k|mid|small|tiny|...] [--impl reference]

A "step" is one pass of the whole hot path (Algorithm 1 lines 10-28: m x [ELDYN, Rho, Vh, XC, Hupdate]) on one
synthetic system.  Default workload: `24k` (104^3 grid, 13,000 orbitals of which 12,000
are occupied, Phi = 117 GB resident: the configuration north_star's metric is quoted on, shaped like the paper's
Ag2160 row of Table 1); one step takes ~24 s, so the default `--steps 3 --warmup 3` run ends in
a few minutes and the driver's `--steps 20 --warmup 5` in ~13.  `--config nano|mid|small|tiny` select the others.
N > 1 (torchrun): ONE system cut into grid slabs over the ranks (the paper's own decomposition, L420-L424; DESIGN
section 10): two NCCL all-reduces per Hamiltonian update, scaling = strong, value = the steps of that one system /
max-over-ranks time.  `--parallel replicas` runs N independent systems instead (weak, no collective).

`--impl reference` times the CPU oracle (oracle/rt_oracle.py, as it stands) on the host cores on a bounded sample
of the same workload; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "RT-TDDFT steps/sec"
UNIT = "steps/s"
SMI_FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={SMI_FIELDS}",
                                       "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, power, reasons = [], None, [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 8:
                continue
            try:
                sm.append(float(parts[0]))
                smax = float(parts[1])
                power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": smax, "reasons": ["no samples"]}
        pmax = max(power)
        load = [c for c, p in zip(sm, power) if p >= 0.5 * pmax] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": smax, "reasons": sorted(reasons),
                "power_w_max": pmax, "samples": len(sm)}


# ------------------------------------------------------------------------------------------------ oracle sample
EIGH_SAMPLE_N = 3000      # largest propagator the bounded oracle sample diagonalises in full (N = 13,000 takes minutes)


def oracle_sample(w, slab_pts, phi_slab=None, seed=0):
    """One bounded sample of the oracle's work for workload `w`: returns a function that runs ONE Hamiltonian update
    of oracle/rt_oracle.py with (i) the density and the projection on a grid slab of `slab_pts` points (all N orbitals),
    (ii) the exact-diagonalisation propagator on the leading n_s x n_s block, n_s = min(N, EIGH_SAMPLE_N), (iii) the
    full-grid Poisson / xc; and the factors that EXTRAPOLATE (i) and (ii) to the whole workload (Ng/slab, (N/n_s)^3)."""
    from oracle import rt_oracle as O
    from paper_2410_09189_b200.workloads import phi_slab_sample
    N, Ng = w.norb, w.ngrid
    rng = np.random.default_rng(seed)
    if phi_slab is None:
        phi_slab = phi_slab_sample(w, slab_pts)
    ns = min(N, EIGH_SAMPLE_N)
    eps = np.sort(rng.uniform(w.eps_range[0], w.eps_range[1], N))
    occ = np.zeros(N)
    occ[: w.nocc] = 2.0
    A = rng.standard_normal((ns, ns)) * 1e-4
    Hbar = np.diag(eps[:ns]) + 0.5 * (A + A.T)
    P0 = np.diag(occ[:ns]).astype(np.complex128)
    ReP = np.diag(occ)
    rho_full = np.abs(rng.standard_normal(Ng)) * (occ.sum() / (Ng * w.dvol))
    rho0_full = rho_full * (1 + 1e-6 * rng.standard_normal(Ng))
    vxc0 = O.vxc_lda(rho0_full)
    VH = np.zeros(Ng)

    def parts():
        t0 = time.perf_counter()
        P1 = O.propagate_eigh(Hbar, P0, w.dt)                       # ELDYN on the n_s block
        t1 = time.perf_counter()
        ReP[:ns, :ns] = P1.real
        rho_s = O.density(phi_slab, ReP)                             # Rho on the slab
        t2 = time.perf_counter()
        vh = O.hartree_mg(VH, rho_full - rho0_full, w.shape, w.h, w.n_vcycles)     # Vh, full grid
        t3 = time.perf_counter()
        dv = vh + O.vxc_lda(rho_full) - vxc0 + O.field_potential(w.shape, w.h, (1e-4, 0, 0))   # XC, full grid
        t4 = time.perf_counter()
        H1 = O.project(phi_slab, dv[:slab_pts] + 0 * rho_s, w.dvol)   # Hupdate on the slab
        t5 = time.perf_counter()
        return {"ELDYN": t1 - t0, "Rho": t2 - t1, "Vh": t3 - t2, "XC": t4 - t3, "Hupdate": t5 - t4}, H1

    return parts, {"grid": Ng / slab_pts, "eldyn": (N / ns) ** 3, "ns": ns}


def oracle_step_seconds(w, parts, scale):
    t, _ = parts()
    per_update = scale["eldyn"] * t["ELDYN"] + t["Vh"] + t["XC"] + scale["grid"] * (t["Rho"] + t["Hupdate"])
    return w.n_hupdates * per_update, t


def sample_text(w, pts, scale):
    return (f"EXTRAPOLATED from a bounded sample: per step {w.n_hupdates} Hamiltonian updates, each = eigh propagator on "
            f"the leading {scale['ns']}^2 block x {scale['eldyn']:.1f} + full-grid Poisson/xc + density & projection on a "
            f"{pts}-point grid slab (all {w.norb} orbitals) x Ng/slab = {scale['grid']:.1f}")


def full_oracle(w):
    from oracle import rt_oracle as O
    from paper_2410_09189_b200.workloads import make_inputs_numpy
    Phi, eps, occ = make_inputs_numpy(w)
    E0 = w.kick if not w.laser else w.E_of_t(0.0)
    return O.RTOracle(w.shape, w.h, Phi, eps, occ, dt=w.dt, E0=E0, n_hupdates=w.n_hupdates, n_vcycles=w.n_vcycles)


def slab_points(w):
    # a few seconds of CPU work per sample: 4 N^2 slab flops per update at ~100 GFLOP/s
    pts = int(2.5e11 / (4.0 * w.norb * w.norb))
    pts = max(1024, min(w.ngrid, pts))
    return (pts // 1024) * 1024 if pts >= 1024 else pts


def threads_used():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count()


# ------------------------------------------------------------------------------------------------ reference arm
def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    big = w.norb * w.ngrid * 8 > 2e9
    times = []
    if big:
        pts = slab_points(w)
        parts, scale = oracle_sample(w, pts, seed=w.seed)
        sample = sample_text(w, pts, scale) + "; Phi slab = the workload generator's raw seeded draw for those points"
        for i in range(args.warmup + args.steps):
            sec, _ = oracle_step_seconds(w, parts, scale)
            if i >= args.warmup:
                times.append(sec)
    else:
        o = full_oracle(w)
        sample = "full oracle steps on the whole workload"
        for i in range(args.warmup + args.steps):
            if w.laser:
                o.set_field(w.E_of_t((i + 1) * w.dt))
            t0 = time.perf_counter()
            o.step(1)
            times.append(time.perf_counter() - t0) if i >= args.warmup else None
    sec = sum(times) / len(times)
    val = 1.0 / sec
    cores = threads_used()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(w, args),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def workload_config(w, args):
    return {"workload": w.name, "grid": list(w.shape), "h_bohr": w.h, "norb": w.norb, "nocc": w.nocc, "dt_au": w.dt,
            "n_hupdates": w.n_hupdates, "n_vcycles": w.n_vcycles, "phi_gb": round(w.norb * w.ngrid * 8 / 1e9, 2),
            "l2": "inputs larger than L2 (Phi streamed twice per Hamiltonian update)" if w.norb * w.ngrid * 8 > 2.5e8
            else "L2 flushed between timed steps is not possible inside a CUDA graph: working set fits L2 (stated)",
            "parallelism": (f"grid slabs over {args.gpus} rank(s), 2 all-reduces per Hamiltonian update"
                            + (", N x N propagator sharded by row blocks (3 all-gathers per update)"
                               if args.gpus > 1 and w.norb >= 2048 else "")
                            if getattr(args, "parallel", "replicas") == "slabs" else
                            "replicas only" if args.gpus > 1 else "single GPU")}


# ------------------------------------------------------------------------------------------------ CUDA arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="24k")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--parallel", default=None, choices=["replicas", "slabs"],
                    help="slabs (default for N > 1) = ONE system cut into grid slabs over the ranks (strong scaling, "
                         "NCCL all-reduces per Hamiltonian update; paper_2410_09189_b200/slab.py); replicas = one "
                         "independent system per rank (weak scaling, no data-path collective)")
    args = ap.parse_args()
    if args.parallel is None:
        args.parallel = "slabs" if args.gpus > 1 or int(os.environ.get("WORLD_SIZE", "1")) > 1 else "replicas"
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup

    from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_device, make_inputs_numpy
    w = WORKLOADS[args.config]
    if args.impl == "reference":
        return run_reference(args, w)

    import torch
    import torch.distributed as dist
    from paper_2410_09189_b200 import replicas
    rank, world, local = replicas.rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the RT-TDDFT path has no CPU fallback")
    torch.cuda.set_device(local)
    slabs = args.parallel == "slabs"
    if world > 1 or slabs:
        if slabs and world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", str(29400 + os.getpid() % 500))
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2410_09189_b200.build import build
    if rank == 0:
        build()
    if world > 1:
        dist.barrier()
    from paper_2410_09189_b200 import binding as B

    # inputs: every rank propagates its own seeded system (replicas; seed offset by rank)
    wr = replicas.replica_workload(w, rank) if not slabs else w
    big = w.norb * w.ngrid * 8 > 2e9
    t_gen = time.perf_counter()
    slab = None
    if slabs:
        from paper_2410_09189_b200 import slab as S
        from paper_2410_09189_b200.workloads import make_inputs_device_slab
        slab = S.slab_partition(w.shape[0], world)[rank]
        comm = S.DistComm()
        nyz = w.shape[1] * w.shape[2]
        if big:
            phi, eps, occ, ortho_err = make_inputs_device_slab(w, slab, rank, comm.all_reduce_sum, device=f"cuda:{local}")
        else:
            Phi, eps, occ = make_inputs_numpy(w)
            phi = torch.from_numpy(np.ascontiguousarray(Phi[:, slab[0] * nyz:(slab[0] + slab[1]) * nyz])).to(f"cuda:{local}")
            ortho_err = float(np.max(np.abs(w.dvol * Phi @ Phi.T - np.eye(w.norb))))
    elif big:
        phi, eps, occ, ortho_err = make_inputs_device(wr, device=f"cuda:{local}")
    else:
        Phi, eps, occ = make_inputs_numpy(wr)
        phi = torch.from_numpy(Phi).to(f"cuda:{local}")
        ortho_err = float(np.max(np.abs(w.dvol * Phi @ Phi.T - np.eye(w.norb))))
    torch.cuda.synchronize()
    torch.cuda.empty_cache()          # hand the generator's scratch back to the driver: the library allocates with cudaMalloc
    t_gen = time.perf_counter() - t_gen

    stream = torch.cuda.Stream(device=local)
    E0 = w.kick if not w.laser else w.E_of_t(0.0)
    with torch.cuda.stream(stream):
        if slabs:
            # past the crossover ("once N exceeds a few thousands") the N x N propagator is sharded too
            shard = dict(prop_shard=(rank, world)) if world > 1 and w.norb >= 2048 else {}
            backend = S.CudaSlabBackend(w.shape, w.h, phi, eps, occ, w.dt, slab, device=local,
                                        stream=stream.cuda_stream, E0=E0, n_hupdates=w.n_hupdates,
                                        n_vcycles=w.n_vcycles, **shard)
            stepper = S.SlabStepper(backend, comm, n_hupdates=w.n_hupdates)
            sim = backend.sim                   # the rt_handle owner: getters, timing and launch counts
            sim.step = stepper.step             # rt_step is not available on a slab handle
        else:
            sim = B.RTTDDFT(w.shape, w.h, phi, eps, occ, w.dt, E0=E0, n_hupdates=w.n_hupdates,
                            n_vcycles=w.n_vcycles, device=local, stream=stream.cuda_stream)
        info = sim.info()
        peak_dmma, peak_dfma = B.rt_probe_fp64_peak(local)

        # stage events inside the timed region when a step is long enough that they cost nothing
        stage_in_timed = w.norb * w.norb * w.ngrid > 1e12 or slabs
        step_no = [0]

        def one_step():
            if w.laser:
                sim.set_field(w.E_of_t((step_no[0] + 1) * w.dt))
            sim.step(1)
            step_no[0] += 1

        for _ in range(args.warmup):
            one_step()
        stream.synchronize()
        if stage_in_timed:
            B.rt_timing_enable(sim.handle, True)
            B.rt_timing_read(sim.handle)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        sampler = ClockSampler(local) if rank == 0 else None
        l0 = B.rt_get_launch_count(sim.handle)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.profiler.start()          # no-op unless run under `ncu --profile-from-start off`
        ev0.record(stream)
        for _ in range(args.steps):
            one_step()
        ev1.record(stream)
        torch.cuda.synchronize()
        torch.cuda.profiler.stop()
        if world > 1:
            dist.barrier()
        ms_total = ev0.elapsed_time(ev1)
        launches = B.rt_get_launch_count(sim.handle) - l0
        clocks = None
        if sampler:
            clocks_how = "nvidia-smi every 200 ms during the timed region"
            if ms_total < 1500.0:
                # the timed region is shorter than a few sampling periods: keep the sampler running over ~1.5 s of the
                # same steps right after it (not timed), so that the clock line describes this workload under load
                t_end = time.perf_counter() + 1.5
                while time.perf_counter() < t_end:
                    for _ in range(max(1, args.steps)):
                        one_step()
                    stream.synchronize()
                clocks_how = ("nvidia-smi every 200 ms over the timed region plus ~1.5 s of the same steps run right "
                              "after it (the timed region alone is shorter than the sampling period)")
            clocks = sampler.stop()
            clocks["sampled"] = clocks_how
        if stage_in_timed:
            stage_ms, stage_calls = B.rt_timing_read(sim.handle)
            B.rt_timing_enable(sim.handle, False)
        else:
            B.rt_timing_enable(sim.handle, True)
            B.rt_timing_read(sim.handle)
            for _ in range(args.steps):
                one_step()
            stage_ms, stage_calls = B.rt_timing_read(sim.handle)
            B.rt_timing_enable(sim.handle, False)

        # end to end through the public API with HOST buffers: field in (pinned host -> device), step, dipole and
        # density out (device -> pinned host), every step
        rho_host = torch.empty(w.ngrid, dtype=torch.float64).pin_memory()
        e_host = torch.zeros(3, dtype=torch.float64).pin_memory()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        # a step of the two largest configs takes seconds: a quarter of the K steps (at least 3) is enough for the wall
        # clock, and keeps the driver's --steps 20 run of the 24k config inside its time limit
        e2e_steps = args.steps if ms_total / args.steps < 1000.0 else min(args.steps, max(3, args.steps // 4))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            E = w.E_of_t((step_no[0] + 1) * w.dt)
            e_host[0], e_host[1], e_host[2] = E
            B._check(sim.handle, B._lib.rt_set_field(sim.handle, e_host.data_ptr()))
            sim.step(1)
            step_no[0] += 1
            mu = sim.dipole()
            B.rt_get_density(sim.handle, rho_host)
        torch.cuda.synchronize()
        e2e_sec = (time.perf_counter() - t0) * args.steps / e2e_steps      # scaled to K steps for the max over ranks
        charge = B.rt_get_charge(sim.handle)

    ms_total, e2e_ms = replicas.max_over_ranks([ms_total, e2e_sec * 1e3], device=f"cuda:{local}")
    if rank != 0:
        sim.close()
        if world > 1 or slabs:
            dist.destroy_process_group()
        return 0

    ms_per_step = ms_total / args.steps
    jobs = 1 if slabs else world                 # slabs: all ranks advance ONE system (strong scaling)
    value = replicas.whole_job_steps_per_s(args.steps, jobs, ms_total)
    e2e_value = replicas.whole_job_steps_per_s(args.steps, jobs, e2e_ms)

    # roofline of the dominant kernel (the stage with the largest share)
    N, Ng = w.norb, w.ngrid
    if slabs:                                    # rank 0's share of the two grid contractions
        Ng = slab[1] * w.shape[1] * w.shape[2]
    alg = {"Hupdate": ("tensor", N * (N + 1.0) * Ng, "a1 projection project_kernel: N(N+1)Ng flop per launch (symmetric output)"),
           "Rho": ("tensor", 1.0 * N * N * Ng, "a5 density density_kernel: N^2 Ng flop per launch (triangular fold)"),
           "ELDYN": (("tensor", (2.0 * (info["exp_order"] // 2 + 1) + 16.0) * N ** 3 / world,
                      "a3+a4 row-sharded: this rank's row block of (q+1) series GEMMs (2N^3 each, no symmetric saving) "
                      "+ U P U^dagger (16N^3), divided by the number of ranks")
                     if slabs and world > 1 and w.norb >= 2048 else
                     ("tensor", ((info["exp_order"] // 2 + 1) + 12.0 - 2.0 * (w.n_hupdates - 1) / w.n_hupdates) * N ** 3,
                      "a3+a4 gemm_abt_tma_kernel: (q+1) symmetric-output series GEMMs (N^3 each) + U P U^dagger "
                      "(2 full dual GEMMs 8N^3 + Hermitian output: Re P1 2N^3 on every update, Im P1 2N^3 on the last "
                      "update of a step only); mean over the m updates")),
           "Vh": ("hbm", 57.0 * w.ngrid * w.n_vcycles, "a7 V-cycles: 57 B/pt/cycle (SURVEY 8d fused-ideal, coarse levels "
                  "included); L2-resident and launch-latency-bound in practice"),
           "XC": ("hbm", 32.0 * w.ngrid, "a8 delta_v_kernel: 32 B/pt")}
    shares = {k: (stage_ms[k] / max(1, stage_calls[k])) for k in stage_ms}
    tot_stage = sum(stage_ms.values())
    dom = max(stage_ms, key=lambda k: stage_ms[k])
    per_kernel = {}
    peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm_peak, hbm_src = 6650.0, "fallback"
    if os.path.exists(peaks_file):
        with open(peaks_file) as f:
            hbm_peak, hbm_src = float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    for k, (bound, work, note) in alg.items():
        if not stage_calls[k]:
            continue
        ms = shares[k]
        if bound == "tensor":
            ach, peak, unit = work / (ms * 1e-3) / 1e12, peak_dmma, "TFLOP/s"
        else:
            ach, peak, unit = work / (ms * 1e-3) / 1e9, hbm_peak, "GB/s"
        per_kernel[k] = {"bound": bound, "ms_per_call": ms, "share": stage_ms[k] / tot_stage if tot_stage else None,
                         "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak, "work": note}
    traffic = None
    tfile = os.path.join(ROOT, "profiles", "roofline_traffic.csv")     # per-launch DRAM bytes from ncu --set full
    if os.path.exists(tfile):
        import csv
        with open(tfile) as f:
            for row in csv.DictReader(f):
                if row["workload"] == w.name and row["stage"] == dom:
                    traffic = float(row["dram_bytes_per_launch"])
    roof = dict(per_kernel[dom])
    roof.update({"kernel": dom, "traffic": traffic,
                 "peak_source": ("FP64 DMMA issue rate measured live by rt_probe_fp64_peak in this run "
                                 f"(DFMA: {peak_dfma:.2f} TFLOP/s)") if roof["bound"] == "tensor" else hbm_src,
                 "timed": "CUDA events around every stage inside the timed region" if stage_in_timed else
                 "CUDA events around every stage in a second pass of K steps (graph bypassed) right after the timed region"})

    # CPU baseline: the oracle as it stands on the host cores, bounded sample
    cpu = None
    if not args.no_cpu_baseline and world == 1:          # the oracle is timed on rank 0 of a one-GPU run only
        cores = threads_used()
        if big:
            pts = slab_points(w)
            slab = phi[:, :pts].contiguous().cpu().numpy()
            parts, scale = oracle_sample(w, pts, phi_slab=slab, seed=w.seed)
            sec, t = oracle_step_seconds(w, parts, scale)
            cpu = {"value": 1.0 / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": (sample_text(w, pts, scale) + "; Phi slab = the first grid points of the SAME Phi; "
                              "measured parts (s): " + ", ".join(f"{k}={v:.2f}" for k, v in t.items()))}
        else:
            o = full_oracle(w)
            n = 0
            t0 = time.perf_counter()
            while n < 3 or (time.perf_counter() - t0 < 10.0 and n < w.nsteps):
                if w.laser:
                    o.set_field(w.E_of_t((n + 1) * w.dt))
                o.step(1)
                n += 1
            sec = (time.perf_counter() - t0) / n
            cpu = {"value": 1.0 / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": f"{n} full oracle steps on the whole workload"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if slabs else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(w, args), "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 24, "d2h_bytes_per_step": 24 + 8 * w.ngrid,
                    "ms_per_step": e2e_ms / args.steps, "steps_timed": e2e_steps},
            "gpu_launches": int(launches), "roofline": roof, "per_kernel": per_kernel, "cpu_baseline": cpu,
            "fp64_peaks_tflops": {"dmma": peak_dmma, "dfma": peak_dfma}, "lib": info,
            "checks": {"ortho_err": ortho_err, "charge": float(charge[0]), "n_electrons": 2.0 * w.nocc,
                       "induced_charge": float(charge[1]), "dipole": [float(x) for x in mu]},
            "setup_s": {"inputs": t_gen}}
    print(json.dumps(line))
    sim.close()
    if world > 1 or slabs:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
