"""Thin ctypes binding of include/rt_tddft.h -- argument marshalling only; every step of the path runs in the
CUDA kernels of librt_tddft.so.  Function names equal the C names.  PyTorch is used by callers for device
memory and streams; this module itself only needs ctypes (+ numpy for host buffers).

There is NO CPU fallback: importing this module raises if the library has not been built
(``python -m paper_2410_09189_b200.build``), and rt_create fails without an sm_100 GPU.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librt_tddft.so")

RT_OK, RT_EINVAL, RT_ENOMEM, RT_ECUDA, RT_ESTATE, RT_ENUMERIC = 0, -1, -2, -3, -4, -5
RT_PHI_DEVICE, RT_NO_HARTREE, RT_NO_XC, RT_NO_GRAPH, RT_NO_TMA, RT_NONORTHOGONAL = 1, 2, 4, 8, 16, 32
RT_XC_LDA_PZ81, RT_XC_PBE = 0, 1
RT_PROP_TAYLOR, RT_PROP_COMMUTATOR = 0, 1
RT_STAGE_NAMES = ("Hupdate", "Rho", "Vh", "ELDYN", "XC")      # Table 1 of the paper, L543-L547
RT_STAGE_COUNT = 5

# every symbol include/rt_tddft.h declares (checked by tests/test_abi.py)
SYMBOLS = (
    "rt_create", "rt_create_general", "rt_get_overlap", "rt_set_field", "rt_step", "rt_get_dipole", "rt_get_density", "rt_get_pmatrix", "rt_get_hmatrix",
    "rt_get_vhartree", "rt_get_time", "rt_get_charge", "rt_get_info", "rt_get_launch_count", "rt_last_error",
    "rt_destroy", "rt_op_project", "rt_op_density", "rt_op_propagate", "rt_op_hartree", "rt_op_vxc",
    "rt_timing_enable", "rt_timing_read", "rt_probe_fp64_peak", "rt_get_convergence",
    "rt_slab_get_buffers", "rt_slab_phase", "rt_slab_get_shard", "rt_slab_more_updates", "rt_get_dipole_series", "rt_spectrum", "rt_spectrum_kick", "rt_get_energy", "rt_state_bytes", "rt_get_state", "rt_set_state",
    "rt_dipole_noalloc",
)

RT_SLAB_INIT, RT_SLAB_PROPAGATE, RT_SLAB_POTENTIAL, RT_SLAB_SHIFT = 0, 1, 2, 3
RT_SLAB_PROP_A, RT_SLAB_PROP_B, RT_SLAB_PROP_C, RT_SLAB_PROP_D, RT_SLAB_CHECK = 4, 5, 6, 7, 8


class rt_config(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("h", C.c_double),
        ("norb", C.c_int32),
        ("dt", C.c_double),
        ("n_hupdates", C.c_int32), ("n_vcycles", C.c_int32),
        ("nu_pre", C.c_int32), ("nu_post", C.c_int32),
        ("jacobi_omega", C.c_double),
        ("exp_order", C.c_int32),
        ("E0", C.c_double * 3),
        ("flags", C.c_uint32),
        ("device", C.c_int32),
        ("stream", C.c_void_p),
        ("propagator", C.c_int32), ("max_order", C.c_int32),
        ("dP_thrs", C.c_double), ("H_thrs", C.c_double),
        ("max_hupdates", C.c_int32),
        ("slab_x0", C.c_int32), ("slab_nx", C.c_int32),
        ("history", C.c_int32),
        ("prop_shards", C.c_int32), ("prop_shard", C.c_int32),
        ("magnus_order", C.c_int32), ("xc_functional", C.c_int32), ("fd_order", C.c_int32),
    ]


class rt_slab_buffers(C.Structure):
    _fields_ = [("xchg_rho", C.c_void_p), ("xchg_rho_count", C.c_int64), ("xchg_H", C.c_void_p),
                ("xchg_H_count", C.c_int64), ("slab_offset", C.c_int64), ("slab_count", C.c_int64)]


class rt_shard_buffers(C.Structure):
    _fields_ = [("Y", C.c_void_p), ("C", C.c_void_p), ("S", C.c_void_p), ("P1re", C.c_void_p), ("P1im", C.c_void_p),
                ("block_count", C.c_int64), ("total_count", C.c_int64), ("prop_shards", C.c_int32),
                ("prop_shard", C.c_int32)]


class RTError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"rt_tddft error {code}: {msg}")
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2410_09189_b200.build` "
            "(the RT-TDDFT path has no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dp, i32, i64p = C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int64)
    sig = {
        "rt_create": [C.POINTER(rt_config), dp, dp, dp, C.POINTER(vp)],
        "rt_create_general": [C.POINTER(rt_config), dp, dp, dp, dp, dp, C.POINTER(vp)], "rt_get_overlap": [vp, dp, dp],
        "rt_set_field": [vp, dp], "rt_step": [vp, i32], "rt_get_dipole": [vp, dp], "rt_get_density": [vp, dp],
        "rt_get_pmatrix": [vp, dp, dp], "rt_get_hmatrix": [vp, dp], "rt_get_vhartree": [vp, dp],
        "rt_get_time": [vp, dp], "rt_get_charge": [vp, dp], "rt_get_info": [vp, dp], "rt_get_launch_count": [vp, i64p],
        "rt_destroy": [vp], "rt_op_project": [vp, dp, dp], "rt_op_density": [vp, dp, dp, dp],
        "rt_op_propagate": [vp, dp, dp, dp, dp, dp], "rt_op_hartree": [vp, dp, dp, i32], "rt_op_vxc": [vp, dp, dp],
        "rt_timing_enable": [vp, i32], "rt_timing_read": [vp, dp, dp], "rt_get_convergence": [vp, dp, dp],
        "rt_slab_get_buffers": [vp, C.POINTER(rt_slab_buffers)], "rt_slab_phase": [vp, i32, i32],
        "rt_slab_get_shard": [vp, C.POINTER(rt_shard_buffers)], "rt_slab_more_updates": [vp, C.POINTER(C.c_int32)],
        "rt_get_dipole_series": [vp, C.c_int64, i32, dp], "rt_get_energy": [vp, C.POINTER(C.c_double)],
        "rt_state_bytes": [vp, i64p], "rt_get_state": [vp, vp], "rt_set_state": [vp, vp],
        "rt_spectrum": [dp, i32, C.c_double, C.c_double, dp, C.c_double, dp, i32, dp, i32, vp],
        "rt_spectrum_kick": [dp, i32, C.c_double, dp, C.c_double, dp, i32, dp, i32, vp],
        "rt_dipole_noalloc": [dp, i32, i32, i32, C.c_double, dp, i32, vp],
    }
    for name, argtypes in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = argtypes
        fn.restype = C.c_int
    lib.rt_probe_fp64_peak.argtypes = [i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.rt_probe_fp64_peak.restype = C.c_int
    lib.rt_last_error.argtypes = [vp]
    lib.rt_last_error.restype = C.c_char_p
    return lib


_lib = _load()


def _ptr(x):
    """Address of a numpy array (host), a torch tensor (host or device), an int address, or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        assert x.dtype == np.float64 and x.flags["C_CONTIGUOUS"], "need C-contiguous float64"
        return x.ctypes.data
    if hasattr(x, "data_ptr"):
        import torch
        assert x.dtype == torch.float64 and x.is_contiguous(), "need contiguous float64 tensor"
        return x.data_ptr()
    raise TypeError(type(x))


def _check(h, rc):
    if rc != RT_OK:
        msg = _lib.rt_last_error(h)
        raise RTError(rc, msg.decode() if msg else "")


# ---- functions with the C names -------------------------------------------------------------------------

def rt_create(cfg: rt_config, phi, eps, occ) -> int:
    h = C.c_void_p()
    eps = np.ascontiguousarray(eps, dtype=np.float64)
    occ = np.ascontiguousarray(occ, dtype=np.float64)
    rc = _lib.rt_create(C.byref(cfg), _ptr(phi), _ptr(eps), _ptr(occ), C.byref(h))
    _check(None, rc)
    return h.value


def rt_create_general(cfg: rt_config, phi, eps, Hks, P0re, P0im=None) -> int:
    h = C.c_void_p()
    eps = np.ascontiguousarray(eps, dtype=np.float64)
    Hks = np.ascontiguousarray(Hks, dtype=np.float64)
    P0re = np.ascontiguousarray(P0re, dtype=np.float64)
    P0im = None if P0im is None else np.ascontiguousarray(P0im, dtype=np.float64)
    rc = _lib.rt_create_general(C.byref(cfg), _ptr(phi), _ptr(eps), _ptr(Hks), _ptr(P0re), _ptr(P0im), C.byref(h))
    _check(None, rc)
    return h.value


def rt_get_overlap(h, S, Sinv):
    _check(h, _lib.rt_get_overlap(h, _ptr(S), _ptr(Sinv)))
    return S, Sinv


def rt_set_field(h, E):
    e = (C.c_double * 3)(*[float(v) for v in E])
    _check(h, _lib.rt_set_field(h, C.cast(e, C.c_void_p)))


def rt_step(h, nsteps=1):
    _check(h, _lib.rt_step(h, int(nsteps)))


def rt_get_dipole(h) -> np.ndarray:
    mu = np.zeros(3)
    _check(h, _lib.rt_get_dipole(h, _ptr(mu)))
    return mu


def rt_get_density(h, out):
    _check(h, _lib.rt_get_density(h, _ptr(out)))
    return out


def rt_get_pmatrix(h, re, im):
    _check(h, _lib.rt_get_pmatrix(h, _ptr(re), _ptr(im)))


def rt_get_hmatrix(h, out):
    _check(h, _lib.rt_get_hmatrix(h, _ptr(out)))
    return out


def rt_get_vhartree(h, out):
    _check(h, _lib.rt_get_vhartree(h, _ptr(out)))
    return out


def rt_get_time(h) -> float:
    t = np.zeros(1)
    _check(h, _lib.rt_get_time(h, _ptr(t)))
    return float(t[0])


def rt_get_charge(h) -> np.ndarray:
    q = np.zeros(2)
    _check(h, _lib.rt_get_charge(h, _ptr(q)))
    return q


def rt_get_info(h) -> dict:
    a = np.zeros(8, dtype=np.int32)
    _check(h, _lib.rt_get_info(h, a.ctypes.data))
    return {"exp_order": int(a[0]), "mg_levels": int(a[1]), "coarsest": (int(a[2]), int(a[3]), int(a[4])),
            "graph": bool(a[5] & 1), "tma": bool(a[5] & 2), "capture_retried": bool(a[5] & 4),
            "paced_projection": bool(a[5] & 8), "paced_density": bool(a[5] & 16),
            "launches_per_step": int(a[6]),
            "project_split_k": int(a[7])}


def rt_get_convergence(h) -> dict:
    n = np.zeros(2, dtype=np.int32)
    err = np.zeros(2)
    _check(h, _lib.rt_get_convergence(h, n.ctypes.data, _ptr(err)))
    return {"hupdates": int(n[0]), "orders": int(n[1]), "H_err": float(err[0]), "dP_err": float(err[1])}


def rt_get_launch_count(h) -> int:
    n = C.c_int64(0)
    _check(h, _lib.rt_get_launch_count(h, C.byref(n)))
    return int(n.value)


def rt_destroy(h):
    if h:
        _lib.rt_destroy(h)


def rt_op_project(h, v, out):
    _check(h, _lib.rt_op_project(h, _ptr(v), _ptr(out)))
    return out


def rt_op_density(h, reP, rho):
    sums = np.zeros(5)
    _check(h, _lib.rt_op_density(h, _ptr(reP), _ptr(rho), _ptr(sums)))
    return rho, sums


def rt_op_propagate(h, Hbar, P0re, P0im, P1re, P1im):
    _check(h, _lib.rt_op_propagate(h, _ptr(Hbar), _ptr(P0re), _ptr(P0im), _ptr(P1re), _ptr(P1im)))
    return P1re, P1im


def rt_op_hartree(h, vh, drho, n_vc):
    _check(h, _lib.rt_op_hartree(h, _ptr(vh), _ptr(drho), int(n_vc)))
    return vh


def rt_op_vxc(h, rho, out):
    _check(h, _lib.rt_op_vxc(h, _ptr(rho), _ptr(out)))
    return out


def rt_timing_enable(h, enable=True):
    _check(h, _lib.rt_timing_enable(h, 1 if enable else 0))


def rt_timing_read(h):
    ms = np.zeros(RT_STAGE_COUNT)
    calls = np.zeros(RT_STAGE_COUNT, dtype=np.int64)
    _check(h, _lib.rt_timing_read(h, _ptr(ms), calls.ctypes.data))
    return dict(zip(RT_STAGE_NAMES, ms.tolist())), dict(zip(RT_STAGE_NAMES, calls.tolist()))


def rt_probe_fp64_peak(device=0):
    """(DMMA TFLOP/s, DFMA TFLOP/s) issue-rate ceilings of the device (calibration instrument)."""
    a, b = C.c_double(0), C.c_double(0)
    rc = _lib.rt_probe_fp64_peak(int(device), C.byref(a), C.byref(b))
    if rc != RT_OK:
        raise RTError(rc, "rt_probe_fp64_peak failed")
    return a.value, b.value


def rt_get_state(h) -> np.ndarray:
    """Checkpoint of the propagation state as a uint8 array (include/rt_tddft.h rt_get_state)."""
    n = C.c_int64()
    _check(h, _lib.rt_state_bytes(h, C.byref(n)))
    buf = np.zeros(n.value, dtype=np.uint8)
    _check(h, _lib.rt_get_state(h, buf.ctypes.data))
    return buf


def rt_set_state(h, buf: np.ndarray):
    buf = np.ascontiguousarray(buf, dtype=np.uint8)
    n = C.c_int64()
    _check(h, _lib.rt_state_bytes(h, C.byref(n)))
    if buf.size != n.value:
        raise RTError(RT_EINVAL, f"state buffer has {buf.size} bytes, the handle needs {n.value}")
    _check(h, _lib.rt_set_state(h, buf.ctypes.data))


def rt_get_energy(h) -> float:
    e = C.c_double()
    _check(h, _lib.rt_get_energy(h, C.byref(e)))
    return e.value


def rt_get_dipole_series(h, first: int, n: int) -> np.ndarray:
    """[n][4]: mu_x, mu_y, mu_z, charge of the time levels first .. first + n - 1 (level 0 is t = 0)."""
    out = np.zeros((int(n), 4))
    _check(h, _lib.rt_get_dipole_series(h, int(first), int(n), _ptr(out)))
    return out


def rt_spectrum(mu, dt, t_kick, kappa, gamma, omega, device=0, stream=0, out=None):
    """Dipole strength function S(omega) of delta-kick runs (include/rt_tddft.h rt_spectrum).  mu: [3][nt] numpy array
    or CUDA tensor; omega: [nw]; returns S as a numpy array unless `out` (numpy / CUDA tensor) is given."""
    if not hasattr(mu, "is_cuda"):
        mu = np.ascontiguousarray(mu, dtype=np.float64)
    nt = int(mu.shape[1])
    if not hasattr(omega, "is_cuda"):
        omega = np.ascontiguousarray(omega, dtype=np.float64)
    nw = int(omega.shape[0])
    if out is None:
        out = np.zeros(nw)
    k = np.ascontiguousarray(kappa, dtype=np.float64)
    rc = _lib.rt_spectrum(_ptr(mu), nt, float(dt), float(t_kick), _ptr(k), float(gamma), _ptr(omega), nw, _ptr(out),
                          int(device), int(stream) if stream else None)
    _check(None, rc)
    return out


RT_NOALLOC_MAX_POINTS = 4194304


def rt_dipole_noalloc(rho, shape, h, out, device=0, stream=0):
    """a6 on a static device scratch array: no handle, no allocation (include/rt_tddft.h).  rho: CUDA tensor [nx*ny*nz],
    out: CUDA tensor [5] = (mu_x, mu_y, mu_z, charge, dVol sum |rho|).  Enqueues on `stream` and does NOT synchronise;
    calls that overlap on the GPU race on the shared scratch."""
    for t in (rho, out):
        if not (hasattr(t, "is_cuda") and t.is_cuda):
            raise ValueError("rt_dipole_noalloc takes device tensors")
    rc = _lib.rt_dipole_noalloc(_ptr(rho), int(shape[0]), int(shape[1]), int(shape[2]), float(h), _ptr(out), int(device),
                                int(stream) if stream else None)
    _check(None, rc)
    return out


def rt_spectrum_kick(mu, dt, E_kick, gamma, omega, device=0, stream=0, out=None):
    """rt_spectrum for the end-point sampled kick of this library: E_kick[q] = field of the run kicked along q; the
    delivered impulse and the effective kick time are formed inside the library (include/rt_tddft.h)."""
    if not hasattr(mu, "is_cuda"):
        mu = np.ascontiguousarray(mu, dtype=np.float64)
    if not hasattr(omega, "is_cuda"):
        omega = np.ascontiguousarray(omega, dtype=np.float64)
    nt, nw = int(mu.shape[1]), int(omega.shape[0])
    if out is None:
        out = np.zeros(nw)
    e = np.ascontiguousarray(E_kick, dtype=np.float64)
    rc = _lib.rt_spectrum_kick(_ptr(mu), nt, float(dt), _ptr(e), float(gamma), _ptr(omega), nw, _ptr(out), int(device),
                               int(stream) if stream else None)
    _check(None, rc)
    return out


def rt_slab_get_buffers(h) -> rt_slab_buffers:
    b = rt_slab_buffers()
    _check(h, _lib.rt_slab_get_buffers(h, C.byref(b)))
    return b


def rt_slab_phase(h, phase: int, it: int = 0):
    _check(h, _lib.rt_slab_phase(h, int(phase), int(it)))


def rt_slab_get_shard(h) -> rt_shard_buffers:
    b = rt_shard_buffers()
    _check(h, _lib.rt_slab_get_shard(h, C.byref(b)))
    return b


def rt_slab_more_updates(h) -> bool:
    m = C.c_int32(0)
    _check(h, _lib.rt_slab_more_updates(h, C.byref(m)))
    return bool(m.value)


# ---- convenience wrapper (the call a user makes) -------------------------------------------------------

class RTTDDFT:
    """Owns one rt_handle.  ``phi`` may be a host numpy array (copied) or a CUDA torch tensor (borrowed)."""

    def __init__(self, shape, h, phi, eps, occ, dt, E0=(0.0, 0.0, 0.0), n_hupdates=2, n_vcycles=2, nu_pre=2,
                 nu_post=2, jacobi_omega=6.0 / 7.0, exp_order=0, hartree=True, xc=True, graph=True, tma=True,
                 device=0, stream=None, propagator="taylor", max_order=0, dP_thrs=0.0, H_thrs=0.0, max_hupdates=0,
                 slab=None, history=0, prop_shard=None, magnus=1, xc_functional="lda", fd_order=2, Hks=None,
                 P0=None, nonorthogonal=False):
        """``slab = (x0, nx_local)``: the handle owns those x-planes and ``phi`` is [norb][nx_local*ny*nz]
        (rt_slab_* entry points; see slab.py).  ``prop_shard = (rank, nranks)``: row-sharded N x N propagator.
        ``Hks`` / ``P0`` ([norb][norb] host arrays; P0 may be complex): the ground state as matrices (rt_create_general);
        ``nonorthogonal``: phi is a non-orthonormal basis.  ``magnus`` = 2: second Magnus term.  ``occ`` may then be None."""
        cfg = rt_config()
        cfg.slab_x0, cfg.slab_nx = (int(slab[0]), int(slab[1])) if slab else (0, 0)
        cfg.history = int(history)
        cfg.prop_shards, cfg.prop_shard = (int(prop_shard[1]), int(prop_shard[0])) if prop_shard else (0, 0)
        cfg.magnus_order = int(magnus)
        cfg.xc_functional = {"lda": RT_XC_LDA_PZ81, "pbe": RT_XC_PBE}[xc_functional]
        cfg.fd_order = int(fd_order)
        cfg.propagator = {"taylor": RT_PROP_TAYLOR, "commutator": RT_PROP_COMMUTATOR}[propagator]
        cfg.max_order, cfg.dP_thrs, cfg.H_thrs, cfg.max_hupdates = int(max_order), float(dP_thrs), float(H_thrs), int(max_hupdates)
        cfg.nx, cfg.ny, cfg.nz = (int(s) for s in shape)
        cfg.h, cfg.norb, cfg.dt = float(h), int(len(eps)), float(dt)
        cfg.n_hupdates, cfg.n_vcycles = int(n_hupdates), int(n_vcycles)
        cfg.nu_pre, cfg.nu_post, cfg.jacobi_omega = int(nu_pre), int(nu_post), float(jacobi_omega)
        cfg.exp_order = int(exp_order)
        cfg.E0 = (C.c_double * 3)(*[float(e) for e in E0])
        flags = 0
        self._phi_ref = None
        if hasattr(phi, "is_cuda"):
            if phi.is_cuda:
                flags |= RT_PHI_DEVICE
                device = phi.device.index if phi.device.index is not None else device
                self._phi_ref = phi           # keep the borrowed tensor alive
            else:
                phi = phi.numpy()
        if not hartree:
            flags |= RT_NO_HARTREE
        if not xc:
            flags |= RT_NO_XC
        if not graph:
            flags |= RT_NO_GRAPH
        if not tma:
            flags |= RT_NO_TMA
        if nonorthogonal:
            flags |= RT_NONORTHOGONAL
        cfg.flags, cfg.device = flags, int(device)
        if stream is None:
            try:
                import torch
                stream = torch.cuda.current_stream(device).cuda_stream if torch.cuda.is_available() else 0
            except ImportError:
                stream = 0
        cfg.stream = int(stream) if stream else None
        self._dt = float(dt)
        self.shape, self.norb = tuple(int(s) for s in shape), int(len(eps))
        self.ngrid = self.shape[0] * self.shape[1] * self.shape[2]
        if Hks is not None or P0 is not None:
            P0 = np.asarray(P0)
            self.handle = rt_create_general(cfg, phi, eps, Hks, P0.real, P0.imag if np.iscomplexobj(P0) else None)
        else:
            self.handle = rt_create(cfg, phi, eps, occ)

    def set_field(self, E):
        rt_set_field(self.handle, E)

    def step(self, n=1):
        rt_step(self.handle, n)

    def dipole(self):
        return rt_get_dipole(self.handle)

    def density(self, out=None):
        if out is None:
            out = np.empty(self.ngrid)
        return rt_get_density(self.handle, out)

    def dipole_series(self, first=0, n=None):
        """Dipole history kept on the device (needs history > 0): [n][4] = mu_x, mu_y, mu_z, charge."""
        if n is None:
            n = int(round(self.time / self._dt)) + 1 - int(first)
        return rt_get_dipole_series(self.handle, first, n)

    def get_state(self):
        return rt_get_state(self.handle)

    def set_state(self, buf):
        rt_set_state(self.handle, buf)

    def energy(self):
        return rt_get_energy(self.handle)

    def pmatrix(self):
        re, im = np.empty((self.norb, self.norb)), np.empty((self.norb, self.norb))
        rt_get_pmatrix(self.handle, re, im)
        return re + 1j * im

    def hmatrix(self):
        return rt_get_hmatrix(self.handle, np.empty((self.norb, self.norb)))

    def overlap(self):
        S, Si = np.empty((self.norb, self.norb)), np.empty((self.norb, self.norb))
        return rt_get_overlap(self.handle, S, Si)

    def vhartree(self):
        return rt_get_vhartree(self.handle, np.empty(self.ngrid))

    @property
    def time(self):
        return rt_get_time(self.handle)

    def info(self):
        return rt_get_info(self.handle)

    def convergence(self):
        return rt_get_convergence(self.handle)

    def close(self):
        if getattr(self, "handle", None):
            rt_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
