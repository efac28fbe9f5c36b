"""Plain, slow, obviously-correct CPU oracle of the RT-TDDFT time step (arXiv 2410.09189).

TEST INFRASTRUCTURE.  NumPy, FP64 / complex128, no blocking, no fusion, no code shared with the CUDA
path.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py`` (cpu_baseline / --impl reference)
may import it.  Citations are ``PAPER.md:L<line>`` (the paper text under /root/reference) plus the
equation / algorithm line; "DESIGN R<n>" is a reading listed in DESIGN.md where the paper is silent.

What is computed (one step, Algorithm 1 lines 9-29, with the dynamic `while`
loops replaced by fixed counts, DESIGN R1):

    H1 = 2 H0 - H-1                                      (Alg. 1 line 11, L365)
    repeat m times:
        Hbar = (H0 + H1)/2                               (Eq. 12; Alg. 1 line 14, L373)
        U    = W exp(-i w dt) W^T,  Hbar = W w W^T       (spectral form, L129, L147: exact)
        P1   = U P0 U^dagger                             (Eq. 15)
        rho  = sum_ij Re(P1)_ij phi_i phi_j              (Eq. 27, Gamma point, real orbitals)
        V_H  = MG(V_H, 4 pi (drho - mean drho), n_vc)    (multigrid, L77; concrete cycle DESIGN R6)
        dV   = V_H + vxc(rho) - vxc(rho0) + E.x          (V_eff terms, L73-L75; length gauge, L325, L412)
        H1   = diag(eps) + dVol * Phi diag(dV) Phi^T     (Alg. 1 line 25, L395; Eq. 4)
    mu = dVol sum_r x(r) rho(r)                          (Alg. 1 line 27, L400)
    H-1, H0, P0 <- H0, H1, P1                            (Alg. 1 line 28, L403)

Parity pins (tests/test_oracle_*.py): zero-field stationarity, tr P = N_e, P Hermitian and P^2 = 2P,
closed-form non-interacting propagation, energy conservation, linear/odd response, commutator series
(Eq. 39) == eigh propagator (L426), converged multigrid == FFT solution of the same stencil,
continuum Gaussian-charge potential (Ewald closed form) with O(h^2) convergence, v_xc = d(rho e_xc)/d rho
and textbook uniform-gas constants, brute-force projection/density on tiny inputs.
Unpinned by anything outside this file: the *value* of the fixed-cycle (unconverged) V_H -- it is
"parity to the definition" (DESIGN R6); everything it converges to is pinned.
"""
from __future__ import annotations

import numpy as np

# --------------------------------------------------------------------------------------------------
# Grid, field
# --------------------------------------------------------------------------------------------------

def axis_coords(n: int, h: float) -> np.ndarray:
    """Centred sawtooth coordinate x(i) = (i - (n-1)/2) h  (length gauge, "sawtooth-like
    potential"; no vacuum dipole correction, DESIGN R4).  Sum_i x(i) = 0."""
    return (np.arange(n, dtype=np.float64) - 0.5 * (n - 1)) * h


def field_potential(shape, h: float, E) -> np.ndarray:
    """V_ext(r) = E . r on the grid, r = (x(ix), y(iy), z(iz)); flat index (ix*ny + iy)*nz + iz."""
    nx, ny, nz = shape
    x, y, z = axis_coords(nx, h), axis_coords(ny, h), axis_coords(nz, h)
    v = E[0] * x[:, None, None] + E[1] * y[None, :, None] + E[2] * z[None, None, :]
    return np.ascontiguousarray(np.broadcast_to(v, shape)).reshape(-1)


# --------------------------------------------------------------------------------------------------
# LDA exchange-correlation: Slater exchange + Perdew-Zunger 1981 correlation, unpolarised (DESIGN R7;
# the paper ran PBE; north_star fixes LDA).  Hartree atomic units.
# --------------------------------------------------------------------------------------------------
PZ_GAMMA, PZ_BETA1, PZ_BETA2 = -0.1423, 1.0529, 0.3334
PZ_A, PZ_B, PZ_C, PZ_D = 0.0311, -0.048, 0.0020, -0.0116
RHO_FLOOR = 1e-30
RHO_RS1 = 3.0 / (4.0 * np.pi)      # density at which r_s = 1; branch is taken on rho (DESIGN R7)


def _rs(rho):
    return (3.0 / (4.0 * np.pi * rho)) ** (1.0 / 3.0)


def vxc_lda(rho: np.ndarray) -> np.ndarray:
    """v_xc(rho) = v_x + v_c.  v_x = -(3 rho/pi)^(1/3).  rho <= RHO_RS1 (r_s >= 1):
    v_c = eps_c (1 + 7/6 b1 sqrt(rs) + 4/3 b2 rs)/(1 + b1 sqrt(rs) + b2 rs); else
    v_c = A ln rs + (B - A/3) + 2/3 C rs ln rs + (2D - C)/3 rs.   rho < RHO_FLOOR -> 0."""
    rho = np.asarray(rho, dtype=np.float64)
    out = np.zeros_like(rho)
    ok = rho >= RHO_FLOOR
    r = rho[ok]
    rs = _rs(r)
    vx = -np.cbrt(3.0 * r / np.pi)
    lo = r <= RHO_RS1
    vc = np.empty_like(r)
    s = np.sqrt(rs[lo])
    den = 1.0 + PZ_BETA1 * s + PZ_BETA2 * rs[lo]
    ec = PZ_GAMMA / den
    vc[lo] = ec * (1.0 + (7.0 / 6.0) * PZ_BETA1 * s + (4.0 / 3.0) * PZ_BETA2 * rs[lo]) / den
    hi = ~lo
    ln = np.log(rs[hi])
    vc[hi] = PZ_A * ln + (PZ_B - PZ_A / 3.0) + (2.0 / 3.0) * PZ_C * rs[hi] * ln + ((2.0 * PZ_D - PZ_C) / 3.0) * rs[hi]
    out[ok] = vx + vc
    return out


def exc_density_lda(rho: np.ndarray) -> np.ndarray:
    """e_xc(rho) = rho (eps_x + eps_c) per unit volume (energy check only).  eps_x = 3/4 v_x."""
    rho = np.asarray(rho, dtype=np.float64)
    out = np.zeros_like(rho)
    ok = rho >= RHO_FLOOR
    r = rho[ok]
    rs = _rs(r)
    ex = -0.75 * np.cbrt(3.0 * r / np.pi)
    lo = r <= RHO_RS1
    ec = np.empty_like(r)
    ec[lo] = PZ_GAMMA / (1.0 + PZ_BETA1 * np.sqrt(rs[lo]) + PZ_BETA2 * rs[lo])
    hi = ~lo
    ln = np.log(rs[hi])
    ec[hi] = PZ_A * ln + PZ_B + PZ_C * rs[hi] * ln + PZ_D * rs[hi]
    out[ok] = r * (ex + ec)
    return out


# --------------------------------------------------------------------------------------------------
# PBE generalised-gradient approximation (the functional the paper ran), unpolarised.
# Perdew, Burke, Ernzerhof, PRL 77, 3865 (1996), restated:  e_xc(n, sigma) = e_x + e_c per unit volume, sigma = |grad n|^2,
#   e_x = n eps_x^unif(n) F_x(s),  eps_x^unif = -(3/4)(3 n/pi)^(1/3),  s = |grad n| / (2 k_F n),  k_F = (3 pi^2 n)^(1/3),
#         F_x = 1 + kappa - kappa / (1 + mu s^2 / kappa),  kappa = 0.804,  mu = beta pi^2 / 3
#   e_c = n [eps_c^unif(r_s) + H(r_s, t)],  t = |grad n| / (2 k_s n),  k_s = sqrt(4 k_F / pi),
#         H = gamma ln{1 + (beta/gamma) t^2 (1 + A t^2) / (1 + A t^2 + A^2 t^4)},  A = (beta/gamma) / (exp(-eps_c^unif/gamma) - 1),
#         beta = 0.06672455060314922,  gamma = (1 - ln 2)/pi^2,  eps_c^unif = Perdew-Wang 1992 (PRB 45, 13244) at zeta = 0.
# On the grid the gradient is a central finite difference D (grad_fd) and E_xc = dVol sum_r e_xc(n_r, |D n|_r^2), whose exact
# derivative with respect to n_r is the potential used here (the grid analogue of v = d e/d n - div(d e/d grad n)):
#   v_xc = d e/d n - sum_q D_q (2 d e/d sigma  D_q n)            (D is antisymmetric, so D^T = -D)
# --------------------------------------------------------------------------------------------------
PBE_KAPPA = 0.804
PBE_BETA = 0.06672455060314922
PBE_GAMMA = (1.0 - np.log(2.0)) / np.pi ** 2
PBE_MU = PBE_BETA * np.pi ** 2 / 3.0
PW92_A, PW92_ALPHA1 = 0.0310907, 0.21370
PW92_B1, PW92_B2, PW92_B3, PW92_B4 = 7.5957, 3.5876, 1.6382, 0.49294
# central-difference first-derivative weights c_1..c_n (f' ~ sum_i c_i (f_{+i} - f_{-i}) / h) of order 2n (Eq. 2's analogue)
FD_GRAD = {2: (0.5,), 4: (2.0 / 3.0, -1.0 / 12.0)}
# second-derivative weights a_0; a_1..a_n of Eq. 2 (L58-L60): f'' ~ (a_0 f_0 + sum_i a_i (f_{+i} + f_{-i})) / h^2, order 2n
FD_LAPL = {2: (-2.0, (1.0,)), 4: (-5.0 / 2.0, (4.0 / 3.0, -1.0 / 12.0))}


def pw92_eps_c(rs):
    """Perdew-Wang 1992 correlation energy per electron of the unpolarised uniform gas, and d eps_c / d r_s."""
    sq = np.sqrt(rs)
    G = PW92_B1 * sq + PW92_B2 * rs + PW92_B3 * rs * sq + PW92_B4 * rs * rs
    dG = 0.5 * PW92_B1 / sq + PW92_B2 + 1.5 * PW92_B3 * sq + 2.0 * PW92_B4 * rs
    lg = np.log(1.0 + 1.0 / (2.0 * PW92_A * G))
    eps = -2.0 * PW92_A * (1.0 + PW92_ALPHA1 * rs) * lg
    deps = -2.0 * PW92_A * PW92_ALPHA1 * lg + (1.0 + PW92_ALPHA1 * rs) * dG / (G * G + G / (2.0 * PW92_A))
    return eps, deps


def pbe_exc(n, sigma):
    """(e_xc, d e_xc / d n, d e_xc / d sigma) of PBE for density n > RHO_FLOOR and sigma = |grad n|^2 (arrays).
    Points with n < RHO_FLOOR give zeros."""
    n = np.asarray(n, dtype=np.float64)
    sigma = np.asarray(sigma, dtype=np.float64)
    e, dn, ds = np.zeros_like(n), np.zeros_like(n), np.zeros_like(n)
    ok = n >= RHO_FLOOR
    r, sg = n[ok], sigma[ok]
    pi = np.pi
    # ---- exchange
    Cx = 0.75 * (3.0 / pi) ** (1.0 / 3.0)
    n13 = np.cbrt(r)
    q = 1.0 / (4.0 * (3.0 * pi * pi) ** (2.0 / 3.0) * n13 ** 8)          # d s^2 / d sigma
    p = sg * q                                                            # s^2
    den = 1.0 + PBE_MU * p / PBE_KAPPA
    F = 1.0 + PBE_KAPPA - PBE_KAPPA / den
    dF = PBE_MU / (den * den)
    ex = -Cx * r * n13 * F
    dex_dn = -Cx * n13 * ((4.0 / 3.0) * F - (8.0 / 3.0) * p * dF)
    dex_ds = -Cx * r * n13 * dF * q
    # ---- correlation
    rs = np.cbrt(3.0 / (4.0 * pi * r))
    eps, deps_drs = pw92_eps_c(rs)
    deps_dn = deps_drs * (-rs / (3.0 * r))
    du_ds = pi / (16.0 * (3.0 * pi * pi) ** (1.0 / 3.0) * n13 ** 7)      # u = t^2 = sigma * du_ds
    u = sg * du_ds
    ex1 = np.exp(-eps / PBE_GAMMA)
    A = (PBE_BETA / PBE_GAMMA) / (ex1 - 1.0)
    dA_deps = A * A * ex1 / PBE_BETA
    Au = A * u
    Dn = 1.0 + Au + Au * Au
    Q = u * (1.0 + Au) / Dn
    H = PBE_GAMMA * np.log(1.0 + (PBE_BETA / PBE_GAMMA) * Q)
    HQ = PBE_BETA / (1.0 + (PBE_BETA / PBE_GAMMA) * Q)
    Qu = (1.0 + 2.0 * Au) / (Dn * Dn)
    QA = -A * u * u * u * (2.0 + Au) / (Dn * Dn)
    du_dn = -(7.0 / 3.0) * u / r
    ec = r * (eps + H)
    dec_dn = eps + H + r * (deps_dn + HQ * (Qu * du_dn + QA * dA_deps * deps_dn))
    dec_ds = r * HQ * Qu * du_ds
    e[ok], dn[ok], ds[ok] = ex + ec, dex_dn + dec_dn, dex_ds + dec_ds
    return e, dn, ds


def grad_fd(u: np.ndarray, h: float, order: int = 2):
    """Central finite-difference gradient (periodic), components along x, y, z; order 2 or 4 (FD_GRAD)."""
    out = []
    for ax in range(3):
        g = np.zeros_like(u)
        for i, c in enumerate(FD_GRAD[order], start=1):
            g = g + c * (np.roll(u, -i, ax) - np.roll(u, i, ax))
        out.append(g / h)
    return out


def vxc_pbe(rho: np.ndarray, shape, h: float, order: int = 2) -> np.ndarray:
    """PBE potential on the grid: v = d e/d n - sum_q D_q (2 d e/d sigma D_q n)  (flat array in, flat array out)."""
    n3 = np.asarray(rho, dtype=np.float64).reshape(shape)
    g = grad_fd(n3, h, order)
    sigma = g[0] * g[0] + g[1] * g[1] + g[2] * g[2]
    _, dn, ds = pbe_exc(n3, sigma)
    v = dn.copy()
    for ax in range(3):
        v = v - grad_fd(2.0 * ds * g[ax], h, order)[ax]
    return v.reshape(-1)


def exc_density_pbe(rho: np.ndarray, shape, h: float, order: int = 2) -> np.ndarray:
    """e_xc(n, |D n|^2) per unit volume on the grid (energy diagnostic)."""
    n3 = np.asarray(rho, dtype=np.float64).reshape(shape)
    g = grad_fd(n3, h, order)
    return pbe_exc(n3, g[0] * g[0] + g[1] * g[1] + g[2] * g[2])[0].reshape(-1)


# --------------------------------------------------------------------------------------------------
# Hartree: periodic 7-point Poisson, fixed count of V(nu1,nu2) cycles, weighted Jacobi (DESIGN R6)
# --------------------------------------------------------------------------------------------------

def apply_A(u: np.ndarray, h: float) -> np.ndarray:
    """A u = -lap_h u = (6 u - sum of the 6 periodic neighbours)/h^2."""
    nb = (np.roll(u, 1, 0) + np.roll(u, -1, 0) + np.roll(u, 1, 1) + np.roll(u, -1, 1)
          + np.roll(u, 1, 2) + np.roll(u, -1, 2))
    return (6.0 * u - nb) / (h * h)


def jacobi_sweep(u: np.ndarray, f: np.ndarray, h: float, omega: float) -> np.ndarray:
    """u <- u + omega D^-1 (f - A u), D = 6/h^2  ==  (1-omega) u + (omega/6)(h^2 f + sum_nb u)."""
    nb = (np.roll(u, 1, 0) + np.roll(u, -1, 0) + np.roll(u, 1, 1) + np.roll(u, -1, 1)
          + np.roll(u, 1, 2) + np.roll(u, -1, 2))
    return (1.0 - omega) * u + (omega / 6.0) * (h * h * f + nb)


def restrict_full_weighting(r: np.ndarray) -> np.ndarray:
    """Tensor-product (1/4, 1/2, 1/4) full weighting; coarse point I sits on fine point 2I (periodic)."""
    for ax in range(3):
        r = 0.25 * np.roll(r, 1, ax) + 0.5 * r + 0.25 * np.roll(r, -1, ax)
        r = np.take(r, np.arange(0, r.shape[ax], 2), axis=ax)
    return r


def prolong_trilinear(e: np.ndarray) -> np.ndarray:
    """Tensor-product linear interpolation: fine 2I <- coarse I ; fine 2I+1 <- (coarse I + coarse I+1)/2."""
    for ax in range(3):
        n = e.shape[ax]
        shp = list(e.shape)
        shp[ax] = 2 * n
        f = np.empty(shp, dtype=np.float64)
        ev = [slice(None)] * 3
        od = [slice(None)] * 3
        ev[ax] = slice(0, 2 * n, 2)
        od[ax] = slice(1, 2 * n, 2)
        f[tuple(ev)] = e
        f[tuple(od)] = 0.5 * (e + np.roll(e, -1, ax))
        e = f
    return e


def lambda_1d(n: int, h: float) -> np.ndarray:
    """Eigenvalues of the periodic 1-D operator (2 u_i - u_{i-1} - u_{i+1})/h^2: (2 - 2 cos 2 pi k/n)/h^2."""
    return (2.0 - 2.0 * np.cos(2.0 * np.pi * np.arange(n) / n)) / (h * h)


def spectral_solve(f: np.ndarray, h: float) -> np.ndarray:
    """Exact solve of A u = f in the zero-mean subspace via the analytic eigenpairs (FFT)."""
    nx, ny, nz = f.shape
    lam = (lambda_1d(nx, h)[:, None, None] + lambda_1d(ny, h)[None, :, None] + lambda_1d(nz, h)[None, None, :])
    fh = np.fft.fftn(f)
    lam[0, 0, 0] = 1.0
    uh = fh / lam
    uh[0, 0, 0] = 0.0
    return np.real(np.fft.ifftn(uh))


def can_coarsen(shape) -> bool:
    """Coarsen while every dimension is even and > 4 (DESIGN R6)."""
    return all((n % 2 == 0) and (n > 4) for n in shape)


def mg_level_shapes(shape):
    shapes = [tuple(shape)]
    while can_coarsen(shapes[-1]):
        shapes.append(tuple(n // 2 for n in shapes[-1]))
    return shapes


def vcycle(u: np.ndarray, f: np.ndarray, h: float, nu1: int, nu2: int, omega: float) -> np.ndarray:
    if not can_coarsen(u.shape):
        return spectral_solve(f, h)                       # coarsest level: exact, zero-mean
    for _ in range(nu1):
        u = jacobi_sweep(u, f, h, omega)
    r = f - apply_A(u, h)
    fc = restrict_full_weighting(r)
    ec = vcycle(np.zeros_like(fc), fc, 2.0 * h, nu1, nu2, omega)   # rediscretised, zero initial guess
    u = u + prolong_trilinear(ec)
    for _ in range(nu2):
        u = jacobi_sweep(u, f, h, omega)
    return u


def apply_A_order(u: np.ndarray, h: float, order: int) -> np.ndarray:
    """A u = -lap_h u with the (2n+1)-point central second difference of Eq. 2 along every axis,
    order = 2n (FD_LAPL): order 2 is the 7-point operator of apply_A, order 4 the 13-point one."""
    a0, an = FD_LAPL[order]
    out = 3.0 * a0 * u
    for ax in range(3):
        for i, a in enumerate(an, start=1):
            out = out + a * (np.roll(u, i, ax) + np.roll(u, -i, ax))
    return -out / (h * h)


def lambda_1d_order(n: int, h: float, order: int) -> np.ndarray:
    """Eigenvalues of the periodic 1-D operator -d2/dx2 discretised with FD_LAPL[order] (plane waves are eigenvectors)."""
    a0, an = FD_LAPL[order]
    th = 2.0 * np.pi * np.arange(n) / n
    return -(a0 + sum(2.0 * a * np.cos(i * th) for i, a in enumerate(an, start=1))) / (h * h)


def spectral_solve_order(f: np.ndarray, h: float, order: int) -> np.ndarray:
    """Exact zero-mean solution of apply_A_order(u) = f (FFT); the potential the order-4 Hartree cycle converges to."""
    nx, ny, nz = f.shape
    lam = (lambda_1d_order(nx, h, order)[:, None, None] + lambda_1d_order(ny, h, order)[None, :, None]
           + lambda_1d_order(nz, h, order)[None, None, :])
    fh = np.fft.fftn(f)
    lam[0, 0, 0] = 1.0
    uh = fh / lam
    uh[0, 0, 0] = 0.0
    return np.real(np.fft.ifftn(uh))


def hartree_mg(VH: np.ndarray, drho: np.ndarray, shape, h: float, n_vc: int,
               nu1: int = 2, nu2: int = 2, omega: float = 6.0 / 7.0, order: int = 2) -> np.ndarray:
    """n_vc V-cycles on  -lap_h V_H = 4 pi (drho - mean drho), warm-started from VH (flat arrays).
    order = 2: the 7-point operator, u <- vcycle(u, f).  order = 4 (the paper's Laplacians are
    high-order, Eq. 2-3): V_H solves the 13-point fourth-order operator A4, and the 7-point multigrid cycle
    acts as its preconditioner -- the way RMG uses multigrid (L77: "multigrid ... as a preconditioner"), DESIGN R17:
        r = f - A4 u ;  d = vcycle(0, r)  [one V(nu1, nu2) cycle of the 7-point hierarchy, zero initial guess] ;  u <- u + d."""
    f = 4.0 * np.pi * (drho - np.mean(drho))
    u = VH.reshape(shape)
    f = f.reshape(shape)
    for _ in range(n_vc):
        if order == 2:
            u = vcycle(u, f, h, nu1, nu2, omega)
        else:
            r = f - apply_A_order(u, h, order)
            u = u + vcycle(np.zeros_like(r), r, h, nu1, nu2, omega)
    return u.reshape(-1)


# --------------------------------------------------------------------------------------------------
# Grid <-> matrix contractions (Eq. 4 quadrature rule)
# --------------------------------------------------------------------------------------------------

def project(Phi: np.ndarray, v: np.ndarray, dVol: float) -> np.ndarray:
    """<phi_i| v |phi_j> = dVol sum_r phi_i(r) v(r) phi_j(r)   (Phi is [N][Ng])."""
    return dVol * ((Phi * v[None, :]) @ Phi.T)


def density(Phi: np.ndarray, ReP: np.ndarray) -> np.ndarray:
    """rho(r) = sum_ij Re(P)_ij phi_i(r) phi_j(r)  (Im P is antisymmetric and drops out for real phi)."""
    return np.sum((ReP @ Phi) * Phi, axis=0)


def dipole(rho: np.ndarray, shape, h: float) -> np.ndarray:
    """mu_q = dVol sum_r x_q(r) rho(r)  (= tr(P M_q), Alg. 1 line 27 with mu_0 folded in, DESIGN R3)."""
    nx, ny, nz = shape
    r3 = rho.reshape(shape)
    dVol = h ** 3
    return dVol * np.array([
        np.sum(axis_coords(nx, h)[:, None, None] * r3),
        np.sum(axis_coords(ny, h)[None, :, None] * r3),
        np.sum(axis_coords(nz, h)[None, None, :] * r3)])


# --------------------------------------------------------------------------------------------------
# Propagators
# --------------------------------------------------------------------------------------------------

def propagator_eigh(Hbar: np.ndarray, dt: float) -> np.ndarray:
    """U = exp(-i Hbar dt) = W exp(-i w dt) W^T by exact diagonalisation."""
    w, W = np.linalg.eigh(Hbar)
    return (W * np.exp(-1j * w * dt)[None, :]) @ W.T


def propagate_eigh(Hbar: np.ndarray, P0: np.ndarray, dt: float) -> np.ndarray:
    """P1 = U P0 U^dagger (Eq. 15)."""
    U = propagator_eigh(Hbar, dt)
    return U @ P0 @ U.conj().T


def propagate_commutator(Hbar: np.ndarray, P0: np.ndarray, dt: float, dP_thrs: float = 1e-14,
                         kmax: int = 200):
    """The paper's own propagator, Eq. 39 (L310-L319) / Alg. 1 lines 15-23 (L375-L390) with S = 1:
    dP^(k) = (1/k)(-i dt)[Hbar, dP^(k-1)],  P1 = P0 + sum_k dP^(k), until max|dP^(k)| <= dP_thrs.
    Garbled lines 17/19 of the listing read as k <- 0, dP <- P0 / k <- k+1 (DESIGN R2).
    Used only as an independent cross-check of propagate_eigh (L426).  Returns (P1, k)."""
    P1 = P0.astype(np.complex128).copy()
    dP = P0.astype(np.complex128).copy()
    k = 0
    err = 2.0 * dP_thrs
    while err > dP_thrs and k < kmax:
        k += 1
        dP = (-1j * dt / k) * (Hbar @ dP - dP @ Hbar)
        P1 = P1 + dP
        err = np.max(np.abs(dP))
    return P1, k


# --------------------------------------------------------------------------------------------------
# Closer-to-paper propagation: second Magnus term (Eq. 13) and a non-orthogonal basis (Eq. 33-38)
# --------------------------------------------------------------------------------------------------

def magnus_omega(H0: np.ndarray, H1: np.ndarray, dt: float, order: int = 1, Sinv=None) -> np.ndarray:
    """Omega of U = exp(Omega) for a Hamiltonian that changes linearly from H0 (at t) to H1 (at t + dt), hbar = 1:
    Omega_1 = -i dt (H0 + H1)/2 (Eq. 12); order 2 adds Omega_2 = (dt^2/12)[H0, H1] (Eq. 13).
    With an overlap matrix S != 1 every H is replaced by S^-1 H (Eq. 36: Omega_1 = -i dt S^-1 Hbar)."""
    if Sinv is not None:
        H0, H1 = Sinv @ H0, Sinv @ H1
    Om = (-1j * dt) * 0.5 * (H0 + H1)
    if order >= 2:
        Om = Om + (dt * dt / 12.0) * (H0 @ H1 - H1 @ H0)
    return Om


def propagate_omega_series(Om: np.ndarray, P0: np.ndarray, dP_thrs: float = 1e-14, kmax: int = 200):
    """The paper's series for a general Omega, Eq. 21-23 (L191-L209) / Eq. 37-38 (L289-L304):
    dP^(k) = (1/k){Omega, dP^(k-1)} = (1/k)(Omega dP^(k-1) + dP^(k-1) Omega^dagger), P1 = P0 + sum_k dP^(k),
    until max|dP^(k)| <= dP_thrs.  Returns (P1, k).  Reduces to propagate_commutator for Omega = -i dt Hbar."""
    P1 = P0.astype(np.complex128).copy()
    dP = P0.astype(np.complex128).copy()
    k = 0
    err = 2.0 * dP_thrs
    while err > dP_thrs and k < kmax:
        k += 1
        dP = (Om @ dP + dP @ Om.conj().T) / k
        P1 = P1 + dP
        err = np.max(np.abs(dP))
    return P1, k


def propagate_exact_general(H0: np.ndarray, H1: np.ndarray, P0: np.ndarray, dt: float, order: int = 1, S=None):
    """P1 = exp(Omega) P0 exp(Omega)^dagger with the exponential by exact diagonalisation (L129, L147).  For S != 1 the
    problem is first taken to an orthogonal basis with the Cholesky factor S = L L^T (L271 / Appendix A):
    H_o = L^-1 H L^-T, P_o = L^T P L; after the propagation P = L^-T P_o L^-1.  Omega_o = magnus_omega(H0_o, H1_o) is
    anti-Hermitian, so i Omega_o is Hermitian and eigh applies."""
    if S is not None:
        L = np.linalg.cholesky(S)
        Li = np.linalg.inv(L)
        H0, H1 = Li @ H0 @ Li.T, Li @ H1 @ Li.T
        P0 = L.T @ P0 @ L
    Om = magnus_omega(H0, H1, dt, order)
    w, W = np.linalg.eigh(1j * Om)                       # Omega = -i (i Omega), i Omega Hermitian
    U = (W * np.exp(-1j * w)[None, :]) @ W.conj().T
    P1 = U @ P0 @ U.conj().T
    if S is not None:
        P1 = Li.T @ P1 @ Li
    return P1


# --------------------------------------------------------------------------------------------------
# The time stepper
# --------------------------------------------------------------------------------------------------

class RTOracle:
    """State machine with the same time semantics as the C-ABI (include/rt_tddft.h).

    After construction t = 0, P = diag(occ), rho = rho0, V_H = 0, H0 = H-1 = diag(eps) + Proj(E0.x)
    (Alg. 1 lines 7-8, L355-L358; delta-kick sampled at the end points, DESIGN R5).  ``step()`` uses
    the field set by the last ``set_field`` (default 0) as E(t_{n+1}).
    """

    def __init__(self, shape, h, Phi, eps, occ, dt, E0=(0.0, 0.0, 0.0), n_hupdates=2, n_vcycles=2,
                 nu_pre=2, nu_post=2, omega=6.0 / 7.0, hartree=True, xc=True,
                 propagator="eigh", dP_thrs=1e-10, max_order=200, H_thrs=0.0, max_hupdates=20,
                 magnus=1, Hks=None, P0=None, nonorthogonal=False, xc_functional="lda", fd_order=2):
        """propagator = "eigh": exact spectral exponential (north_star).  propagator = "commutator": the
        paper's own series applied to P (Eq. 39, Alg. 1 lines 15-23) until max|dP^(k)| <= dP_thrs
        (Alg. 1 line 5: 1e-10).  H_thrs > 0 turns the fixed count of Hamiltonian updates into the paper's
        dynamic loop (Alg. 1 lines 12-13, 24-26; L483): repeat while max|H1 - H1_old| > H_thrs, at most
        max_hupdates times.  ``last_hupdates``, ``last_H_err``, ``last_orders`` report what the last step did.
        magnus = 2 adds the second Magnus term Omega_2 = dt^2/12 [H0, H1] (Eq. 13).  nonorthogonal = True: Phi is
        any basis of real functions, S = dVol Phi Phi^T != 1 and P is propagated with Eq. 33-38 (L262-L304); the
        ground state then enters as a Hamiltonian matrix ``Hks`` [N][N] (instead of eps) and a density matrix ``P0``
        [N][N] with tr(P0 S) = N_e (instead of occ).  Both options route the propagation through magnus_omega.
        xc_functional = "pbe": the GGA the paper ran (L453) instead of north_star's LDA; fd_order = 2 or 4: order of the
        finite-difference operators on the grid (gradient of the GGA, Laplacian the Hartree potential solves)."""
        assert xc_functional in ("lda", "pbe") and fd_order in (2, 4)
        self.xc_functional, self.fd_order = xc_functional, int(fd_order)
        assert propagator in ("eigh", "commutator")
        self.propagator, self.dP_thrs, self.max_order = propagator, float(dP_thrs), int(max_order)
        self.H_thrs, self.max_hupdates = float(H_thrs), int(max_hupdates)
        self.last_hupdates, self.last_H_err, self.last_H_errs, self.last_orders = 0, 0.0, [], []
        self.shape = tuple(int(n) for n in shape)
        self.h = float(h)
        self.dVol = self.h ** 3
        self.Phi = np.asarray(Phi, dtype=np.float64)
        self.N, self.Ng = self.Phi.shape
        assert self.Ng == int(np.prod(self.shape))
        self.eps = np.asarray(eps, dtype=np.float64).copy()
        self.occ = np.asarray(occ, dtype=np.float64).copy()
        self.dt = float(dt)
        self.m, self.n_vc = int(n_hupdates), int(n_vcycles)
        self.nu1, self.nu2, self.omega = int(nu_pre), int(nu_post), float(omega)
        self.hartree, self.xc = bool(hartree), bool(xc)
        self.t = 0.0
        self.magnus, self.nonorth = int(magnus), bool(nonorthogonal)
        self.Hks = np.diag(self.eps) if Hks is None else np.asarray(Hks, dtype=np.float64).copy()
        self.P0 = (np.diag(self.occ) if P0 is None else np.asarray(P0)).astype(np.complex128)
        self.S = project(self.Phi, np.ones(self.Ng), self.dVol) if self.nonorth else None      # overlap, Eq. 30
        self.Sinv = np.linalg.inv(self.S) if self.nonorth else None
        self.rho0 = density(self.Phi, self.P0.real)
        self.rho = self.rho0.copy()
        self.vxc0 = self._vxc(self.rho0) if self.xc else np.zeros(self.Ng)
        self.VH = np.zeros(self.Ng)
        self.E_next = np.zeros(3)
        self.H0 = self.Hks + project(self.Phi, field_potential(self.shape, self.h, np.asarray(E0, float)), self.dVol)
        self.Hm1 = self.H0.copy()

    def _vxc(self, rho):
        if self.xc_functional == "pbe":
            return vxc_pbe(rho, self.shape, self.h, self.fd_order)
        return vxc_lda(rho)

    def _exc(self, rho):
        if self.xc_functional == "pbe":
            return exc_density_pbe(rho, self.shape, self.h, self.fd_order)
        return exc_density_lda(rho)

    def set_field(self, E):
        self.E_next = np.asarray(E, dtype=np.float64).copy()

    def delta_v(self, rho):
        """dV(r) = V_H[drho] + v_xc(rho) - v_xc(rho0) + E(t_{n+1}).x ; updates the warm-started V_H."""
        dv = field_potential(self.shape, self.h, self.E_next)
        if self.hartree:
            self.VH = hartree_mg(self.VH, rho - self.rho0, self.shape, self.h, self.n_vc,
                                 self.nu1, self.nu2, self.omega, self.fd_order)
            dv = dv + self.VH
        if self.xc:
            dv = dv + self._vxc(rho) - self.vxc0
        return dv

    def _propagate(self, Hbar, H1=None):
        if self.magnus >= 2 or self.nonorth:              # general Omega (Eq. 13 / Eq. 36)
            if self.propagator == "eigh":
                return propagate_exact_general(self.H0, H1, self.P0, self.dt, self.magnus, self.S)
            Om = magnus_omega(self.H0, H1, self.dt, self.magnus, self.Sinv)
            P1, k = propagate_omega_series(Om, self.P0, self.dP_thrs, self.max_order)      # Eq. 37-38
            self.last_orders.append(k)
            return P1
        if self.propagator == "eigh":
            return propagate_eigh(Hbar, self.P0, self.dt)                  # Eq. 15
        P1, k = propagate_commutator(Hbar, self.P0, self.dt, self.dP_thrs, self.max_order)   # lines 15-23
        self.last_orders.append(k)
        return P1

    def step(self, nsteps: int = 1):
        for _ in range(nsteps):
            H1 = 2.0 * self.H0 - self.Hm1                                  # Alg. 1 line 11
            self.last_orders, self.last_H_errs = [], []
            it = 0
            H_err = 2.0 * self.H_thrs                                      # line 12
            while (it < self.m) if self.H_thrs <= 0.0 else (H_err > self.H_thrs and it < self.max_hupdates):
                Hbar = 0.5 * (self.H0 + H1)                                # line 14 / Eq. 12
                P1 = self._propagate(Hbar, H1)
                rho = density(self.Phi, P1.real)                           # Eq. 27
                H1_old = H1
                H1 = self.Hks + project(self.Phi, self.delta_v(rho), self.dVol)            # line 25
                H_err = float(np.max(np.abs(H1 - H1_old)))                 # line 24 (after the update, DESIGN R2)
                self.last_H_errs.append(H_err)
                it += 1
            self.last_hupdates, self.last_H_err = it, H_err
            self.rho = rho
            self.Hm1, self.H0, self.P0 = self.H0, H1, P1                   # line 28
            self.t += self.dt

    def dipole(self):
        return dipole(self.rho, self.shape, self.h)                        # line 27

    def density(self):
        return self.rho

    def energy(self):
        """E = sum_i eps_i Re P_ii + 1/2 dVol sum drho V_H + dVol sum [e_xc(rho) - e_xc(rho0) - vxc0 drho]
        (+ dVol sum E.x drho while a field is on).  Its functional derivative w.r.t. rho is delta_v, so it
        is conserved by the exact dynamics when E = 0 (test aid; uses the current, unconverged V_H)."""
        drho = self.rho - self.rho0
        e = float(np.sum(self.Hks * self.P0.real))        # tr(H_KS P); = sum_i eps_i Re P_ii in the KS basis
        if self.hartree:
            e += 0.5 * self.dVol * float(np.sum(drho * self.VH))
        if self.xc:
            e += self.dVol * float(np.sum(self._exc(self.rho) - self._exc(self.rho0) - self.vxc0 * drho))
        e += self.dVol * float(np.sum(field_potential(self.shape, self.h, self.E_next) * drho))
        return e


# --------------------------------------------------------------------------------------------------
# Photoabsorption spectrum of delta-kick runs (DESIGN R16)
# --------------------------------------------------------------------------------------------------

def dipole_strength(mu: np.ndarray, dt: float, t_kick: float, kappa, gamma: float, omega: np.ndarray) -> np.ndarray:
    """S(w) = -(2 w / (n_used pi)) sum_q (1/kappa_q) Im dt sum_n c_n [mu_q(t_n) - mu_q(0)] exp((i w - gamma)(t_n - t_kick)).

    "Photoabsorption spectra are calculated as a sum of Fourier transforms of mu_x(t), mu_y(t) and mu_z(t) obtained
    from three independent simulations with the kick ... along x, y, and z" (L453).  mu[q] is the q-component of the
    dipole of the run kicked along q with delivered impulse kappa_q (rows with kappa_q = 0 are skipped); trapezoid
    weights c_n, exponential damping gamma, phases counted from the effective kick time t_kick.  Plain loop over
    frequencies; no FFT, so omega may be any grid."""
    mu = np.asarray(mu, dtype=np.float64)
    omega = np.asarray(omega, dtype=np.float64)
    nt = mu.shape[1]
    t = np.arange(nt) * dt - t_kick
    c = np.ones(nt)
    c[0] = c[-1] = 0.5
    used = [q for q in range(3) if kappa[q] != 0.0]
    S = np.zeros(omega.shape[0])
    for iw, w in enumerate(omega):
        acc = 0.0
        for q in used:
            ft = dt * np.sum(c * (mu[q] - mu[q, 0]) * np.exp((1j * w - gamma) * t))
            acc += ft.imag / kappa[q]
        S[iw] = -(2.0 * w / (len(used) * np.pi)) * acc
    return S
