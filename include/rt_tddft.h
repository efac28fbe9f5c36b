/* rt_tddft.h -- C ABI of the B200-native RT-TDDFT time step (arXiv 2410.09189, "RMG" RT-TDDFT).
 *
 * The library propagates the one-particle density matrix P(t) in the basis of N real ground-state
 * Kohn-Sham orbitals Phi sampled on a periodic uniform grid ("orthogonal basis set for
 * density matrix propagation", overlap = identity; Gamma point, L337).  One rt_step is Algorithm 1 lines
 * 10-28 with the two dynamic `while` loops replaced by fixed counts (DESIGN R1, R8):
 *
 *   H1 = 2 H0 - H-1                                   line 11
 *   repeat n_hupdates times:                          lines 13-26
 *     Hbar = (H0 + H1)/2 ; U = exp(-i Hbar dt)        line 14, Eq. 12 (L123); series of real FP64 GEMMs
 *     P1 = U P0 U^dagger                              Eq. 15 (L143-L145)
 *     rho(r) = sum_ij Re(P1)_ij phi_i(r) phi_j(r)     Eq. 27 (L232)
 *     V_H <- n_vcycles V-cycles on -lap V_H = 4 pi (rho - rho0 - mean)   ("Vh", Table 1; DESIGN R6)
 *     dV = V_H + vxc(rho) - vxc(rho0) + E(t+dt).r     ("exchange/correlation", L547; length gauge L325)
 *     H1 = diag(eps) + dVol Phi diag(dV) Phi^T        line 25 ("Hupdate", L543; quadrature Eq. 4)
 *   mu = dVol sum_r r rho(r)                          line 27
 *   H-1 <- H0 ; H0 <- H1 ; P0 <- P1                   line 28
 *
 * Conventions
 *   - Grid: periodic nx x ny x nz, flat index r = (ix*ny + iy)*nz + iz (z fastest), Ng = nx*ny*nz, dVol = h^3.
 *     Coordinates are the centred sawtooth x(ix) = (ix - (nx-1)/2) h (DESIGN R4).
 *   - Phi is row-major [norb][Ng] FP64 (orbital-major, grid index contiguous), dVol*sum_r phi_i phi_j = delta_ij.
 *   - All N x N matrices are row-major FP64; complex P is passed as separate real / imaginary planes.
 *   - Every pointer argument is documented as HOST, DEVICE or EITHER (EITHER = any pointer cudaMemcpy with
 *     cudaMemcpyDefault accepts; the copy is stream-ordered and the call returns after it has completed).
 *   - Every function returns RT_OK (0) or a negative code; no exceptions, no exit(); rt_last_error gives text.
 *     A CUDA error poisons the handle: later calls return RT_ESTATE.
 *   - Nothing is allocated inside rt_step; all workspaces are created in rt_create.
 *   - There is no CPU fallback: without an sm_100 device rt_create returns RT_ECUDA.
 */
#ifndef RT_TDDFT_H
#define RT_TDDFT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RT_OK       0
#define RT_EINVAL  -1   /* bad argument / unsupported shape            */
#define RT_ENOMEM  -2   /* not enough device memory for the workspaces */
#define RT_ECUDA   -3   /* CUDA runtime error (message in rt_last_error) */
#define RT_ESTATE  -4   /* handle poisoned by an earlier error, or NULL */
#define RT_ENUMERIC -5  /* non-finite value on the device, or a dynamic loop of Alg. 1 ran out of iterations */

/* rt_config.flags */
#define RT_PHI_DEVICE  1u   /* `phi` is a DEVICE pointer that the library BORROWS (never copies, never writes)
                               for the lifetime of the handle; otherwise phi is HOST memory and is copied   */
#define RT_NO_HARTREE  2u   /* test aid: drop V_H from dV                                                */
#define RT_NO_XC       4u   /* test aid: drop vxc(rho) - vxc(rho0) from dV                               */
#define RT_NO_GRAPH    8u   /* launch kernels directly instead of replaying a CUDA graph of one step     */
#define RT_NO_TMA     16u   /* use the cp.async versions of the DMMA kernels even where TMA applies (the
                               library falls back to them by itself when Ng is odd or phi is not 16-byte aligned) */

#define RT_NONORTHOGONAL 32u /* Phi is a NON-orthonormal basis of real functions: S = dVol Phi Phi^T != 1 and P is propagated
                               with Eq. 33-38.  Needs rt_create_general and RT_PROP_COMMUTATOR      */

/* rt_config.propagator */
#define RT_PROP_TAYLOR      0   /* U = exp(-i Hbar dt) by a fixed-degree Taylor polynomial, then P1 = U P0 U^dagger      */
#define RT_XC_LDA_PZ81 0
#define RT_XC_PBE      1
#define RT_PROP_COMMUTATOR  1   /* the paper's own series applied to P: dP^(k) = (-i dt/k)[Hbar, dP^(k-1)],
                                   P1 = P0 + sum_k dP^(k) until max|dP^(k)| <= dP_thrs (Eq. 39, Alg. 1 lines
                                   15-23 L375-L392; real/imaginary split of Eq. 40)                          */

typedef struct rt_ctx* rt_handle;

typedef struct {
  int32_t  nx, ny, nz;      /* periodic grid, each >= 2; Ng = nx*ny*nz                                       */
  double   h;               /* spacing (bohr) > 0                                                            */
  int32_t  norb;            /* N = N_occ + N_virt >= 1 (Alg. 1 line 2)                                       */
  double   dt;              /* time step (a.u.) > 0                                                          */
  int32_t  n_hupdates;      /* m >= 1 Hamiltonian updates per step; 0 -> 2                   */
  int32_t  n_vcycles;       /* V-cycles per Poisson solve >= 0; there are m solves per step (DESIGN R9)      */
  int32_t  nu_pre, nu_post; /* Jacobi sweeps before / after the coarse correction; 0,0 -> 2,2                */
  double   jacobi_omega;    /* damping; 0 -> 6/7                                                             */
  int32_t  exp_order;       /* K = degree in X of the Taylor polynomial of exp(-iX); 0 -> chosen from the
                               spectral bound so that the truncation term <= 1e-17 (DESIGN R8)               */
  double   E0[3];           /* field in force at t = 0 (the delta-"kick", Eq. 41, DESIGN R5)            */
  uint32_t flags;           /* RT_* flags above                                                              */
  int32_t  device;          /* CUDA device ordinal                                                           */
  void*    stream;          /* cudaStream_t all work is enqueued on (e.g. torch.cuda.current_stream()); NULL = legacy default */
  /* -- the paper's dynamic loops (Alg. 1 line 5, L351); all zero = the fixed-count step described above -- */
  int32_t  propagator;      /* RT_PROP_TAYLOR (0) or RT_PROP_COMMUTATOR                                       */
  int32_t  max_order;       /* commutator series: largest order k; 0 -> from the spectral bound (<= 96)       */
  double   dP_thrs;         /* commutator series: stop when max|dP^(k)| <= dP_thrs; 0 -> 1e-10                */
  double   H_thrs;          /* > 0: repeat the Hamiltonian update while max|H1 - H1_old| > H_thrs (Alg. 1 lines
                               12-13, 24-26; L483) instead of n_hupdates times.  rt_step then synchronises the
                               host once per update (it reads the 8-byte error norm)                           */
  int32_t  max_hupdates;    /* bound on the updates per step when H_thrs > 0; 0 -> 20                          */
  /* -- grid-slab sharding (the paper's own decomposition): this handle owns the x-planes
   *    [slab_x0, slab_x0 + slab_nx) of the nx*ny*nz grid and `phi` holds only those: [norb][slab_nx*ny*nz].
   *    slab_nx = 0: the whole grid (single GPU; every entry point above).  slab_nx > 0: see rt_slab_* below.   */
  int32_t  slab_x0, slab_nx;
  /* -- dipole history: > 0 keeps the dipole of the last `history` time levels on the device, appended by the step
   *    itself (no host synchronisation per step); read with rt_get_dipole_series.  0 = off.                        */
  int32_t  history;
  /* -- row-sharded N x N propagator on slab handles (the replicated N^3 work is replaced by a
   *    multi-GPU product "once N exceeds a few thousands"): rank prop_shard of prop_shards owns a block of whole
   *    128-row tiles of every N x N product of a2-a4; the caller all-gathers the blocks at three points of a
   *    Hamiltonian update (rt_slab_get_shard, RT_SLAB_PROP_A..D).  0 or 1 = replicated propagator.  Taylor mode only. */
  int32_t  prop_shards, prop_shard;
  /* -- closer-to-paper physics; all zero = the north_star step ------------------------------- */
  int32_t  magnus_order;    /* 0 or 1: Omega = Omega_1 (Eq. 12, "mid-point"); 2: + Omega_2 = dt^2/12 [H0, H1] (Eq. 13,
                               L125), fourth order in dt.  Needs RT_PROP_COMMUTATOR (the series takes any Omega)     */
  int32_t  xc_functional;   /* RT_XC_LDA_PZ81 (0, north_star) or RT_XC_PBE (the functional the paper ran, L453, L501):
                               v_xc = de/dn - sum_q D_q (2 de/dsigma D_q rho) with central differences D of fd_order    */
  int32_t  fd_order;        /* order of the finite-difference operators on the grid (Eq. 2): 0 or 2 = 7-point
                               Laplacian in the Hartree solve and 2-point gradients; 4 = the 13-point fourth-order
                               Laplacian as the operator V_H solves -- each of the n_vcycles cycles is then
                               r = f - A4 u, d = one 7-point V-cycle on (0, r), u += d (multigrid as the preconditioner,
                               L77; DESIGN R17) -- and 4-point gradients                                              */
} rt_config;

/* Alg. 1 lines 4-8 (L348-L358): t = 0, P0 = diag(occ), rho0, vxc(rho0), V_H = 0,
 * H0 = H-1 = diag(eps) + Proj(E0.r).   phi: [norb][Ng] HOST (copied) or DEVICE (borrowed, RT_PHI_DEVICE);
 * eps, occ: [norb] HOST, copied; occ in [0,2].  *out receives the handle (owned by the caller -> rt_destroy). */
int rt_create(const rt_config* cfg, const double* phi, const double* eps, const double* occ, rt_handle* out);

/* The same with the ground state given as MATRICES in the basis Phi (all HOST, row-major [norb][norb], copied):
 * Hks = <phi_i|H_KS|phi_j>, P0re/P0im = the density matrix at t = 0 (P0im may be NULL = 0; tr(P0 S) = N_e), eps[norb] =
 * the Kohn-Sham eigenvalues (only their range is used: spectral shift and the bound that sizes the series).  With
 * RT_NONORTHOGONAL the library forms S = dVol Phi Phi^T and S^-1 itself.  H0 = H-1 = Hks + Proj(E0.r). */
int rt_create_general(const rt_config* cfg, const double* phi, const double* eps, const double* Hks, const double* P0re,
                      const double* P0im, rt_handle* out);

/* Field E(t_{n+1}) used by the following step(s): HOST double[3]; sticky; default (0,0,0).  The three values are read
 * before the call returns (they travel to the device as kernel arguments), so the buffer may be reused at once.
 * RT_EINVAL when |E| is so large that the series order fixed at rt_create (DESIGN R8: spectral bound with E0 and a
 * 0.5 Ha margin) would leave a truncation term above 1e-15 -- create the handle with that E0 or an explicit order. */
int rt_set_field(rt_handle h, const double E[3]);

/* Enqueue nsteps >= 0 time steps on the stream.  Does not synchronise the host. */
int rt_step(rt_handle h, int32_t nsteps);

/* Dipole mu[3] (HOST) at the current time: dVol sum_r r rho(r) (Alg. 1 line 27).  Synchronises the stream. */
int rt_get_dipole(rt_handle h, double mu[3]);

/* Density rho(r) at the current time into rho[Ng] (EITHER).  Synchronises the stream. */
int rt_get_density(rt_handle h, double* rho);

/* Dipole time series mu(t_k), k = first .. first + n - 1 (k = 0 is t = 0), into out[n][4] (HOST): mu_x, mu_y, mu_z and
 * the charge dVol sum rho.  Needs rt_config.history > 0; only the last `history` levels are kept (RT_EINVAL for
 * older or future ones, and for levels before the one restored by rt_set_state).  Synchronises the stream once,
 * however many steps were enqueued. */
int rt_get_dipole_series(rt_handle h, int64_t first, int32_t n, double* out);

/* ---- checkpoint / resume ---------------------------------------------------------------------------
 * The propagation state of Algorithm 1 between two steps: t, P0 (re, im), H0, H-1 (line 28), the warm-start V_H, the
 * field E(t_next), rho and its five sums -- (4 norb^2 + 2 Ng + 16) doubles plus a 64-byte header; Phi, eps, occ and the
 * configuration are NOT part of it (the caller owns them).  A run restored into a handle created with the same
 * configuration continues bit-identically.  buf: HOST memory of rt_state_bytes() bytes.  Both calls synchronise.
 * rt_set_state returns RT_EINVAL when the header does not match the handle (norb, grid, dt) and leaves it untouched.
 * The dipole history (rt_config.history) restarts at the restored time level. */
int rt_state_bytes(rt_handle h, int64_t* nbytes);
int rt_get_state(rt_handle h, void* buf);
int rt_set_state(rt_handle h, const void* buf);

/* ---- diagnostics / test aids ------------------------------------------------------------------ */

/* P(t) = re + i im, each [norb][norb] (EITHER; either pointer may be NULL).  Synchronises. */
int rt_get_pmatrix(rt_handle h, double* re, double* im);
/* H0 (the Hamiltonian at the current time, [norb][norb], EITHER).  Synchronises. */
int rt_get_hmatrix(rt_handle h, double* H0);
/* Energy diagnostic (HOST double): E = sum_i eps_i Re P_ii + dVol sum_r [1/2 drho V_H + e_xc(rho) - e_xc(rho0)
 * - v_xc(rho0) drho + E(t_next).r drho] with the current (fixed-cycle) V_H; its derivative with respect to rho is the dV
 * of the step, so it is conserved once the field is off ("conservation of energy", Figs. 3-4).
 * Three small kernels; synchronises. */
int rt_get_energy(rt_handle h, double* energy);
/* Warm-start Hartree potential V_H[Ng] (EITHER).  Synchronises. */
int rt_get_vhartree(rt_handle h, double* vh);
/* Overlap matrix S = dVol Phi Phi^T and its inverse as the library computed them (RT_NONORTHOGONAL handles; each
 * [norb][norb], EITHER, either may be NULL).  Synchronises. */
int rt_get_overlap(rt_handle h, double* S, double* Sinv);
/* Current time t (HOST). */
int rt_get_time(rt_handle h, double* t);
/* Integrals of the current density, HOST double[2]: { dVol sum rho , dVol sum (rho - rho0) }.  Synchronises. */
int rt_get_charge(rt_handle h, double q[2]);
/* info[0] = exp_order K actually used, info[1] = number of multigrid levels, info[2..4] = coarsest nx,ny,nz,
 * info[5] = 1 if steps (or slab phases) replay a CUDA graph, +2 if the TMA-fed DMMA kernels are in use, +4 if a slab
 * phase capture was ever invalidated from outside (that phase was then enqueued directly), +8 / +16 if the projection /
 * density launches run persistent CTAs in lock-step (producer pacing, large systems only), info[6] = kernels launched
 * per step, info[7] = split-K of the projection.  HOST int32[8]. */
int rt_get_info(rt_handle h, int32_t info[8]);
/* Total number of this library's kernel launches enqueued through the handle so far (graph replays count the
 * kernels inside the graph).  HOST. */
int rt_get_launch_count(rt_handle h, int64_t* n);
/* What the loops of Alg. 1 did in the most recent step.  HOST: n[0] = Hamiltonian updates (n_hupdates unless
 * H_thrs > 0), n[1] = orders summed by the commutator series in the last update (0 with RT_PROP_TAYLOR);
 * err[0] = last max|H1 - H1_old| (0 unless H_thrs > 0), err[1] = last max|dP^(k)|.  Synchronises.  Returns
 * RT_ENUMERIC (outputs filled) when the last commutator series went non-finite or used max_order terms without
 * reaching dP_thrs; with H_thrs > 0 rt_step itself returns RT_ENUMERIC in those cases. */
int rt_get_convergence(rt_handle h, int32_t n[2], double err[2]);
/* Text of the last error on this handle (or of the last failed rt_create when h == NULL).  Never NULL. */
const char* rt_last_error(rt_handle h);
/* Frees every workspace (not a borrowed phi).  NULL is accepted. */
int rt_destroy(rt_handle h);

/* ---- per-stage entry points: the rows of the hot path one at a time (parity tests, roofline timing) ----
 * They use the handle's Phi, grid, stream and scratch space but do NOT touch the propagation state
 * (P, H history, V_H, t).  All enqueue on the stream and synchronise before returning. */

/* a1 "Hupdate": out[N][N] = dVol * Phi diag(v) Phi^T   (v[Ng], out: EITHER).  Eq. 4 (L68-L71), Alg. 1 line 25. */
int rt_op_project(rt_handle h, const double* v, double* out);
/* a5 "Rho" + a6: rho[Ng] = sum_ij S_ij phi_i phi_j for a real SYMMETRIC S[N][N] (reP, rho: EITHER);
 * sums (HOST double[5], may be NULL) = { sum rho, sum x rho, sum y rho, sum z rho, sum (rho - rho0) } (no dVol). */
int rt_op_density(rt_handle h, const double* reP, double* rho, double sums[5]);
/* a2-a4 "ELDYN": P1 = U P0 U^dagger with U = exp(-i Hbar dt), Hbar real symmetric, P0 Hermitian
 * (all [N][N], EITHER).  Eq. 12 (L123), Eq. 15 (L143). */
int rt_op_propagate(rt_handle h, const double* Hbar, const double* P0re, const double* P0im,
                    double* P1re, double* P1im);
/* a7 "Vh": n_vc V-cycles on -lap_h V = 4 pi (drho - mean drho), warm-started from vh (in/out) (EITHER); lap_h and the
 * cycle follow rt_config.fd_order. */
int rt_op_hartree(rt_handle h, double* vh, const double* drho, int32_t n_vc);
/* a8 "exchange/correlation": vxc[Ng] = potential of rho[Ng] (EITHER): Slater + PZ81, or PBE with rt_config.xc_functional. */
int rt_op_vxc(rt_handle h, const double* rho, double* vxc);

/* ---- grid-slab sharding: one handle per rank, phases separated by the two exchanges of the method --------
 * The grid contractions are local to a slab (a5: rho on the slab; a1: a partial sum of dH over the slab, L424);
 * the N x N propagator (a2-a4) and the O(Ng) Poisson / xc stages (a7, a8) are replicated on every rank.  Between the
 * phases the CALLER combines two library-owned device buffers across ranks with a SUM all-reduce (NCCL through
 * torch.distributed in paper_2410_09189_b200/slab.py):
 *   xchg_rho [Ng + 8]    : rho on the full grid (each rank writes its slab, zeros elsewhere) followed by the five
 *                          partial sums { sum rho, sum x rho, sum y rho, sum z rho, sum (rho - rho0) } + 3 pad
 *   xchg_H   [norb*ldn]  : partial H1 = dVol Phi_slab diag(dV) Phi_slab^T (+ diag(eps) on the rank with slab_x0 = 0)
 * A handle created with slab_nx > 0 accepts rt_slab_*, the getters and rt_set_field; rt_step and rt_op_* return
 * RT_ESTATE.  Sequence (every rank, same order):
 *   rt_create                      -> local rho0 slab in xchg_rho, partial H(t=0) in xchg_H
 *   [all-reduce xchg_rho, xchg_H]     rt_slab_phase(h, RT_SLAB_INIT, 0)
 *   per time step, it = 0, 1, ... :
 *     rt_slab_phase(h, RT_SLAB_PROPAGATE, it)  (a2-a5, a6 partial)   [all-reduce xchg_rho]
 *     rt_slab_phase(h, RT_SLAB_POTENTIAL, it)  (a7, a8, a1 partial)  [all-reduce xchg_H]
 *     rt_slab_phase(h, RT_SLAB_CHECK, it)      (Alg. 1 lines 12-13, 24: one more update?)  rt_slab_more_updates
 *   rt_slab_phase(h, RT_SLAB_SHIFT, 0)         (Alg. 1 line 28)
 * With rt_config.prop_shards > 1 RT_SLAB_PROPAGATE is replaced by four phases with all-gathers of row blocks between
 * them (buffers from rt_slab_get_shard; every rank's block is block_count doubles at offset prop_shard * block_count):
 *     RT_SLAB_PROP_A (a2, Y = X^2 rows)                    [all-gather Y]
 *     RT_SLAB_PROP_B (a3 series, first half of a4, rows)   [all-gather C, S]
 *     RT_SLAB_PROP_C (second half of a4, rows)             [all-gather P1re, P1im]
 *     RT_SLAB_PROP_D (P1 made exactly Hermitian, a5, a6 partial)   [all-reduce xchg_rho]
 * Phases enqueue on the handle's stream and do not synchronise (RT_SLAB_CHECK does when H_thrs > 0: it reads the 8-byte
 * error norm); the collectives must run on the same stream (or be ordered after it).  Each phase is captured into a
 * CUDA graph on first use and replayed afterwards (unless RT_NO_GRAPH). */
#define RT_SLAB_INIT      0
#define RT_SLAB_PROPAGATE 1
#define RT_SLAB_POTENTIAL 2
#define RT_SLAB_SHIFT     3
#define RT_SLAB_PROP_A    4
#define RT_SLAB_PROP_B    5
#define RT_SLAB_PROP_C    6
#define RT_SLAB_PROP_D    7
#define RT_SLAB_CHECK     8
typedef struct {
  double* xchg_rho;  int64_t xchg_rho_count;   /* DEVICE, Ng + 8 doubles                          */
  double* xchg_H;    int64_t xchg_H_count;     /* DEVICE, norb * ldn doubles (ldn = norb rounded up to 8) */
  int64_t slab_offset, slab_count;             /* this rank's range of grid points inside xchg_rho */
} rt_slab_buffers;
typedef struct {
  double *Y, *C, *S, *P1re, *P1im;             /* DEVICE, total_count doubles each: [prop_shards * rows_per_rank][ldn]   */
  int64_t block_count;                         /* doubles per rank block (rows_per_rank * ldn)                          */
  int64_t total_count;                         /* >= prop_shards * block_count                                           */
  int32_t prop_shards, prop_shard;
} rt_shard_buffers;
int rt_slab_get_buffers(rt_handle h, rt_slab_buffers* out);
int rt_slab_get_shard(rt_handle h, rt_shard_buffers* out);
int rt_slab_phase(rt_handle h, int32_t phase, int32_t it);
/* After RT_SLAB_CHECK(it) (or RT_SLAB_POTENTIAL(it) on a fixed-count handle): *more (HOST) = 1 if Algorithm 1 wants
 * another Hamiltonian update in this time step (fixed count: it + 1 < n_hupdates; H_thrs > 0: max|H1 - H1_old| >
 * H_thrs and it + 1 < max_hupdates), else 0.  Identical on every rank. */
int rt_slab_more_updates(rt_handle h, int32_t* more);

/* ---- per-stage timing (CUDA events on the launching stream) ------------------------------------
 * Stage ids follow Table 1 (L543-L547) plus the rest of the step. */
#define RT_STAGE_HUPDATE 0   /* a1 projection (+ split-K reduce)          */
#define RT_STAGE_RHO     1   /* a5 density (+ partial reduce, a6 dipole)  */
#define RT_STAGE_VH      2   /* a7 multigrid Poisson                      */
#define RT_STAGE_ELDYN   3   /* a2-a4 mean Hamiltonian, exp series, UPU^+ */
#define RT_STAGE_XC      4   /* a8 vxc + dV assembly                      */
#define RT_STAGE_COUNT   5
/* enable != 0: later rt_step calls bracket every stage with cudaEvents (and bypass the CUDA graph). */
int rt_timing_enable(rt_handle h, int32_t enable);
/* Synchronises; ms[RT_STAGE_COUNT] (HOST) = accumulated device milliseconds per stage since the last call,
 * calls[RT_STAGE_COUNT] (HOST) = number of times each stage ran.  Resets the accumulators. */
int rt_timing_read(rt_handle h, double ms[RT_STAGE_COUNT], int64_t calls[RT_STAGE_COUNT]);

/* ---- photoabsorption spectrum from delta-kick runs (post-processing kernel, stateless) ------------------
 * "Photoabsorption spectra are calculated as a sum of Fourier transforms of mu_x(t), mu_y(t) and mu_z(t) obtained from
 * three independent simulations with the kick ... along x, y, and z".  The paper prints no formula;
 * DESIGN R16 takes the standard dipole strength function
 *   S(w) = -(2 w / (3 pi)) sum_q (1/kappa_q) Im  dt sum_n' c_n [mu_q(t_n) - mu_q(0)] exp((i w - gamma)(t_n - t_kick))
 * with trapezoid weights c_n (1/2 at both ends), t_n = n dt, n = 0..nt-1, kappa_q the delivered impulse (E_kick dt / 2
 * for the end-point sampled kick of DESIGN R5, with t_kick = dt / 2) and an exponential damping gamma.
 * mu: [3][nt] (HOST or DEVICE), row q = the q-component of the dipole of the run kicked along q; a row whose
 * kappa_q == 0 is skipped (and the 1/3 becomes 1/(number of rows used)).  omega: [nw], S: [nw] (HOST or DEVICE).
 * Runs on `device` / `stream` (cudaStream_t) and synchronises the stream before returning. */
int rt_spectrum(const double* mu, int32_t nt, double dt, double t_kick, const double kappa[3], double gamma,
                const double* omega, int32_t nw, double* S, int32_t device, void* stream);

/* Same, for the end-point sampled kick of this library (DESIGN R5): E_kick[3] (HOST) is the rt_config.E0 of the three
 * runs (component q = field of the run kicked along q); kappa_q = E_q dt / 2 and t_kick = dt / 2 are formed here. */
int rt_spectrum_kick(const double* mu, int32_t nt, double dt, const double E_kick[3], double gamma, const double* omega,
                     int32_t nw, double* S, int32_t device, void* stream);

/* ---- an entry point that allocates nothing --------------------------------------------------------------------
 * a6 (Alg. 1 line 27: mu = dVol sum_r r rho(r), charge = dVol sum_r rho(r)) of a density that is already
 * on the device, for callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops, harnesses
 * that forbid it): no handle, no cudaMalloc / cudaFree / allocating library call inside.  The block partial sums of
 * the two-stage reduction live in ONE file-scope device array (160 KB, held by every GPU that loads the library until
 * the process exits), which bounds the grid: nx*ny*nz <= RT_NOALLOC_MAX_POINTS, larger grids are refused with RT_EINVAL
 * and the limit in rt_last_error(NULL).
 * rho: [nx*ny*nz] DEVICE, read only.  out: DEVICE double[5], written = { mu_x, mu_y, mu_z, dVol sum rho, dVol sum |rho| }
 * with the centred coordinates of this library (x(i) = (i - (nx-1)/2) h, DESIGN R4) and dVol = h^3.
 * Enqueues two kernels on `stream` (cudaStream_t) of `device` and returns without synchronising (RT_ECUDA if a launch
 * is refused).  Nothing in the scratch needs clearing between calls (every partial that is read was written by the
 * same call), but ALL calls share it -- from any thread, stream or handle of the process: two calls that overlap on the
 * GPU race on it and both results are undefined.  Serialise them (same stream, or an event between the streams). */
#define RT_NOALLOC_MAX_POINTS 4194304
int rt_dipole_noalloc(const double* rho, int32_t nx, int32_t ny, int32_t nz, double h, double* out, int32_t device,
                      void* stream);

/* ---- calibration instrument (not on the hot path) ----------------------------------------------------
 * Measures the FP64 issue-rate ceilings of `device` with register-resident operands: DMMA.8x8x4 (mma.sync
 * m8n8k4 f64) and DFMA, in TFLOP/s (HOST doubles).  Takes ~0.5 s.  The roofline fractions bench.py reports for
 * the a1/a3/a4/a5 kernels are quoted against the DMMA figure measured in the same run. */
int rt_probe_fp64_peak(int32_t device, double* dmma_tflops, double* dfma_tflops);

#ifdef __cplusplus
}
#endif
#endif /* RT_TDDFT_H */
