// rt_internal.h -- launcher prototypes shared between the kernel translation units and rt_api.cu.
// Not part of the public ABI (that is include/rt_tddft.h).
#pragma once
#include <string>
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace rt {

constexpr int TILE = 128;        // CTA tile edge of the DMMA kernels (orbital index)

struct GridDims { int nx, ny, nz; };

// ---- a1 projection: W[s][i][j] = sum_{r in chunk s} phi_i(r) w(r) phi_j(r) for upper tiles (ti <= tj) -----
// Three classes of tiles, listed in this order: the Tfull full off-diagonal tiles, the Tn off-diagonal tiles of a ragged
// last tile column with at most 96 valid columns (the TMA kernel runs them with 64 x 24 warp tiles at ~0.78 of the cost),
// and the ntile diagonal tiles (~0.65: blocks below the diagonal are not issued).  Each class has its own split-K count
// so that every CTA of the launch costs about the same, and the blocks are ordered class by class, (split, tile) s-major
// inside a class: CTAs that run together then have equal durations and stay in lock-step along k, which is what
// keeps the Phi row panels they share in L2 (measured: 50 % L2 hits with mixed durations against 80 % in lock-step).
struct ProjectPlan {
  int N;                 // orbitals
  long long Ng;          // grid points (contraction length), also the leading dimension of Phi
  int ntile;             // ceil(N / TILE)
  int T;                 // number of upper-triangular tiles
  int Tfull;             // full off-diagonal tiles
  int Tn;                // narrow off-diagonal tiles (0 unless the last tile column has <= 96 valid columns)
  int S;                 // split-K factor of the full tiles
  long long kchunk;      // grid points per split (multiple of 16)
  int Sn;                // ... of the narrow tiles (<= S)
  long long kchunk_n;
  int Sd;                // ... of the diagonal tiles (<= S)
  long long kchunk_d;
  int ldn;               // leading dimension of the N x N outputs
  int grid() const { return S * Tfull + Sn * Tn + Sd * ntile; }
};
struct ProjBlock { int s, t; long long kbeg, kend; };
#ifdef __CUDACC__
__device__ __forceinline__ ProjBlock project_decode(int b, const ProjectPlan& p) {
  ProjBlock r;
  long long kc;
  const int n0 = p.S * p.Tfull, n1 = n0 + p.Sn * p.Tn;
  if (b < n0) { r.s = b / p.Tfull; r.t = b - r.s * p.Tfull; kc = p.kchunk; }
  else if (b < n1) { const int bb = b - n0; r.s = bb / p.Tn; r.t = p.Tfull + (bb - r.s * p.Tn); kc = p.kchunk_n; }
  else { const int bb = b - n1; r.s = bb / p.ntile; r.t = p.Tfull + p.Tn + (bb - r.s * p.ntile); kc = p.kchunk_d; }
  r.kbeg = (long long)r.s * kc;
  r.kend = (r.kbeg + kc < p.Ng) ? r.kbeg + kc : p.Ng;
  return r;
}
#endif
void launch_project(const ProjectPlan& p, const double* phi, const double* w, const int2* tiles, double* W,
                    cudaStream_t st);
// H[i][j] = scale * sum_s W[s][i][j] (+ eps_i if i == j and eps != nullptr) (+ Hadd[i][j] if Hadd != nullptr), mirrored to
// the lower triangle.
void launch_project_reduce(const ProjectPlan& p, const double* W, const double* eps, double scale, double* H,
                           cudaStream_t st, const double* Hadd = nullptr);
size_t project_smem_bytes();

// ---- a5 density: rho_part[p][r] = sum over the j-tiles of pair p of sum_j phi_j(r) (Pfold Phi)_j(r) -------
struct DensityPlan {
  int N;
  long long Ng;
  int ntile;             // j tiles
  int npairs;            // ceil(ntile / 2): CTA handles j-tiles (p, ntile-1-p)
  long long nrt;         // r tiles = ceil(Ng / TILE)
  int ldn;
  int group_r;           // raster: r-tiles per supertile
  int group_t;           // TMA kernel: work types per supertile (group_t * group_r ~ number of SMs)
  int ntypes;            // TMA kernel: work types per r-tile (each owns one partial row); >= npairs
};
// TMA density kernel: one k-segment of j-tile jt: stages s0, s0 + dir, ... (ns of them), stage s covering the
// contraction rows jt*TILE + 16 s ... + 15.  A work type is two consecutive DensSeg (the second may have ns = 0).
struct DensSeg { int jt, s0, ns, dir; };
void launch_density(const DensityPlan& p, const double* phi, const double* Pfold, double* rho_part, cudaStream_t st);
size_t density_smem_bytes();
// Pfold[j][i] = 2 P[j][i] (i > j), P[j][j] (i == j), 0 (i < j)
void launch_fold_upper(int N, int ldn, const double* P, double* Pfold, cudaStream_t st);

// ---- a3/a4 N x N GEMM:  D = alpha0 * A0 B0^T + alpha1 * A1 B1^T ; optional Z1 += beta1 D, Z2 += beta2 D --------
struct GemmArgs {
  int N, ldn;
  const double* A0; const double* B0; double alpha0;
  const double* A1; const double* B1; double alpha1;     // A1 == nullptr -> single term
  double* D;                                            // may be nullptr (only the axpys are wanted)
  double* Z1; double beta1;                             // may be nullptr
  double* Z2; double beta2;
  const int* skip;                                      // device flag (may be nullptr): non-zero -> the launch is a no-op
  int row_beg, row_end;                                 // rows of D computed by this launch (multiples of TILE; row_end
                                                        // clipped to N); 0, N = the whole matrix.  A row block is what
                                                        // one rank of the sharded propagator owns
};
// N <= GEMM_SMALL_N32: 32 x 32 CTA tiles; N <= GEMM_SMALL_N: 64 x 64; above: 128 x 128 (rt_api.cu sends N > GEMM_SMALL_N
// to the TMA-fed kernel when TMA is available)
constexpr int GEMM_SMALL_N32 = 512, GEMM_SMALL_N = 1536;
void launch_gemm_abt(const GemmArgs& g, cudaStream_t st);
size_t gemm_smem_bytes();

// ---- TMA-fed, warp-specialised versions (gemm_tma.cu): default on sm_100a when Phi rows are 16-byte aligned ----
int    init_tma_kernels();                 // sets the dynamic shared-memory attribute; returns a cudaError_t value
size_t tma_smem_bytes();
// tmPhi: Phi [N][Ng] with box {16 k, 128 rows}; w must be readable up to roundup(Ng, 16) doubles
size_t project_tma_pace_ints(const ProjectPlan& p, int sms);   // checkpoint counters of a paced launch (0: not paced)
void launch_project_tma(const ProjectPlan& p, const CUtensorMap& tmPhi, const double* w, const int2* tiles, double* W,
                        int sms, int* pace_cnt, int pace_w, cudaStream_t st);
// tmP: Pfold [N][N] (ld = ldn) box {16, 128}; tmPhiN: Phi with box {16 r, 16 k-rows} (b3d = 0: 8 loads per stage)
// or, when Ng % 16 == 0, the 3-D view {16 r-low, N k, Ng/16 r-high} with box {16, 16, 8} (b3d = 1: one load)
size_t density_tma_pace_ints(const DensityPlan& p, int sms);
void launch_density_tma(const DensityPlan& p, const CUtensorMap& tmP, const CUtensorMap& tmPhiN, int b3d,
                        const double* phi, const DensSeg* segs, double* rho_part, int sms, int* pace_cnt, int pace_w,
                        int hint, cudaStream_t st);
// sym = +1 / -1: the product is known to be symmetric / antisymmetric (polynomials of the symmetric X commute; P1 is
// Hermitian): only the upper tiles (list `tiles`, ti <= tj) are computed and the mirror image is written too
// `tiles` / `ntiles`: the 128 x 128 output tiles of this launch (sym != 0: upper tiles only).  Stream-K: the (tile, stage)
// units are cut into one contiguous range per CTA; ws / sync are the fix-up workspace and flags (gemm_tma_ws_doubles,
// gemm_tma_sync_ints; sync must be zero before the first launch and is left zero by every launch).
void launch_gemm_abt_tma(const GemmArgs& g, const CUtensorMap& tmA0, const CUtensorMap& tmB0, const CUtensorMap& tmA1,
                         const CUtensorMap& tmB1, int sym, const int2* tiles, int ntiles, double* ws, int* sync, int sms,
                         cudaStream_t st);
size_t gemm_tma_ws_doubles(int sms);
size_t gemm_tma_sync_ints(int sms);

// ---- elementwise N x N (a2 and series glue) -------------------------------------------------------------
// first != 0: H1 = 2 H0 - Hm1 first.  X = dt * ((H0 + H1)/2 - sigma I)
// S != nullptr (non-orthogonal basis): X = dt * ((H0 + H1)/2 - sigma S)
void launch_hbar(int N, int ldn, const double* Hm1, const double* H0, double* H1, double* X, double dt,
                 double sigma, int first, cudaStream_t st, const double* S = nullptr);
// dP' = (M + M^dagger)/k from R = Re M, I = Im M: Sn = (R + R^T)/k, An = (I - I^T)/k, P1r += Sn, P1i += An  (L434-L438)
void launch_transpose_add(int N, int ldn, const double* R, const double* I, double inv_k, double* Sn, double* An,
                          double* P1r, double* P1i, const int* skip, cudaStream_t st);
void launch_axpby(int N, int ldn, double a, const double* X, double b, const double* Y, double* out, cudaStream_t st);
// C = I + c1 Y ; S = I + s1 Y
void launch_series_init(int N, int ldn, const double* Y, double* C, double c1, double* S, double s1, cudaStream_t st);
// C = 1 + sum_k c[k-1] Y^k, S = 1 + sum_k s[k-1] Y^k, k = 1..q, from the stored powers pw[k-1] = Y^k
constexpr int SERIES_MAX_Q = 12;
struct SeriesArgs { const double* pw[SERIES_MAX_Q]; double c[SERIES_MAX_Q], s[SERIES_MAX_Q]; int q; };
void launch_series_combine(int N, int ldn, const SeriesArgs& a, double* C, double* S, int row_beg, int row_end,
                           cudaStream_t st);    // rows [row_beg, row_end) only (a rank's block of the sharded propagator)
// dst = src for n matrices (state shift, line 28)
void launch_copy5(int N, int ldn, double* d0, const double* s0, double* d1, const double* s1, double* d2,
                  const double* s2, double* d3, const double* s3, cudaStream_t st);
void launch_set_diag(int N, int ldn, double* M, const double* diag, cudaStream_t st);   // M = diag(d)
// Re[j][i] = Re[i][j], Im[j][i] = -Im[i][j] for j > i, Im[i][i] = 0: makes P exactly Hermitian from its upper triangle
// (the row-sharded propagator computes both triangles separately)
void launch_hermitize(int N, int ldn, double* Re, double* Im, cudaStream_t st);

// ---- grid kernels (a6, a7, a8) ---------------------------------------------------------------------------
// rho[r] = sum_p rho_part[p][r]; block partial sums of {rho, x rho, y rho, z rho, rho - rho0} -> bsums[nb][5]
int  reduce_rho_blocks(long long Ng);
// Ng points starting at x-plane x0 of the grid gd (a grid slab; x0 = 0 and Ng = nx*ny*nz for the whole grid); part,
// rho0, rho point at the first point of the slab
void launch_reduce_rho(const double* rho_part, int nparts, long long Ng, GridDims gd, double h, int x0,
                       const double* rho0, double* rho, double* bsums, double* sums, cudaStream_t st);
// w[r] = (hartree ? VH : 0) + (xc ? vxc(rho) - vxc0 : 0) + E.x(r)
void launch_delta_v(long long Ng, GridDims gd, double h, const double* rho, const double* vxc0, const double* VH,
                    const double* E, int use_h, int use_xc, double* w, cudaStream_t st);
void launch_vxc(long long Ng, const double* rho, double* vxc, cudaStream_t st);
// PBE on the grid (oracle.vxc_pbe): pass 1 a = d e/d n, b_q = 2 d e/d sigma D_q rho (scr: 4 arrays of Ng, [a | bx | by | bz]);
// pass 2 out = a - sum_q D_q b_q; order = 2 or 4 (central differences).  exc != nullptr: also e_xc per point (energy).
void launch_vxc_pbe(GridDims gd, double h, int order, const double* rho, double* scr, double* out, double* exc,
                    cudaStream_t st);
// out[r] = fld(r) + (VH ? VH[r] : 0) + (vxc ? vxc[r] - vxc0[r] : 0)   (dV assembly when v_xc was computed separately)
void launch_energy_exc(long long Ng, GridDims gd, double h, const double* rho, const double* rho0, const double* vxc0,
                       const double* VH, const double* E, const double* exc, const double* exc0, int use_h, int N, int ldn,
                       const double* eps, const double* P0r, double* bsums, double* out, cudaStream_t st);
void launch_delta_v_assemble(long long Ng, GridDims gd, double h, const double* vxc, const double* vxc0, const double* VH,
                             const double* E, double* w, cudaStream_t st);
void launch_field(long long Ng, GridDims gd, double h, const double* E, double* w, cudaStream_t st);
void launch_set_field(double* dE, double ex, double ey, double ez, cudaStream_t st);   // dE[0..2] = E, by value
// f = 4 pi (rho - rho0 - sums[4]/Ng)      (rho0 may be nullptr: f = 4 pi (rho - sums[4]/Ng))
void launch_poisson_rhs(long long Ng, const double* rho, const double* rho0, const double* sums, double* f,
                        cudaStream_t st);

// ---- convergence state of the paper's dynamic loops (Alg. 1 lines 12-13, 16-23) ----
// Lives in device memory; the host reads it only in the dynamic-H_thrs mode and in rt_get_convergence.
constexpr int MAX_ORDER = 96;
struct ConvState {
  unsigned long long dP_bits[MAX_ORDER + 1];   // max|dP^(k)|, bit pattern of a non-negative double (atomicMax)
  unsigned int arrived[MAX_ORDER + 1];         // blocks of commutator_check that have contributed to order k
  int done;                                    // dP_err <= dP_thrs reached: the GEMMs of later orders skip themselves
  int k_used;                                  // orders summed into P1
  unsigned long long H_bits;                   // max|H1 - H1_old| of this Hamiltonian update
};
// after the two GEMMs of order k: dP_err = max(|dPr|, |dPi|) over the matrix; the last block to arrive sets
// k_used = k and done = (dP_err <= thrs).  A no-op once done is set.
void launch_commutator_check(int N, int ldn, const double* dPr, const double* dPi, int k, double thrs, ConvState* cs,
                             cudaStream_t st);
// cs->H_bits = max |A - B| over the N x N matrices (line 24)
void launch_maxabs_diff(int N, int ldn, const double* A, const double* B, ConvState* cs, cudaStream_t st);
void launch_maxabs_minus_identity(int N, int ldn, const double* T, ConvState* cs, cudaStream_t st);
void launch_trace_product(int N, int ldn, const double* A, const double* B, double* out, cudaStream_t st);   // out[5]

// energy diagnostic: out[0] = sum_r [1/2 drho VH + exc(rho) - exc(rho0) - vxc0 drho + E.r drho], out[5] = sum_i eps_i P_ii
void launch_energy(long long Ng, GridDims gd, double h, const double* rho, const double* rho0, const double* vxc0,
                   const double* VH, const double* E, int use_h, int use_xc, int N, int ldn, const double* eps,
                   const double* P0r, double* bsums, double* out, cudaStream_t st);
// dipole history: hist[(count % cap)][4] = { dvol sums[1..3], dvol sums[0] }; count += 1   (one thread)
void launch_record_dipole(const double* sums, double dvol, double* hist, int cap, unsigned long long* count,
                          cudaStream_t st);
// S[iw] per the formula in include/rt_tddft.h (rt_spectrum); one warp per frequency, fixed summation order
void launch_spectrum(const double* mu, int nt, double dt, double t_kick, const double* kappa3, int nused, double gamma,
                     const double* omega, int nw, double* S, cudaStream_t st);

struct MgLevel {
  GridDims gd; double h; long long n;
  double* u; double* tmp; double* f; double* r;     // solution, ping-pong scratch, rhs, residual
};
// One Poisson solve (a7): rhs = 4 pi (rho - rho0 - sums[4]/n), then n_vc V(nu1,nu2) cycles on lv[0].u (warm start).
// The coarse end of the hierarchy runs inside one single-CTA shared-memory kernel per cycle; larger levels use
// shared-memory tile kernels (mg_kernels.cu).  Returns the number of kernels enqueued.
constexpr int MG_MAX_LEVELS = 12;
struct MgSolveArgs {
  const MgLevel* lv; int nlev;
  int n_vc, nu1, nu2; double omega;
  const double *Qx, *Qy, *Qz, *lx, *ly, *lz;     // eigenbasis of the coarsest level (exact zero-mean solve)
  const double* rho; const double* rho0;         // rho0 may be nullptr
  const double* sums;                            // sums[4] = sum(rho - rho0)
  int zero0 = 0;                                 // level 0 starts from a zero guess (the cycle is used as a preconditioner)
  int rhs_given = 0;                             // lv[0].f already holds the right-hand side (rho, rho0, sums unused)
};
int init_mg_kernels();                           // dynamic shared-memory attributes; returns a cudaError_t value
int launch_mg_solve(const MgSolveArgs& s, cudaStream_t st);
// fourth-order operator, the 7-point cycle as preconditioner (mg_kernels.cu); dl0: level-0 arrays of the correction, f4: rhs
int launch_mg_solve_order4(const MgSolveArgs& s, const MgLevel& dl0, double* f4, cudaStream_t st);
// block sums of drho for rt_op_hartree (mean removal): sums[4] = sum(drho)
void launch_sum_only(const double* v, long long n, double* bsums, double* sums, cudaStream_t st);

// ---- noalloc.cu: the a6 reduction on a static device scratch array (no allocation, no handle) ----
long long dipole_noalloc_max_points();
int launch_dipole_noalloc(const double* rho, int nx, int ny, int nz, double h, double* out, int device, cudaStream_t st,
                          std::string* err);

}  // namespace rt
