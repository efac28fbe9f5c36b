// grid_kernels.cu -- HBM/L2-bound stages on the real-space grid and the small N x N glue kernels.
//
//   a6  reduce_rho      : rho = sum of the density kernel's partials, fused dipole / charge reduction
//                         (Alg. 1 line 27) with a fixed-order second stage (bit-reproducible).
//   a7  poisson_rhs     : right-hand side of the Poisson solve (the multigrid cycle itself is in mg_kernels.cu).
//   a8  delta_v / vxc   : Slater exchange + PZ81 correlation and the dV assembly ("exchange/correlation", L547).
//   a2  hbar etc.       : Alg. 1 lines 11, 14, 28 on N x N matrices.
#include "rt_internal.h"

namespace rt {

constexpr int RB = 256;                 // threads per block of the streaming kernels
constexpr int RED_BLOCKS_MAX = 1024;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// block-wide sums of NV values; result valid in thread 0
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double (*sh)[NV]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < NV; ++q) v[q] = warp_sum(v[q]);
  if (lane == 0)
#pragma unroll
    for (int q = 0; q < NV; ++q) sh[warp][q] = v[q];
  __syncthreads();
  if (threadIdx.x == 0) {
    const int nw = blockDim.x >> 5;
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      double s = 0.0;
      for (int w = 0; w < nw; ++w) s += sh[w][q];
      v[q] = s;
    }
  }
}

// ---------------------------------------------------------------------------------------------- a6
int reduce_rho_blocks(long long Ng) {
  long long nb = (Ng + RB * 4 - 1) / (RB * 4);
  return (int)(nb < 1 ? 1 : (nb > RED_BLOCKS_MAX ? RED_BLOCKS_MAX : nb));
}

__global__ void __launch_bounds__(RB)
reduce_rho_kernel(const double* __restrict__ part, int nparts, long long Ng, GridDims gd, double h, int x0,
                  const double* __restrict__ rho0, double* __restrict__ rho, double* __restrict__ bsums) {
  __shared__ double sh[RB / 32][5];
  double v[5] = {0, 0, 0, 0, 0};
  const double cx = 0.5 * (gd.nx - 1), cy = 0.5 * (gd.ny - 1), cz = 0.5 * (gd.nz - 1);
  const long long nyz = (long long)gd.ny * gd.nz;
  for (long long r = (long long)blockIdx.x * RB + threadIdx.x; r < Ng; r += (long long)gridDim.x * RB) {
    double s = 0.0;
    for (int p = 0; p < nparts; ++p) s += part[(long long)p * Ng + r];
    rho[r] = s;
    const int ixl = (int)(r / nyz);                  // plane inside the slab; x0 = first plane of the slab
    const int rem = (int)(r - (long long)ixl * nyz);
    const int iy = rem / gd.nz, iz = rem - iy * gd.nz;
    const int ix = ixl + x0;
    v[0] += s;
    v[1] += ((double)ix - cx) * h * s;
    v[2] += ((double)iy - cy) * h * s;
    v[3] += ((double)iz - cz) * h * s;
    v[4] += rho0 ? (s - rho0[r]) : s;
  }
  block_sum<5>(v, sh);
  if (threadIdx.x == 0)
#pragma unroll
    for (int q = 0; q < 5; ++q) bsums[blockIdx.x * 5 + q] = v[q];
}

__global__ void final_sums_kernel(const double* __restrict__ bsums, int nb, int nv, double* __restrict__ sums) {
  // one warp per value; fixed order: lane-strided partials, then a shuffle tree
  const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (q >= nv) return;
  double s = 0.0;
  for (int b = lane; b < nb; b += 32) s += bsums[b * nv + q];
  s = warp_sum(s);
  if (lane == 0) sums[q] = s;
}

void launch_reduce_rho(const double* rho_part, int nparts, long long Ng, GridDims gd, double h, int x0,
                       const double* rho0, double* rho, double* bsums, double* sums, cudaStream_t st) {
  const int nb = reduce_rho_blocks(Ng);
  reduce_rho_kernel<<<nb, RB, 0, st>>>(rho_part, nparts, Ng, gd, h, x0, rho0, rho, bsums);
  final_sums_kernel<<<1, 32 * 5, 0, st>>>(bsums, nb, 5, sums);
}

__global__ void __launch_bounds__(RB)
sum_only_kernel(const double* __restrict__ v, long long n, double* __restrict__ bsums) {
  __shared__ double sh[RB / 32][5];
  double a[5] = {0, 0, 0, 0, 0};
  for (long long r = (long long)blockIdx.x * RB + threadIdx.x; r < n; r += (long long)gridDim.x * RB) a[4] += v[r];
  block_sum<5>(a, sh);
  if (threadIdx.x == 0)
#pragma unroll
    for (int q = 0; q < 5; ++q) bsums[blockIdx.x * 5 + q] = a[q];
}

void launch_sum_only(const double* v, long long n, double* bsums, double* sums, cudaStream_t st) {
  const int nb = reduce_rho_blocks(n);
  sum_only_kernel<<<nb, RB, 0, st>>>(v, n, bsums);
  final_sums_kernel<<<1, 32 * 5, 0, st>>>(bsums, nb, 5, sums);
}

// ------------------------------------------------------------------------- dipole history and spectrum
__global__ void record_dipole_kernel(const double* __restrict__ sums, double dvol, double* __restrict__ hist, int cap,
                                     unsigned long long* __restrict__ count) {
  if (threadIdx.x == 0) {
    const unsigned long long k = *count;
    double* e = hist + (k % (unsigned long long)cap) * 4;
    e[0] = dvol * sums[1]; e[1] = dvol * sums[2]; e[2] = dvol * sums[3]; e[3] = dvol * sums[0];
    *count = k + 1;
  }
}
void launch_record_dipole(const double* sums, double dvol, double* hist, int cap, unsigned long long* count,
                          cudaStream_t st) {
  record_dipole_kernel<<<1, 32, 0, st>>>(sums, dvol, hist, cap, count);
}

// Dipole strength function (include/rt_tddft.h rt_spectrum).  One warp per frequency: lanes stride over
// the time samples, shuffle tree at the end (fixed order).
__global__ void __launch_bounds__(128)
spectrum_kernel(const double* __restrict__ mu, int nt, double dt, double t_kick, double k0, double k1, double k2,
                int nused, double gamma, const double* __restrict__ omega, int nw, double* __restrict__ S) {
  const int iw = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (iw >= nw) return;
  const double w = omega[iw];
  const double kap[3] = {k0, k1, k2};
  double acc = 0.0;
  for (int q = 0; q < 3; ++q) {
    if (kap[q] == 0.0) continue;
    const double* m = mu + (long long)q * nt;
    const double m0 = m[0];
    double im = 0.0;
    for (int n = lane; n < nt; n += 32) {
      const double t = (double)n * dt - t_kick;
      const double cn = (n == 0 || n == nt - 1) ? 0.5 : 1.0;
      im += cn * (m[n] - m0) * exp(-gamma * t) * sin(w * t);
    }
    im = warp_sum(im);
    acc += im / kap[q];
  }
  if (lane == 0) S[iw] = -(2.0 * w / ((double)nused * 3.14159265358979323846)) * dt * acc;
}
void launch_spectrum(const double* mu, int nt, double dt, double t_kick, const double* kappa3, int nused, double gamma,
                     const double* omega, int nw, double* S, cudaStream_t st) {
  spectrum_kernel<<<(nw + 3) / 4, 128, 0, st>>>(mu, nt, dt, t_kick, kappa3[0], kappa3[1], kappa3[2], nused, gamma, omega,
                                                 nw, S);
}

// ---------------------------------------------------------------------------------------------- a8
// Slater exchange + Perdew-Zunger 1981 correlation, unpolarised (DESIGN R7); branch on rho <= 3/(4 pi).
__device__ __forceinline__ double vxc_pz81(double rho) {
  if (!(rho >= 1e-30)) return 0.0;
  const double PI = 3.14159265358979323846;
  const double vx = -cbrt(3.0 * rho / PI);
  const double rs = cbrt(3.0 / (4.0 * PI * rho));
  double vc;
  if (rho <= 3.0 / (4.0 * PI)) {
    const double sq = sqrt(rs);
    const double den = 1.0 + 1.0529 * sq + 0.3334 * rs;
    const double ec = -0.1423 / den;
    vc = ec * (1.0 + (7.0 / 6.0) * 1.0529 * sq + (4.0 / 3.0) * 0.3334 * rs) / den;
  } else {
    const double ln = log(rs);
    vc = 0.0311 * ln + (-0.048 - 0.0311 / 3.0) + (2.0 / 3.0) * 0.0020 * rs * ln + ((2.0 * -0.0116 - 0.0020) / 3.0) * rs;
  }
  return vx + vc;
}

// e_xc(rho) = rho (eps_x + eps_c) per unit volume, eps_x = 3/4 v_x (energy diagnostic only)
__device__ __forceinline__ double exc_pz81(double rho) {
  if (!(rho >= 1e-30)) return 0.0;
  const double PI = 3.14159265358979323846;
  const double ex = -0.75 * cbrt(3.0 * rho / PI);
  const double rs = cbrt(3.0 / (4.0 * PI * rho));
  double ec;
  if (rho <= 3.0 / (4.0 * PI)) ec = -0.1423 / (1.0 + 1.0529 * sqrt(rs) + 0.3334 * rs);
  else { const double ln = log(rs); ec = 0.0311 * ln + -0.048 + 0.0020 * rs * ln + -0.0116 * rs; }
  return rho * (ex + ec);
}

__device__ __forceinline__ double field_at(long long r, GridDims gd, double h, const double* __restrict__ E) {
  const long long nyz = (long long)gd.ny * gd.nz;
  const int ix = (int)(r / nyz);
  const int rem = (int)(r - (long long)ix * nyz);
  const int iy = rem / gd.nz, iz = rem - iy * gd.nz;
  return E[0] * (((double)ix - 0.5 * (gd.nx - 1)) * h) + E[1] * (((double)iy - 0.5 * (gd.ny - 1)) * h) +
         E[2] * (((double)iz - 0.5 * (gd.nz - 1)) * h);
}

__global__ void __launch_bounds__(RB)
delta_v_kernel(long long Ng, GridDims gd, double h, const double* __restrict__ rho, const double* __restrict__ vxc0,
               const double* __restrict__ VH, const double* __restrict__ E, int use_h, int use_xc,
               double* __restrict__ w) {
  const long long r = (long long)blockIdx.x * RB + threadIdx.x;
  if (r >= Ng) return;
  double v = field_at(r, gd, h, E);
  if (use_h) v += VH[r];
  if (use_xc) v += vxc_pz81(rho[r]) - vxc0[r];
  w[r] = v;
}

__global__ void __launch_bounds__(RB) vxc_kernel(long long Ng, const double* __restrict__ rho, double* __restrict__ out) {
  const long long r = (long long)blockIdx.x * RB + threadIdx.x;
  if (r < Ng) out[r] = vxc_pz81(rho[r]);
}

__global__ void __launch_bounds__(RB)
field_kernel(long long Ng, GridDims gd, double h, const double* __restrict__ E, double* __restrict__ w) {
  const long long r = (long long)blockIdx.x * RB + threadIdx.x;
  if (r < Ng) w[r] = field_at(r, gd, h, E);
}

__global__ void trace_eps_kernel(int N, int ldn, const double* __restrict__ eps, const double* __restrict__ P,
                                 double* __restrict__ out);
// ---------------------------------------------------------------------------------------------- a8, GGA
// PBE (Perdew, Burke, Ernzerhof, PRL 77, 3865), unpolarised, with PW92 uniform-gas correlation -- the functional the
// paper ran.  Same formulas, symbols and operation order as oracle.pbe_exc:
//   e = e_x + e_c,  de/dn,  de/dsigma  at (n, sigma = |D n|^2).
__device__ __forceinline__ void pbe_point(double n, double sigma, double& e, double& dn, double& ds) {
  e = dn = ds = 0.0;
  if (!(n >= 1e-30)) return;
  const double PI = 3.14159265358979323846;
  const double KAPPA = 0.804, BETA = 0.06672455060314922;
  const double GAMMA = (1.0 - 0.6931471805599453) / (PI * PI);
  const double MU = BETA * PI * PI / 3.0;
  const double A0 = 0.0310907, AL1 = 0.21370, B1 = 7.5957, B2 = 3.5876, B3 = 1.6382, B4 = 0.49294;
  // exchange
  const double Cx = 0.75 * cbrt(3.0 / PI);
  const double n13 = cbrt(n);
  const double n23 = n13 * n13, n43 = n23 * n23, n83 = n43 * n43;
  const double c32 = cbrt(3.0 * PI * PI);
  const double q = 1.0 / (4.0 * c32 * c32 * n83);
  const double p = sigma * q;
  const double den = 1.0 + MU * p / KAPPA;
  const double F = 1.0 + KAPPA - KAPPA / den;
  const double dF = MU / (den * den);
  const double ex = -Cx * n * n13 * F;
  const double dex_dn = -Cx * n13 * ((4.0 / 3.0) * F - (8.0 / 3.0) * p * dF);
  const double dex_ds = -Cx * n * n13 * dF * q;
  // correlation (PW92 + H)
  const double rs = cbrt(3.0 / (4.0 * PI * n));
  const double sq = sqrt(rs);
  const double G = B1 * sq + B2 * rs + B3 * rs * sq + B4 * rs * rs;
  const double dG = 0.5 * B1 / sq + B2 + 1.5 * B3 * sq + 2.0 * B4 * rs;
  const double lg = log(1.0 + 1.0 / (2.0 * A0 * G));
  const double eps = -2.0 * A0 * (1.0 + AL1 * rs) * lg;
  const double deps_drs = -2.0 * A0 * AL1 * lg + (1.0 + AL1 * rs) * dG / (G * G + G / (2.0 * A0));
  const double deps_dn = deps_drs * (-rs / (3.0 * n));
  const double du_ds = PI / (16.0 * c32 * n43 * n);            // n^(7/3)
  const double u = sigma * du_ds;
  const double ex1 = exp(-eps / GAMMA);
  const double A = (BETA / GAMMA) / (ex1 - 1.0);
  const double dA_deps = A * A * ex1 / BETA;
  const double Au = A * u;
  const double Dn = 1.0 + Au + Au * Au;
  const double Q = u * (1.0 + Au) / Dn;
  const double H = GAMMA * log(1.0 + (BETA / GAMMA) * Q);
  const double HQ = BETA / (1.0 + (BETA / GAMMA) * Q);
  const double Qu = (1.0 + 2.0 * Au) / (Dn * Dn);
  const double QA = -A * u * u * u * (2.0 + Au) / (Dn * Dn);
  const double du_dn = -(7.0 / 3.0) * u / n;
  const double ec = n * (eps + H);
  const double dec_dn = eps + H + n * (deps_dn + HQ * (Qu * du_dn + QA * dA_deps * deps_dn));
  const double dec_ds = n * HQ * Qu * du_ds;
  e = ex + ec; dn = dex_dn + dec_dn; ds = dex_ds + dec_ds;
}

__device__ __forceinline__ int wrap_idx(int i, int n) { i %= n; return i < 0 ? i + n : i; }

// central-difference derivative along one axis at point (ix, iy, iz); ORDER = 2: (f+ - f-)/2h, 4: (2/3)(f+1 - f-1) - (1/12)(f+2 - f-2)
template <int ORDER>
__device__ __forceinline__ double ddx(const double* __restrict__ f, GridDims gd, int ix, int iy, int iz, int axis,
                                      double inv_h) {
  auto at = [&](int d) {
    const int x = axis == 0 ? wrap_idx(ix + d, gd.nx) : ix;
    const int y = axis == 1 ? wrap_idx(iy + d, gd.ny) : iy;
    const int z = axis == 2 ? wrap_idx(iz + d, gd.nz) : iz;
    return f[((long long)x * gd.ny + y) * gd.nz + z];
  };
  double g = (ORDER == 2 ? 0.5 : 2.0 / 3.0) * (at(1) - at(-1));
  if (ORDER == 4) g += (-1.0 / 12.0) * (at(2) - at(-2));
  return g * inv_h;
}

template <int ORDER>
__global__ void __launch_bounds__(RB)
pbe_pass1_kernel(GridDims gd, double inv_h, const double* __restrict__ rho, double* __restrict__ scr,
                 double* __restrict__ exc) {
  const long long n = (long long)gd.nx * gd.ny * gd.nz;
  const long long r = (long long)blockIdx.x * RB + threadIdx.x;
  if (r >= n) return;
  const int nyz = gd.ny * gd.nz;
  const int ix = (int)(r / nyz), rem = (int)(r - (long long)ix * nyz), iy = rem / gd.nz, iz = rem - iy * gd.nz;
  const double gx = ddx<ORDER>(rho, gd, ix, iy, iz, 0, inv_h);
  const double gy = ddx<ORDER>(rho, gd, ix, iy, iz, 1, inv_h);
  const double gz = ddx<ORDER>(rho, gd, ix, iy, iz, 2, inv_h);
  const double sigma = gx * gx + gy * gy + gz * gz;
  double e, dn, ds;
  pbe_point(rho[r], sigma, e, dn, ds);
  scr[r] = dn;
  scr[n + r] = 2.0 * ds * gx;
  scr[2 * n + r] = 2.0 * ds * gy;
  scr[3 * n + r] = 2.0 * ds * gz;
  if (exc) exc[r] = e;
}
template <int ORDER>
__global__ void __launch_bounds__(RB)
pbe_pass2_kernel(GridDims gd, double inv_h, const double* __restrict__ scr, double* __restrict__ out) {
  const long long n = (long long)gd.nx * gd.ny * gd.nz;
  const long long r = (long long)blockIdx.x * RB + threadIdx.x;
  if (r >= n) return;
  const int nyz = gd.ny * gd.nz;
  const int ix = (int)(r / nyz), rem = (int)(r - (long long)ix * nyz), iy = rem / gd.nz, iz = rem - iy * gd.nz;
  double v = scr[r];
  v -= ddx<ORDER>(scr + n, gd, ix, iy, iz, 0, inv_h);
  v -= ddx<ORDER>(scr + 2 * n, gd, ix, iy, iz, 1, inv_h);
  v -= ddx<ORDER>(scr + 3 * n, gd, ix, iy, iz, 2, inv_h);
  out[r] = v;
}
void launch_vxc_pbe(GridDims gd, double h, int order, const double* rho, double* scr, double* out, double* exc,
                    cudaStream_t st) {
  const long long n = (long long)gd.nx * gd.ny * gd.nz;
  const unsigned nb = (unsigned)((n + RB - 1) / RB);
  if (order == 4) {
    pbe_pass1_kernel<4><<<nb, RB, 0, st>>>(gd, 1.0 / h, rho, scr, exc);
    if (out) pbe_pass2_kernel<4><<<nb, RB, 0, st>>>(gd, 1.0 / h, scr, out);
  } else {
    pbe_pass1_kernel<2><<<nb, RB, 0, st>>>(gd, 1.0 / h, rho, scr, exc);
    if (out) pbe_pass2_kernel<2><<<nb, RB, 0, st>>>(gd, 1.0 / h, scr, out);
  }
}

__global__ void __launch_bounds__(RB)
delta_v_assemble_kernel(long long Ng, GridDims gd, double h, const double* __restrict__ vxc,
                        const double* __restrict__ vxc0, const double* __restrict__ VH, const double* __restrict__ E,
                        double* __restrict__ w) {
  const long long r = (long long)blockIdx.x * RB + threadIdx.x;
  if (r >= Ng) return;
  double v = field_at(r, gd, h, E);
  if (VH) v += VH[r];
  if (vxc) v += vxc[r] - vxc0[r];
  w[r] = v;
}
void launch_delta_v_assemble(long long Ng, GridDims gd, double h, const double* vxc, const double* vxc0, const double* VH,
                             const double* E, double* w, cudaStream_t st) {
  delta_v_assemble_kernel<<<(unsigned)((Ng + RB - 1) / RB), RB, 0, st>>>(Ng, gd, h, vxc, vxc0, VH, E, w);
}

// energy sum for a functional whose e_xc per point was computed separately: sum [1/2 drho VH + exc - exc0 - vxc0 drho + E.r drho]
__global__ void __launch_bounds__(RB)
energy_exc_kernel(long long Ng, GridDims gd, double h, const double* __restrict__ rho, const double* __restrict__ rho0,
                  const double* __restrict__ vxc0, const double* __restrict__ VH, const double* __restrict__ E,
                  const double* __restrict__ exc, const double* __restrict__ exc0, int use_h, double* __restrict__ bsums) {
  __shared__ double sh[RB / 32][5];
  double v[5] = {0, 0, 0, 0, 0};
  for (long long r = (long long)blockIdx.x * RB + threadIdx.x; r < Ng; r += (long long)gridDim.x * RB) {
    const double d = rho[r] - rho0[r];
    double e = field_at(r, gd, h, E) * d;
    if (use_h) e += 0.5 * d * VH[r];
    if (exc) e += exc[r] - exc0[r] - vxc0[r] * d;
    v[0] += e;
  }
  block_sum<5>(v, sh);
  if (threadIdx.x == 0)
#pragma unroll
    for (int q = 0; q < 5; ++q) bsums[blockIdx.x * 5 + q] = v[q];
}
void launch_energy_exc(long long Ng, GridDims gd, double h, const double* rho, const double* rho0, const double* vxc0,
                       const double* VH, const double* E, const double* exc, const double* exc0, int use_h, int N, int ldn,
                       const double* eps, const double* P0r, double* bsums, double* out, cudaStream_t st) {
  const int nb = reduce_rho_blocks(Ng);
  energy_exc_kernel<<<nb, RB, 0, st>>>(Ng, gd, h, rho, rho0, vxc0, VH, E, exc, exc0, use_h, bsums);
  final_sums_kernel<<<1, 32 * 5, 0, st>>>(bsums, nb, 5, out);
  trace_eps_kernel<<<1, 1024, 0, st>>>(N, ldn, eps, P0r, out);
}

// Energy diagnostic (conserved after the kick; Figs. 3-4):
//   E = sum_i eps_i Re P_ii + dVol sum_r [ 1/2 drho V_H + e_xc(rho) - e_xc(rho0) - vxc0 drho + E.r drho ]
__global__ void __launch_bounds__(RB)
energy_kernel(long long Ng, GridDims gd, double h, const double* __restrict__ rho, const double* __restrict__ rho0,
              const double* __restrict__ vxc0, const double* __restrict__ VH, const double* __restrict__ E, int use_h,
              int use_xc, double* __restrict__ bsums) {
  __shared__ double sh[RB / 32][5];
  double v[5] = {0, 0, 0, 0, 0};
  for (long long r = (long long)blockIdx.x * RB + threadIdx.x; r < Ng; r += (long long)gridDim.x * RB) {
    const double d = rho[r] - rho0[r];
    double e = field_at(r, gd, h, E) * d;
    if (use_h) e += 0.5 * d * VH[r];
    if (use_xc) e += exc_pz81(rho[r]) - exc_pz81(rho0[r]) - vxc0[r] * d;
    v[0] += e;
  }
  block_sum<5>(v, sh);
  if (threadIdx.x == 0)
#pragma unroll
    for (int q = 0; q < 5; ++q) bsums[blockIdx.x * 5 + q] = v[q];
}
__global__ void trace_eps_kernel(int N, int ldn, const double* __restrict__ eps, const double* __restrict__ P,
                                 double* __restrict__ out) {
  __shared__ double sh[32][5];
  double v[5] = {0, 0, 0, 0, 0};
  for (int i = threadIdx.x; i < N; i += blockDim.x) v[0] += eps[i] * P[(long long)i * ldn + i];
  block_sum<5>(v, sh);
  if (threadIdx.x == 0) out[5] = v[0];
}
void launch_energy(long long Ng, GridDims gd, double h, const double* rho, const double* rho0, const double* vxc0,
                   const double* VH, const double* E, int use_h, int use_xc, int N, int ldn, const double* eps,
                   const double* P0r, double* bsums, double* out, cudaStream_t st) {
  const int nb = reduce_rho_blocks(Ng);
  energy_kernel<<<nb, RB, 0, st>>>(Ng, gd, h, rho, rho0, vxc0, VH, E, use_h, use_xc, bsums);
  final_sums_kernel<<<1, 32 * 5, 0, st>>>(bsums, nb, 5, out);          // out[0] = grid part (without dVol)
  trace_eps_kernel<<<1, 1024, 0, st>>>(N, ldn, eps, P0r, out);          // out[5] = sum_i eps_i P_ii
}

static inline unsigned nblk(long long n) { return (unsigned)((n + RB - 1) / RB); }

void launch_delta_v(long long Ng, GridDims gd, double h, const double* rho, const double* vxc0, const double* VH,
                    const double* E, int use_h, int use_xc, double* w, cudaStream_t st) {
  delta_v_kernel<<<nblk(Ng), RB, 0, st>>>(Ng, gd, h, rho, vxc0, VH, E, use_h, use_xc, w);
}
void launch_vxc(long long Ng, const double* rho, double* vxc, cudaStream_t st) {
  vxc_kernel<<<nblk(Ng), RB, 0, st>>>(Ng, rho, vxc);
}
// E(t_{n+1}) passed BY VALUE (a kernel argument is captured at launch: the caller's buffer can be reused at once)
__global__ void set_field_kernel(double* __restrict__ dE, double ex, double ey, double ez) {
  if (threadIdx.x == 0) { dE[0] = ex; dE[1] = ey; dE[2] = ez; }
}
void launch_set_field(double* dE, double ex, double ey, double ez, cudaStream_t st) {
  set_field_kernel<<<1, 32, 0, st>>>(dE, ex, ey, ez);
}
void launch_field(long long Ng, GridDims gd, double h, const double* E, double* w, cudaStream_t st) {
  field_kernel<<<nblk(Ng), RB, 0, st>>>(Ng, gd, h, E, w);
}

// ---------------------------------------------------------------------------------------------- a7
__global__ void __launch_bounds__(RB)
poisson_rhs_kernel(long long Ng, const double* __restrict__ rho, const double* __restrict__ rho0,
                   const double* __restrict__ sums, double* __restrict__ f) {
  const long long r = (long long)blockIdx.x * RB + threadIdx.x;
  if (r >= Ng) return;
  const double mean = sums[4] / (double)Ng;
  const double d = rho0 ? rho[r] - rho0[r] : rho[r];
  f[r] = 4.0 * 3.14159265358979323846 * (d - mean);
}
void launch_poisson_rhs(long long Ng, const double* rho, const double* rho0, const double* sums, double* f,
                        cudaStream_t st) {
  poisson_rhs_kernel<<<nblk(Ng), RB, 0, st>>>(Ng, rho, rho0, sums, f);
}

// ---------------------------------------------------------------------------------------------- a2 and glue
// S == nullptr: orthonormal basis, X = dt (Hbar - sigma I); else X = dt (Hbar - sigma S)  (then S^-1 X = dt (S^-1 Hbar - sigma I))
__global__ void hbar_kernel(int N, int ldn, const double* __restrict__ Hm1, const double* __restrict__ H0,
                            double* __restrict__ H1, double* __restrict__ X, double dt, double sigma, int first,
                            const double* __restrict__ S) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j >= N) return;
  const long long o = (long long)i * ldn + j;
  const double h0 = H0[o];
  double h1;
  if (first) { h1 = 2.0 * h0 - Hm1[o]; H1[o] = h1; } else { h1 = H1[o]; }
  double x = 0.5 * (h0 + h1);
  if (S) x -= sigma * S[o];
  else if (i == j) x -= sigma;
  X[o] = dt * x;
}
void launch_hbar(int N, int ldn, const double* Hm1, const double* H0, double* H1, double* X, double dt, double sigma,
                 int first, cudaStream_t st, const double* S) {
  hbar_kernel<<<dim3((N + 127) / 128, N), 128, 0, st>>>(N, ldn, Hm1, H0, H1, X, dt, sigma, first, S);
}

// ---- the paper's "one multiply + transpose" form of a commutator step (DGEAM) -------------
// R, I: real and imaginary part of M = Omega dP (full N x N products).  dP' = (M + M^dagger)/k:
//   Sn = (R + R^T)/k (symmetric), An = (I - I^T)/k (antisymmetric);  P1r += Sn, P1i += An.
// 32 x 32 tiles through shared memory so that both the (i, j) and the (j, i) accesses are coalesced; only tiles
// bj >= bi are visited and both images are written, so the outputs are exactly (anti)symmetric.
__global__ void __launch_bounds__(256)
transpose_add_kernel(int N, int ldn, const double* __restrict__ R, const double* __restrict__ I, double inv_k,
                     double* __restrict__ Sn, double* __restrict__ An, double* __restrict__ P1r,
                     double* __restrict__ P1i, const int* __restrict__ skip) {
  if (skip && *skip) return;
  const int bi = blockIdx.y, bj = blockIdx.x;
  if (bj < bi) return;
  __shared__ double tR[32][33], tI[32][33];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;      // 32 x 8
  for (int r = ty; r < 32; r += 8) {                            // tile (bj, bi), read row-wise
    const int row = bj * 32 + r, col = bi * 32 + tx;
    const bool ok = row < N && col < N;
    tR[r][tx] = ok ? R[(long long)row * ldn + col] : 0.0;
    tI[r][tx] = ok ? I[(long long)row * ldn + col] : 0.0;
  }
  __syncthreads();
  double sv[4], av[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {                                 // tile (bi, bj): element (row, col) needs (col, row)
    const int r = ty + 8 * q;
    const int row = bi * 32 + r, col = bj * 32 + tx;
    sv[q] = av[q] = 0.0;
    if (row < N && col < N) {
      const long long o = (long long)row * ldn + col;
      sv[q] = (R[o] + tR[tx][r]) * inv_k;
      av[q] = (row == col) ? 0.0 : (I[o] - tI[tx][r]) * inv_k;
      if (bj > bi || col >= row) { Sn[o] = sv[q]; An[o] = av[q]; P1r[o] += sv[q]; P1i[o] += av[q]; }
    }
  }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < 4; ++q) { tR[ty + 8 * q][tx] = sv[q]; tI[ty + 8 * q][tx] = av[q]; }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {                            // mirror image into tile (bj, bi), written row-wise
    const int row = bj * 32 + r, col = bi * 32 + tx;            // = transpose of element (col, row) of tile (bi, bj)
    if (row < N && col < N && (bj > bi || col < row)) {
      const long long o = (long long)row * ldn + col;
      const double s = tR[tx][r], a = -tI[tx][r];
      Sn[o] = s; An[o] = a; P1r[o] += s; P1i[o] += a;
    }
  }
}
void launch_transpose_add(int N, int ldn, const double* R, const double* I, double inv_k, double* Sn, double* An,
                          double* P1r, double* P1i, const int* skip, cudaStream_t st) {
  const int nb = (N + 31) / 32;
  transpose_add_kernel<<<dim3(nb, nb), 256, 0, st>>>(N, ldn, R, I, inv_k, Sn, An, P1r, P1i, skip);
}

// out = a X + b Y (whole N x ldn buffers; padding stays zero)
__global__ void axpby_kernel(long long n, double a, const double* X, double b, const double* Y, double* out) {   // out may alias X
  for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < n; r += (long long)gridDim.x * blockDim.x)
    out[r] = a * X[r] + b * Y[r];
}
void launch_axpby(int N, int ldn, double a, const double* X, double b, const double* Y, double* out, cudaStream_t st) {
  const long long n = (long long)N * ldn;
  long long nb = (n + 255) / 256;
  if (nb > 148 * 16) nb = 148 * 16;
  axpby_kernel<<<(unsigned)nb, 256, 0, st>>>(n, a, X, b, Y, out);
}

__global__ void series_init_kernel(int N, int ldn, const double* __restrict__ Y, double* __restrict__ C, double c1,
                                   double* __restrict__ S, double s1) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j >= N) return;
  const long long o = (long long)i * ldn + j;
  const double y = Y[o], d = (i == j) ? 1.0 : 0.0;
  C[o] = d + c1 * y;
  S[o] = d + s1 * y;
}
void launch_series_init(int N, int ldn, const double* Y, double* C, double c1, double* S, double s1, cudaStream_t st) {
  series_init_kernel<<<dim3((N + 127) / 128, N), 128, 0, st>>>(N, ldn, Y, C, c1, S, s1);
}

// cos / sinc series from the stored powers of Y = X^2:  C = 1 + sum_k c_k Y^k,  Sc = 1 + sum_k s_k Y^k  (k = 1..q), summed
// in the order k = 1, 2, ... -- the same order, and the same operations, as series_init_kernel followed by the
// read-modify-write accumulation in the GEMM epilogues that this kernel replaces.
__global__ void series_combine_kernel(int N, int ldn, SeriesArgs a, double* __restrict__ C, double* __restrict__ S,
                                      int row_beg) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = row_beg + blockIdx.y;
  if (j >= N) return;
  const long long o = (long long)i * ldn + j;
  const double d = (i == j) ? 1.0 : 0.0;
  const double y1 = a.pw[0][o];
  double cv = d + a.c[0] * y1, sv = d + a.s[0] * y1;
#pragma unroll 1
  for (int k = 1; k < a.q; ++k) {
    const double y = a.pw[k][o];
    cv += a.c[k] * y;
    sv += a.s[k] * y;
  }
  C[o] = cv;
  S[o] = sv;
}
void launch_series_combine(int N, int ldn, const SeriesArgs& a, double* C, double* S, int row_beg, int row_end,
                           cudaStream_t st) {
  if (row_end <= row_beg) return;
  series_combine_kernel<<<dim3((N + 127) / 128, row_end - row_beg), 128, 0, st>>>(N, ldn, a, C, S, row_beg);
}

// Line 28 shifts H-1 <- H0 and H0 <- H1 in ONE launch, so H0 is both a source and a destination: no __restrict__
// here, and every element is read into registers before any store.
__global__ void copy4_kernel(long long n, double* d0, const double* s0, double* d1, const double* s1, double* d2,
                             const double* s2, double* d3, const double* s3) {
  for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < n; r += (long long)gridDim.x * blockDim.x) {
    const double a = s0[r], b = s1[r], c = s2[r], d = s3[r];
    d0[r] = a; d1[r] = b; d2[r] = c; d3[r] = d;
  }
}
void launch_copy5(int N, int ldn, double* d0, const double* s0, double* d1, const double* s1, double* d2,
                  const double* s2, double* d3, const double* s3, cudaStream_t st) {
  const long long n = (long long)N * ldn;
  long long nb = (n + 255) / 256;
  if (nb > 148 * 16) nb = 148 * 16;
  copy4_kernel<<<(unsigned)nb, 256, 0, st>>>(n, d0, s0, d1, s1, d2, s2, d3, s3);
}

// ---------------------------------------------------------------- dynamic-loop error norms (Alg. 1 lines 22, 24)
// max that does not drop NaN/Inf: a non-finite operand turns the result into +inf, so a blown-up series or Hamiltonian
// can never read as "converged" (fmax alone discards NaN)
__device__ __forceinline__ double max_nf(double m, double x) {
  return (x != x || m != m) ? __longlong_as_double(0x7ff0000000000000LL) : (x > m ? x : m);
}
__device__ __forceinline__ double block_max(double m) {
  __shared__ double shm[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max_nf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if (lane == 0) shm[warp] = m;
  __syncthreads();
  if (warp == 0) {
    m = lane < (int)(blockDim.x >> 5) ? shm[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max_nf(m, __shfl_xor_sync(0xffffffffu, m, o));
  }
  return m;      // valid in thread 0
}

__global__ void __launch_bounds__(RB)
commutator_check_kernel(long long n, const double* __restrict__ a, const double* __restrict__ b, int k, double thrs,
                        ConvState* __restrict__ cs) {
  // `done` can only be set by the last block of an EARLIER launch (every block of this one arrives first)
  if (*reinterpret_cast<volatile int*>(&cs->done)) return;
  double m = 0.0;
  for (long long r = (long long)blockIdx.x * RB + threadIdx.x; r < n; r += (long long)gridDim.x * RB)
    m = max_nf(max_nf(m, fabs(a[r])), fabs(b[r]));
  m = block_max(m);
  if (threadIdx.x == 0) {
    atomicMax(&cs->dP_bits[k], (unsigned long long)__double_as_longlong(m));
    __threadfence();
    if (atomicAdd(&cs->arrived[k], 1u) == gridDim.x - 1) {
      __threadfence();
      const double err = __longlong_as_double((long long)atomicMax(&cs->dP_bits[k], 0ull));
      cs->k_used = k;
      if (!(err > thrs)) cs->done = 1;          // Alg. 1 line 18: while (dP_err > dP_thrs)
    }
  }
}
static int norm_blocks(long long n) {
  long long nb = (n + RB * 4 - 1) / (RB * 4);
  return (int)(nb < 1 ? 1 : (nb > 148 * 8 ? 148 * 8 : nb));
}
void launch_commutator_check(int N, int ldn, const double* dPr, const double* dPi, int k, double thrs, ConvState* cs,
                             cudaStream_t st) {
  const long long n = (long long)N * ldn;      // padding columns hold zeros
  commutator_check_kernel<<<norm_blocks(n), RB, 0, st>>>(n, dPr, dPi, k, thrs, cs);
}

__global__ void __launch_bounds__(RB)
maxabs_diff_kernel(long long n, const double* __restrict__ a, const double* __restrict__ b, ConvState* __restrict__ cs) {
  double m = 0.0;
  for (long long r = (long long)blockIdx.x * RB + threadIdx.x; r < n; r += (long long)gridDim.x * RB)
    m = max_nf(m, fabs(a[r] - b[r]));
  m = block_max(m);
  if (threadIdx.x == 0) atomicMax(&cs->H_bits, (unsigned long long)__double_as_longlong(m));
}
void launch_maxabs_diff(int N, int ldn, const double* A, const double* B, ConvState* cs, cudaStream_t st) {
  const long long n = (long long)N * ldn;
  maxabs_diff_kernel<<<norm_blocks(n), RB, 0, st>>>(n, A, B, cs);
}

// cs->H_bits = max |T - 1| (Newton-Schulz residual of the overlap inverse)
__global__ void __launch_bounds__(RB)
maxabs_minus_identity_kernel(int N, int ldn, const double* __restrict__ T, ConvState* __restrict__ cs) {
  double m = 0.0;
  const long long n = (long long)N * ldn;
  for (long long r = (long long)blockIdx.x * RB + threadIdx.x; r < n; r += (long long)gridDim.x * RB) {
    const int i = (int)(r / ldn), j = (int)(r - (long long)i * ldn);
    if (j < N) m = max_nf(m, fabs(T[r] - (i == j ? 1.0 : 0.0)));
  }
  m = block_max(m);
  if (threadIdx.x == 0) atomicMax(&cs->H_bits, (unsigned long long)__double_as_longlong(m));
}
void launch_maxabs_minus_identity(int N, int ldn, const double* T, ConvState* cs, cudaStream_t st) {
  maxabs_minus_identity_kernel<<<norm_blocks((long long)N * ldn), RB, 0, st>>>(N, ldn, T, cs);
}

// out[5] = sum_ij A_ij B_ij  (tr(H_KS Re P) for symmetric matrices); one block, fixed order
__global__ void trace_product_kernel(int N, int ldn, const double* __restrict__ A, const double* __restrict__ B,
                                     double* __restrict__ out) {
  __shared__ double sh[32][5];
  double v[5] = {0, 0, 0, 0, 0};
  const long long n = (long long)N * ldn;
  for (long long r = threadIdx.x; r < n; r += blockDim.x) v[0] += A[r] * B[r];
  block_sum<5>(v, sh);
  if (threadIdx.x == 0) out[5] = v[0];
}
void launch_trace_product(int N, int ldn, const double* A, const double* B, double* out, cudaStream_t st) {
  trace_product_kernel<<<1, 1024, 0, st>>>(N, ldn, A, B, out);
}

__global__ void set_diag_kernel(int N, int ldn, double* __restrict__ M, const double* __restrict__ d) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j >= ldn) return;
  M[(long long)i * ldn + j] = (i == j) ? d[i] : 0.0;
}
__global__ void hermitize_kernel(int N, int ldn, double* Re, double* Im) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;      // (i, j), j > i is the source
  if (j >= N) return;
  if (j > i) {
    Re[(long long)j * ldn + i] = Re[(long long)i * ldn + j];
    Im[(long long)j * ldn + i] = -Im[(long long)i * ldn + j];
  } else if (j == i) {
    Im[(long long)i * ldn + i] = 0.0;
  }
}
void launch_hermitize(int N, int ldn, double* Re, double* Im, cudaStream_t st) {
  hermitize_kernel<<<dim3((N + 127) / 128, N), 128, 0, st>>>(N, ldn, Re, Im);
}

void launch_set_diag(int N, int ldn, double* M, const double* diag, cudaStream_t st) {
  set_diag_kernel<<<dim3((ldn + 127) / 128, N), 128, 0, st>>>(N, ldn, M, diag);
}

}  // namespace rt
