// mg_kernels.cu -- a7 "Vh": periodic 7-point Poisson solve, fixed count of V(nu1,nu2) cycles, weighted Jacobi,
// full weighting, trilinear prolongation, exact separable solve on the coarsest level (DESIGN R6; the paper only
// says "multigrid", Table 1 "Vh" L545).
//
// Two kinds of kernels:
//   * large levels: shared-memory tiles with halos, 3 launches per level per cycle
//       mg_smooth_kernel<false>  : nu (1 or 2) Jacobi sweeps fused; the tile is loaded once with a halo of nu
//       mg_resid_restrict_kernel : residual on a (2c+1)^3 fine patch kept in shared memory, full weighting -> coarse rhs
//       mg_smooth_kernel<true>   : u + P e (coarse patch staged in shared memory) followed by the post-sweeps
//   * the levels from which the rest of the hierarchy fits one CTA's shared memory (<= 200 KB: 16^3 and below, 13^3):
//       ONE launch of mg_coarse_kernel<true> per cycle (per solve when even the finest level fits): a single CTA walks
//       down and up the hierarchy on shared-memory arrays, phases separated by __syncthreads (~0.1 us) instead of
//       kernel boundaries (~2 us).  A coarsest level too large for that (a grid that cannot be halved) is solved by
//       mg_coarse_kernel<false>: a cluster of 8 CTAs on global memory, phases separated by the cluster barrier
//       (measured ~2 us per phase including the L2 round trips, so it is only the fallback).
// Every value is computed with the same formula and operand order as before the fusion (one thread per output).
#include "rt_internal.h"

#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace rt {

namespace {

constexpr int MG_THREADS = 512;          // tile kernels
constexpr int CL_THREADS = 1024;         // cluster kernel, per CTA
constexpr int CL_SIZE = 8;               // CTAs per cluster (portable maximum)

__device__ __forceinline__ int wrapi(int i, int n) {
  i %= n;
  return i < 0 ? i + n : i;
}
// Linear index -> (x, y, z) of a box with y-z extents (ny, nz) without integer division: q = floor(i / d) as
// umulhi(i, ceil(2^32 / d)), exact for i, d < 2^16 (every box here has fewer than 2^16 points; the division was the
// bottleneck of the first version of these kernels: ~100 instructions per point against ~15 of useful work).
struct Dec3 {
  int ny, nz, nyz;
  unsigned myz, mz;
  __host__ __device__ static Dec3 make(int ny_, int nz_) {      // two 64-bit divisions: done on the host or once per CTA
    Dec3 d;
    d.ny = ny_; d.nz = nz_; d.nyz = ny_ * nz_;
    d.myz = d.nyz > 1 ? (unsigned)((0x100000000ull + (unsigned)d.nyz - 1) / (unsigned)d.nyz) : 0u;
    d.mz = nz_ > 1 ? (unsigned)((0x100000000ull + (unsigned)nz_ - 1) / (unsigned)nz_) : 0u;
    return d;
  }
  __device__ __forceinline__ void operator()(int i, int& x, int& y, int& z) const {
    x = nyz > 1 ? (int)__umulhi((unsigned)i, myz) : i;
    const int rem = i - x * nyz;
    y = nz > 1 ? (int)__umulhi((unsigned)rem, mz) : rem;
    z = rem - y * nz;
  }
};

// ------------------------------------------------------------------------------------------- tile kernels
struct SmoothArgs {
  GridDims gd;           // this level
  GridDims gc;           // next coarser level (PROLONG only)
  int bx, by, bz;        // interior tile
  int tx, ty, tz;        // tiles per dimension
  int nsweep;            // 0 (PROLONG only), 1 or 2
  double h2, omega;
  const double* uin;     // nullptr: zero initial guess
  const double* f;
  const double* ec;      // PROLONG: coarse-level correction
  double* uout;
  Dec3 decA, decB, decC, decI;   // halo box, halo-1 box, coarse patch, interior
};

// out = (1 - omega) c + (omega / 6) (h^2 f + neighbours), neighbours summed x-, x+, y-, y+, z-, z+
__device__ __forceinline__ double jacobi_point(const double* __restrict__ s, int sy, int sz, int o, double fv,
                                               double h2, double omega) {
  const int px = sy * sz;
  const double nb = s[o - px] + s[o + px] + s[o - sz] + s[o + sz] + s[o - 1] + s[o + 1];
  return (1.0 - omega) * s[o] + (omega / 6.0) * (h2 * fv + nb);
}

template <bool PROLONG>
__global__ void __launch_bounds__(MG_THREADS) mg_smooth_kernel(const SmoothArgs a) {
  extern __shared__ __align__(16) double sm[];
  const int H = a.nsweep;
  const int rx = a.bx + 2 * H, ry = a.by + 2 * H, rz = a.bz + 2 * H;
  const int nA = rx * ry * rz;
  const int nB = (H == 2) ? (rx - 2) * (ry - 2) * (rz - 2) : 0;
  // coarse patch (PROLONG): covers fine coordinates [x0 - H, x0 + bx + H)
  const int cx = PROLONG ? (rx / 2 + 2) : 0, cy = PROLONG ? (ry / 2 + 2) : 0, cz = PROLONG ? (rz / 2 + 2) : 0;
  // f on the box of the first sweep (halo H-1), loaded in the same round trip as u
  const int fx = rx - 2, fy = ry - 2, fz = rz - 2;
  const int nF = H > 0 ? fx * fy * fz : 0;
  double* A = sm;
  double* B = A + nA;
  double* C = B + nB;
  double* F = C + cx * cy * cz;
  int* xs = reinterpret_cast<int*>(F + nF);
  int* ys = xs + rx;
  int* zs = ys + ry;

  const int tid = threadIdx.x;
  int b = blockIdx.x;
  const int tiz = b % a.tz; b /= a.tz;
  const int tiy = b % a.ty;
  const int tix = b / a.ty;
  const int x0 = tix * a.bx, y0 = tiy * a.by, z0 = tiz * a.bz;
  const int nx = a.gd.nx, ny = a.gd.ny, nz = a.gd.nz;

  for (int i = tid; i < rx; i += MG_THREADS) xs[i] = wrapi(x0 - H + i, nx);
  for (int i = tid; i < ry; i += MG_THREADS) ys[i] = wrapi(y0 - H + i, ny);
  for (int i = tid; i < rz; i += MG_THREADS) zs[i] = wrapi(z0 - H + i, nz);
  int c0x = 0, c0y = 0, c0z = 0;
  if (PROLONG) {
    c0x = (x0 - H) >> 1; c0y = (y0 - H) >> 1; c0z = (z0 - H) >> 1;      // arithmetic shift = floor
    const int ncx = a.gc.nx, ncy = a.gc.ny, ncz = a.gc.nz;
    const Dec3 decC = a.decC;
    for (int i = tid; i < cx * cy * cz; i += MG_THREADS) {
      int lx, ly, lz;
      decC(i, lx, ly, lz);
      C[i] = a.ec[((long long)wrapi(c0x + lx, ncx) * ncy + wrapi(c0y + ly, ncy)) * ncz + wrapi(c0z + lz, ncz)];
    }
  }
  __syncthreads();

  // load the tile with its halo (periodic wrap); PROLONG: add the trilinear interpolation of the coarse patch
  const Dec3 decA = a.decA;
  for (int i = tid; i < nA; i += MG_THREADS) {
    int lx, ly, lz;
    decA(i, lx, ly, lz);
    double v = a.uin ? a.uin[((long long)xs[lx] * ny + ys[ly]) * nz + zs[lz]] : 0.0;
    if (PROLONG) {
      const int X = x0 - H + lx, Y = y0 - H + ly, Z = z0 - H + lz;
      const int I0 = (X >> 1) - c0x, J0 = (Y >> 1) - c0y, K0 = (Z >> 1) - c0z;
      const int I1 = I0 + (X & 1), J1 = J0 + (Y & 1), K1 = K0 + (Z & 1);
      auto at = [&](int I, int J, int K) { return C[(I * cy + J) * cz + K]; };
      // 0.5 (p + q) with p == q on even points reproduces the injected value exactly
      const double z00 = 0.5 * (at(I0, J0, K0) + at(I0, J0, K1));
      const double z01 = 0.5 * (at(I0, J1, K0) + at(I0, J1, K1));
      const double z10 = 0.5 * (at(I1, J0, K0) + at(I1, J0, K1));
      const double z11 = 0.5 * (at(I1, J1, K0) + at(I1, J1, K1));
      const double y0v = 0.5 * (z00 + z01), y1v = 0.5 * (z10 + z11);
      v += 0.5 * (y0v + y1v);
    }
    A[i] = v;
  }
  if (H > 0) {
    const Dec3 decF = a.decB;
    for (int i = tid; i < nF; i += MG_THREADS) {
      int lx, ly, lz;
      decF(i, lx, ly, lz);
      F[i] = a.f[((long long)xs[lx + 1] * ny + ys[ly + 1]) * nz + zs[lz + 1]];
    }
  }
  __syncthreads();

  if (H == 2) {       // first sweep: halo-1 region, stays in shared memory
    const Dec3 decB = a.decB;
    for (int i = tid; i < nB; i += MG_THREADS) {
      int lx, ly, lz;
      decB(i, lx, ly, lz);
      B[i] = jacobi_point(A, ry, rz, ((lx + 1) * ry + ly + 1) * rz + lz + 1, F[i], a.h2, a.omega);
    }
    __syncthreads();
  }
  if (H == 0) {       // no sweep: u + P e only
    for (int i = tid; i < nA; i += MG_THREADS) {
      int lx, ly, lz;
      decA(i, lx, ly, lz);
      const int X = x0 + lx, Y = y0 + ly, Z = z0 + lz;
      if (X >= nx || Y >= ny || Z >= nz) continue;
      a.uout[((long long)X * ny + Y) * nz + Z] = A[i];
    }
  } else {            // last sweep: interior, to global memory
    const double* S = (H == 2) ? B : A;
    const int sy = ry - (H == 2 ? 2 : 0), sz = rz - (H == 2 ? 2 : 0);
    const int nI = a.bx * a.by * a.bz;
    const Dec3 decI = a.decI;
    for (int i = tid; i < nI; i += MG_THREADS) {
      int lx, ly, lz;
      decI(i, lx, ly, lz);
      const int X = x0 + lx, Y = y0 + ly, Z = z0 + lz;
      if (X >= nx || Y >= ny || Z >= nz) continue;
      const long long g = ((long long)X * ny + Y) * nz + Z;
      // f of the interior point: offset 1 inside the halo-1 box when H == 2, the box itself when H == 1
      const double fv = (H == 2) ? F[((lx + 1) * fy + ly + 1) * fz + lz + 1] : F[(lx * fy + ly) * fz + lz];
      a.uout[g] = jacobi_point(S, sy, sz, ((lx + 1) * sy + ly + 1) * sz + lz + 1, fv, a.h2, a.omega);
    }
  }
}

size_t smooth_smem_bytes(int bx, int by, int bz, int H, bool prolong) {
  const int rx = bx + 2 * H, ry = by + 2 * H, rz = bz + 2 * H;
  size_t d = (size_t)rx * ry * rz + (H == 2 ? (size_t)(rx - 2) * (ry - 2) * (rz - 2) : 0);
  if (prolong) d += (size_t)(rx / 2 + 2) * (ry / 2 + 2) * (rz / 2 + 2);
  if (H > 0) d += (size_t)(rx - 2) * (ry - 2) * (rz - 2);
  return d * 8 + (size_t)(rx + ry + rz) * 4 + 16;
}

struct ResRestArgs {
  GridDims gf, gc;
  int cbx, cby, cbz;     // coarse tile
  int tx, ty, tz;
  double inv_h2;
  const double* u;
  const double* f;
  double* fc;
  Dec3 decU, decQ, decT;         // u box, residual box, coarse tile
};

// coarse rhs = R (f - A u): residual on the (2c+1)^3 fine patch around the coarse tile, then (1/4,1/2,1/4)^3
__global__ void __launch_bounds__(MG_THREADS) mg_resid_restrict_kernel(const ResRestArgs a) {
  extern __shared__ __align__(16) double sm[];
  const int ux = 2 * a.cbx + 3, uy = 2 * a.cby + 3, uz = 2 * a.cbz + 3;
  const int qx = ux - 2, qy = uy - 2, qz = uz - 2;
  double* U = sm;
  double* R = U + ux * uy * uz;
  int* xs = reinterpret_cast<int*>(R + qx * qy * qz);
  int* ys = xs + ux;
  int* zs = ys + uy;
  const int tid = threadIdx.x;
  int b = blockIdx.x;
  const int tiz = b % a.tz; b /= a.tz;
  const int tiy = b % a.ty;
  const int tix = b / a.ty;
  const int C0x = tix * a.cbx, C0y = tiy * a.cby, C0z = tiz * a.cbz;
  const int nx = a.gf.nx, ny = a.gf.ny, nz = a.gf.nz;
  for (int i = tid; i < ux; i += MG_THREADS) xs[i] = wrapi(2 * C0x - 2 + i, nx);
  for (int i = tid; i < uy; i += MG_THREADS) ys[i] = wrapi(2 * C0y - 2 + i, ny);
  for (int i = tid; i < uz; i += MG_THREADS) zs[i] = wrapi(2 * C0z - 2 + i, nz);
  __syncthreads();
  const Dec3 decU = a.decU, decQ = a.decQ, decT = a.decT;
  for (int i = tid; i < ux * uy * uz; i += MG_THREADS) {
    int lx, ly, lz;
    decU(i, lx, ly, lz);
    U[i] = a.u[((long long)xs[lx] * ny + ys[ly]) * nz + zs[lz]];
  }
  for (int i = tid; i < qx * qy * qz; i += MG_THREADS) {      // f on the residual box, same round trip
    int lx, ly, lz;
    decQ(i, lx, ly, lz);
    R[i] = a.f[((long long)xs[lx + 1] * ny + ys[ly + 1]) * nz + zs[lz + 1]];
  }
  __syncthreads();
  for (int i = tid; i < qx * qy * qz; i += MG_THREADS) {
    int lx, ly, lz;
    decQ(i, lx, ly, lz);
    const int o = ((lx + 1) * uy + ly + 1) * uz + lz + 1, px = uy * uz;
    const double nb = U[o - px] + U[o + px] + U[o - uz] + U[o + uz] + U[o - 1] + U[o + 1];
    R[i] = R[i] - (6.0 * U[o] - nb) * a.inv_h2;
  }
  __syncthreads();
  const int ncx = a.gc.nx, ncy = a.gc.ny, ncz = a.gc.nz;
  for (int i = tid; i < a.cbx * a.cby * a.cbz; i += MG_THREADS) {
    int I, J, K;
    decT(i, I, J, K);
    if (C0x + I >= ncx || C0y + J >= ncy || C0z + K >= ncz) continue;
    double s = 0.0;
#pragma unroll
    for (int da = -1; da <= 1; ++da) {
      const double wa = da == 0 ? 0.5 : 0.25;
      double sy = 0.0;
#pragma unroll
      for (int db = -1; db <= 1; ++db) {
        const double wb = db == 0 ? 0.5 : 0.25;
        const double* p = R + ((2 * I + 1 + da) * qy + 2 * J + 1 + db) * qz + 2 * K + 1;
        sy += wb * (0.25 * p[-1] + 0.5 * p[0] + 0.25 * p[1]);
      }
      s += wa * sy;
    }
    a.fc[((long long)(C0x + I) * ncy + C0y + J) * ncz + C0z + K] = s;
  }
}

size_t resrest_smem_bytes(int cbx, int cby, int cbz) {
  const int ux = 2 * cbx + 3, uy = 2 * cby + 3, uz = 2 * cbz + 3;
  return ((size_t)ux * uy * uz + (size_t)(ux - 2) * (uy - 2) * (uz - 2)) * 8 + (size_t)(ux + uy + uz) * 4 + 16;
}

}  // namespace

// ------------------------------------------------------------------------------------------- cluster kernel
namespace {

struct ClusterArgs {
  int nlev;                    // levels lv[0 .. nlev-1]; lv[nlev-1] is solved exactly
  int ncycles;                 // V-cycles on lv[0]
  int zero_guess;              // lv[0].u starts from zero (called as the coarse part of a larger cycle)
  int nu1, nu2;
  double omega;
  MgLevel lv[MG_MAX_LEVELS];
  const double *Qx, *Qy, *Qz, *lx, *ly, *lz;
  int do_rhs;                  // lv[0].f = 4 pi (rho - rho0 - sums[4]/n) first (rho0 may be nullptr)
  const double* rho;
  const double* rho0;
  const double* sums;
};

// Phase barrier of the coarse kernel.  SMEM: one CTA, every array in shared memory, __syncthreads.
// !SMEM: a cluster of CL_SIZE CTAs on arrays in global memory (L2), hardware cluster barrier (flushes L1).
template <bool SMEM>
struct CoarseCtx {
  int gtid, gthreads;
  __device__ __forceinline__ void sync() {
    if (SMEM) __syncthreads();
    else { __threadfence(); cg::this_cluster().sync(); }
  }
};

__device__ __forceinline__ double nb_sum_g(const double* u, const GridDims& gd, int ix, int iy, int iz) {
  const int nyz = gd.ny * gd.nz;
  const int xm = ix == 0 ? gd.nx - 1 : ix - 1, xp = ix == gd.nx - 1 ? 0 : ix + 1;
  const int ym = iy == 0 ? gd.ny - 1 : iy - 1, yp = iy == gd.ny - 1 ? 0 : iy + 1;
  const int zm = iz == 0 ? gd.nz - 1 : iz - 1, zp = iz == gd.nz - 1 ? 0 : iz + 1;
  const int row = iy * gd.nz, pl = ix * nyz;
  return u[xm * nyz + row + iz] + u[xp * nyz + row + iz] + u[pl + ym * gd.nz + iz] + u[pl + yp * gd.nz + iz] +
         u[pl + row + zm] + u[pl + row + zp];
}

template <class Ctx>
__device__ void cl_jacobi(Ctx& c, const MgLevel& L, const Dec3& dec, const double* in, double* out, double omega) {
  const int n = (int)L.n;
  const double h2 = L.h * L.h;
  for (int r = c.gtid; r < n; r += c.gthreads) {
    if (!in) { out[r] = (1.0 - omega) * 0.0 + (omega / 6.0) * (h2 * L.f[r] + 0.0); continue; }
    int ix, iy, iz;
    dec(r, ix, iy, iz);
    out[r] = (1.0 - omega) * in[r] + (omega / 6.0) * (h2 * L.f[r] + nb_sum_g(in, L.gd, ix, iy, iz));
  }
  c.sync();
}

template <class Ctx>
__device__ void cl_residual(Ctx& c, const MgLevel& L, const Dec3& dec, const double* u) {
  const int n = (int)L.n;
  const double inv_h2 = 1.0 / (L.h * L.h);
  for (int r = c.gtid; r < n; r += c.gthreads) {
    int ix, iy, iz;
    dec(r, ix, iy, iz);
    L.r[r] = L.f[r] - (6.0 * u[r] - nb_sum_g(u, L.gd, ix, iy, iz)) * inv_h2;
  }
  c.sync();
}

template <class Ctx>
__device__ void cl_restrict(Ctx& c, const MgLevel& F, const MgLevel& Cc, const Dec3& dec) {
  const int nc = (int)Cc.n;
  const GridDims gf = F.gd;
  const int nyz = gf.ny * gf.nz;
  for (int r = c.gtid; r < nc; r += c.gthreads) {
    int I, J, K;
    dec(r, I, J, K);
    double s = 0.0;
#pragma unroll
    for (int a = -1; a <= 1; ++a) {
      int x = 2 * I + a; x = x < 0 ? x + gf.nx : (x >= gf.nx ? x - gf.nx : x);
      const double wa = a == 0 ? 0.5 : 0.25;
      double sy = 0.0;
#pragma unroll
      for (int b = -1; b <= 1; ++b) {
        int y = 2 * J + b; y = y < 0 ? y + gf.ny : (y >= gf.ny ? y - gf.ny : y);
        const double wb = b == 0 ? 0.5 : 0.25;
        const double* p = F.r + x * nyz + y * gf.nz;
        const int z0 = 2 * K;
        const int zm = z0 == 0 ? gf.nz - 1 : z0 - 1, zp = z0 + 1 >= gf.nz ? z0 + 1 - gf.nz : z0 + 1;
        sy += wb * (0.25 * p[zm] + 0.5 * p[z0] + 0.25 * p[zp]);
      }
      s += wa * sy;
    }
    Cc.f[r] = s;
  }
  c.sync();
}

template <class Ctx>
__device__ void cl_prolong_add(Ctx& c, const MgLevel& Cc, const double* ec, const MgLevel& F, const Dec3& dec,
                               double* u) {
  const int nf = (int)F.n;
  const GridDims gc = Cc.gd;
  const int nyz = gc.ny * gc.nz;
  for (int r = c.gtid; r < nf; r += c.gthreads) {
    int ix, iy, iz;
    dec(r, ix, iy, iz);
    const int I0 = ix >> 1, J0 = iy >> 1, K0 = iz >> 1;
    const int I1 = (ix & 1) ? (I0 + 1 == gc.nx ? 0 : I0 + 1) : I0;
    const int J1 = (iy & 1) ? (J0 + 1 == gc.ny ? 0 : J0 + 1) : J0;
    const int K1 = (iz & 1) ? (K0 + 1 == gc.nz ? 0 : K0 + 1) : K0;
    auto at = [&](int I, int J, int K) { return ec[I * nyz + J * gc.nz + K]; };
    const double z00 = 0.5 * (at(I0, J0, K0) + at(I0, J0, K1));
    const double z01 = 0.5 * (at(I0, J1, K0) + at(I0, J1, K1));
    const double z10 = 0.5 * (at(I1, J0, K0) + at(I1, J0, K1));
    const double z11 = 0.5 * (at(I1, J1, K0) + at(I1, J1, K1));
    const double y0 = 0.5 * (z00 + z01), y1 = 0.5 * (z10 + z11);
    u[r] += 0.5 * (y0 + y1);
  }
  c.sync();
}

// Exact solve on the coarsest level in the zero-mean subspace: u = (Qx x Qy x Qz) L^+ (Qx x Qy x Qz)^T f with the
// real orthonormal eigenvectors of the periodic 1-D operator (columns of Q) and eigenvalues lx + ly + lz.
// Six axis passes through the scratch arrays L.r and L.tmp.
template <class Ctx>
__device__ void cl_coarse_solve(Ctx& c, const MgLevel& L, const Dec3& dec, const ClusterArgs& a, double* u) {
  const int nx = L.gd.nx, ny = L.gd.ny, nz = L.gd.nz;
  const int n = nx * ny * nz;
  const double* f = L.f;
  double* s0 = L.r;
  double* s1 = L.tmp;
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // x: f -> s0, contract with Q^T
    int q, b_, k_;
    dec(o, q, b_, k_);
    const int rest = o - q * ny * nz;
    double s = 0.0;
    for (int i = 0; i < nx; ++i) s += a.Qx[i * nx + q] * f[i * ny * nz + rest];
    s0[o] = s;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // y: s0 -> s1
    int q, b, k;
    dec(o, q, b, k);
    double s = 0.0;
    for (int j = 0; j < ny; ++j) s += a.Qy[j * ny + b] * s0[(q * ny + j) * nz + k];
    s1[o] = s;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // z and the division: s1 -> s0
    int q, b, cc;
    dec(o, q, b, cc);
    double s = 0.0;
    for (int k = 0; k < nz; ++k) s += a.Qz[k * nz + cc] * s1[(q * ny + b) * nz + k];
    const double lam = a.lx[q] + a.ly[b] + a.lz[cc];
    s0[o] = (q == 0 && b == 0 && cc == 0) ? 0.0 : s / lam;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // back, z: s0 -> s1, contract with Q
    int q, b, k;
    dec(o, q, b, k);
    double s = 0.0;
    for (int cc = 0; cc < nz; ++cc) s += a.Qz[k * nz + cc] * s0[(q * ny + b) * nz + cc];
    s1[o] = s;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // y: s1 -> s0
    int q, j, k;
    dec(o, q, j, k);
    double s = 0.0;
    for (int b = 0; b < ny; ++b) s += a.Qy[j * ny + b] * s1[(q * ny + b) * nz + k];
    s0[o] = s;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // x: s0 -> u
    int i, b_, k_;
    dec(o, i, b_, k_);
    const int rest = o - i * ny * nz;
    double s = 0.0;
    for (int q = 0; q < nx; ++q) s += a.Qx[i * nx + q] * s0[q * ny * nz + rest];
    u[o] = s;
  }
  c.sync();
}

// Shared-memory footprint of levels l0.. of a hierarchy (u, tmp, f, r per level)
__host__ __device__ inline size_t coarse_smem_doubles(const MgLevel* lv, int nlev) {
  size_t d = 0;
  for (int l = 0; l < nlev; ++l) d += 4 * (size_t)lv[l].n;
  return d;
}

template <bool SMEM>
__global__ void __launch_bounds__(CL_THREADS) mg_coarse_kernel(const __grid_constant__ ClusterArgs a) {
  extern __shared__ __align__(16) double sm[];
  __shared__ MgLevel slv[MG_MAX_LEVELS];
  __shared__ Dec3 sdec[MG_MAX_LEVELS];
  CoarseCtx<SMEM> c{(int)threadIdx.x, CL_THREADS};
  if (!SMEM) {
    c.gtid = (int)cg::this_cluster().block_rank() * CL_THREADS + threadIdx.x;
    c.gthreads = CL_SIZE * CL_THREADS;
  }
  const int last = a.nlev - 1;
  if (threadIdx.x == 0) {
    double* p = sm;
    for (int l = 0; l < a.nlev; ++l) {
      MgLevel L = a.lv[l];
      if (SMEM) { L.u = p; L.tmp = p + L.n; L.f = p + 2 * L.n; L.r = p + 3 * L.n; p += 4 * L.n; }
      slv[l] = L;
    }
  }
  if ((int)threadIdx.x < a.nlev) sdec[threadIdx.x] = Dec3::make(a.lv[threadIdx.x].gd.ny, a.lv[threadIdx.x].gd.nz);
  __syncthreads();
  const MgLevel& G0 = a.lv[0];          // level 0 in global memory (input / output of the SMEM variant)

  if (a.do_rhs) {
    const MgLevel& L = slv[0];
    const int n = (int)L.n;
    const double mean = a.sums[4] / (double)n;
    for (int r = c.gtid; r < n; r += c.gthreads) {
      const double d = a.rho0 ? a.rho[r] - a.rho0[r] : a.rho[r];
      L.f[r] = 4.0 * 3.14159265358979323846 * (d - mean);
    }
  } else if (SMEM) {
    for (int r = c.gtid; r < (int)G0.n; r += c.gthreads) slv[0].f[r] = G0.f[r];
  }
  if (SMEM && !a.zero_guess)
    for (int r = c.gtid; r < (int)G0.n; r += c.gthreads) slv[0].u[r] = G0.u[r];
  c.sync();

  // where each level's current solution lives (u or tmp); sweeps ping-pong between the two
  double* cur[MG_MAX_LEVELS];
  for (int l = 0; l < a.nlev; ++l) cur[l] = slv[l].u;

  for (int cyc = 0; cyc < a.ncycles; ++cyc) {
    for (int l = 0; l < last; ++l) {
      const MgLevel& L = slv[l];
      bool zero = (l > 0) || (a.zero_guess && cyc == 0);
      for (int s = 0; s < a.nu1; ++s) {
        // zero guess: nothing is read, so start in the buffer from which the remaining sweeps end in u
        double* out = zero ? (((a.nu1 - 1 + a.nu2) & 1) ? L.tmp : L.u) : (cur[l] == L.u ? L.tmp : L.u);
        cl_jacobi(c, L, sdec[l], zero ? nullptr : cur[l], out, a.omega);
        cur[l] = out;
        zero = false;
      }
      if (zero) {           // nu1 == 0 with a zero guess: the residual needs an actual array of zeros
        for (int r = c.gtid; r < (int)L.n; r += c.gthreads) L.u[r] = 0.0;
        cur[l] = L.u;
        c.sync();
      }
      cl_residual(c, L, sdec[l], cur[l]);
      cl_restrict(c, L, slv[l + 1], sdec[l + 1]);
    }
    cl_coarse_solve(c, slv[last], sdec[last], a, slv[last].u);
    cur[last] = slv[last].u;
    for (int l = last - 1; l >= 0; --l) {
      const MgLevel& L = slv[l];
      cl_prolong_add(c, slv[l + 1], cur[l + 1], L, sdec[l], cur[l]);
      for (int s = 0; s < a.nu2; ++s) {
        double* out = cur[l] == L.u ? L.tmp : L.u;
        cl_jacobi(c, L, sdec[l], cur[l], out, a.omega);
        cur[l] = out;
      }
    }
  }
  if (SMEM || cur[0] != G0.u)
    for (int r = c.gtid; r < (int)G0.n; r += c.gthreads) G0.u[r] = cur[0][r];
}

}  // namespace

// ------------------------------------------------------------------------------------------- host side
namespace {

int tile_edge(int n, int bmax) {            // equal tiles of at most bmax points covering n
  const int nt = (n + bmax - 1) / bmax;
  return (n + nt - 1) / nt;
}

struct TileGeom { int bx, by, bz, tx, ty, tz; };
// Largest tile is (mx, my, mz); on small levels the tile is halved (x, y, then z, in turn) until there are at least
// ~148 CTAs or the tile is down to 256 points: these launches are latency-bound, so more SMs in flight is what counts.
TileGeom make_geom(const GridDims& g, int mx, int my, int mz) {
  for (int turn = 0; turn < 12; ++turn) {
    const long long nt = (long long)((g.nx + mx - 1) / mx) * ((g.ny + my - 1) / my) * ((g.nz + mz - 1) / mz);
    if (nt >= 148 || mx * my * mz <= 256) break;
    if (turn % 3 == 0 && mx > 2) mx /= 2;
    else if (turn % 3 == 1 && my > 2) my /= 2;
    else if (turn % 3 == 2 && mz > 8) mz /= 2;
  }
  TileGeom t;
  t.bx = tile_edge(g.nx, mx); t.by = tile_edge(g.ny, my); t.bz = tile_edge(g.nz, mz);
  t.tx = (g.nx + t.bx - 1) / t.bx; t.ty = (g.ny + t.by - 1) / t.by; t.tz = (g.nz + t.bz - 1) / t.bz;
  return t;
}

// nsweep in {0,1,2}; ec != nullptr: u + P ec first
void launch_smooth(const MgLevel& L, const MgLevel* coarse, const double* ec, const double* uin, double* uout,
                   int nsweep, double omega, cudaStream_t st) {
  const TileGeom t = make_geom(L.gd, 8, 8, 32);
  SmoothArgs a{};
  a.gd = L.gd;
  if (coarse) a.gc = coarse->gd;
  a.bx = t.bx; a.by = t.by; a.bz = t.bz; a.tx = t.tx; a.ty = t.ty; a.tz = t.tz;
  a.nsweep = nsweep; a.h2 = L.h * L.h; a.omega = omega;
  a.uin = uin; a.f = L.f; a.ec = ec; a.uout = uout;
  {
    const int H = nsweep, ry = t.by + 2 * H, rz = t.bz + 2 * H;
    a.decA = Dec3::make(ry, rz);
    a.decB = Dec3::make(ry > 2 ? ry - 2 : 1, rz > 2 ? rz - 2 : 1);
    a.decC = Dec3::make(ry / 2 + 2, rz / 2 + 2);
    a.decI = Dec3::make(t.by, t.bz);
  }
  const unsigned grid = (unsigned)(t.tx * t.ty * t.tz);
  const size_t smem = smooth_smem_bytes(t.bx, t.by, t.bz, nsweep, ec != nullptr);
  if (ec) mg_smooth_kernel<true><<<grid, MG_THREADS, smem, st>>>(a);
  else mg_smooth_kernel<false><<<grid, MG_THREADS, smem, st>>>(a);
}

void launch_resid_restrict(const MgLevel& F, const MgLevel& C, const double* u, cudaStream_t st) {
  const TileGeom t = make_geom(C.gd, 4, 4, 16);
  ResRestArgs a{};
  a.gf = F.gd; a.gc = C.gd;
  a.cbx = t.bx; a.cby = t.by; a.cbz = t.bz; a.tx = t.tx; a.ty = t.ty; a.tz = t.tz;
  a.inv_h2 = 1.0 / (F.h * F.h);
  a.u = u; a.f = F.f; a.fc = C.f;
  a.decU = Dec3::make(2 * t.by + 3, 2 * t.bz + 3);
  a.decQ = Dec3::make(2 * t.by + 1, 2 * t.bz + 1);
  a.decT = Dec3::make(t.by, t.bz);
  mg_resid_restrict_kernel<<<(unsigned)(t.tx * t.ty * t.tz), MG_THREADS, resrest_smem_bytes(t.bx, t.by, t.bz), st>>>(a);
}

// ---- exact coarsest-level solve on global memory, whole-GPU version ---------------------------------------------
// The paper's grids (N_x x 132 x 132) halve only twice: 1176 x 132 x 132 -> 294 x 33 x 33 = 320 k points,
// far beyond what one CTA (or the 8-CTA cluster, whose index decode is exact below 2^16 points per plane pair) can
// hold.  The separable solve u = (Qx x Qy x Qz) L^+ (Qx x Qy x Qz)^T f is six batched small dense transforms; here each
// is one launch with one thread per output point (plain 64-bit index arithmetic), contraction along one axis.
// axis pass: out[.., o_axis, ..] = sum_i M(i, o_axis) in[.., i, ..]; TRANS = false: M(i, o) = Q[i * n + o] (Q^T f);
// TRANS = true: M(i, o) = Q[o * n + i] (Q g).  DIV: divide by lx + ly + lz afterwards (zero for the constant mode).
template <int AXIS, bool TRANS, bool DIV>
__global__ void __launch_bounds__(256)
coarse_axis_kernel(GridDims gd, const double* __restrict__ Q, const double* __restrict__ in, double* __restrict__ out,
                   const double* __restrict__ lx, const double* __restrict__ ly, const double* __restrict__ lz) {
  const long long n = (long long)gd.nx * gd.ny * gd.nz;
  const long long o = (long long)blockIdx.x * 256 + threadIdx.x;
  if (o >= n) return;
  const long long nyz = (long long)gd.ny * gd.nz;
  const int ix = (int)(o / nyz);
  const int rem = (int)(o - ix * nyz);
  const int iy = rem / gd.nz, iz = rem - iy * gd.nz;
  const int na = AXIS == 0 ? gd.nx : (AXIS == 1 ? gd.ny : gd.nz);
  const int oa = AXIS == 0 ? ix : (AXIS == 1 ? iy : iz);
  const long long stride = AXIS == 0 ? nyz : (AXIS == 1 ? gd.nz : 1);
  const double* p = in + (o - (long long)oa * stride);
  double s = 0.0;
  for (int i = 0; i < na; ++i) s += (TRANS ? Q[(long long)oa * na + i] : Q[(long long)i * na + oa]) * p[(long long)i * stride];
  if (DIV) {
    const double lam = lx[ix] + ly[iy] + lz[iz];
    s = (ix == 0 && iy == 0 && iz == 0) ? 0.0 : s / lam;
  }
  out[o] = s;
}

// same six passes, in the same order and through the same scratch arrays (L.r, L.tmp), as cl_coarse_solve
void launch_coarse_exact_global(const MgLevel& L, const MgSolveArgs& s, cudaStream_t st) {
  const unsigned nb = (unsigned)((L.n + 255) / 256);
  coarse_axis_kernel<0, false, false><<<nb, 256, 0, st>>>(L.gd, s.Qx, L.f, L.r, nullptr, nullptr, nullptr);
  coarse_axis_kernel<1, false, false><<<nb, 256, 0, st>>>(L.gd, s.Qy, L.r, L.tmp, nullptr, nullptr, nullptr);
  coarse_axis_kernel<2, false, true><<<nb, 256, 0, st>>>(L.gd, s.Qz, L.tmp, L.r, s.lx, s.ly, s.lz);
  coarse_axis_kernel<2, true, false><<<nb, 256, 0, st>>>(L.gd, s.Qz, L.r, L.tmp, nullptr, nullptr, nullptr);
  coarse_axis_kernel<1, true, false><<<nb, 256, 0, st>>>(L.gd, s.Qy, L.tmp, L.r, nullptr, nullptr, nullptr);
  coarse_axis_kernel<0, true, false><<<nb, 256, 0, st>>>(L.gd, s.Qx, L.r, L.u, nullptr, nullptr, nullptr);
}
constexpr long long CLUSTER_MAX_POINTS = 32768;    // largest coarsest level the 8-CTA cluster kernel handles

constexpr size_t COARSE_SMEM_MAX = 200 * 1024;     // bytes of level arrays the single-CTA kernel may hold

bool fits_smem(const MgSolveArgs& s, int l0) {
  return coarse_smem_doubles(s.lv + l0, s.nlev - l0) * 8 <= COARSE_SMEM_MAX;
}

// levels l0.. : single CTA on shared memory when they fit, else the 8-CTA cluster on global memory
int launch_coarse(const MgSolveArgs& s, int l0, int ncycles, int zero_guess, int do_rhs, cudaStream_t st) {
  if (!fits_smem(s, l0) && l0 == s.nlev - 1 && s.lv[l0].n > CLUSTER_MAX_POINTS) {
    // a large coarsest level: the exact solve as six whole-GPU launches (it ignores the initial guess; cycles beyond the
    // first would reproduce the same exact solution)
    int launches = 6;
    if (do_rhs) { launch_poisson_rhs(s.lv[l0].n, s.rho, s.rho0, s.sums, s.lv[l0].f, st); ++launches; }
    if (ncycles > 0) launch_coarse_exact_global(s.lv[l0], s, st);
    else launches -= 6;
    return launches;
  }
  ClusterArgs a{};
  a.nlev = s.nlev - l0; a.ncycles = ncycles; a.zero_guess = zero_guess;
  a.nu1 = s.nu1; a.nu2 = s.nu2; a.omega = s.omega;
  for (int l = l0; l < s.nlev; ++l) a.lv[l - l0] = s.lv[l];
  a.Qx = s.Qx; a.Qy = s.Qy; a.Qz = s.Qz; a.lx = s.lx; a.ly = s.ly; a.lz = s.lz;
  a.do_rhs = do_rhs; a.rho = s.rho; a.rho0 = s.rho0; a.sums = s.sums;
  if (fits_smem(s, l0)) {
    mg_coarse_kernel<true><<<1, CL_THREADS, coarse_smem_doubles(a.lv, a.nlev) * 8, st>>>(a);
  } else {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(CL_SIZE); cfg.blockDim = dim3(CL_THREADS); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CL_SIZE; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, mg_coarse_kernel<false>, a);
  }
  return 1;
}

struct BigCycle {
  const MgSolveArgs& s;
  int lc;
  cudaStream_t st;
  int launches = 0;
  double* cur[MG_MAX_LEVELS];

  void smooth(int l, int nsweeps, bool zero) {        // plain sweeps, <= 2 per launch
    const MgLevel& L = s.lv[l];
    while (nsweeps > 0) {
      const int k = nsweeps >= 2 ? 2 : 1;
      double* out = zero ? L.u : (cur[l] == L.u ? L.tmp : L.u);
      launch_smooth(L, nullptr, nullptr, zero ? nullptr : cur[l], out, k, s.omega, st);
      ++launches;
      cur[l] = out;
      zero = false;
      nsweeps -= k;
    }
  }
  void vcycle(int l) {
    const MgLevel& L = s.lv[l];
    const bool zero = l > 0 || s.zero0;
    if (zero && s.nu1 == 0) { cudaMemsetAsync(L.u, 0, (size_t)L.n * 8, st); cur[l] = L.u; }
    else smooth(l, s.nu1, zero);
    launch_resid_restrict(L, s.lv[l + 1], cur[l], st);
    ++launches;
    if (l + 1 == lc) {
      launches += launch_coarse(s, lc, 1, 1, 0, st);
      cur[l + 1] = s.lv[l + 1].u;
    } else {
      vcycle(l + 1);
    }
    const int k = s.nu2 >= 2 ? 2 : s.nu2;
    double* out = cur[l] == L.u ? L.tmp : L.u;
    launch_smooth(L, &s.lv[l + 1], cur[l + 1], cur[l], out, k, s.omega, st);
    ++launches;
    cur[l] = out;
    smooth(l, s.nu2 - k, false);
  }
};

}  // namespace

int init_mg_kernels() {
  cudaError_t e = cudaFuncSetAttribute(mg_smooth_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(mg_smooth_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(mg_resid_restrict_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(mg_coarse_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)COARSE_SMEM_MAX);
  return (int)e;
}

int launch_mg_solve(const MgSolveArgs& s, cudaStream_t st) {
  // lc = first level from which the rest of the hierarchy fits one CTA's shared memory; if even the coarsest level
  // does not, the levels above it use the tile kernels and the exact solve runs on the cluster
  int lc = 0;
  while (lc < s.nlev - 1 && !fits_smem(s, lc)) ++lc;
  if (lc == 0) {           // the whole hierarchy is small: rhs + every cycle in one launch
    return launch_coarse(s, 0, s.n_vc, s.zero0, s.rhs_given ? 0 : 1, st);
  }
  if (!s.rhs_given) launch_poisson_rhs(s.lv[0].n, s.rho, s.rho0, s.sums, s.lv[0].f, st);
  BigCycle bc{s, lc, st};
  for (int l = 0; l < s.nlev; ++l) bc.cur[l] = s.lv[l].u;
  for (int v = 0; v < s.n_vc; ++v) bc.vcycle(0);
  if (bc.cur[0] != s.lv[0].u)
    cudaMemcpyAsync(s.lv[0].u, bc.cur[0], (size_t)s.lv[0].n * 8, cudaMemcpyDeviceToDevice, st);
  return bc.launches + (s.rhs_given ? 0 : 1);
}

// ---- fourth-order operator (Eq. 2 with n = 2): r = f - A4 u, A4 = -(13-point Laplacian) ---------
// One thread per point, periodic wrap by index arithmetic; the arrays are L2-resident at every config.
__global__ void __launch_bounds__(256)
resid_order4_kernel(GridDims gd, double inv_h2, const double* __restrict__ u, const double* __restrict__ f,
                    double* __restrict__ r) {
  const long long n = (long long)gd.nx * gd.ny * gd.nz;
  const long long p = (long long)blockIdx.x * 256 + threadIdx.x;
  if (p >= n) return;
  const int nyz = gd.ny * gd.nz;
  const int ix = (int)(p / nyz), rem = (int)(p - (long long)ix * nyz), iy = rem / gd.nz, iz = rem - iy * gd.nz;
  auto at = [&](int x, int y, int z) { return u[((long long)x * gd.ny + y) * gd.nz + z]; };
  auto wrap = [](int i, int n_) { i %= n_; return i < 0 ? i + n_ : i; };
  const double c0 = -2.5, c1 = 4.0 / 3.0, c2 = -1.0 / 12.0;
  double acc = 3.0 * c0 * u[p];
  // same accumulation order as oracle.apply_A_order: axis by axis, distance 1 then 2, (minus side + plus side)
  acc += c1 * (at(wrap(ix + 1, gd.nx), iy, iz) + at(wrap(ix - 1, gd.nx), iy, iz));
  acc += c2 * (at(wrap(ix + 2, gd.nx), iy, iz) + at(wrap(ix - 2, gd.nx), iy, iz));
  acc += c1 * (at(ix, wrap(iy + 1, gd.ny), iz) + at(ix, wrap(iy - 1, gd.ny), iz));
  acc += c2 * (at(ix, wrap(iy + 2, gd.ny), iz) + at(ix, wrap(iy - 2, gd.ny), iz));
  acc += c1 * (at(ix, iy, wrap(iz + 1, gd.nz)) + at(ix, iy, wrap(iz - 1, gd.nz)));
  acc += c2 * (at(ix, iy, wrap(iz + 2, gd.nz)) + at(ix, iy, wrap(iz - 2, gd.nz)));
  r[p] = f[p] - (-acc * inv_h2);
}
__global__ void __launch_bounds__(256) add_inplace_kernel(long long n, double* __restrict__ u, const double* __restrict__ d) {
  const long long p = (long long)blockIdx.x * 256 + threadIdx.x;
  if (p < n) u[p] += d[p];
}

// Hartree solve with the fourth-order operator: the 7-point V-cycle is the preconditioner (oracle.hartree_mg, order = 4):
//   f4 = 4 pi (rho - rho0 - mean);  n_vc times:  r = f4 - A4 u ;  d = Vcycle_7pt(0, r) ;  u += d.
// `s.lv[0].u` is the warm-started potential; `dl0` supplies level-0 arrays of the correction hierarchy (u = d, f = r) and
// f4 the right-hand side.  Returns the number of kernels enqueued.
int launch_mg_solve_order4(const MgSolveArgs& s, const MgLevel& dl0, double* f4, cudaStream_t st) {
  const MgLevel& L0 = s.lv[0];
  const unsigned nb = (unsigned)((L0.n + 255) / 256);
  launch_poisson_rhs(L0.n, s.rho, s.rho0, s.sums, f4, st);
  int launches = 1;
  MgLevel lv[MG_MAX_LEVELS];
  for (int l = 0; l < s.nlev; ++l) lv[l] = s.lv[l];
  lv[0] = dl0;
  MgSolveArgs d = s;
  d.lv = lv; d.n_vc = 1; d.zero0 = 1; d.rhs_given = 1;
  for (int v = 0; v < s.n_vc; ++v) {
    resid_order4_kernel<<<nb, 256, 0, st>>>(L0.gd, 1.0 / (L0.h * L0.h), L0.u, f4, dl0.f);
    launches += 1 + launch_mg_solve(d, st);
    add_inplace_kernel<<<nb, 256, 0, st>>>(L0.n, L0.u, dl0.u);
    launches += 1;
  }
  return launches;
}

}  // namespace rt
