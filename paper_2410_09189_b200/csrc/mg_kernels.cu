// mg_kernels.cu -- a7 "Vh": periodic 7-point Poisson solve, fixed count of V(nu1,nu2) cycles, weighted Jacobi,
// full weighting, trilinear prolongation, exact separable solve on the coarsest level (DESIGN R6; the paper only
// says "multigrid", Table 1 "Vh" L545).
//
// Two kinds of kernels:
//   * levels with more than MG_CLUSTER_MAX_PTS points: shared-memory tiles with halos, 3 launches per level per cycle
//       mg_smooth_kernel<false>  : nu (1 or 2) Jacobi sweeps fused; the tile is loaded once with a halo of nu
//       mg_resid_restrict_kernel : residual on a (2c+1)^3 fine patch kept in shared memory, full weighting -> coarse rhs
//       mg_smooth_kernel<true>   : u + P e (coarse patch staged in shared memory) followed by the post-sweeps
//   * all smaller levels: ONE launch of mg_cluster_kernel per cycle (or per solve when the finest level is small):
//       a thread-block cluster of 8 CTAs walks down and up the hierarchy, phases separated by the hardware cluster
//       barrier (~0.2 us, flushes L1) instead of kernel boundaries (~2 us each); arrays stay in L2.
// Every value is computed with the same formula and operand order as before the fusion (one thread per output).
#include "rt_internal.h"

#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace rt {

namespace {

constexpr int MG_THREADS = 256;          // tile kernels
constexpr int CL_THREADS = 1024;         // cluster kernel, per CTA
constexpr int CL_SIZE = 8;               // CTAs per cluster (portable maximum)

__device__ __forceinline__ int wrapi(int i, int n) {
  i %= n;
  return i < 0 ? i + n : i;
}
__device__ __forceinline__ void decode3(int i, int ny, int nz, int& x, int& y, int& z) {
  const int nyz = ny * nz;
  x = i / nyz;
  const int rem = i - x * nyz;
  y = rem / nz;
  z = rem - y * nz;
}

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
  double* A = sm;
  double* B = A + nA;
  double* C = B + nB;
  int* xs = reinterpret_cast<int*>(C + cx * cy * cz);
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
    for (int i = tid; i < cx * cy * cz; i += MG_THREADS) {
      int lx, ly, lz;
      decode3(i, cy, cz, lx, ly, lz);
      C[i] = a.ec[((long long)wrapi(c0x + lx, ncx) * ncy + wrapi(c0y + ly, ncy)) * ncz + wrapi(c0z + lz, ncz)];
    }
  }
  __syncthreads();

  // load the tile with its halo (periodic wrap); PROLONG: add the trilinear interpolation of the coarse patch
  for (int i = tid; i < nA; i += MG_THREADS) {
    int lx, ly, lz;
    decode3(i, ry, rz, lx, ly, lz);
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
  __syncthreads();

  if (H == 2) {       // first sweep: halo-1 region, stays in shared memory
    const int dy = ry - 2, dz = rz - 2;
    for (int i = tid; i < nB; i += MG_THREADS) {
      int lx, ly, lz;
      decode3(i, dy, dz, lx, ly, lz);
      const double fv = a.f[((long long)xs[lx + 1] * ny + ys[ly + 1]) * nz + zs[lz + 1]];
      B[i] = jacobi_point(A, ry, rz, ((lx + 1) * ry + ly + 1) * rz + lz + 1, fv, a.h2, a.omega);
    }
    __syncthreads();
  }
  if (H == 0) {       // no sweep: u + P e only
    for (int i = tid; i < nA; i += MG_THREADS) {
      int lx, ly, lz;
      decode3(i, ry, rz, lx, ly, lz);
      const int X = x0 + lx, Y = y0 + ly, Z = z0 + lz;
      if (X >= nx || Y >= ny || Z >= nz) continue;
      a.uout[((long long)X * ny + Y) * nz + Z] = A[i];
    }
  } else {            // last sweep: interior, to global memory
    const double* S = (H == 2) ? B : A;
    const int sy = ry - (H == 2 ? 2 : 0), sz = rz - (H == 2 ? 2 : 0);
    const int nI = a.bx * a.by * a.bz;
    for (int i = tid; i < nI; i += MG_THREADS) {
      int lx, ly, lz;
      decode3(i, a.by, a.bz, lx, ly, lz);
      const int X = x0 + lx, Y = y0 + ly, Z = z0 + lz;
      if (X >= nx || Y >= ny || Z >= nz) continue;
      const long long g = ((long long)X * ny + Y) * nz + Z;
      a.uout[g] = jacobi_point(S, sy, sz, ((lx + 1) * sy + ly + 1) * sz + lz + 1, a.f[g], a.h2, a.omega);
    }
  }
}

size_t smooth_smem_bytes(int bx, int by, int bz, int H, bool prolong) {
  const int rx = bx + 2 * H, ry = by + 2 * H, rz = bz + 2 * H;
  size_t d = (size_t)rx * ry * rz + (H == 2 ? (size_t)(rx - 2) * (ry - 2) * (rz - 2) : 0);
  if (prolong) d += (size_t)(rx / 2 + 2) * (ry / 2 + 2) * (rz / 2 + 2);
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
  for (int i = tid; i < ux * uy * uz; i += MG_THREADS) {
    int lx, ly, lz;
    decode3(i, uy, uz, lx, ly, lz);
    U[i] = a.u[((long long)xs[lx] * ny + ys[ly]) * nz + zs[lz]];
  }
  __syncthreads();
  for (int i = tid; i < qx * qy * qz; i += MG_THREADS) {
    int lx, ly, lz;
    decode3(i, qy, qz, lx, ly, lz);
    const int o = ((lx + 1) * uy + ly + 1) * uz + lz + 1, px = uy * uz;
    const double nb = U[o - px] + U[o + px] + U[o - uz] + U[o + uz] + U[o - 1] + U[o + 1];
    const double fv = a.f[((long long)xs[lx + 1] * ny + ys[ly + 1]) * nz + zs[lz + 1]];
    R[i] = fv - (6.0 * U[o] - nb) * a.inv_h2;
  }
  __syncthreads();
  const int ncx = a.gc.nx, ncy = a.gc.ny, ncz = a.gc.nz;
  for (int i = tid; i < a.cbx * a.cby * a.cbz; i += MG_THREADS) {
    int I, J, K;
    decode3(i, a.cby, a.cbz, I, J, K);
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

struct ClusterCtx {
  cg::cluster_group cl;
  int gtid, gthreads;
  __device__ __forceinline__ void sync() { __threadfence(); cl.sync(); }
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

__device__ void cl_jacobi(ClusterCtx& c, const MgLevel& L, const double* in, double* out, double omega) {
  const int n = (int)L.n;
  const double h2 = L.h * L.h;
  for (int r = c.gtid; r < n; r += c.gthreads) {
    if (!in) { out[r] = (1.0 - omega) * 0.0 + (omega / 6.0) * (h2 * L.f[r] + 0.0); continue; }
    int ix, iy, iz;
    decode3(r, L.gd.ny, L.gd.nz, ix, iy, iz);
    out[r] = (1.0 - omega) * in[r] + (omega / 6.0) * (h2 * L.f[r] + nb_sum_g(in, L.gd, ix, iy, iz));
  }
  c.sync();
}

__device__ void cl_residual(ClusterCtx& c, const MgLevel& L, const double* u) {
  const int n = (int)L.n;
  const double inv_h2 = 1.0 / (L.h * L.h);
  for (int r = c.gtid; r < n; r += c.gthreads) {
    int ix, iy, iz;
    decode3(r, L.gd.ny, L.gd.nz, ix, iy, iz);
    L.r[r] = L.f[r] - (6.0 * u[r] - nb_sum_g(u, L.gd, ix, iy, iz)) * inv_h2;
  }
  c.sync();
}

__device__ void cl_restrict(ClusterCtx& c, const MgLevel& F, const MgLevel& Cc) {
  const int nc = (int)Cc.n;
  const GridDims gf = F.gd, gc = Cc.gd;
  const int nyz = gf.ny * gf.nz;
  for (int r = c.gtid; r < nc; r += c.gthreads) {
    int I, J, K;
    decode3(r, gc.ny, gc.nz, I, J, K);
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

__device__ void cl_prolong_add(ClusterCtx& c, const MgLevel& Cc, const double* ec, const MgLevel& F, double* u) {
  const int nf = (int)F.n;
  const GridDims gf = F.gd, gc = Cc.gd;
  const int nyz = gc.ny * gc.nz;
  for (int r = c.gtid; r < nf; r += c.gthreads) {
    int ix, iy, iz;
    decode3(r, gf.ny, gf.nz, ix, iy, iz);
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
__device__ void cl_coarse_solve(ClusterCtx& c, const MgLevel& L, const ClusterArgs& a, double* u) {
  const int nx = L.gd.nx, ny = L.gd.ny, nz = L.gd.nz;
  const int n = nx * ny * nz;
  const double* f = L.f;
  double* s0 = L.r;
  double* s1 = L.tmp;
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // x: f -> s0, contract with Q^T
    const int q = o / (ny * nz), rest = o % (ny * nz);
    double s = 0.0;
    for (int i = 0; i < nx; ++i) s += a.Qx[i * nx + q] * f[i * ny * nz + rest];
    s0[o] = s;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // y: s0 -> s1
    const int q = o / (ny * nz), b = (o / nz) % ny, k = o % nz;
    double s = 0.0;
    for (int j = 0; j < ny; ++j) s += a.Qy[j * ny + b] * s0[(q * ny + j) * nz + k];
    s1[o] = s;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // z and the division: s1 -> s0
    const int q = o / (ny * nz), b = (o / nz) % ny, cc = o % nz;
    double s = 0.0;
    for (int k = 0; k < nz; ++k) s += a.Qz[k * nz + cc] * s1[(q * ny + b) * nz + k];
    const double lam = a.lx[q] + a.ly[b] + a.lz[cc];
    s0[o] = (q == 0 && b == 0 && cc == 0) ? 0.0 : s / lam;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // back, z: s0 -> s1, contract with Q
    const int q = o / (ny * nz), b = (o / nz) % ny, k = o % nz;
    double s = 0.0;
    for (int cc = 0; cc < nz; ++cc) s += a.Qz[k * nz + cc] * s0[(q * ny + b) * nz + cc];
    s1[o] = s;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // y: s1 -> s0
    const int q = o / (ny * nz), j = (o / nz) % ny, k = o % nz;
    double s = 0.0;
    for (int b = 0; b < ny; ++b) s += a.Qy[j * ny + b] * s1[(q * ny + b) * nz + k];
    s0[o] = s;
  }
  c.sync();
  for (int o = c.gtid; o < n; o += c.gthreads) {                    // x: s0 -> u
    const int i = o / (ny * nz), rest = o % (ny * nz);
    double s = 0.0;
    for (int q = 0; q < nx; ++q) s += a.Qx[i * nx + q] * s0[q * ny * nz + rest];
    u[o] = s;
  }
  c.sync();
}

__global__ void __cluster_dims__(CL_SIZE, 1, 1) __launch_bounds__(CL_THREADS)
mg_cluster_kernel(const __grid_constant__ ClusterArgs a) {
  ClusterCtx c{cg::this_cluster(), 0, 0};
  c.gtid = (int)c.cl.block_rank() * CL_THREADS + threadIdx.x;
  c.gthreads = CL_SIZE * CL_THREADS;
  const int last = a.nlev - 1;

  if (a.do_rhs) {
    const MgLevel& L = a.lv[0];
    const int n = (int)L.n;
    const double mean = a.sums[4] / (double)n;
    for (int r = c.gtid; r < n; r += c.gthreads) {
      const double d = a.rho0 ? a.rho[r] - a.rho0[r] : a.rho[r];
      L.f[r] = 4.0 * 3.14159265358979323846 * (d - mean);
    }
    c.sync();
  }

  // where each level's current solution lives (u or tmp); sweeps ping-pong between the two
  double* cur[MG_MAX_LEVELS];
  for (int l = 0; l < a.nlev; ++l) cur[l] = a.lv[l].u;

  for (int cyc = 0; cyc < a.ncycles; ++cyc) {
    for (int l = 0; l < last; ++l) {
      const MgLevel& L = a.lv[l];
      bool zero = (l > 0) || (a.zero_guess && cyc == 0);
      for (int s = 0; s < a.nu1; ++s) {
        // zero guess: nothing is read, so start in the buffer from which the remaining sweeps end in u
        double* out = zero ? (((a.nu1 - 1 + a.nu2) & 1) ? L.tmp : L.u) : (cur[l] == L.u ? L.tmp : L.u);
        cl_jacobi(c, L, zero ? nullptr : cur[l], out, a.omega);
        cur[l] = out;
        zero = false;
      }
      if (zero) {           // nu1 == 0 with a zero guess: the residual needs an actual array of zeros
        for (int r = c.gtid; r < (int)L.n; r += c.gthreads) L.u[r] = 0.0;
        cur[l] = L.u;
        c.sync();
      }
      cl_residual(c, L, cur[l]);
      cl_restrict(c, L, a.lv[l + 1]);
    }
    cl_coarse_solve(c, a.lv[last], a, a.lv[last].u);
    cur[last] = a.lv[last].u;
    for (int l = last - 1; l >= 0; --l) {
      const MgLevel& L = a.lv[l];
      cl_prolong_add(c, a.lv[l + 1], cur[l + 1], L, cur[l]);
      for (int s = 0; s < a.nu2; ++s) {
        double* out = cur[l] == L.u ? L.tmp : L.u;
        cl_jacobi(c, L, cur[l], out, a.omega);
        cur[l] = out;
      }
    }
  }
  if (cur[0] != a.lv[0].u) {
    const MgLevel& L = a.lv[0];
    for (int r = c.gtid; r < (int)L.n; r += c.gthreads) L.u[r] = cur[0][r];
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------- host side
namespace {

int tile_edge(int n, int bmax) {            // equal tiles of at most bmax points covering n
  const int nt = (n + bmax - 1) / bmax;
  return (n + nt - 1) / nt;
}

struct TileGeom { int bx, by, bz, tx, ty, tz; };
TileGeom make_geom(const GridDims& g, int mx, int my, int mz) {
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
  mg_resid_restrict_kernel<<<(unsigned)(t.tx * t.ty * t.tz), MG_THREADS, resrest_smem_bytes(t.bx, t.by, t.bz), st>>>(a);
}

void launch_cluster(const MgSolveArgs& s, int l0, int ncycles, int zero_guess, int do_rhs, cudaStream_t st) {
  ClusterArgs a{};
  a.nlev = s.nlev - l0; a.ncycles = ncycles; a.zero_guess = zero_guess;
  a.nu1 = s.nu1; a.nu2 = s.nu2; a.omega = s.omega;
  for (int l = l0; l < s.nlev; ++l) a.lv[l - l0] = s.lv[l];
  a.Qx = s.Qx; a.Qy = s.Qy; a.Qz = s.Qz; a.lx = s.lx; a.ly = s.ly; a.lz = s.lz;
  a.do_rhs = do_rhs; a.rho = s.rho; a.rho0 = s.rho0; a.sums = s.sums;
  mg_cluster_kernel<<<CL_SIZE, CL_THREADS, 0, st>>>(a);
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
    const bool zero = l > 0;
    if (zero && s.nu1 == 0) { cudaMemsetAsync(L.u, 0, (size_t)L.n * 8, st); cur[l] = L.u; }
    else smooth(l, s.nu1, zero);
    launch_resid_restrict(L, s.lv[l + 1], cur[l], st);
    ++launches;
    if (l + 1 == lc) {
      launch_cluster(s, lc, 1, 1, 0, st);
      ++launches;
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
  return (int)e;
}

int launch_mg_solve(const MgSolveArgs& s, cudaStream_t st) {
  int lc = 0;
  while (lc < s.nlev - 1 && s.lv[lc].n > MG_CLUSTER_MAX_PTS) ++lc;
  if (lc == 0) {           // the whole hierarchy is small: rhs + every cycle in one launch
    launch_cluster(s, 0, s.n_vc, 0, 1, st);
    return 1;
  }
  launch_poisson_rhs(s.lv[0].n, s.rho, s.rho0, s.sums, s.lv[0].f, st);
  BigCycle bc{s, lc, st};
  for (int l = 0; l < s.nlev; ++l) bc.cur[l] = s.lv[l].u;
  for (int v = 0; v < s.n_vc; ++v) bc.vcycle(0);
  if (bc.cur[0] != s.lv[0].u)
    cudaMemcpyAsync(s.lv[0].u, bc.cur[0], (size_t)s.lv[0].n * 8, cudaMemcpyDeviceToDevice, st);
  return bc.launches + 1;
}

}  // namespace rt
