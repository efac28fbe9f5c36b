// gemm_kernels.cu -- the three FP64 tensor-core (DMMA) stages of the RT-TDDFT step.
//
//   a1 project_kernel  : dH_ij = sum_r phi_i(r) dV(r) phi_j(r)   ("Hupdate", Table 1; Alg. 1 line 25)
//                        M = N = norb, K = Ng; dV fused as a scale on the B fragments (no scaled copy of Phi);
//                        upper-triangular tiles only, split-K with a fixed-order second-stage reduction.
//   a5 density_kernel  : rho(r) = sum_j phi_j(r) (Pfold Phi)_j(r) ("Rho", L544; Eq. 27)
//                        M = norb (j), N = Ng (r), K = norb (i >= j only: Pfold is the upper-triangular fold);
//                        the Ng x N product is never stored: fused row-dot epilogue.
//   a3/a4 gemm_abt     : D = a0 A0 B0^T + a1 A1 B1^T   ("ELDYN", L546): series for cos/sin(X), U P0 U^dagger.
//
// All: 128 x 128 CTA tile, 8 warps (2 x 4), warp tile 64 x 32 = 8 x 4 DMMA tiles, BK = 16, 4-stage cp.async ring.
#include "dmma_core.cuh"
#include "rt_internal.h"

namespace rt {

constexpr int FA = 8, FB = 4, WM = 2, WN = 4;
constexpr int BM = 8 * FA * WM, BN = 8 * FB * WN;      // 128 x 128
constexpr int NT = 32 * WM * WN;                       // 256 threads
constexpr int STAGES = 4;
static_assert(BM == TILE && BN == TILE, "tile mismatch");

// ======================================================================================================
// a1 projection
// ======================================================================================================
constexpr int PROJ_STAGE = BM * BK + BN * BK + BK;     // doubles per stage: A tile, B tile, weights

__global__ void __launch_bounds__(NT, 1)
project_kernel(const double* __restrict__ phi, const double* __restrict__ w, const int2* __restrict__ tiles,
               double* __restrict__ W, const ProjectPlan pl) {
  extern __shared__ __align__(16) double smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, c = lane & 3;
  const int wrow = (warp / WN) * (8 * FA), wcol = (warp % WN) * (8 * FB);
  const int N = pl.N, ldn = pl.ldn;
  const long long Ng = pl.Ng;
  const ProjBlock pb = project_decode(blockIdx.x, pl);
  const int s = pb.s;
  const int2 tt = tiles[pb.t];
  const int i0 = tt.x * TILE, j0 = tt.y * TILE;
  const long long kbeg = pb.kbeg, kend = pb.kend;
  const int nk = (int)((kend - kbeg + BK - 1) / BK);
  const bool vec = ((Ng & 1) == 0) && ((reinterpret_cast<uintptr_t>(phi) & 15) == 0);

  double acc[FA][FB][2];
#pragma unroll
  for (int a = 0; a < FA; ++a)
#pragma unroll
    for (int b = 0; b < FB; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

  auto load = [&](int kt, int slot) {
    double* sA = smem + slot * PROJ_STAGE;
    double* sB = sA + BM * BK;
    double* sW = sB + BN * BK;
    const long long k0 = kbeg + (long long)kt * BK;
    load_tile_kc<BM, NT>(sA, phi, Ng, i0, N, k0, kend, vec, tid);
    load_tile_kc<BN, NT>(sB, phi, Ng, j0, N, k0, kend, vec, tid);
    if (tid < 8) {
      const long long k = k0 + 2 * tid, rem = kend - k;
      if ((reinterpret_cast<uintptr_t>(w) & 15) == 0) {
        int bytes = rem > 0 ? (rem >= 2 ? 16 : 8) : 0;
        cp_async16(sW + 2 * tid, bytes ? (const void*)(w + k) : (const void*)w, bytes);
      } else {
        int b0 = rem > 0 ? 8 : 0, b1 = rem > 1 ? 8 : 0;
        cp_async8(sW + 2 * tid, b0 ? (const void*)(w + k) : (const void*)w, b0);
        cp_async8(sW + 2 * tid + 1, b1 ? (const void*)(w + k + 1) : (const void*)w, b1);
      }
    }
  };

#pragma unroll
  for (int p = 0; p < STAGES - 1; ++p) {
    if (p < nk) load(p, p);
    cp_async_commit();
  }
  for (int kt = 0; kt < nk; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    const int nxt = kt + STAGES - 1;
    if (nxt < nk) load(nxt, nxt % STAGES);
    cp_async_commit();
    const double* sA = smem + (kt % STAGES) * PROJ_STAGE;
    mma_stage_kc<FA, FB, true>(acc, sA, sA + BM * BK, sA + BM * BK + BN * BK, wrow, wcol, g, c);
  }
  cp_async_wait<0>();

  // epilogue: raw partial sums into slab s (upper tiles only; the reduce kernel scales / mirrors)
  double* Ws = W + (long long)s * N * ldn;
#pragma unroll
  for (int a = 0; a < FA; ++a) {
    const int row = i0 + wrow + 8 * a + g;
    if (row < N) {
#pragma unroll
      for (int b = 0; b < FB; ++b) {
        const int col = j0 + wcol + 8 * b + 2 * c;
        if (col < N) *reinterpret_cast<double2*>(Ws + (long long)row * ldn + col) = make_double2(acc[a][b][0], acc[a][b][1]);
      }
    }
  }
}

__global__ void project_reduce_kernel(const double* __restrict__ W, const double* __restrict__ eps, double scale,
                                      double* __restrict__ H, int N, int ldn, int S, int Sn, int Sd, int narrow_tile,
                                      const double* __restrict__ Hadd) {
  // one thread per (i, j) with j >= i; fixed summation order over the splits
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int i = blockIdx.y;
  if (j >= N || j < i) return;
  const long long slab = (long long)N * ldn;
  const double* p = W + (long long)i * ldn + j;
  double sum = 0.0;
  // diagonal tiles and the tiles of a narrow last column have their own split counts (ProjectPlan)
  const int ns = (i / TILE == j / TILE) ? Sd : (j / TILE == narrow_tile ? Sn : S);
  // 16 loads in flight per thread, added in split order (with one load per add the kernel is a chain of ns L2 round
  // trips: 67 us for the 148 splits of `small`, 9 % of its step)
  int s = 0;
  for (; s + 16 <= ns; s += 16) {
    double v[16];
#pragma unroll
    for (int u = 0; u < 16; ++u) v[u] = p[(long long)(s + u) * slab];
#pragma unroll
    for (int u = 0; u < 16; ++u) sum += v[u];
  }
  for (; s < ns; ++s) sum += p[(long long)s * slab];
  double v = scale * sum;
  if (i == j && eps) v += eps[i];
  if (Hadd) v += Hadd[(long long)i * ldn + j];
  H[(long long)i * ldn + j] = v;
  H[(long long)j * ldn + i] = v;
}

size_t project_smem_bytes() { return (size_t)STAGES * PROJ_STAGE * sizeof(double); }

void launch_project(const ProjectPlan& p, const double* phi, const double* w, const int2* tiles, double* W,
                    cudaStream_t st) {
  static bool attr = false;
  if (!attr) {
    cudaFuncSetAttribute(project_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)project_smem_bytes());
    attr = true;
  }
  project_kernel<<<p.grid(), NT, project_smem_bytes(), st>>>(phi, w, tiles, W, p);
}

void launch_project_reduce(const ProjectPlan& p, const double* W, const double* eps, double scale, double* H,
                           cudaStream_t st, const double* Hadd) {
  dim3 grid((p.N + 127) / 128, p.N);
  project_reduce_kernel<<<grid, 128, 0, st>>>(W, eps, scale, H, p.N, p.ldn, p.S, p.Sn, p.Sd, p.Tn > 0 ? p.ntile - 1 : -1,
                                              Hadd);
}

// ======================================================================================================
// a5 density
// ======================================================================================================
constexpr int DENS_STAGE = BM * BK + BK * BN;          // A tile (Pfold, K-contiguous) + B tile (Phi, N-contiguous)

__global__ void __launch_bounds__(NT, 1)
density_kernel(const double* __restrict__ phi, const double* __restrict__ Pf, double* __restrict__ rho_part, int N,
               long long Ng, int ntile, int npairs, long long nrt, int ldn, int group_r) {
  extern __shared__ __align__(16) double smem[];
  __shared__ double colred[WM][BN];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, c = lane & 3;
  const int wm = warp / WN, wn = warp % WN;
  const int wrow = wm * (8 * FA), wcol = wn * (8 * FB);

  // raster: supertiles of group_r r-tiles x all pairs, pair index fastest inside a supertile column
  const long long L = blockIdx.x;
  const long long per_group = (long long)group_r * npairs;
  const long long grp = L / per_group;
  const long long in = L % per_group;
  const long long r_first = grp * group_r;
  const long long gr_here = (nrt - r_first < group_r) ? (nrt - r_first) : group_r;
  const int pair = (int)(in / gr_here);
  const long long rt_ = r_first + in % gr_here;
  if (pair >= npairs || rt_ >= nrt) return;
  const long long r0 = rt_ * TILE;
  const bool vecP = true;   // Pfold is library-owned: ldn is a multiple of 8, base cudaMalloc-aligned
  const bool vecF = ((Ng & 1) == 0) && ((reinterpret_cast<uintptr_t>(phi) & 15) == 0);

  double colsum[FB / 2][4];
#pragma unroll
  for (int t = 0; t < FB / 2; ++t)
#pragma unroll
    for (int q = 0; q < 4; ++q) colsum[t][q] = 0.0;

  for (int which = 0; which < 2; ++which) {
    const int jt = which == 0 ? pair : ntile - 1 - pair;
    if (which == 1 && jt <= pair) break;
    const int j0 = jt * TILE;
    const int kbeg = j0;                       // Pfold is zero below the diagonal: i >= j0 only
    const int nk = (N - kbeg + BK - 1) / BK;

    double acc[FA][FB][2];
#pragma unroll
    for (int a = 0; a < FA; ++a)
#pragma unroll
      for (int b = 0; b < FB; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

    auto load = [&](int kt, int slot) {
      double* sA = smem + slot * DENS_STAGE;
      double* sB = sA + BM * BK;
      const int k0 = kbeg + kt * BK;
      load_tile_kc<BM, NT>(sA, Pf, ldn, j0, N, k0, N, vecP, tid);
      load_tile_nc<BN, NT>(sB, phi, Ng, k0, N, r0, Ng, vecF, tid);
    };
    __syncthreads();   // previous j-tile's last stage fully consumed before its slots are refilled
#pragma unroll
    for (int p = 0; p < STAGES - 1; ++p) {
      if (p < nk) load(p, p);
      cp_async_commit();
    }
    for (int kt = 0; kt < nk; ++kt) {
      cp_async_wait<STAGES - 2>();
      __syncthreads();
      const int nxt = kt + STAGES - 1;
      if (nxt < nk) load(nxt, nxt % STAGES);
      cp_async_commit();
      const double* sA = smem + (kt % STAGES) * DENS_STAGE;
      mma_stage_nc<FA, FB, BN>(acc, sA, sA + BM * BK, wrow, wcol, g, c);
    }
    cp_async_wait<0>();

    // fused row-dot: colsum(r) += sum_j phi_j(r) * T_j(r); lane owns columns wcol + 16 t + 4 c + {0..3}
#pragma unroll
    for (int a = 0; a < FA; ++a) {
      const int j = j0 + wrow + 8 * a + g;
      if (j < N) {
        const double* prow = phi + (long long)j * Ng + r0 + wcol + 4 * c;
#pragma unroll
        for (int t = 0; t < FB / 2; ++t) {
          const long long col = r0 + wcol + 16 * t + 4 * c;
          double f[4];
          if (vecF && col + 3 < Ng) {
            const double2 f01 = *reinterpret_cast<const double2*>(prow + 16 * t);
            const double2 f23 = *reinterpret_cast<const double2*>(prow + 16 * t + 2);
            f[0] = f01.x; f[1] = f01.y; f[2] = f23.x; f[3] = f23.y;
          } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) f[q] = (col + q < Ng) ? prow[16 * t + q] : 0.0;
          }
          // column offset q = 2 e + p  <->  acc[a][2 t + p][e]
          colsum[t][0] += f[0] * acc[a][2 * t][0];
          colsum[t][1] += f[1] * acc[a][2 * t + 1][0];
          colsum[t][2] += f[2] * acc[a][2 * t][1];
          colsum[t][3] += f[3] * acc[a][2 * t + 1][1];
        }
      }
    }
  }

  // reduce over the 8 row groups g of the warp (lanes with equal c), then over the WM warps sharing columns
#pragma unroll
  for (int t = 0; t < FB / 2; ++t)
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      double v = colsum[t][q];
      v += __shfl_xor_sync(0xffffffffu, v, 4);
      v += __shfl_xor_sync(0xffffffffu, v, 8);
      v += __shfl_xor_sync(0xffffffffu, v, 16);
      colsum[t][q] = v;
    }
  if (g == 0) {
#pragma unroll
    for (int t = 0; t < FB / 2; ++t)
#pragma unroll
      for (int q = 0; q < 4; ++q) colred[wm][wcol + 16 * t + 4 * c + q] = colsum[t][q];
  }
  __syncthreads();
  if (tid < BN) {
    const long long r = r0 + tid;
    if (r < Ng) {
      double v = 0.0;
#pragma unroll
      for (int m = 0; m < WM; ++m) v += colred[m][tid];
      rho_part[(long long)pair * Ng + r] = v;
    }
  }
}

size_t density_smem_bytes() { return (size_t)STAGES * DENS_STAGE * sizeof(double); }

void launch_density(const DensityPlan& p, const double* phi, const double* Pfold, double* rho_part, cudaStream_t st) {
  static bool attr = false;
  if (!attr) {
    cudaFuncSetAttribute(density_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)density_smem_bytes());
    attr = true;
  }
  const long long ngroups = (p.nrt + p.group_r - 1) / p.group_r;
  const long long nblocks = ngroups * p.group_r * p.npairs;
  density_kernel<<<(unsigned)nblocks, NT, density_smem_bytes(), st>>>(phi, Pfold, rho_part, p.N, p.Ng, p.ntile,
                                                                      p.npairs, p.nrt, p.ldn, p.group_r);
}

__global__ void fold_upper_kernel(const double* __restrict__ P, double* __restrict__ Pf, int N, int ldn) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;   // column
  const int j = blockIdx.y;                              // row
  if (i >= ldn) return;
  double v = 0.0;
  if (i < N) {
    const double p = P[(long long)j * ldn + i];
    v = (i > j) ? 2.0 * p : (i == j ? p : 0.0);
  }
  Pf[(long long)j * ldn + i] = v;
}

void launch_fold_upper(int N, int ldn, const double* P, double* Pfold, cudaStream_t st) {
  dim3 grid((ldn + 127) / 128, N);
  fold_upper_kernel<<<grid, 128, 0, st>>>(P, Pfold, N, ldn);
}

// ======================================================================================================
// a3/a4 N x N GEMM, D = a0 A0 B0^T + a1 A1 B1^T
// ======================================================================================================
// Tile variants: 128 x 128 (8 warps, warp tile 64 x 32) for large N; 64 x 64 and 32 x 32 CTA tiles for small N, where
// 128 x 128 tiles would leave most of the 148 SMs idle (N = 128 is ONE such tile, N = 512 sixteen).
template <int FA, int FB, int WM, int WN>
__global__ void __launch_bounds__(32 * WM * WN)
gemm_abt_kernel(GemmArgs ga) {
  constexpr int BM = 8 * FA * WM, BN = 8 * FB * WN, NT = 32 * WM * WN;
  constexpr int GEMM_STAGE = BM * BK + BN * BK;
  if (ga.skip && *ga.skip) return;
  extern __shared__ __align__(16) double smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, c = lane & 3;
  const int wrow = (warp / WN) * (8 * FA), wcol = (warp % WN) * (8 * FB);
  const int N = ga.N, ldn = ga.ldn;
  const int i0 = ga.row_beg + blockIdx.y * BM, j0 = blockIdx.x * BN;
  const int nk1 = (N + BK - 1) / BK;
  const int nk = ga.A1 ? 2 * nk1 : nk1;

  double acc[FA][FB][2];
#pragma unroll
  for (int a = 0; a < FA; ++a)
#pragma unroll
    for (int b = 0; b < FB; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

  auto load = [&](int kt, int slot) {
    double* sA = smem + slot * GEMM_STAGE;
    double* sB = sA + BM * BK;
    const bool second = kt >= nk1;
    const double* A = second ? ga.A1 : ga.A0;
    const double* B = second ? ga.B1 : ga.B0;
    const int k0 = (second ? kt - nk1 : kt) * BK;
    load_tile_kc<BM, NT>(sA, A, ldn, i0, N, k0, N, true, tid);
    load_tile_kc<BN, NT>(sB, B, ldn, j0, N, k0, N, true, tid);
  };
#pragma unroll
  for (int p = 0; p < STAGES - 1; ++p) {
    if (p < nk) load(p, p);
    cp_async_commit();
  }
  const double ratio = ga.A1 ? ga.alpha1 / ga.alpha0 : 1.0;
  for (int kt = 0; kt < nk; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    const int nxt = kt + STAGES - 1;
    if (nxt < nk) load(nxt, nxt % STAGES);
    cp_async_commit();
    const double* sA = smem + (kt % STAGES) * GEMM_STAGE;
    if (kt == nk1 && ratio != 1.0) {
      // switch terms: fold alpha1/alpha0 into the accumulators so that the final scale is alpha0 for both
      const double inv = 1.0 / ratio;            // ratios used by the library are +-1: exact
#pragma unroll
      for (int a = 0; a < FA; ++a)
#pragma unroll
        for (int b = 0; b < FB; ++b) { acc[a][b][0] *= inv; acc[a][b][1] *= inv; }
    }
    mma_stage_kc<FA, FB, false>(acc, sA, sA + BM * BK, nullptr, wrow, wcol, g, c);
  }
  cp_async_wait<0>();
  const double fin = (ga.A1 && ratio != 1.0) ? ga.alpha0 * ratio : ga.alpha0;

#pragma unroll
  for (int a = 0; a < FA; ++a) {
    const int row = i0 + wrow + 8 * a + g;
    if (row < N) {
#pragma unroll
      for (int b = 0; b < FB; ++b) {
        const int col = j0 + wcol + 8 * b + 2 * c;
        if (col < N) {
          const long long o = (long long)row * ldn + col;
          const double2 d = make_double2(fin * acc[a][b][0], fin * acc[a][b][1]);
          if (ga.D) *reinterpret_cast<double2*>(ga.D + o) = d;
          if (ga.Z1) {
            double2 z = *reinterpret_cast<double2*>(ga.Z1 + o);
            z.x += ga.beta1 * d.x; z.y += ga.beta1 * d.y;
            *reinterpret_cast<double2*>(ga.Z1 + o) = z;
          }
          if (ga.Z2) {
            double2 z = *reinterpret_cast<double2*>(ga.Z2 + o);
            z.x += ga.beta2 * d.x; z.y += ga.beta2 * d.y;
            *reinterpret_cast<double2*>(ga.Z2 + o) = z;
          }
        }
      }
    }
  }
}

size_t gemm_smem_bytes() { return (size_t)STAGES * (BM * BK + BN * BK) * sizeof(double); }

template <int FA_, int FB_, int WM_, int WN_>
static void launch_gemm_variant(const GemmArgs& g, cudaStream_t st) {
  constexpr int bm = 8 * FA_ * WM_, bn = 8 * FB_ * WN_;
  const size_t smem = (size_t)STAGES * (bm + bn) * BK * sizeof(double);
  static bool attr = false;
  if (!attr) {
    cudaFuncSetAttribute(gemm_abt_kernel<FA_, FB_, WM_, WN_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    attr = true;
  }
  const int rows = g.row_end - g.row_beg;
  if (rows <= 0) return;
  gemm_abt_kernel<FA_, FB_, WM_, WN_><<<dim3((g.N + bn - 1) / bn, (rows + bm - 1) / bm), 32 * WM_ * WN_, smem, st>>>(g);
}

void launch_gemm_abt(const GemmArgs& g, cudaStream_t st) {
  if (g.N <= GEMM_SMALL_N32) launch_gemm_variant<2, 2, 2, 2>(g, st);          // 32 x 32 tiles, 4 warps
  else if (g.N <= GEMM_SMALL_N) launch_gemm_variant<4, 2, 2, 4>(g, st);        // 64 x 64 tiles, 8 warps
  else launch_gemm_variant<FA, FB, WM, WN>(g, st);                             // 128 x 128 tiles
}

}  // namespace rt
