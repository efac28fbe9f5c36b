// dmma_core.cuh -- FP64 tensor-core (DMMA.8x8x4) tile machinery shared by the three GEMM-shaped stages
// (a1 projection, a5 density, a3/a4 N x N propagator GEMMs).  sm_100a only.
//
// FP64 is not a tcgen05 kind, so the contraction runs on warp-level mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4)
// with register accumulators; operands are staged global -> shared with 16-byte cp.async (LDGSTS) in a
// multi-stage ring, and read back with conflict-free 128-bit LDS thanks to an XOR chunk swizzle.
//
// Tile geometry (all kernels): CTA tile BM x BN, BK = 16 doubles per stage, warp tile (8*FA) x (8*FB).
//
// Shared layouts (a "chunk" is 16 bytes = 2 doubles):
//   K-contiguous operand  [rows][16]      : chunk ch of row r lives at chunk (ch ^ ((r & 1) << 2))
//   N-contiguous operand  [16 k-rows][BN] : chunk ch of k-row k lives at chunk (ch ^ (((k >> 1) & 3) << 1))
//
// Fragment <-> k mapping.  m8n8k4 sums over 4 k values held by the 4 lanes c = lane & 3 of a quad; WHICH k a
// lane holds is free as long as A and B agree.  One LDS.128 gives a lane two consecutive doubles, so inside a
// 16-wide stage we use, for half in {0,1}, e in {0,1}:   k(c, half, e) = 2 c + 8 half + e
// (4 MMA k-steps per stage, each A/B 128-bit load feeding two of them).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rt {

constexpr int BK = 16;   // doubles per pipeline stage along the contraction

__device__ __forceinline__ void dmma884(double& d0, double& d1, const double a, const double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem, int src_bytes) {
  uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- global -> shared tile loaders -----------------------------------------------------------------

// K-contiguous tile: ROWS rows x 16 doubles from g[(row0 + r) * ld + k0 ...], rows >= nrows and k >= kend are
// zero-filled.  vec16: rows are 16-byte aligned (ld even, base aligned, k0 even).
template <int ROWS, int NT>
__device__ __forceinline__ void load_tile_kc(double* sm, const double* __restrict__ g, long long ld, int row0,
                                             int nrows, long long k0, long long kend, bool vec16, int tid) {
#pragma unroll
  for (int i = 0; i < (ROWS * 8) / NT; ++i) {
    const int idx = tid + i * NT;
    const int r = idx >> 3, ch = idx & 7;
    const int gr = row0 + r;
    const long long k = k0 + 2 * ch;
    double* dst = sm + r * BK + ((ch ^ ((r & 1) << 2)) << 1);
    const long long rem = kend - k;
    const bool rok = gr < nrows;
    const double* src = g + (long long)gr * ld + k;
    if (vec16) {
      int bytes = (rok && rem > 0) ? (rem >= 2 ? 16 : 8) : 0;
      cp_async16(dst, bytes ? (const void*)src : (const void*)g, bytes);
    } else {
      int b0 = (rok && rem > 0) ? 8 : 0, b1 = (rok && rem > 1) ? 8 : 0;
      cp_async8(dst, b0 ? (const void*)src : (const void*)g, b0);
      cp_async8(dst + 1, b1 ? (const void*)(src + 1) : (const void*)g, b1);
    }
  }
}

// N-contiguous tile: 16 k-rows x COLS doubles from g[(k0 + kr) * ld + col0 ...]; k >= kend and col >= ncols
// are zero-filled.
template <int COLS, int NT>
__device__ __forceinline__ void load_tile_nc(double* sm, const double* __restrict__ g, long long ld, long long k0,
                                             long long kend, long long col0, long long ncols, bool vec16, int tid) {
  constexpr int CH = COLS / 2;   // chunks per k-row
#pragma unroll
  for (int i = 0; i < (BK * CH) / NT; ++i) {
    const int idx = tid + i * NT;
    const int kr = idx / CH, ch = idx % CH;
    const long long k = k0 + kr;
    const long long col = col0 + 2 * ch;
    double* dst = sm + kr * COLS + ((ch ^ (((kr >> 1) & 3) << 1)) << 1);
    const long long rem = ncols - col;
    const bool kok = k < kend;
    const double* src = g + k * ld + col;
    if (vec16) {
      int bytes = (kok && rem > 0) ? (rem >= 2 ? 16 : 8) : 0;
      cp_async16(dst, bytes ? (const void*)src : (const void*)g, bytes);
    } else {
      int b0 = (kok && rem > 0) ? 8 : 0, b1 = (kok && rem > 1) ? 8 : 0;
      cp_async8(dst, b0 ? (const void*)src : (const void*)g, b0);
      cp_async8(dst + 1, b1 ? (const void*)(src + 1) : (const void*)g, b1);
    }
  }
}

// ---- one pipeline stage of MMAs ------------------------------------------------------------------------
// acc[FA][FB][2]; smA: K-contiguous [BM][16]; warp rows start at wrow; lane = (g = lane >> 2, c = lane & 3).

// B K-contiguous ([BN][16]); optional per-k weights wk (16 doubles in shared, may be nullptr when !SCALE).
template <int FA, int FB, bool SCALE>
__device__ __forceinline__ void mma_stage_kc(double (&acc)[FA][FB][2], const double* __restrict__ smA,
                                             const double* __restrict__ smB, const double* __restrict__ wk,
                                             int wrow, int wcol, int g, int c) {
  const int swz = (g & 1) << 2;
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    const int off = (((c + 4 * half) ^ swz) << 1);
    double2 af[FA], bf[FB];
#pragma unroll
    for (int a = 0; a < FA; ++a) af[a] = *reinterpret_cast<const double2*>(smA + (wrow + 8 * a + g) * BK + off);
#pragma unroll
    for (int b = 0; b < FB; ++b) bf[b] = *reinterpret_cast<const double2*>(smB + (wcol + 8 * b + g) * BK + off);
    if (SCALE) {
      const double2 w = *reinterpret_cast<const double2*>(wk + ((c + 4 * half) << 1));
#pragma unroll
      for (int b = 0; b < FB; ++b) { bf[b].x *= w.x; bf[b].y *= w.y; }
    }
#pragma unroll
    for (int a = 0; a < FA; ++a)
#pragma unroll
      for (int b = 0; b < FB; ++b) dmma884(acc[a][b][0], acc[a][b][1], af[a].x, bf[b].x);
#pragma unroll
    for (int a = 0; a < FA; ++a)
#pragma unroll
      for (int b = 0; b < FB; ++b) dmma884(acc[a][b][0], acc[a][b][1], af[a].y, bf[b].y);
  }
}

// B N-contiguous ([16][BN]).  n-tile (2t + p) of the warp holds columns wcol + 16 t + 2 n' + p (n' = B lane g),
// so that a lane's accumulators acc[a][2t+p][e] sit on columns wcol + 16 t + 4 c + 2 e + p.
template <int FA, int FB, int BN>
__device__ __forceinline__ void mma_stage_nc(double (&acc)[FA][FB][2], const double* __restrict__ smA,
                                             const double* __restrict__ smB, int wrow, int wcol, int g, int c) {
  static_assert(FB % 2 == 0, "FB must be even for the N-contiguous B path");
  const int swz = (g & 1) << 2;
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    const int off = (((c + 4 * half) ^ swz) << 1);
    double2 af[FA];
#pragma unroll
    for (int a = 0; a < FA; ++a) af[a] = *reinterpret_cast<const double2*>(smA + (wrow + 8 * a + g) * BK + off);
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int k = 2 * c + 8 * half + e;
      double2 bf[FB / 2];
#pragma unroll
      for (int t = 0; t < FB / 2; ++t) {
        const int ch = (wcol >> 1) + g + 8 * t;
        bf[t] = *reinterpret_cast<const double2*>(smB + k * BN + ((ch ^ (c << 1)) << 1));
      }
#pragma unroll
      for (int a = 0; a < FA; ++a)
#pragma unroll
        for (int t = 0; t < FB / 2; ++t) {
          const double av = e ? af[a].y : af[a].x;
          dmma884(acc[a][2 * t][0], acc[a][2 * t][1], av, bf[t].x);
          dmma884(acc[a][2 * t + 1][0], acc[a][2 * t + 1][1], av, bf[t].y);
        }
    }
  }
}

}  // namespace rt
