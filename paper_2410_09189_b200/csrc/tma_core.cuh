// tma_core.cuh -- TMA + mbarrier producer/consumer machinery for the FP64 DMMA kernels (sm_100a).
//
// One producer thread issues cp.async.bulk.tensor (SASS UTMALDG) loads of hardware-swizzled (SWIZZLE_128B) tiles
// into a ring of shared-memory stages and arms a "full" mbarrier with the byte count; 8 consumer warps wait on it,
// run LDS.128 + DMMA.8x8x4 only, and release the stage through an "empty" mbarrier (one arrival per warp).  No
// CTA-wide barrier and no address arithmetic sits on the MMA warps (the first ncu capture showed 1.4 bookkeeping
// instructions per DMMA and a per-stage __syncthreads holding the tensor pipe at ~80 %).
//
// Shared tile layouts produced by TMA with CU_TENSOR_MAP_SWIZZLE_128B (16-byte chunk index ^= 128-byte-row index & 7):
//   K-contiguous operand: box {16 doubles (k), 128 rows}  -> [128][16] doubles, chunk ch of row r at ch ^ (r & 7)
//   N-contiguous operand: 8 boxes {16 doubles (n), 16 k-rows}, box bx covers columns 16 bx .. 16 bx + 15
//                         -> [8][16][16] doubles, chunk ch of k-row k at ch ^ (k & 7)
// Conflict-free 128-bit fragment reads need the two rows a quarter-warp touches to differ in bit 2 of (r & 7), so
// MMA row g of an 8-row block reads shared row perm(g) = (g >> 1) | ((g & 1) << 2); the epilogues undo the permutation.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "dmma_core.cuh"

namespace rt {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
// Waits for the phase with the given parity (single-thread callers: the TMA producer).  A pipeline bug would otherwise hang the GPU until the driver's
// watchdog fires, so after ~10 s of polling the kernel traps (the launch then fails loudly with a CUDA error).
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  if (mbar_try_wait(bar, parity)) return;
  const long long t0 = clock64();
  while (!mbar_try_wait(bar, parity)) {
    if (clock64() - t0 > 20000000000LL) __trap();
  }
}
// The same for a whole (converged) consumer warp in front of warp-level MMAs: every lane polls, and the vote makes the
// exit from the polling loop warp-uniform (the compiler emits no reconvergence point between the loop and the stage's
// mma.sync, which must be executed by the whole warp together).
__device__ __forceinline__ void mbar_wait_warp(uint32_t bar, uint32_t parity) {
  if (__all_sync(0xffffffffu, mbar_try_wait(bar, parity))) return;
  const long long t0 = clock64();
  while (!__all_sync(0xffffffffu, mbar_try_wait(bar, parity))) {
    if (clock64() - t0 > 20000000000LL) __trap();
  }
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// 2-D tiled TMA load: coordinates (c0 = inner/contiguous element index, c1 = row index)
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
// The same with an L2 eviction-priority hint (createpolicy): evict_last for the operand the launch keeps resident in L2,
// evict_first for data that streams through once.
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void tma_load_2d_hint(void* dst, const CUtensorMap* map, int c0, int c1, uint32_t bar,
                                                 uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3}], [%4], %5;"
      ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(bar), "l"(policy) : "memory");
}
__device__ __forceinline__ void tma_load_3d_hint(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar,
                                                 uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4}], [%5], %6;"
      ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(policy) : "memory");
}
// 1-D bulk copy (bytes multiple of 16, both addresses 16-byte aligned)
__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}
// barrier among the consumer warps only (named barrier 1)
__device__ __forceinline__ void consumer_sync(int nthreads) {
  asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}

// Consumer side of the ring: hand a stage back to the producer.  The fence is what makes this safe.  ptxas schedules the
// arrive BEFORE the last DMMAs of the stage (SASS: SYNCS.ARRIVE followed by 24 DMMA.8x8x4), and the scoreboard wait for the
// last fragment loads sits at their first use -- after the arrive.  The LDS of those fragments can therefore still be in
// flight when the eighth arrival lets the producer's next TMA overwrite the slot, and they then return the NEW tile:
// rows 48-63 of a warp tile (the last A fragments) built from the wrong grid points, once every few thousand stages when
// the producer is already waiting for the slot.  __threadfence_block (MEMBAR.CTA) completes every earlier load of the
// lane; __syncwarp extends that to the warp; then one lane arrives.  Latent since round 1; it surfaced in round 2 when
// producer pacing (and, in the N x N GEMM, a faster epilogue) changed who waits for whom.
__device__ __forceinline__ void release_stage(uint32_t empty_bar, int lane) {
  __threadfence_block();
  __syncwarp();
  if (lane == 0) mbar_arrive(empty_bar);
}

__device__ __forceinline__ int perm8(int g) { return (g >> 1) | ((g & 1) << 2); }

// ---- one pipeline stage of MMAs on TMA-swizzled tiles ---------------------------------------------------
// A, B K-contiguous ([128][16], 128B swizzle).  pg = perm8(lane >> 2), c = lane & 3.
// NA0 / NA1: number of row blocks (from the top of the warp tile) computed for the column blocks b < FB/2 / b >= FB/2.
// On a diagonal CTA tile of a symmetric product the 8 x 8 blocks strictly below the diagonal are never read; a
// PREDICATED-off DMMA still costs its statically scheduled issue slot (measured: no gain), so the skipped blocks are
// removed at compile time and the kernel branches between a few instantiations.
template <int FA, int FB, bool SCALE, int NA0 = FA, int NA1 = FA>
__device__ __forceinline__ void mma_stage_kc_tma(double (&acc)[FA][FB][2], const double* __restrict__ smA,
                                                 const double* __restrict__ smB, const double* __restrict__ wk,
                                                 int wrow, int wcol, int pg, int c) {
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    const int off = pg * BK + (((c + 4 * half) ^ pg) << 1);
    constexpr int NAM = NA0 > NA1 ? NA0 : NA1;
    double2 af[FA], bf[FB];
#pragma unroll
    for (int a = 0; a < NAM; ++a) af[a] = *reinterpret_cast<const double2*>(smA + (wrow + 8 * a) * BK + off);
#pragma unroll
    for (int b = 0; b < FB; ++b) bf[b] = *reinterpret_cast<const double2*>(smB + (wcol + 8 * b) * BK + off);
    if (SCALE) {
      const double2 w = *reinterpret_cast<const double2*>(wk + ((c + 4 * half) << 1));
#pragma unroll
      for (int b = 0; b < FB; ++b) { bf[b].x *= w.x; bf[b].y *= w.y; }
    }
#pragma unroll
    for (int a = 0; a < FA; ++a)
#pragma unroll
      for (int b = 0; b < FB; ++b)
        if (a < (b < FB / 2 ? NA0 : NA1)) dmma884(acc[a][b][0], acc[a][b][1], af[a].x, bf[b].x);
#pragma unroll
    for (int a = 0; a < FA; ++a)
#pragma unroll
      for (int b = 0; b < FB; ++b)
        if (a < (b < FB / 2 ? NA0 : NA1)) dmma884(acc[a][b][0], acc[a][b][1], af[a].y, bf[b].y);
  }
}

// A K-contiguous, B N-contiguous in 8 boxes of [16 k][16 n].  Lane g = lane >> 2 reads chunk g of box
// (wcol/16 + t) at k-row k: columns 16 t + 2 g + {0,1} -> n-tiles 2t, 2t+1 (same interleave as dmma_core.cuh).
// NA: number of row blocks (from the top of the warp tile) that are computed.  On the diagonal block of the upper-
// triangular fold the A fragments of the lower row blocks are all zeros (compile-time removal: see above).
template <int FA, int FB, int NA = FA>
__device__ __forceinline__ void mma_stage_nc_tma(double (&acc)[FA][FB][2], const double* __restrict__ smA,
                                                 const double* __restrict__ smB, int wrow, int wcol, int g, int pg,
                                                 int c) {
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    const int off = pg * BK + (((c + 4 * half) ^ pg) << 1);
    double2 af[FA];
#pragma unroll
    for (int a = 0; a < NA; ++a) af[a] = *reinterpret_cast<const double2*>(smA + (wrow + 8 * a) * BK + off);
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int k = 2 * c + 8 * half + e;
      double2 bf[FB / 2];
#pragma unroll
      for (int t = 0; t < FB / 2; ++t)
        bf[t] = *reinterpret_cast<const double2*>(smB + ((wcol >> 4) + t) * 256 + k * BK + ((g ^ (k & 7)) << 1));
#pragma unroll
      for (int a = 0; a < NA; ++a)
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
