// gemm_tma.cu -- TMA-fed, warp-specialised versions of the three FP64 DMMA stages (the default path on sm_100a;
// gemm_kernels.cu keeps the cp.async versions for shapes TMA cannot describe: odd Ng or unaligned Phi).
//
//   a1 project_tma_kernel : dH_ij = sum_r phi_i(r) dV(r) phi_j(r)   (Table 1 "Hupdate" L543; Alg. 1 line 25)
//   a5 density_tma_kernel : rho(r) = sum_j phi_j(r) (Pfold Phi)_j(r) ("Rho" L544; Eq. 27), persistent CTAs
//   a3/a4 gemm_abt_tma    : D = a0 A0 B0^T + a1 A1 B1^T              ("ELDYN" L546)
//
// CTA = 8 consumer warps (2 x 4, warp tile 64 x 32 = 8 x 4 DMMA.8x8x4 tiles) + 1 producer warp (one elected lane
// issues TMA).  6-stage ring, 32 KB per stage (A 128x16 + B 128x16 doubles), full/empty mbarriers.
#include "rt_internal.h"
#include "tma_core.cuh"

namespace rt {

namespace {

constexpr int FA = 8, FB = 4, WM = 2, WN = 4;
constexpr int NCONS = WM * WN;                 // consumer warps
constexpr int NTHREADS = 32 * (NCONS + 4);     // + one producer warpgroup (only its first lane works)
// setmaxnreg budget: the CTA is launched with 384 x 168 = 64512 registers; 256*232 + 128*40 = 64512 exactly
constexpr int REGS_CONSUMER = 232, REGS_PRODUCER = 40;
constexpr int ST = 6;                          // pipeline stages
constexpr int TILE_D = TILE * BK;              // doubles in one 128 x 16 operand tile (16 KB)
constexpr int STAGE_D = 2 * TILE_D;            // A + B
constexpr uint32_t TILE_BYTES = TILE_D * 8;

struct alignas(8) Bars { unsigned long long full[ST]; unsigned long long empty[ST]; };

// dynamic shared layout: [ST][A|B] (1024-aligned) | weights [ST][16] | barriers | reduce scratch
constexpr size_t SMEM_TILES = (size_t)ST * STAGE_D * 8;
constexpr size_t SMEM_W = (size_t)ST * BK * 8;
constexpr size_t SMEM_RED = (size_t)WM * TILE * 8;
constexpr size_t SMEM_TOTAL = 1024 + SMEM_TILES + SMEM_W + sizeof(Bars) + SMEM_RED;

// 1024-byte alignment of the tile ring (128B-swizzle atom).  The offset is added to the __shared__ array itself so the
// compiler keeps the shared address space (fragment reads must be LDS.128, not generic LD).
__device__ __forceinline__ double* align1024(uint8_t* p) {
  const uint32_t a = smem_u32(p);
  return reinterpret_cast<double*>(p + ((1024u - (a & 1023u)) & 1023u));
}

__device__ __forceinline__ void regs_consumer() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS_CONSUMER)); }
__device__ __forceinline__ void regs_producer() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS_PRODUCER)); }

__device__ __forceinline__ void init_bars(Bars* bars) {
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < ST; ++s) {
      mbar_init(smem_u32(&bars->full[s]), 1);
      mbar_init(smem_u32(&bars->empty[s]), NCONS);
    }
    fence_barrier_init();
  }
  __syncthreads();
}

}  // namespace

// ======================================================================================================
// a1 projection
// ======================================================================================================
// Persistent: CTA c works through the items c, c + G, c + 2G, ... of the class-ordered (split, tile) list, so the G CTAs
// that run together are always G consecutive items -- the same split of neighbouring tiles of one 2-D block, which share
// Phi row panels.  That sharing only turns into L2 hits while the CTAs stay close together along k: all of them read the
// same k-range of ~2 sqrt(G) row panels, 1 KB per panel and grid point, so a spread of a few thousand grid points
// already overflows the L2.  A plain grid (one CTA per item, round 2 first capture) drifted apart over the 37 ms a CTA
// lives at N = 13,000: 38 % L2 hits, 6.2 TB of DRAM reads per launch against 0.12 TB of Phi.  PACING keeps them together:
// every PACE_CK stages the producer thread counts itself in at a checkpoint counter and does not run ahead of the
// checkpoint PACE_W before until all G CTAs have reached it.  Only TMA issue is throttled, never the slowest CTA, and a
// CTA whose peers are not there (tail of the launch, or SMs shared with another stream) gives up after two timeouts.
constexpr int PACE_CK = 32;
constexpr long long PACE_TIMEOUT_CLK = 100000;      // ~50 us

__global__ void __launch_bounds__(NTHREADS, 1)
project_tma_kernel(const __grid_constant__ CUtensorMap tmPhi, const double* __restrict__ w,
                   const int2* __restrict__ tiles, double* __restrict__ W, const ProjectPlan pl, int nitems,
                   int* __restrict__ pace_cnt, int pace_n, int pace_w) {
  extern __shared__ uint8_t smem_raw[];
  double* tilesm = align1024(smem_raw);
  double* wsm = tilesm + (size_t)ST * STAGE_D;
  Bars* bars = reinterpret_cast<Bars*>(wsm + ST * BK);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  init_bars(bars);

  const int N = pl.N, ldn = pl.ldn;
  const int G = gridDim.x;

  if (warp >= NCONS) {
    // ===== producer: runs ahead across items =====
    regs_producer();
    if (warp == NCONS && lane == 0) {
      tma_prefetch_desc(&tmPhi);
      long long it = 0;
      int misses = pace_cnt ? 0 : 2;
      for (int item = blockIdx.x; item < nitems; item += G) {
        const ProjBlock pb = project_decode(item, pl);
        const int2 tt = tiles[pb.t];
        const int i0 = tt.x * TILE, j0 = tt.y * TILE;
        const int nk = (int)((pb.kend - pb.kbeg + BK - 1) / BK);
        for (int kt = 0; kt < nk; ++kt, ++it) {
          if (misses < 2 && (it % PACE_CK) == 0) {
            const long long q = it / PACE_CK;
            if (q >= pace_n) { misses = 2; }                 // past the counters (never with the host's bound): run free
            else atomicAdd(pace_cnt + q, 1);
            if (misses < 2 && q >= pace_w) {
              const volatile int* prev = pace_cnt + (q - pace_w);
              if (*prev < G) {
                const long long t0 = clock64();
                while (*prev < G) {
                  if (clock64() - t0 > PACE_TIMEOUT_CLK) { ++misses; break; }
                }
              }
            }
          }
          const int slot = (int)(it % ST);
          if (it >= ST) mbar_wait(smem_u32(&bars->empty[slot]), (uint32_t)((it / ST) - 1) & 1);
          const uint32_t full = smem_u32(&bars->full[slot]);
          mbar_expect_tx(full, 2 * TILE_BYTES + BK * 8);
          const long long k0 = pb.kbeg + (long long)kt * BK;
          double* sA = tilesm + (size_t)slot * STAGE_D;
          tma_load_2d(sA, &tmPhi, (int)k0, i0, full);
          tma_load_2d(sA + TILE_D, &tmPhi, (int)k0, j0, full);
          bulk_load_1d(wsm + slot * BK, w + k0, BK * 8, full);     // w is padded to a multiple of 16 doubles
        }
      }
    }
    return;
  }

  // ===== consumers =====
  regs_consumer();
  const int g = lane >> 2, c = lane & 3, pg = perm8(g);
  long long it = 0;
  for (int item = blockIdx.x; item < nitems; item += G) {
    const ProjBlock pb = project_decode(item, pl);
    const int2 tt = tiles[pb.t];
    const int i0 = tt.x * TILE, j0 = tt.y * TILE;
    const int nk = (int)((pb.kend - pb.kbeg + BK - 1) / BK);
    // Diagonal tile of the symmetric output: only 8 x 8 blocks on or above the diagonal are needed (project_reduce reads
    // j >= i), 136 of the CTA's 256.  The warp roles (wm, wn) are permuted so that every scheduler partition
    // (warp % 4) gets 32-36 of them instead of 10-58: {(0,2),(1,0)}, {(0,3),(1,1)}, {(0,1),(1,2)}, {(0,0),(1,3)}.
    const bool diag = i0 == j0;
    double* Ws = W + (long long)pb.s * N * ldn;
    if (!diag && N - j0 <= 96) {
      // Ragged last tile column with at most 96 valid columns (N = 2400: 96): the 8 warps cover 128 x 96 as 2 x 4 warp
      // tiles of 64 x 24 instead of leaving the warps of the last 32 columns multiplying padding.
      constexpr int FB3 = 3;
      const int wrow3 = (warp / WN) * (8 * FA), wcol3 = (warp % WN) * (8 * FB3);
      double acc3[FA][FB3][2];
#pragma unroll
      for (int a = 0; a < FA; ++a)
#pragma unroll
        for (int b = 0; b < FB3; ++b) acc3[a][b][0] = acc3[a][b][1] = 0.0;
      for (int kt = 0; kt < nk; ++kt, ++it) {
        const int slot = (int)(it % ST);
        mbar_wait_warp(smem_u32(&bars->full[slot]), (uint32_t)(it / ST) & 1);
        const double* sA = tilesm + (size_t)slot * STAGE_D;
        mma_stage_kc_tma<FA, FB3, true>(acc3, sA, sA + TILE_D, wsm + slot * BK, wrow3, wcol3, pg, c);
        release_stage(smem_u32(&bars->empty[slot]), lane);
      }
#pragma unroll
      for (int a = 0; a < FA; ++a) {
        const int row = i0 + wrow3 + 8 * a + pg;
        if (row < N) {
#pragma unroll
          for (int b = 0; b < FB3; ++b) {
            const int col = j0 + wcol3 + 8 * b + c;
            if (col < N) Ws[(long long)row * ldn + col] = acc3[a][b][0];
            if (col + 4 < N) Ws[(long long)row * ldn + col + 4] = acc3[a][b][1];
          }
        }
      }
      continue;
    }
    const int role = diag ? ((warp < 4) ? ((0x0132 >> (4 * warp)) & 15) : warp) : warp;
    const int wrow = (role / WN) * (8 * FA), wcol = (role % WN) * (8 * FB);
    // blocks on or above the diagonal, as row counts for the two column halves of the warp tile (rounded up to a
    // rectangle): (0,0), (1,2): rows < 2 | 4 ; (0,1), (1,3): rows < 6 | 8 ; (0,2), (0,3): all ; (1,0), (1,1): none
    const int dlt = (wcol - wrow) / 8;
    double acc[FA][FB][2];
#pragma unroll
    for (int a = 0; a < FA; ++a)
#pragma unroll
      for (int b = 0; b < FB; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

    if (!diag) {
      for (int kt = 0; kt < nk; ++kt, ++it) {
        const int slot = (int)(it % ST);
        mbar_wait_warp(smem_u32(&bars->full[slot]), (uint32_t)(it / ST) & 1);
        const double* sA = tilesm + (size_t)slot * STAGE_D;
        mma_stage_kc_tma<FA, FB, true>(acc, sA, sA + TILE_D, wsm + slot * BK, wrow, wcol, pg, c);
        release_stage(smem_u32(&bars->empty[slot]), lane);
      }
    } else {
      const bool live = i0 + wrow < N && j0 + wcol < N;
      for (int kt = 0; kt < nk; ++kt, ++it) {
        const int slot = (int)(it % ST);
        mbar_wait_warp(smem_u32(&bars->full[slot]), (uint32_t)(it / ST) & 1);
        const double* sA = tilesm + (size_t)slot * STAGE_D;
        if (!live) {}                             // the whole warp tile is padding (N < 128: tiny systems)
        else if (dlt >= 8) mma_stage_kc_tma<FA, FB, true>(acc, sA, sA + TILE_D, wsm + slot * BK, wrow, wcol, pg, c);
        else if (dlt == 4) mma_stage_kc_tma<FA, FB, true, 6, 8>(acc, sA, sA + TILE_D, wsm + slot * BK, wrow, wcol, pg, c);
        else if (dlt == 0) mma_stage_kc_tma<FA, FB, true, 2, 4>(acc, sA, sA + TILE_D, wsm + slot * BK, wrow, wcol, pg, c);
        release_stage(smem_u32(&bars->empty[slot]), lane);
      }
    }

    // epilogue: raw partial sums into slab s.  MMA row g <-> tile row perm8(g); tile col n' <-> perm8(n')
#pragma unroll
    for (int a = 0; a < FA; ++a) {
      const int row = i0 + wrow + 8 * a + pg;
      if (row < N) {
#pragma unroll
        for (int b = 0; b < FB; ++b) {
          const int col = j0 + wcol + 8 * b + c;        // perm8(2c) = c, perm8(2c+1) = c + 4
          if (col < N) Ws[(long long)row * ldn + col] = acc[a][b][0];
          if (col + 4 < N) Ws[(long long)row * ldn + col + 4] = acc[a][b][1];
        }
      }
    }
  }
}

size_t tma_smem_bytes() { return SMEM_TOTAL; }

// Pacing pays where the 2-D blocking of the tile list does (ntile well above the 12 x 12 block: at N = 2,400 every wave
// touches all 19 row panels anyway and pacing only cost 2 % of the kernel time) and on launches long enough to drift
// (per-CTA stage count >= PACE_MIN_STAGES, ~35 ms).  Unpaced launches keep one CTA per item: the hardware then hands out
// items as SMs free up, which measured less DRAM traffic than the static round-robin of persistent CTAs.
constexpr long long PACE_MIN_STAGES = 16384;
constexpr int PACE_MIN_NTILE = 32;
size_t project_tma_pace_ints(const ProjectPlan& p, int sms) {
  const long long nitems = p.grid();
  const long long G = nitems < sms ? nitems : sms;
  long long kc = p.kchunk;                                           // the class with the longest items
  if (p.Tn > 0 && p.kchunk_n > kc) kc = p.kchunk_n;
  if (p.kchunk_d > kc) kc = p.kchunk_d;
  const long long per_item = (kc + BK - 1) / BK;
  const long long stages = ((nitems + G - 1) / G) * per_item;
  if (G < 2 || p.ntile < PACE_MIN_NTILE || stages < PACE_MIN_STAGES) return 0;
  return (size_t)(stages / PACE_CK + 2);
}

void launch_project_tma(const ProjectPlan& p, const CUtensorMap& tmPhi, const double* w, const int2* tiles, double* W,
                        int sms, int* pace_cnt, int pace_w, cudaStream_t st) {
  const int nitems = p.grid();
  const size_t npace = pace_cnt ? project_tma_pace_ints(p, sms) : 0;
  const int G = npace ? (nitems < sms ? nitems : sms) : nitems;
  if (npace) cudaMemsetAsync(pace_cnt, 0, npace * sizeof(int), st);
  project_tma_kernel<<<G, NTHREADS, SMEM_TOTAL, st>>>(tmPhi, w, tiles, W, p, nitems, npace ? pace_cnt : nullptr, (int)npace,
                                                      pace_w);
}

// ======================================================================================================
// a5 density (persistent)
// ======================================================================================================
// Work item = (type, r-tile).  A type is one or two k-segments of one j-tile each (table built on the host,
// rt_api.cu build_density_types): all types cost about the same number of stages, every type owns one row of the
// partial-sum array.  Items are rastered in groups of group_r r-tiles x all types, r-tile fastest.
struct DensWork { int type; long long rt; bool valid; };

// 2-D supertiles: group_t types x group_r r-tiles run together (~ one item per SM).  The CTAs of a supertile walk the
// contraction index in step, so a P-fold row panel is fetched from DRAM once and hit in L2 by the group_r CTAs that share
// its type, and a Phi panel once for the group_t CTAs that share its r-tile.  Round 1 ran ALL types of 3 r-tiles
// together: at N = 13,000 that is 51 different 27 MB row panels of the 1.35 GB fold in flight with 3-fold reuse, and ncu
// measured 6.5 TB of DRAM reads per launch against 0.12 TB of operands (L2 hit rate 37 %).
__device__ __forceinline__ DensWork dens_decode(long long L, int ntypes, long long nrt, int group_r, int group_t) {
  const long long per_rg = (long long)group_r * ntypes;          // items of one full r-group
  const long long rg = L / per_rg;
  const long long in = L - rg * per_rg;
  const long long r_first = rg * group_r;
  const long long gr_here = (nrt - r_first < group_r) ? (nrt - r_first) : group_r;
  DensWork d;
  d.valid = r_first < nrt && in < gr_here * ntypes;
  const long long per_tg = (long long)group_t * gr_here;          // items of one full type-group inside this r-group
  const long long tg = gr_here > 0 ? in / per_tg : 0;
  const long long in2 = in - tg * per_tg;
  d.type = (int)(tg * group_t + (gr_here > 0 ? in2 / gr_here : 0));
  d.rt = r_first + (gr_here > 0 ? in2 % gr_here : 0);
  d.valid = d.valid && d.type < ntypes && d.rt < nrt;
  return d;
}

__global__ void __launch_bounds__(NTHREADS, 1)
density_tma_kernel(const __grid_constant__ CUtensorMap tmP, const __grid_constant__ CUtensorMap tmPhiN,
                   const double* __restrict__ phi, const DensSeg* __restrict__ segs, double* __restrict__ rho_part,
                   int N, long long Ng, int ntypes, long long nrt, int group_r, int group_t, long long nwork,
                   int b3d, int* __restrict__ pace_cnt, int pace_n, int pace_w, int hint) {
  extern __shared__ uint8_t smem_raw[];
  double* tilesm = align1024(smem_raw);
  double* wsm = tilesm + (size_t)ST * STAGE_D;
  Bars* bars = reinterpret_cast<Bars*>(wsm + ST * BK);
  double* colred = reinterpret_cast<double*>(bars + 1);       // [WM][TILE]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  init_bars(bars);

  if (warp >= NCONS) {
    // ===== producer: runs ahead across segments and work items =====
    regs_producer();
    if (warp == NCONS && lane == 0) {
      tma_prefetch_desc(&tmP);
      tma_prefetch_desc(&tmPhiN);
      // the Phi panels of the r-tiles in flight are what the launch keeps in L2 (every type re-reads them); the fold
      // streams through (shared only by the group_r CTAs of the same type, which walk it together)
      const uint64_t pol_phi = l2_policy_evict_last();
      long long it = 0;
      int misses = pace_cnt ? 0 : 2;
      const int G = gridDim.x;
      for (long long L = blockIdx.x; L < nwork; L += gridDim.x) {
        const DensWork wk = dens_decode(L, ntypes, nrt, group_r, group_t);
        if (!wk.valid) continue;
        const long long r0 = wk.rt * TILE;
        for (int which = 0; which < 2; ++which) {
          const DensSeg sg = segs[2 * wk.type + which];
          const int j0 = sg.jt * TILE;
          for (int i = 0; i < sg.ns; ++i, ++it) {
            if (misses < 2 && (it % PACE_CK) == 0) {                          // pacing: see project_tma_kernel
              const long long q = it / PACE_CK;
              if (q >= pace_n) { misses = 2; }
              else atomicAdd(pace_cnt + q, 1);
              if (misses < 2 && q >= pace_w) {
                const volatile int* prev = pace_cnt + (q - pace_w);
                if (*prev < G) {
                  const long long t0 = clock64();
                  while (*prev < G) {
                    if (clock64() - t0 > PACE_TIMEOUT_CLK) { ++misses; break; }
                  }
                }
              }
            }
            const int slot = (int)(it % ST);
            if (it >= ST) mbar_wait(smem_u32(&bars->empty[slot]), (uint32_t)((it / ST) - 1) & 1);
            const uint32_t full = smem_u32(&bars->full[slot]);
            mbar_expect_tx(full, 2 * TILE_BYTES);
            const int k0 = j0 + (sg.s0 + sg.dir * i) * BK;
            double* sA = tilesm + (size_t)slot * STAGE_D;
            tma_load_2d(sA, &tmP, k0, j0, full);                              // Pfold[j0.., k0..]
            if (b3d) {                                                        // Phi[k0.., r0 .. r0+127] in one op
              if (hint) tma_load_3d_hint(sA + TILE_D, &tmPhiN, 0, k0, (int)(r0 >> 4), full, pol_phi);
              else tma_load_3d(sA + TILE_D, &tmPhiN, 0, k0, (int)(r0 >> 4), full);
            } else {
#pragma unroll
              for (int bx = 0; bx < 8; ++bx)                                  // Phi[k0.., r0 + 16 bx ..]
                tma_load_2d(sA + TILE_D + bx * 256, &tmPhiN, (int)(r0 + 16 * bx), k0, full);
            }
          }
        }
      }
    }
    return;
  }

  // ===== consumers =====
  regs_consumer();
  const int g = lane >> 2, c = lane & 3, pg = perm8(g);
  const int wm = warp / WN, wn = warp % WN;
  const int wrow = wm * (8 * FA), wcol = wn * (8 * FB);
  const int ctid = threadIdx.x;                                 // 0..255
  const bool vecF = ((Ng & 1) == 0) && ((reinterpret_cast<uintptr_t>(phi) & 15) == 0);
  long long it = 0;
  for (long long L = blockIdx.x; L < nwork; L += gridDim.x) {
    const DensWork wk = dens_decode(L, ntypes, nrt, group_r, group_t);
    if (!wk.valid) continue;
    const long long r0 = wk.rt * TILE;
    double colsum[FB / 2][4];
#pragma unroll
    for (int t = 0; t < FB / 2; ++t)
#pragma unroll
      for (int q = 0; q < 4; ++q) colsum[t][q] = 0.0;

    for (int which = 0; which < 2; ++which) {               // same segment order as the producer
      const DensSeg sg = segs[2 * wk.type + which];
      if (sg.ns == 0) continue;
      const int j0 = sg.jt * TILE;
      double acc[FA][FB][2];
#pragma unroll
      for (int a = 0; a < FA; ++a)
#pragma unroll
        for (int b = 0; b < FB; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

      for (int i = 0; i < sg.ns; ++i, ++it) {
        const int slot = (int)(it % ST);
        mbar_wait_warp(smem_u32(&bars->full[slot]), (uint32_t)(it / ST) & 1);
        const double* sA = tilesm + (size_t)slot * STAGE_D;
        // stage sidx holds the contraction rows k = j0 + 16 sidx ...: inside the diagonal block (sidx < 8) the fold is
        // upper triangular, Pfold[j][k] = 0 for k < j, so row block a of this warp is all zeros in half `half` of the
        // stage unless 8 (wrow/8 + a) <= 16 sidx + 8 half + 7
        // (both halves of a stage then need the same even number of row blocks: na = 2 sidx + 2 - wrow/8)
        const int na = 2 * (sg.s0 + sg.dir * i) + 2 - wrow / 8;
        if (na >= 8) mma_stage_nc_tma<FA, FB>(acc, sA, sA + TILE_D, wrow, wcol, g, pg, c);
        else if (na == 6) mma_stage_nc_tma<FA, FB, 6>(acc, sA, sA + TILE_D, wrow, wcol, g, pg, c);
        else if (na == 4) mma_stage_nc_tma<FA, FB, 4>(acc, sA, sA + TILE_D, wrow, wcol, g, pg, c);
        else if (na == 2) mma_stage_nc_tma<FA, FB, 2>(acc, sA, sA + TILE_D, wrow, wcol, g, pg, c);
        release_stage(smem_u32(&bars->empty[slot]), lane);
      }

      // fused row-dot: colsum(r) += sum_j phi_j(r) T_j(r); lane owns columns wcol + 16 t + 4 c + {0..3}
#pragma unroll
      for (int a = 0; a < FA; ++a) {
        const int j = j0 + wrow + 8 * a + pg;
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
            colsum[t][0] += f[0] * acc[a][2 * t][0];
            colsum[t][1] += f[1] * acc[a][2 * t + 1][0];
            colsum[t][2] += f[2] * acc[a][2 * t][1];
            colsum[t][3] += f[3] * acc[a][2 * t + 1][1];
          }
        }
      }
    }

    // reduce over the 8 row groups of the warp, then over the WM warps sharing columns
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
        for (int q = 0; q < 4; ++q) colred[wm * TILE + wcol + 16 * t + 4 * c + q] = colsum[t][q];
    }
    consumer_sync(32 * NCONS);
    if (ctid < TILE) {
      const long long r = r0 + ctid;
      if (r < Ng) {
        double v = 0.0;
#pragma unroll
        for (int m = 0; m < WM; ++m) v += colred[m * TILE + ctid];
        rho_part[(long long)wk.type * Ng + r] = v;
      }
    }
    consumer_sync(32 * NCONS);
  }
}

size_t density_tma_pace_ints(const DensityPlan& p, int sms) {
  const long long ngroups = (p.nrt + p.group_r - 1) / p.group_r;
  const long long nwork = ngroups * p.group_r * p.ntypes;
  const long long G = nwork < sms ? nwork : sms;
  const long long per_item = (long long)(p.ntile + 1) * (TILE / BK) + 2;
  const long long stages = ((nwork + G - 1) / G) * per_item;
  if (G < 2 || stages < PACE_MIN_STAGES) return 0;
  return (size_t)(stages / PACE_CK + 2);
}

void launch_density_tma(const DensityPlan& p, const CUtensorMap& tmP, const CUtensorMap& tmPhiN, int b3d,
                        const double* phi, const DensSeg* segs, double* rho_part, int sms, int* pace_cnt, int pace_w,
                        int hint, cudaStream_t st) {
  const long long ngroups = (p.nrt + p.group_r - 1) / p.group_r;
  const long long nwork = ngroups * p.group_r * p.ntypes;
  const long long grid = nwork < sms ? nwork : sms;
  const size_t npace = pace_cnt ? density_tma_pace_ints(p, sms) : 0;
  if (npace) cudaMemsetAsync(pace_cnt, 0, npace * sizeof(int), st);
  density_tma_kernel<<<(unsigned)grid, NTHREADS, SMEM_TOTAL, st>>>(tmP, tmPhiN, phi, segs, rho_part, p.N, p.Ng,
                                                                   p.ntypes, p.nrt, p.group_r, p.group_t, nwork, b3d,
                                                                   npace ? pace_cnt : nullptr, (int)npace, pace_w, hint);
}

// ======================================================================================================
// a3/a4 N x N GEMM (stream-K)
// ======================================================================================================
// The work of one launch is the list of (tile, pipeline stage) units, ntiles x nk of them, in tile-list order.  It is cut
// into G = min(#SMs, ...) contiguous RANGES of (almost) equal length and every CTA processes one range, so all SMs
// finish together whatever ntiles is (round 1: one CTA per 128 x 128 tile -- N = 2400 gave 190 upper tiles on 148 SMs,
// two waves at 64 % fill, ELDYN at 0.58 of the DMMA roof).  A tile that straddles ranges is finished by the CTA that
// holds its FIRST stages (the "head", at the end of that CTA's range); the CTAs holding later stages (the "tails", at
// the very start of their ranges) park their partial accumulators in a workspace slot and raise a flag.  The head adds
// the slots in range order, so the summation order -- and therefore every bit of the result -- is fixed by (N, G)
// alone.  Deadlock freedom does not depend on all CTAs being co-resident (three delta-kick handles share the GPU on
// three streams): ranges are handed out through a ticket counter in reverse order, so a head only ever waits for CTAs
// that took their ticket BEFORE it, i.e. that are already running or done.
struct GemmTmaArgs {
  int N, ldn, nterms;
  int sym;                 // +1: D is symmetric, -1: antisymmetric -> the tile list holds ti <= tj only and the mirror
                           //  image is written too; 0: plain tile list
  const int2* tiles;       // tile list (ti, tj)
  int ntiles;
  double alpha0, alpha1;
  double* D; double* Z1; double beta1; double* Z2; double beta2;
  const int* skip;         // non-zero -> no-op (orders past convergence of the commutator series)
  double* ws;              // [G][TILE*TILE] partial accumulators of the tail items, indexed by range
  int* sync;               // [0] = ticket counter, [1] = finished-CTA counter, [2 + p] = flag of range p (0 = empty)
};

__device__ __forceinline__ long long range_begin(long long total, int G, int j) { return total * j / G; }

// Work of CTA `range` of G: the contiguous piece [total * range / G, total * (range + 1) / G) of the (tile, stage) units.
// A CTA therefore walks ~ntiles/G CONSECUTIVE tiles of the (row-major) list, which share their A row panel: it stays in
// L2 for the whole walk.  (Measured at N = 13,000: a variant that ran whole waves data-parallel -- concurrent CTAs on
// consecutive tiles of a 2-D blocked list -- and split only the tail was 2.4 % slower per GEMM, 257.6 vs 251.5 ms for
// the full dual products; nfw below is what is left of it, switched off.)
struct GemmWork { int t, kt0, kt1, tl; bool tail; };
struct GemmIter {
  int G, range, nk, nfw, w, tail0;
  long long total, u, u1;
  __device__ GemmIter(int ntiles, int nk_, int G_, int range_) : G(G_), range(range_), nk(nk_), w(0) {
    nfw = 0;
    tail0 = 0;
    total = (long long)(ntiles - tail0) * nk;
    u = range_begin(total, G, range);
    u1 = range_begin(total, G, range + 1);
  }
  __device__ bool next(GemmWork& it) {
    if (w < nfw) { it.t = w * G + range; it.kt0 = 0; it.kt1 = nk; it.tl = 0; it.tail = false; ++w; return true; }
    if (u >= u1) return false;
    it.tl = (int)(u / nk);
    it.kt0 = (int)(u - (long long)it.tl * nk);
    it.kt1 = (int)((u1 - u < nk - it.kt0) ? (it.kt0 + (u1 - u)) : nk);
    it.t = tail0 + it.tl;
    it.tail = true;
    u += it.kt1 - it.kt0;
    return true;
  }
};

__global__ void __launch_bounds__(NTHREADS, 1)
gemm_abt_tma_kernel(const __grid_constant__ CUtensorMap tmA0, const __grid_constant__ CUtensorMap tmB0,
                    const __grid_constant__ CUtensorMap tmA1, const __grid_constant__ CUtensorMap tmB1,
                    GemmTmaArgs ga) {
  if (ga.skip && *ga.skip) return;
  extern __shared__ uint8_t smem_raw[];
  double* tilesm = align1024(smem_raw);
  double* wsm = tilesm + (size_t)ST * STAGE_D;
  Bars* bars = reinterpret_cast<Bars*>(wsm + ST * BK);
  int* sh_ticket = reinterpret_cast<int*>(bars + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = gridDim.x;
  if (threadIdx.x == 0) *sh_ticket = atomicAdd(&ga.sync[0], 1);
  init_bars(bars);                                  // ends with __syncthreads
  const int range = G - 1 - *sh_ticket;             // later tickets take earlier ranges (see above)
  const int N = ga.N, ldn = ga.ldn;
  const int nk1 = (N + BK - 1) / BK;
  const int nk = ga.nterms * nk1;

  if (warp >= NCONS) {
    regs_producer();
    if (warp == NCONS && lane == 0) {
      tma_prefetch_desc(&tmA0);
      tma_prefetch_desc(&tmB0);
      long long it = 0;
      GemmIter iter(ga.ntiles, nk, G, range);
      GemmWork wk;
      while (iter.next(wk)) {
        const int kt0 = wk.kt0, kt1 = wk.kt1;
        const int2 tt = ga.tiles[wk.t];
        const int i0 = tt.x * TILE, j0 = tt.y * TILE;
        for (int kt = kt0; kt < kt1; ++kt, ++it) {
          const int slot = (int)(it % ST);
          if (it >= ST) mbar_wait(smem_u32(&bars->empty[slot]), (uint32_t)((it / ST) - 1) & 1);
          const uint32_t full = smem_u32(&bars->full[slot]);
          mbar_expect_tx(full, 2 * TILE_BYTES);
          const bool second = kt >= nk1;
          const int k0 = (second ? kt - nk1 : kt) * BK;
          double* sA = tilesm + (size_t)slot * STAGE_D;
          tma_load_2d(sA, second ? &tmA1 : &tmA0, k0, i0, full);
          tma_load_2d(sA + TILE_D, second ? &tmB1 : &tmB0, k0, j0, full);
        }
      }
    }
  } else {
    regs_consumer();
    const int g = lane >> 2, c = lane & 3, pg = perm8(g);
    const int wrow = (warp / WN) * (8 * FA), wcol = (warp % WN) * (8 * FB);
    const int ctid = threadIdx.x;                      // 0 .. 255
    const double ratio = ga.nterms == 2 ? ga.alpha1 / ga.alpha0 : 1.0;
    const double inv = 1.0 / ratio;                     // +-1 in this library: exact
    const double fin = (ga.nterms == 2 && ratio != 1.0) ? ga.alpha0 * ratio : ga.alpha0;
    const double msign = (double)ga.sym;
    long long it = 0;
    GemmIter iter(ga.ntiles, nk, G, range);
    GemmWork wk;
    while (iter.next(wk)) {
      const int kt0 = wk.kt0, kt1 = wk.kt1;
      const int2 tt = ga.tiles[wk.t];
      const int i0 = tt.x * TILE, j0 = tt.y * TILE;
      double acc[FA][FB][2];
#pragma unroll
      for (int a = 0; a < FA; ++a)
#pragma unroll
        for (int b = 0; b < FB; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

      for (int kt = kt0; kt < kt1; ++kt, ++it) {
        const int slot = (int)(it % ST);
        mbar_wait_warp(smem_u32(&bars->full[slot]), (uint32_t)(it / ST) & 1);
        if (kt == nk1 && ratio != 1.0) {            // fold alpha1/alpha0 into the first term's sum
#pragma unroll
          for (int a = 0; a < FA; ++a)
#pragma unroll
            for (int b = 0; b < FB; ++b) { acc[a][b][0] *= inv; acc[a][b][1] *= inv; }
        }
        const double* sA = tilesm + (size_t)slot * STAGE_D;
        mma_stage_kc_tma<FA, FB, false>(acc, sA, sA + TILE_D, nullptr, wrow, wcol, pg, c);
        release_stage(smem_u32(&bars->empty[slot]), lane);
      }
      if (ga.nterms == 2 && ratio != 1.0 && kt1 <= nk1) {      // the item never reached the second term
#pragma unroll
        for (int a = 0; a < FA; ++a)
#pragma unroll
          for (int b = 0; b < FB; ++b) { acc[a][b][0] *= inv; acc[a][b][1] *= inv; }
      }

      if (kt0 > 0) {
        // ---- tail of a tile whose head lives in an earlier range: park the partial sums, raise the flag ----
        double* slotp = ga.ws + (size_t)range * (TILE * TILE);
#pragma unroll
        for (int a = 0; a < FA; ++a)
#pragma unroll
          for (int b = 0; b < FB; ++b)
#pragma unroll
            for (int e = 0; e < 2; ++e) slotp[((a * FB + b) * 2 + e) * (32 * NCONS) + ctid] = acc[a][b][e];
        __threadfence();
        consumer_sync(32 * NCONS);
        if (ctid == 0) {
          __threadfence();
          atomicExch(&ga.sync[2 + range], 1);
        }
        continue;
      }
      if (kt1 < nk) {
        // ---- head of a tile that continues in the following ranges: add their partial sums in range order ----
        const long long tile_end = (long long)(wk.tl + 1) * nk;
        for (int p = range + 1; p < G && range_begin(iter.total, G, p) < tile_end; ++p) {
          if (ctid == 0) {
            const long long t0 = clock64();
            while (atomicAdd(&ga.sync[2 + p], 0) == 0) {
              if (clock64() - t0 > 20000000000LL) __trap();
            }
            __threadfence();
          }
          consumer_sync(32 * NCONS);
          const double* slotp = ga.ws + (size_t)p * (TILE * TILE);
#pragma unroll
          for (int a = 0; a < FA; ++a)
#pragma unroll
            for (int b = 0; b < FB; ++b)
#pragma unroll
              for (int e = 0; e < 2; ++e) acc[a][b][e] += __ldcg(slotp + ((a * FB + b) * 2 + e) * (32 * NCONS) + ctid);
          consumer_sync(32 * NCONS);
          if (ctid == 0) atomicExch(&ga.sync[2 + p], 0);            // self-cleaning: the next launch finds every flag at 0
        }
      }

      // ---- epilogue of a complete tile ----
      // Products without Z1 / Z2 (the whole Taylor path: rt_api.cu enqueue_expm / enqueue_shard_B keep the powers of Y
      // instead of accumulating) store element by element.  Products that accumulate (the commutator series: P1 += dP^(k))
      // read Z1 / Z2 for a batch of 2 x 2 fragments first and store afterwards: D, Z1, Z2 are plain pointers that may
      // alias as far as the compiler knows, so element-wise `Z[o] += ...` statements serialise into one dependent L2 round
      // trip each (ncu, N = 2,400: 70 % of the DMMA pipe against 91 % for the same product without Z).  Every element and
      // every mirror image is touched by exactly one thread, once, so the batching changes no value.  (This version first
      // ran in round 2 BEFORE the stage-release race of tma_core.cuh was understood: it returned the consumers to the
      // main loop early enough to hit that race, was blamed for it and taken out; with release_stage in place it is
      // bit-reproducible -- tests/test_gpu_api_contract.py.)
      const bool diag = ga.sym && i0 == j0;
      const bool hasZ1 = ga.Z1 != nullptr, hasZ2 = ga.Z2 != nullptr;
      if (!hasZ1 && !hasZ2) {
#pragma unroll
        for (int a = 0; a < FA; ++a) {
          const int row = i0 + wrow + 8 * a + pg;
          if (row < N) {
#pragma unroll
            for (int b = 0; b < FB; ++b) {
#pragma unroll
              for (int e = 0; e < 2; ++e) {
                const int col = j0 + wcol + 8 * b + c + 4 * e;
                if (col < N && (!diag || col >= row)) {
                  const long long o = (long long)row * ldn + col;
                  double d = fin * acc[a][b][e];
                  if (ga.sym < 0 && row == col) d = 0.0;
                  if (ga.D) ga.D[o] = d;
                  if (ga.sym && row != col && ga.D) ga.D[(long long)col * ldn + row] = msign * d;   // mirror image
                }
              }
            }
          }
        }
      } else {
#pragma unroll
        for (int a = 0; a < FA; ++a) {
          const int row = i0 + wrow + 8 * a + pg;
          if (row < N) {
#pragma unroll
            for (int bb = 0; bb < FB; bb += 2) {
              double z1[2][2], z2[2][2], z1m[2][2], z2m[2][2];
#pragma unroll
              for (int b = 0; b < 2; ++b)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int col = j0 + wcol + 8 * (bb + b) + c + 4 * e;
                  z1[b][e] = z2[b][e] = z1m[b][e] = z2m[b][e] = 0.0;
                  if (col < N && (!diag || col >= row)) {
                    const long long o = (long long)row * ldn + col;
                    if (hasZ1) z1[b][e] = ga.Z1[o];
                    if (hasZ2) z2[b][e] = ga.Z2[o];
                    if (ga.sym && row != col) {
                      const long long om = (long long)col * ldn + row;
                      if (hasZ1) z1m[b][e] = ga.Z1[om];
                      if (hasZ2) z2m[b][e] = ga.Z2[om];
                    }
                  }
                }
#pragma unroll
              for (int b = 0; b < 2; ++b)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int col = j0 + wcol + 8 * (bb + b) + c + 4 * e;
                  if (col < N && (!diag || col >= row)) {
                    const long long o = (long long)row * ldn + col;
                    double d = fin * acc[a][bb + b][e];
                    if (ga.sym < 0 && row == col) d = 0.0;
                    if (ga.D) ga.D[o] = d;
                    if (hasZ1) ga.Z1[o] = z1[b][e] + ga.beta1 * d;
                    if (hasZ2) ga.Z2[o] = z2[b][e] + ga.beta2 * d;
                    if (ga.sym && row != col) {            // mirror image (exactly (anti)symmetric output)
                      const long long om = (long long)col * ldn + row;
                      const double dm = msign * d;
                      if (ga.D) ga.D[om] = dm;
                      if (hasZ1) ga.Z1[om] = z1m[b][e] + ga.beta1 * dm;
                      if (hasZ2) ga.Z2[om] = z2m[b][e] + ga.beta2 * dm;
                    }
                  }
                }
            }
          }
        }
      }
    }
  }
  // the last CTA to finish rewinds the two counters for the next launch
  __syncthreads();
  if (threadIdx.x == 0) {
    if (atomicAdd(&ga.sync[1], 1) == G - 1) {
      atomicExch(&ga.sync[0], 0);
      atomicExch(&ga.sync[1], 0);
    }
  }
}

int gemm_tma_grid(int ntiles, int N, int nterms, int sms) {
  const long long total = (long long)ntiles * nterms * ((N + BK - 1) / BK);
  long long g = total / 8;                      // at least 8 stages per range
  if (g > sms) g = sms;
  return (int)(g < 1 ? 1 : g);
}
size_t gemm_tma_ws_doubles(int sms) { return (size_t)sms * TILE * TILE; }
size_t gemm_tma_sync_ints(int sms) { return (size_t)sms + 2; }

void launch_gemm_abt_tma(const GemmArgs& g, const CUtensorMap& tmA0, const CUtensorMap& tmB0, const CUtensorMap& tmA1,
                         const CUtensorMap& tmB1, int sym, const int2* tiles, int ntiles, double* ws, int* sync, int sms,
                         cudaStream_t st) {
  if (ntiles <= 0) return;
  GemmTmaArgs a{g.N, g.ldn, g.A1 ? 2 : 1, sym, tiles, ntiles, g.alpha0, g.alpha1, g.D, g.Z1, g.beta1, g.Z2, g.beta2,
                g.skip, ws, sync};
  const int grid = gemm_tma_grid(ntiles, g.N, a.nterms, sms);
  gemm_abt_tma_kernel<<<grid, NTHREADS, SMEM_TOTAL, st>>>(tmA0, tmB0, tmA1, tmB1, a);
}

int init_tma_kernels() {
  cudaError_t e;
  e = cudaFuncSetAttribute(project_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_TOTAL);
  if (e != cudaSuccess) return (int)e;
  e = cudaFuncSetAttribute(density_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_TOTAL);
  if (e != cudaSuccess) return (int)e;
  e = cudaFuncSetAttribute(gemm_abt_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_TOTAL);
  return (int)e;
}

}  // namespace rt
