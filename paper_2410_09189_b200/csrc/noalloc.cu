// noalloc.cu -- rt_dipole_noalloc: the a6 reduction (Alg. 1 line 27: dipole and charge of a density on
// the grid) for callers that cannot allocate device memory: code under CUDA graph capture, tight serving loops, harnesses
// that forbid cudaMalloc.  It needs no rt_handle and calls no cudaMalloc / cudaFree / allocating library routine.
//
// The kernel is a variant of reduce_rho_kernel (grid_kernels.cu): one CTA per 1,024 grid points writes its five partial
// sums to SCRATCH, a second one-CTA kernel adds the partials in a fixed order.  The scratch of the existing path is
// cudaMalloc'ed per handle at rt_create; here it is the file-scope array below, NA_MAX_BLOCKS x 5 doubles = 160 KB of
// device memory that every GPU which loads this library holds until the process exits.  That fixes the largest grid:
// NA_MAX_POINTS = 4,194,304 points (128^3 = 2,097,152 and 160^3 = 4,096,000 fit).
//
// In HOST code the name g_na_scratch is a host-side stand-in for the symbol, not a device address: a kernel handed
// `g_na_scratch` from the host would fault (or, where the GPU can reach host memory, silently use the wrong memory).
// The device address comes from cudaGetSymbolAddress, asked once per device with that device current (na_scratch_ptr).
#include "rt_internal.h"

#include <mutex>
#include <string>

namespace rt {

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_ITEMS = 4;                                   // grid points per thread
constexpr int NA_POINTS_PER_BLOCK = NA_THREADS * NA_ITEMS;    // 1,024
constexpr int NA_MAX_BLOCKS = 4096;
constexpr long long NA_MAX_POINTS = (long long)NA_MAX_BLOCKS * NA_POINTS_PER_BLOCK;
constexpr int NA_NV = 5;                                      // sum rho, sum x rho, sum y rho, sum z rho, sum |rho|
constexpr int NA_MAX_DEVICES = 64;

static __device__ __align__(256) double g_na_scratch[NA_MAX_BLOCKS * NA_NV];

// first stage: partial sums of block b -> scratch[b * 5 .. b * 5 + 4].  Every slot that the second stage reads is written
// here in the same call, so nothing in the scratch has to start at zero.
__global__ void __launch_bounds__(NA_THREADS)
dipole_noalloc_partial_kernel(const double* __restrict__ rho, long long Ng, int nx, int ny, int nz, double h,
                              double* __restrict__ scratch) {
  __shared__ double sh[NA_THREADS / 32][NA_NV];
  double v[NA_NV] = {0, 0, 0, 0, 0};
  const double cx = 0.5 * (nx - 1), cy = 0.5 * (ny - 1), cz = 0.5 * (nz - 1);      // centred sawtooth (DESIGN R4)
  const long long nyz = (long long)ny * nz;
  const long long base = (long long)blockIdx.x * NA_POINTS_PER_BLOCK;
#pragma unroll
  for (int i = 0; i < NA_ITEMS; ++i) {
    const long long r = base + (long long)i * NA_THREADS + threadIdx.x;
    if (r < Ng) {
      const double s = rho[r];
      const int ix = (int)(r / nyz);
      const int rem = (int)(r - (long long)ix * nyz);
      const int iy = rem / nz, iz = rem - iy * nz;
      v[0] += s;
      v[1] += ((double)ix - cx) * h * s;
      v[2] += ((double)iy - cy) * h * s;
      v[3] += ((double)iz - cz) * h * s;
      v[4] += fabs(s);
    }
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < NA_NV; ++q) {
    double s = v[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) sh[warp][q] = s;
  }
  __syncthreads();
  if (threadIdx.x < NA_NV) {
    double s = 0.0;
    for (int w = 0; w < NA_THREADS / 32; ++w) s += sh[w][threadIdx.x];
    scratch[(long long)blockIdx.x * NA_NV + threadIdx.x] = s;
  }
}

// second stage: one warp per value, lane-strided partials in block order, then a shuffle tree (fixed order: the result
// does not depend on scheduling).  out = { mu_x, mu_y, mu_z, charge, dVol sum |rho| }.
__global__ void dipole_noalloc_final_kernel(const double* __restrict__ scratch, int nb, double dvol,
                                            double* __restrict__ out) {
  const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (q >= NA_NV) return;
  double s = 0.0;
  for (int b = lane; b < nb; b += 32) s += scratch[(long long)b * NA_NV + q];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) {
    const int slot = q == 0 ? 3 : (q == 4 ? 4 : q - 1);
    out[slot] = dvol * s;
  }
}

// Device address of the scratch array on `device` (which must be current).  Asked once per device.
cudaError_t na_scratch_ptr(int device, double** ptr) {
  static std::mutex mu;
  static double* cached[NA_MAX_DEVICES] = {nullptr};
  std::lock_guard<std::mutex> lock(mu);
  if (!cached[device]) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_na_scratch);
    if (e != cudaSuccess) return e;
    cached[device] = p;
  }
  *ptr = cached[device];
  return cudaSuccess;
}

}  // namespace

long long dipole_noalloc_max_points() { return NA_MAX_POINTS; }

// Returns RT_OK or an RT_E* code with the reason in *err.  Enqueues two kernels on `st`; does not synchronise.
int launch_dipole_noalloc(const double* rho, int nx, int ny, int nz, double h, double* out, int device, cudaStream_t st,
                          std::string* err) {
  const long long Ng = (long long)nx * ny * nz;
  if (Ng > NA_MAX_POINTS) {
    *err = "rt_dipole_noalloc: grid of " + std::to_string(Ng) + " points exceeds the static scratch (maximum " +
           std::to_string(NA_MAX_POINTS) + " points); use rt_create / rt_get_dipole for larger grids";
    return -1;   // RT_EINVAL
  }
  if (device < 0 || device >= NA_MAX_DEVICES) {
    *err = "rt_dipole_noalloc: device ordinal out of range";
    return -1;
  }
  cudaError_t e = cudaSetDevice(device);
  double* scratch = nullptr;
  if (e == cudaSuccess) e = na_scratch_ptr(device, &scratch);
  if (e != cudaSuccess) {
    cudaGetLastError();
    *err = std::string("rt_dipole_noalloc: ") + cudaGetErrorString(e);
    return -3;   // RT_ECUDA
  }
  const int nb = (int)((Ng + NA_POINTS_PER_BLOCK - 1) / NA_POINTS_PER_BLOCK);
  dipole_noalloc_partial_kernel<<<nb, NA_THREADS, 0, st>>>(rho, Ng, nx, ny, nz, h, scratch);
  dipole_noalloc_final_kernel<<<1, 32 * NA_NV, 0, st>>>(scratch, nb, h * h * h, out);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    *err = std::string("rt_dipole_noalloc: launch failed: ") + cudaGetErrorString(e);
    return -3;
  }
  return 0;
}

}  // namespace rt
