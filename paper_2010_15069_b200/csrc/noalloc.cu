// noalloc.cu -- spgpe_norm_noalloc (include/spgpe.h): the component norms N_c = dx dy sum_r |psi_c|^2 (R-8) of a
// caller-owned order parameter, computed WITHOUT any allocation: for callers that cannot call cudaMalloc (code under
// CUDA graph capture, tight serving loops, harnesses that forbid it).  It is a variant of the norm reduction of aux.cu
// (norm_partials_kernel + sum_partials_kernel behind spgpe_norm), whose scratch -- one pair of partial sums per CTA --
// comes from a handle's cudaMalloc'd buffer there and from a fixed file-scope device array here.
//
// The scratch.  g_norm_scratch below: NOALLOC_BLOCKS x 2 doubles = 16 KiB, aligned to 256 bytes; every GPU that loads
// the library holds it until the process exits.  In HOST code the name g_norm_scratch is only a host-side stand-in of
// the symbol, not a device address (a kernel handed &g_norm_scratch[0] from the host would fault, or silently use the
// wrong memory where the GPU can reach host memory): the device address is looked up with cudaGetSymbolAddress, in
// this file, once per device, with that device current, and that pointer is what the kernels receive.
//
// Sharing.  Every call on a device uses the same array and finds the previous call's contents in it.  Nothing in it
// has to start at zero: the first kernel overwrites every one of the NOALLOC_BLOCKS slots before the second kernel
// reads them (all NOALLOC_BLOCKS CTAs are always launched; a CTA without points writes zeros), and no counter or flag
// lives in it.  Calls that overlap on the GPU (two streams, or two host threads on one device) race on it: keep the
// calls of a device on one stream, or order them with events.
//
// Nothing here calls cudaMalloc, cudaFree or an allocating library routine; the results leave through the caller's
// device pointer, asynchronously on the caller's stream.
#include <atomic>

#include <cuda_runtime.h>

#include "../../include/spgpe.h"
#include "common.cuh"

namespace spgpe {

constexpr int NOALLOC_BLOCKS = 1024;    // CTAs of the first kernel = slots of the scratch (the grid of spgpe_norm)
constexpr int NOALLOC_THREADS = 256;
constexpr int NOALLOC_MAX_AXIS = 8192;  // largest nx, ny accepted (the library's largest grid: 2^26 points)
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) double g_norm_scratch[NOALLOC_BLOCKS * 2];

// partial[blk][c] = sum over the points of CTA blk of |psi_c|^2 (grid-stride, fixed order; fp64 accumulation)
template <int DT>
__global__ void __launch_bounds__(NOALLOC_THREADS) norm_partials_static_kernel(const void* __restrict__ psi, size_t points,
                                                                              double* __restrict__ partial) {
  __shared__ double red[2][NOALLOC_THREADS / 32];
  double x0 = 0.0, x1 = 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < points; i += (size_t)gridDim.x * blockDim.x) {
    const cplx u = Store<DT>::ld(psi, 2 * i), d = Store<DT>::ld(psi, 2 * i + 1);
    x0 += fma(u.re, u.re, u.im * u.im);
    x1 += fma(d.re, d.re, d.im * d.im);
  }
#pragma unroll
  for (int m = 16; m >= 1; m >>= 1) {
    x0 += __shfl_xor_sync(0xffffffffu, x0, m);
    x1 += __shfl_xor_sync(0xffffffffu, x1, m);
  }
  if ((threadIdx.x & 31) == 0) {
    red[0][threadIdx.x >> 5] = x0;
    red[1][threadIdx.x >> 5] = x1;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double s0 = 0.0, s1 = 0.0;
    for (int i = 0; i < NOALLOC_THREADS / 32; ++i) {
      s0 += red[0][i];
      s1 += red[1][i];
    }
    partial[2 * blockIdx.x] = s0;  // every slot is written by every call (see the header comment)
    partial[2 * blockIdx.x + 1] = s1;
  }
}

// out[c] = cell * sum_blk partial[blk][c]; one CTA, fixed order
__global__ void __launch_bounds__(NOALLOC_THREADS) norm_finish_static_kernel(const double* __restrict__ partial, double cell,
                                                                            double* __restrict__ out) {
  __shared__ double red[NOALLOC_THREADS / 32];
  for (int c = 0; c < 2; ++c) {
    double x = 0.0;
    for (int b = threadIdx.x; b < NOALLOC_BLOCKS; b += blockDim.x) x += partial[2 * b + c];
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) x += __shfl_xor_sync(0xffffffffu, x, m);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x == 0) {
      double s = 0.0;
      for (int i = 0; i < NOALLOC_THREADS / 32; ++i) s += red[i];
      out[c] = cell * s;
    }
    __syncthreads();
  }
}

// Device address of g_norm_scratch on the CURRENT device: looked up once per device (set-up of that device), kept in
// a per-device slot.  Racing threads look up the same value.
static std::atomic<double*> g_scratch_addr[NOALLOC_MAX_DEVICES];

static cudaError_t scratch_of_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
  double* p = g_scratch_addr[dev].load(std::memory_order_acquire);
  if (p == nullptr) {
    e = cudaGetSymbolAddress((void**)&p, g_norm_scratch);  // `dev` is current: the address is that device's copy
    if (e != cudaSuccess) return e;
    if (p == nullptr) return cudaErrorInvalidSymbol;
    g_scratch_addr[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return cudaSuccess;
}

}  // namespace spgpe

using namespace spgpe;

extern "C" int spgpe_norm_noalloc(const void* d_psi, int dtype, int nx, int ny, double Lx, double Ly, double* d_out,
                                  void* cuda_stream) {
  if (!d_psi || !d_out || nx < 1 || ny < 1 || !(Lx > 0.0) || !(Ly > 0.0)) return SPGPE_ERR_INVALID_ARG;
  if (dtype != SPGPE_C128 && dtype != SPGPE_C64) return SPGPE_ERR_INVALID_ARG;
  if (nx > NOALLOC_MAX_AXIS || ny > NOALLOC_MAX_AXIS) return SPGPE_ERR_TOO_LARGE;
  double* scratch = nullptr;
  if (scratch_of_current_device(&scratch) != cudaSuccess) return SPGPE_ERR_CUDA;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const size_t points = (size_t)nx * (size_t)ny;
  const double cell = (Lx / nx) * (Ly / ny);
  if (dtype == SPGPE_C128) norm_partials_static_kernel<0><<<NOALLOC_BLOCKS, NOALLOC_THREADS, 0, s>>>(d_psi, points, scratch);
  else norm_partials_static_kernel<1><<<NOALLOC_BLOCKS, NOALLOC_THREADS, 0, s>>>(d_psi, points, scratch);
  if (cudaGetLastError() != cudaSuccess) return SPGPE_ERR_CUDA;
  norm_finish_static_kernel<<<1, NOALLOC_THREADS, 0, s>>>(scratch, cell, d_out);
  if (cudaGetLastError() != cudaSuccess) return SPGPE_ERR_CUDA;
  return SPGPE_OK;
}
