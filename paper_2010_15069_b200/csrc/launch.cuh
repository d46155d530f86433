// launch.cuh -- launch configuration per line length and the macro that instantiates the row/column
// pass kernels of one length in its own translation unit (inst_<N>.cu), so that lengths compile in parallel.
#pragma once
#include <stdlib.h>
#include "pass_x.cuh"
#include "pass_y.cuh"

namespace spgpe {

// lines (rows or columns) per CTA: at most 256 threads per CTA up to N = 2048, 512 at N = 4096.  Rows of 512 points go two
// to a CTA (128 threads, like the four rows of 256 points): with four (256 threads at 128 registers) the back-to-back
// step at 512 x 256 / 512 x 512 was as long as the two serialised launches (25.1 / 32.1 us against 18.0 / 25.2 us with
// two: profiles/r2_eta_sweep.md).  Rows of 1024 points go one to a CTA (128 threads; with two, 1024 x 1024 took 35.2 us per
// row pass against 31.0 us: config 3 73.0 -> 69.6 us/step).  Columns of 512 points stay four to a CTA (two: better at
// 512 x 512 and 2048 x 512, worse at 1024 x 512); one row of 512 points per CTA is no better than two.
template <int N> struct Lines {
  static constexpr int X = (N >= 1024) ? 1 : (N >= 512 ? 2 : 4);
  static constexpr int Y = (N >= 4096) ? 1 : (N >= 1024 ? 2 : 4);
  static constexpr int YDB = (N == 2048) ? 1 : (N == 1024 ? 2 : 0);  // columns per tile of pass_y_db_kernel (0: none)
};

constexpr int SPGPE_MAX_DEVICES = 64;

// Number of CTAs of `kernel` that can be resident on env.device at once, and the one-time opt-in to `smem` bytes
// of dynamic shared memory.  Both are per-device properties: the cache is indexed by the device ordinal (a second
// handle on another GPU of the same process sets the attribute there too).  Racing threads compute the same value.
template <typename K>
cudaError_t resident_ctas(K kernel, int threads, size_t smem, const LaunchEnv& env, int* cache, int* out) {
  const int slot = (env.device >= 0 && env.device < SPGPE_MAX_DEVICES) ? env.device : -1;
  int r = slot >= 0 ? __atomic_load_n(&cache[slot], __ATOMIC_ACQUIRE) : 0;
  if (r == 0) {
    int sms = 0, occ = 0;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, env.device);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem);
    if (e != cudaSuccess) return e;
    r = sms * (occ > 0 ? occ : 1);
    if (slot >= 0) __atomic_store_n(&cache[slot], r, __ATOMIC_RELEASE);
  }
  if (env.ctas_per_sm > 0) {  // diagnostic cap (not cached)
    int sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, env.device);
    if (e != cudaSuccess) return e;
    if (env.ctas_per_sm * sms < r) r = env.ctas_per_sm * sms;
  }
  *out = r;
  return cudaSuccess;
}

template <int DT, int N, int MODE>
cudaError_t launch_x(const PassXArgs& a, int ny, cudaStream_t s, const LaunchEnv& env, int* grid_out);

// launch with programmatic stream serialization (common.cuh, pdl_wait): the kernel may start its prologue while
// the previous kernel on the stream drains
template <typename K, typename A>
cudaError_t launch_pdl(K kernel, int grid, int threads, size_t smem, cudaStream_t s, const A& args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, args);
}

// grid_out: number of CTAs launched (= rows of PassXArgs::partial written by MODE_EPI)
template <int DT, int N, int MODE, int XS, bool NEST, int TIME>
cudaError_t launch_x_time(const PassXArgs& a, int ny, cudaStream_t s, const LaunchEnv& env, int* grid_out) {
  constexpr int L = Lines<N>::X;
  auto k = pass_x_kernel<DT, N, L, MODE, XS, NEST, TIME>;
  constexpr size_t smem = XSmem<N, L>::BYTES;
  static int cache[SPGPE_MAX_DEVICES] = {};
  int resident = 0;
  cudaError_t e = resident_ctas(k, L * (N / 8), smem, env, cache, &resident);
  if (e != cudaSuccess) return e;
  const int groups = ny / L;
  const int grid = groups < resident ? groups : resident;
  *grid_out = grid;
  return launch_pdl(k, grid, L * (N / 8), smem, s, a);
}

// real or imaginary time is a compile-time property of the default opening / closing passes (TIME = 0 | 1); the
// steady-state pass exists in real time only; the nested instantiations decide at run time (TIME = 2)
template <int DT, int N, int MODE, int XS, bool NEST>
cudaError_t launch_x_xs(const PassXArgs& a, int ny, cudaStream_t s, const LaunchEnv& env, int* grid_out) {
  if constexpr (NEST) return launch_x_time<DT, N, MODE, XS, true, 2>(a, ny, s, env, grid_out);
  else if constexpr (MODE == MODE_MID || MODE == MODE_FWD) return launch_x_time<DT, N, MODE, XS, false, 0>(a, ny, s, env, grid_out);
  else return a.imag ? launch_x_time<DT, N, MODE, XS, false, 1>(a, ny, s, env, grid_out)
                     : launch_x_time<DT, N, MODE, XS, false, 0>(a, ny, s, env, grid_out);
}

template <int DT, int N, int MODE>
cudaError_t launch_x(const PassXArgs& a, int ny, cudaStream_t s, const LaunchEnv& env, int* grid_out) {
  if constexpr (MODE != MODE_FWD) {  // the transform-only mode has no real-space part
    if (a.nest)
      return a.xs == 1 ? launch_x_xs<DT, N, MODE, 1, true>(a, ny, s, env, grid_out)
                       : launch_x_xs<DT, N, MODE, 2, true>(a, ny, s, env, grid_out);
  }
  return a.xs == 1 ? launch_x_xs<DT, N, MODE, 1, false>(a, ny, s, env, grid_out)
                   : launch_x_xs<DT, N, MODE, 2, false>(a, ny, s, env, grid_out);
}

template <int DT, int N, int YMODE>
cudaError_t launch_y(const PassYArgs& a, cudaStream_t s, const LaunchEnv& env, int* grid_out) {
  constexpr int L = Lines<N>::Y;
  auto k = pass_y_kernel<DT, N, L, YMODE>;
  constexpr size_t smem = YSmem<N, L>::BYTES;
  static int cache[SPGPE_MAX_DEVICES] = {};
  int resident = 0;
  cudaError_t e = resident_ctas(k, L * (N / 8), smem, env, cache, &resident);
  if (e != cudaSuccess) return e;
  const int groups = a.nx / L;
  const int grid = groups < resident ? groups : resident;
  *grid_out = grid;
  return launch_pdl(k, grid, L * (N / 8), smem, s, a);
}

template <int DT, int N>
cudaError_t launch_y_db(const PassYArgs& a, cudaStream_t s, const LaunchEnv& env, int* grid_out) {
  constexpr int L = Lines<N>::YDB > 0 ? Lines<N>::YDB : 1;
  auto k = pass_y_db_kernel<DT, N, L>;
  constexpr size_t smem = YSmemDB<N, L>::BYTES;
  static int cache[SPGPE_MAX_DEVICES] = {};
  int resident = 0;
  cudaError_t e = resident_ctas(k, L * (N / 8), smem, env, cache, &resident);
  if (e != cudaSuccess) return e;
  const int groups = a.nx / L;
  const int grid = groups < resident ? groups : resident;
  *grid_out = grid;
  return launch_pdl(k, grid, L * (N / 8), smem, s, a);
}
// YMODE_STEP goes to the double-buffered kernel where one exists.  complex64 storage keeps the two-column kernel:
// a one-column tile of float2 pairs is only 16 bytes wide, too narrow for efficient TMA boxes (measured at 2048^2:
// 86 us against 78 us).
template <int DT, int N>
cudaError_t launch_y_step(const PassYArgs& a, cudaStream_t s, const LaunchEnv& env, int* g) {
  if constexpr (Lines<N>::YDB > 0 && DT == 0) {
    if (!env.no_ydb) return launch_y_db<DT, N>(a, s, env, g);
  }
  return launch_y<DT, N, YMODE_STEP>(a, s, env, g);
}

#define SPGPE_DEFINE_LAUNCHERS(N_)                                                               \
  cudaError_t launch_pass_x_##N_(int dt, int mode, const PassXArgs& a, int ny, cudaStream_t s, \
                                 const LaunchEnv& env, int* g) { \
    if (dt == 0) {                                                                               \
      switch (mode) {                                                                            \
        case MODE_PRO: return launch_x<0, N_, MODE_PRO>(a, ny, s, env, g);                               \
        case MODE_MID: return launch_x<0, N_, MODE_MID>(a, ny, s, env, g);                               \
        case MODE_EPI: return launch_x<0, N_, MODE_EPI>(a, ny, s, env, g);                               \
        case MODE_EPI_OBS: return launch_x<0, N_, MODE_EPI_OBS>(a, ny, s, env, g);                       \
        default: return launch_x<0, N_, MODE_FWD>(a, ny, s, env, g);                                     \
      }                                                                                          \
    }                                                                                            \
    switch (mode) {                                                                              \
      case MODE_PRO: return launch_x<1, N_, MODE_PRO>(a, ny, s, env, g);                                 \
      case MODE_MID: return launch_x<1, N_, MODE_MID>(a, ny, s, env, g);                                 \
      case MODE_EPI: return launch_x<1, N_, MODE_EPI>(a, ny, s, env, g);                                 \
      case MODE_EPI_OBS: return launch_x<1, N_, MODE_EPI_OBS>(a, ny, s, env, g);                         \
      default: return launch_x<1, N_, MODE_FWD>(a, ny, s, env, g);                                       \
    }                                                                                            \
  }                                                                                              \
  cudaError_t launch_pass_y_##N_(int dt, int ymode, const PassYArgs& a, cudaStream_t s, \
                                 const LaunchEnv& env, int* g) { \
    if (dt == 0) {                                                                               \
      switch (ymode) {                                                                           \
        case YMODE_STEP: return launch_y_step<0, N_>(a, s, env, g);                            \
        case YMODE_ENERGY: return launch_y<0, N_, YMODE_ENERGY>(a, s, env, g);                        \
        case YMODE_FWDONLY: return launch_y<0, N_, YMODE_FWDONLY>(a, s, env, g);                      \
        case YMODE_STEP_OBS: return launch_y<0, N_, YMODE_STEP_OBS>(a, s, env, g);                    \
        default: return launch_y<0, N_, YMODE_INVONLY>(a, s, env, g);                                 \
      }                                                                                          \
    }                                                                                            \
    switch (ymode) {                                                                             \
      case YMODE_STEP: return launch_y_step<1, N_>(a, s, env, g);                              \
      case YMODE_ENERGY: return launch_y<1, N_, YMODE_ENERGY>(a, s, env, g);                          \
      case YMODE_FWDONLY: return launch_y<1, N_, YMODE_FWDONLY>(a, s, env, g);                        \
      case YMODE_STEP_OBS: return launch_y<1, N_, YMODE_STEP_OBS>(a, s, env, g);                      \
      default: return launch_y<1, N_, YMODE_INVONLY>(a, s, env, g);                                   \
    }                                                                                            \
  }

}  // namespace spgpe
