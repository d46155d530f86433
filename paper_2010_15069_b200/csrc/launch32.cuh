// launch32.cuh -- launchers of the fp32 pass kernels (pass32.cuh), one translation unit per line length (inst32_<N>.cu).
#pragma once
#include "launch.cuh"
#include "pass32.cuh"

namespace spgpe {

template <int N, int MODE, int XS>
cudaError_t launch_row32_xs(const PassXArgs& a, int ny, cudaStream_t s, const LaunchEnv& env, int* grid_out) {
  constexpr int L = (XS == 2) ? 2 : Lines32<N>::X;
  auto k = row32_kernel<N, L, MODE, XS>;
  constexpr size_t smem = (XS == 2) ? Smem32<N, L>::BYTES_Y : Smem32<N, L>::BYTES_X;
  static int cache[SPGPE_MAX_DEVICES] = {};
  int resident = 0;
  cudaError_t e = resident_ctas(k, L * (N / 16), smem, env, cache, &resident);
  if (e != cudaSuccess) return e;
  const int groups = ny / L;
  const int grid = groups < resident ? groups : resident;
  *grid_out = grid;
  return launch_pdl(k, grid, L * (N / 16), smem, s, a);
}

// a split x axis (xs = 2) is handled by the fp32 kernels from sub-line length 512 up (full warps per line pair)
template <int N, int MODE>
cudaError_t launch_row32(const PassXArgs& a, int ny, cudaStream_t s, const LaunchEnv& env, int* grid_out) {
  if constexpr (N >= 512) {
    if (a.xs == 2) return launch_row32_xs<N, MODE, 2>(a, ny, s, env, grid_out);
  }
  return launch_row32_xs<N, MODE, 1>(a, ny, s, env, grid_out);
}

template <int N, int YMODE>
cudaError_t launch_col32(const PassYArgs& a, cudaStream_t s, const LaunchEnv& env, int* grid_out) {
  constexpr int L = Lines32<N>::Y;
  auto k = col32_kernel<N, L, YMODE>;
  constexpr size_t smem = Smem32<N, L>::BYTES_Y;
  static int cache[SPGPE_MAX_DEVICES] = {};
  int resident = 0;
  cudaError_t e = resident_ctas(k, L * (N / 16), smem, env, cache, &resident);
  if (e != cudaSuccess) return e;
  const int groups = a.nx / L;
  const int grid = groups < resident ? groups : resident;
  *grid_out = grid;
  return launch_pdl(k, grid, L * (N / 16), smem, s, a);
}

#define SPGPE_DEFINE_LAUNCHERS32(N_)                                                                              \
  cudaError_t launch_row32_##N_(int mode, const PassXArgs& a, int ny, cudaStream_t s, const LaunchEnv& env,      \
                                int* g) {                                                                          \
    switch (mode) {                                                                                                \
      case MODE_PRO: return launch_row32<N_, MODE_PRO>(a, ny, s, env, g);                                          \
      case MODE_MID: return launch_row32<N_, MODE_MID>(a, ny, s, env, g);                                          \
      default: return launch_row32<N_, MODE_EPI>(a, ny, s, env, g);                                                \
    }                                                                                                              \
  }                                                                                                                \
  cudaError_t launch_col32_##N_(int ymode, const PassYArgs& a, cudaStream_t s, const LaunchEnv& env, int* g) {   \
    switch (ymode) {                                                                                               \
      case YMODE_STEP: return launch_col32<N_, YMODE_STEP>(a, s, env, g);                                          \
      case YMODE_FWDONLY: return launch_col32<N_, YMODE_FWDONLY>(a, s, env, g);                                    \
      default: return launch_col32<N_, YMODE_INVONLY>(a, s, env, g);                                               \
    }                                                                                                              \
  }

}  // namespace spgpe
