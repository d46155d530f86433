// launch.cuh -- launch configuration per line length and the macro that instantiates the row/column
// pass kernels of one length in its own translation unit (inst_<N>.cu), so that lengths compile in parallel.
#pragma once
#include "pass_x.cuh"
#include "pass_y.cuh"

namespace spgpe {

// lines (rows or columns) per CTA: 256 threads per CTA up to N = 2048, 512 at N = 4096
template <int N> struct Lines { static constexpr int X = (N >= 2048) ? 1 : (N == 1024 ? 2 : 4), Y = X; };

template <int DT, int N, int MODE>
cudaError_t launch_x(const PassXArgs& a, int ny, cudaStream_t s) {
  constexpr int L = Lines<N>::X;
  auto k = pass_x_kernel<DT, N, L, MODE>;
  constexpr size_t smem = (size_t)L * Plan<N>::PTS * 2 * sizeof(double2);
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  k<<<ny / L, L * (N / 8), smem, s>>>(a);
  return cudaGetLastError();
}

template <int DT, int N, int YMODE>
cudaError_t launch_y(const PassYArgs& a, cudaStream_t s) {
  constexpr int L = Lines<N>::Y;
  auto k = pass_y_kernel<DT, N, L, YMODE>;
  constexpr size_t smem = (size_t)L * YLayout<N, L>::LINE_PTS * 2 * sizeof(double2);
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  k<<<a.nx / L, L * (N / 8), smem, s>>>(a);
  return cudaGetLastError();
}

#define SPGPE_DEFINE_LAUNCHERS(N_)                                                               \
  cudaError_t launch_pass_x_##N_(int dt, int mode, const PassXArgs& a, int ny, cudaStream_t s) { \
    if (dt == 0) {                                                                               \
      switch (mode) {                                                                            \
        case MODE_PRO: return launch_x<0, N_, MODE_PRO>(a, ny, s);                               \
        case MODE_MID: return launch_x<0, N_, MODE_MID>(a, ny, s);                               \
        case MODE_EPI: return launch_x<0, N_, MODE_EPI>(a, ny, s);                               \
        default: return launch_x<0, N_, MODE_FWD>(a, ny, s);                                     \
      }                                                                                          \
    }                                                                                            \
    switch (mode) {                                                                              \
      case MODE_PRO: return launch_x<1, N_, MODE_PRO>(a, ny, s);                                 \
      case MODE_MID: return launch_x<1, N_, MODE_MID>(a, ny, s);                                 \
      case MODE_EPI: return launch_x<1, N_, MODE_EPI>(a, ny, s);                                 \
      default: return launch_x<1, N_, MODE_FWD>(a, ny, s);                                       \
    }                                                                                            \
  }                                                                                              \
  cudaError_t launch_pass_y_##N_(int dt, int ymode, const PassYArgs& a, cudaStream_t s) {        \
    if (dt == 0)                                                                                 \
      return ymode == YMODE_STEP ? launch_y<0, N_, YMODE_STEP>(a, s)                             \
                                 : launch_y<0, N_, YMODE_ENERGY>(a, s);                          \
    return ymode == YMODE_STEP ? launch_y<1, N_, YMODE_STEP>(a, s)                               \
                               : launch_y<1, N_, YMODE_ENERGY>(a, s);                            \
  }

}  // namespace spgpe
