// internal.h -- declarations shared by the translation units of libspgpe (host side).
#pragma once
#include <cuda_runtime.h>

#include "pass_x.cuh"
#include "pass_y.cuh"

namespace spgpe {

// per-length launchers (inst_<N>.cu)
#define SPGPE_DECL(N_)                                                                          \
  cudaError_t launch_pass_x_##N_(int dt, int mode, const PassXArgs& a, int ny, cudaStream_t s,           \
                                 const LaunchEnv& env, int* grid);                                        \
  cudaError_t launch_pass_y_##N_(int dt, int ymode, const PassYArgs& a, cudaStream_t s, const LaunchEnv& env, \
                                 int* grid);
SPGPE_DECL(64)
SPGPE_DECL(128)
SPGPE_DECL(256)
SPGPE_DECL(512)
SPGPE_DECL(1024)
SPGPE_DECL(2048)
SPGPE_DECL(4096)
#undef SPGPE_DECL
// fp32 kernels of the complex64 path (inst32_<N>.cu, pass32.cuh)
#define SPGPE_DECL32(N_)                                                                                      \
  cudaError_t launch_row32_##N_(int mode, const PassXArgs& a, int ny, cudaStream_t s, const LaunchEnv& env,  \
                                int* grid);                                                                    \
  cudaError_t launch_col32_##N_(int ymode, const PassYArgs& a, cudaStream_t s, const LaunchEnv& env, int* grid);
SPGPE_DECL32(64)
SPGPE_DECL32(128)
SPGPE_DECL32(256)
SPGPE_DECL32(512)
SPGPE_DECL32(1024)
SPGPE_DECL32(2048)
SPGPE_DECL32(4096)
#undef SPGPE_DECL32

// join of the two interleaved sub-transforms of an axis longer than 4096 (split.cu)
struct SplitArgs {
  void* psi;           // [ny][nx][2]
  int nx, ny;          // full grid
  const int* fx;       // [nx/2] true frequency (0..nx/2-1) of sub-transform position pos; split x axis only
  const int* fy;       // [ny/2]
  const double2* wx;   // [nx/2] exp(-2 pi i fx[pos] / nx)
  const double2* wy;   // [ny/2]
  const double2* phx;  // [2][nx] k_x phase: entry i*mx + pos of the join (split x axis) or stored position (unsplit)
  const double2* phy;  // [ny]    k_y phase, entry j*my + pos of the join, 1/(nx ny) included (split y axis only)
  const double* Kx;    // [2][nx] energy mode: same order as phx
  const double* Ky;    // [ny]
  double* partial;     // [gridDim.x] energy mode
  // two-float copies of wx, wy, phx, phy for the fp32 join of complex64 storage (split32_kernel); NULL: fp64 arithmetic
  const float4 *wx32, *wy32, *phx32, *phy32;
};
cudaError_t launch_split(int dt, const SplitArgs& a, int sx, int sy, int energy, int nblk, cudaStream_t s);

// host-side plan queries (tables.cu)
int plan_tw_total(int n);                       // number of twiddle entries of length n
void plan_fill_twiddles(int n, double2* host);  // exp(-2 pi i k lo / (16 M_j)) blocks, see common.cuh
int plan_lines_ydb(int n);                      // columns per tile of the double-buffered column pass (0: none)
int plan_lines_x(int n);                        // rows per CTA of the row pass of length n
int plan_lines_y(int n);                        // columns per CTA of the column pass of length n
int plan_lines_x32(int n);                      // rows / columns per CTA of the fp32 kernels (pass32.cuh)
int plan_lines_y32(int n);
void plan_fill_twiddles32(int n, float4* host); // the twiddles of plan_fill_twiddles as two-float values
int plan_freq_of_pos(int n, int pos);           // signed-less frequency index f in [0, n) stored at position pos

// small kernels (aux.cu); all enqueue on s and return cudaGetLastError()
cudaError_t aux_phase_tables(const double* Kx, const double* Ky, int nx, int ny, double dt, int imag,
                             double2* exk, double2* eyk, float4* exk32, float4* eyk32, cudaStream_t s);
// partial[nblk][ncol] -> out[col] = factor * sum_blk partial[blk][col]   (fixed summation order)
cudaError_t aux_sum_partials(const double* partial, int nblk, int ncol, double factor, double* out,
                             cudaStream_t s);
cudaError_t aux_apply_scale(int dt, void* psi, size_t points, const double* scale, cudaStream_t s);
// real-space observables from partial[ngroups][stride] (aux.cu, obs_finish_kernel); out[6]
cudaError_t aux_obs_finish(const double* partial, int ngroups, int stride, double cell, const double* scale,
                           double* out, cudaStream_t s);
// partial[nblk][2]: sum |psi_c|^2 ; returns nblk used through *nblk (<= max_blk)
cudaError_t aux_norm_partials(int dt, const void* psi, size_t points, double* partial, int nblk,
                              cudaStream_t s);
// partial[nblk][3]: potential+Zeeman, interaction, Raman sums (without dx dy)
cudaError_t aux_energy_partials(int dt, const void* psi, const void* V, const void* Om, const void* De,
                                size_t points, double g_uu, double g_dd, double g_ud, double* partial,
                                int nblk, cudaStream_t s);
cudaError_t aux_set_targets(double* target, double n_up, double n_dn, cudaStream_t s);
// out[0] = max |field| (0 for a NULL field)
cudaError_t aux_absmax(int dt, const void* field, size_t points, double* out, cudaStream_t s);
// probes (bench roofline denominators)
cudaError_t aux_probe_dfma(cudaStream_t s, double* tflops);
cudaError_t aux_probe_ffma(cudaStream_t s, double* tflops);
cudaError_t aux_probe_copy(cudaStream_t s, long long bytes, double* gbs);

}  // namespace spgpe
