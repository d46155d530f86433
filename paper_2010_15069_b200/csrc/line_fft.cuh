// line_fft.cuh -- length-N complex transform of one line held 16 points per thread in registers,
// radix-16 stages exchanged through shared memory (one __syncthreads per exchange).
//
// Forward (decimation in frequency): input v[n] = x[t + n*T] (natural order), output v[g*RL + s] =
// X[f] where the "stored position" of that register is (t + g*T) + (N/RL)*s and f = freq_of_pos(N, pos)
// (host-side table, see tables.cu).  Inverse is the exact mirror (unnormalised: inverse(forward(x)) = N x).
// Between the two no reordering is needed, so pointwise k-space factors are applied on registers.
//
// Shared-memory line buffer: point p of component c lives at double2 index (p + (p >> PADSHIFT))*2 + c.
#pragma once
#include "radix.cuh"

namespace spgpe {

template <int N>
__device__ __forceinline__ int smem_idx(int p, int c) {
  return ((p + (p >> Plan<N>::PADSHIFT)) << 1) + c;
}

// positions of radix-16 stage j (1-based): hi*16*M + n*M + lo with t = hi*M + lo, M = N >> (4j)
template <int N, int J>
struct StagePos {
  static constexpr int M = N >> (4 * J);
  int base, lo;
  __device__ __forceinline__ StagePos(int t) {
    lo = t & (M - 1);
    base = ((t - lo) << 4) + lo;  // hi*M*16 + lo
  }
  __device__ __forceinline__ int pos(int n) const { return base + n * M; }
};

template <int N>
__device__ __forceinline__ void sts_last(double2* buf, int t, int c, const cplx* v) {
  typedef Plan<N> P;
#pragma unroll
  for (int g = 0; g < P::G; ++g)
#pragma unroll
    for (int s = 0; s < P::RL; ++s)
      buf[smem_idx<N>((t + g * P::T) * P::RL + s, c)] = make_double2(v[g * P::RL + s].re, v[g * P::RL + s].im);
}
template <int N>
__device__ __forceinline__ void lds_last(const double2* buf, int t, int c, cplx* v) {
  typedef Plan<N> P;
#pragma unroll
  for (int g = 0; g < P::G; ++g)
#pragma unroll
    for (int s = 0; s < P::RL; ++s) {
      double2 d = buf[smem_idx<N>((t + g * P::T) * P::RL + s, c)];
      v[g * P::RL + s] = mk(d.x, d.y);
    }
}
template <int N, int J>
__device__ __forceinline__ void sts_stage(double2* buf, int t, int c, const cplx* v) {
  StagePos<N, J> sp(t);
#pragma unroll
  for (int n = 0; n < 16; ++n) buf[smem_idx<N>(sp.pos(n), c)] = make_double2(v[n].re, v[n].im);
}
template <int N, int J>
__device__ __forceinline__ void lds_stage(const double2* buf, int t, int c, cplx* v) {
  StagePos<N, J> sp(t);
#pragma unroll
  for (int n = 0; n < 16; ++n) {
    double2 d = buf[smem_idx<N>(sp.pos(n), c)];
    v[n] = mk(d.x, d.y);
  }
}

// v[k] *= w_j[k][lo] (forward) or conj (inverse); w_j[k][lo] = exp(-2 pi i k lo / (16 M_j))
template <int N, int J, int D>
__device__ __forceinline__ void twiddle(const double2* __restrict__ tw, int t, cplx* v) {
  constexpr int M = N >> (4 * J);
  const int lo = t & (M - 1);
  const double2* w = tw + tw_offset<N>(J) + lo;
#pragma unroll
  for (int k = 1; k < 16; ++k) {
    // the address depends on v[k] (late_zero), so that ptxas cannot hoist the table load far above its use
    double2 d = __ldg(w + (k - 1) * M + late_zero(v[k].re));
    v[k] = (D < 0) ? cmul(v[k], mk(d.x, d.y)) : cmulc(v[k], mk(d.x, d.y));
  }
}

// one forward radix-16 stage J followed by the exchange into stage J+1's (or the last stage's) registers
template <int N, int J>
__device__ __forceinline__ void fwd_stages(double2* buf, const double2* __restrict__ tw, int t, int c, cplx* v) {
  if constexpr (J < Plan<N>::NS) {
    dft16<-1>(v);
    twiddle<N, J, -1>(tw, t, v);
    sts_stage<N, J>(buf, t, c, v);
    __syncthreads();
    if constexpr (J + 1 < Plan<N>::NS) lds_stage<N, J + 1>(buf, t, c, v);
    else lds_last<N>(buf, t, c, v);
    fwd_stages<N, J + 1>(buf, tw, t, c, v);
  }
}
template <int N>
__device__ __forceinline__ void line_fft_fwd(double2* buf, const double2* __restrict__ tw, int t, int c, cplx* v) {
  fwd_stages<N, 1>(buf, tw, t, c, v);
  dft_last<-1, Plan<N>::RL>(v);
}

template <int N, int J>
__device__ __forceinline__ void inv_stages(double2* buf, const double2* __restrict__ tw, int t, int c, cplx* v) {
  if constexpr (J >= 1) {
    if constexpr (J + 1 < Plan<N>::NS) sts_stage<N, J + 1>(buf, t, c, v);
    else sts_last<N>(buf, t, c, v);
    __syncthreads();
    lds_stage<N, J>(buf, t, c, v);
    twiddle<N, J, +1>(tw, t, v);
    dft16<+1>(v);
    inv_stages<N, J - 1>(buf, tw, t, c, v);
  }
}
template <int N>
__device__ __forceinline__ void line_fft_inv(double2* buf, const double2* __restrict__ tw, int t, int c, cplx* v) {
  dft_last<+1, Plan<N>::RL>(v);
  inv_stages<N, Plan<N>::NS - 1>(buf, tw, t, c, v);
}

}  // namespace spgpe
