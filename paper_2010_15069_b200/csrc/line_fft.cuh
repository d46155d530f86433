// line_fft.cuh -- length-N complex transform of one line held 16 points per thread in registers,
// radix-16 stages exchanged through shared memory (one __syncthreads per exchange).
//
// Forward (decimation in frequency): input v[n] = x[t + n*T] (natural order), output v[g*RL + s] =
// X[f] where the "stored position" of that register is (t + g*T) + (N/RL)*s and f = freq_of_pos(N, pos)
// (host-side table, see tables.cu).  Inverse is the exact mirror (unnormalised: inverse(forward(x)) = N x).
// Between the two no reordering is needed, so pointwise k-space factors are applied on registers.
//
// Three-stage plans (N >= 512): after the first radix-16 stage the line splits into 16 independent blocks of
// N/16 points, each owned by the RL threads t with the same t / RL (times two components): these threads sit in
// ONE warp, so the exchange between the second stage and the last one needs only __syncwarp().  The last-stage
// groups of thread t = (hi, lo) are q = hi*16 + lo + g*RL (inside its own block).
//
// Twiddles are read from a table in shared memory (copied there once per CTA by the pass kernels).
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

// first last-stage group of thread t; its groups are group0 + g * GSTEP
template <int N>
__device__ __forceinline__ int last_group0(int t) {
  typedef Plan<N> P;
  if (P::NS == 3) return (t / P::RL) * 16 + (t % P::RL);
  return t;
}
template <int N> struct LastStep { static constexpr int GSTEP = (Plan<N>::NS == 3) ? Plan<N>::RL : Plan<N>::T; };

// double2 index of element (group q0 + g*GSTEP, s) of the last stage.  When RL == 2^PADSHIFT the padded index is
// affine in (g, s): one base per thread plus compile-time offsets.
template <int N>
struct LastIdx {
  typedef Plan<N> P;
  static constexpr bool AFFINE = (P::RL == (1 << P::PADSHIFT));
  int base;
  __device__ __forceinline__ LastIdx(int t, int c) {
    const int q0 = last_group0<N>(t);
    base = AFFINE ? (q0 * (P::RL + 1) * 2 + c) : (q0 * P::RL * 2 + c);
    q0_ = q0; c_ = c;
  }
  __device__ __forceinline__ int at(int g, int s) const {
    if (AFFINE) return base + (g * LastStep<N>::GSTEP * (P::RL + 1) + s) * 2;
    return smem_idx<N>((q0_ + g * LastStep<N>::GSTEP) * P::RL + s, c_);
  }
  int q0_, c_;
};

template <int N>
__device__ __forceinline__ void sts_last(double2* buf, int t, int c, const cplx* v) {
  typedef Plan<N> P;
  const LastIdx<N> ix(t, c);
#pragma unroll
  for (int g = 0; g < P::G; ++g)
#pragma unroll
    for (int s = 0; s < P::RL; ++s)
      buf[ix.at(g, s)] = make_double2(v[g * P::RL + s].re, v[g * P::RL + s].im);
}
template <int N>
__device__ __forceinline__ void lds_last(const double2* buf, int t, int c, cplx* v) {
  typedef Plan<N> P;
  const LastIdx<N> ix(t, c);
#pragma unroll
  for (int g = 0; g < P::G; ++g)
#pragma unroll
    for (int s = 0; s < P::RL; ++s) {
      double2 d = buf[ix.at(g, s)];
      v[g * P::RL + s] = mk(d.x, d.y);
    }
}
// barrier of the exchange next to the last stage: warp-local for three-stage plans
template <int N>
__device__ __forceinline__ void sync_last() {
  if (Plan<N>::NS == 3) __syncwarp();
  else __syncthreads();
}
// double2 index of element n of radix-16 stage J: affine in n when the stride M is a multiple of the padding period
template <int N, int J>
struct StageIdx {
  static constexpr int M = N >> (4 * J);
  static constexpr int S = Plan<N>::PADSHIFT;
  static constexpr bool AFFINE = (M % (1 << S)) == 0;
  StagePos<N, J> sp;
  int base, c_;
  __device__ __forceinline__ StageIdx(int t, int c) : sp(t), c_(c) { base = smem_idx<N>(sp.base, c); }
  __device__ __forceinline__ int at(int n) const {
    if (AFFINE) return base + n * ((M + (M >> S)) * 2);
    return smem_idx<N>(sp.pos(n), c_);
  }
};
template <int N, int J>
__device__ __forceinline__ void sts_stage(double2* buf, int t, int c, const cplx* v) {
  const StageIdx<N, J> ix(t, c);
#pragma unroll
  for (int n = 0; n < 16; ++n) buf[ix.at(n)] = make_double2(v[n].re, v[n].im);
}
template <int N, int J>
__device__ __forceinline__ void lds_stage(const double2* buf, int t, int c, cplx* v) {
  const StageIdx<N, J> ix(t, c);
#pragma unroll
  for (int n = 0; n < 16; ++n) {
    double2 d = buf[ix.at(n)];
    v[n] = mk(d.x, d.y);
  }
}

// v[k] *= w_j[k][lo] (forward) or conj (inverse); w_j[k][lo] = exp(-2 pi i k lo / (16 M_j))
//
// flip (0 or 0x80000000, stage 1 only) negates the twiddles of odd k.  With it a thread may hold its 16 points
// rotated by 8 (register n = point (n + 8) mod 16) on the natural-order side of the transform: rotating the
// input of a 16-point DFT by 8 multiplies output k by (-1)^k, and multiplying input k by (-1)^k rotates the output.
__device__ __forceinline__ double flip_sign(double x, int flip) {
  return __hiloint2double(__double2hiint(x) ^ flip, __double2loint(x));
}
template <int N, int J, int D>
__device__ __forceinline__ void twiddle(const double2* tw, int t, cplx* v, int flip) {
  constexpr int M = N >> (4 * J);
  const int lo = t & (M - 1);
  const double2* w = tw + tw_offset<N>(J) + lo;
#pragma unroll
  for (int k = 1; k < 16; ++k) {
    double2 d = w[(k - 1) * M];
    if (J == 1 && (k & 1)) {
      d.x = flip_sign(d.x, flip);
      d.y = flip_sign(d.y, flip);
    }
    v[k] = (D < 0) ? cmul(v[k], mk(d.x, d.y)) : cmulc(v[k], mk(d.x, d.y));
  }
}

// Synchronisation policy of a line transform.  sync(): barrier over the threads that share the line buffers;
// acquire()/release(): bracket every exchange (the shared-memory stores, the barrier and the loads after it).
// CtaSync: the whole CTA works on the same lines, no bracket.  GroupSync (pass_x.cuh): two thread groups of one
// CTA work on different lines and take turns at their exchanges.
// REG_TW1: the policy object carries the thread's 15 stage-1 twiddles in registers (tw1[k-1] = w_1[k][lo]); used by
// kernels with registers to spare, it takes those reads off the shared-memory path.
struct CtaSync {
  static constexpr bool REG_TW1 = false;
  __device__ __forceinline__ void sync() const { __syncthreads(); }
  __device__ __forceinline__ void acquire() const {}
  __device__ __forceinline__ void release() const {}
};
template <int N, typename Sy>
__device__ __forceinline__ void sync_last_p(const Sy& sy) {
  if (Plan<N>::NS == 3) __syncwarp();
  else sy.sync();
}

// stage-1 twiddles from registers (see REG_TW1)
template <int D>
__device__ __forceinline__ void twiddle_reg(const double2* w, cplx* v, int flip) {
#pragma unroll
  for (int k = 1; k < 16; ++k) {
    double2 d = w[k - 1];
    if (k & 1) {
      d.x = flip_sign(d.x, flip);
      d.y = flip_sign(d.y, flip);
    }
    v[k] = (D < 0) ? cmul(v[k], mk(d.x, d.y)) : cmulc(v[k], mk(d.x, d.y));
  }
}
template <int N, int J, int D, typename Sy>
__device__ __forceinline__ void twiddle_p(const double2* tw, int t, cplx* v, int flip, const Sy& sy) {
  if constexpr (Sy::REG_TW1 && J == 1) twiddle_reg<D>(sy.tw1, v, flip);
  else twiddle<N, J, D>(tw, t, v, flip);
}

// one forward radix-16 stage J followed by the exchange into stage J+1's (or the last stage's) registers
template <int N, int J, typename Sy>
__device__ __forceinline__ void fwd_stages(double2* buf, const double2* tw, int t, int c, cplx* v, int flip,
                                           const Sy& sy) {
  if constexpr (J < Plan<N>::NS) {
    dft16<-1>(v);
    twiddle_p<N, J, -1>(tw, t, v, flip, sy);
    sy.acquire();
    sts_stage<N, J>(buf, t, c, v);
    if constexpr (J + 1 < Plan<N>::NS) {
      sy.sync();
      lds_stage<N, J + 1>(buf, t, c, v);
    } else {
      sync_last_p<N>(sy);
      lds_last<N>(buf, t, c, v);
    }
    sy.release();
    fwd_stages<N, J + 1>(buf, tw, t, c, v, flip, sy);
  }
}
template <int N, typename Sy = CtaSync>
__device__ __forceinline__ void line_fft_fwd(double2* buf, const double2* tw, int t, int c, cplx* v, int flip = 0,
                                             const Sy& sy = Sy()) {
  fwd_stages<N, 1>(buf, tw, t, c, v, flip, sy);
  dft_last<-1, Plan<N>::RL>(v);
}

struct NoHook {
  __device__ __forceinline__ void operator()() const {}
};
// hook() runs right after the last read of the line buffer (the loads of stage 1): from there on the buffer is
// free as soon as every warp has passed that point
template <int N, int J, typename Hook, typename Sy>
__device__ __forceinline__ void inv_stages(double2* buf, const double2* tw, int t, int c, cplx* v, int flip,
                                           const Hook& hook, const Sy& sy) {
  if constexpr (J >= 1) {
    sy.acquire();
    if constexpr (J + 1 < Plan<N>::NS) {
      sts_stage<N, J + 1>(buf, t, c, v);
      sy.sync();
    } else {
      sts_last<N>(buf, t, c, v);
      sync_last_p<N>(sy);
    }
    lds_stage<N, J>(buf, t, c, v);
    sy.release();
    if constexpr (J == 1) hook();
    twiddle_p<N, J, +1>(tw, t, v, flip, sy);
    dft16<+1>(v);
    inv_stages<N, J - 1>(buf, tw, t, c, v, flip, hook, sy);
  }
}
template <int N, typename Hook = NoHook, typename Sy = CtaSync>
__device__ __forceinline__ void line_fft_inv(double2* buf, const double2* tw, int t, int c, cplx* v, int flip = 0,
                                             const Hook& hook = Hook(), const Sy& sy = Sy()) {
  dft_last<+1, Plan<N>::RL>(v);
  inv_stages<N, Plan<N>::NS - 1>(buf, tw, t, c, v, flip, hook, sy);
}

}  // namespace spgpe
