// fft32.cuh -- single-precision line transforms of the complex64 path (R-14): a thread holds 16 points of
// BOTH spin components (u[16], d[16]) in registers, radix-16 stages as in line_fft.cuh (same plans, same stored
// order, so the k-space tables and the two families of kernels are interchangeable), exchanged through shared memory
// as one float4 (up.re, up.im, dn.re, dn.im) per point.
//
// Precision.  Butterfly additions are fp32 (rounding errors without a preferred direction).  Every multiplication by
// a fixed factor -- the inter-stage twiddles, the constants of the radix-16 butterfly, the k-space phase factors --
// uses the factor as a two-float sum hi + lo (hi = fp32 rounding of the fp64 value, lo = fp32 rounding of the rest):
// rounding a fixed factor to fp32 once makes every step non-unitary by ~1e-7 in the same direction, which the
// nonlinear term turns into a wave-function error of 1e-4 ... 1e-3 after 2000 steps (measured
// again in round 2: 2.2e-3 with rounded twiddles against 4e-6 with exact ones).
#pragma once
#include "common.cuh"

namespace spgpe {

// One complex number of one component = one 64-bit register pair (re, im).  Arithmetic uses Blackwell's packed fp32
// instructions (FADD2 / FMUL2 / FFMA2 through __fadd2_rn / __fmul2_rn / __ffma2_rn): a complex addition is one
// instruction, a complex product with a scalar pair (w_re, w_im) two -- the hardware takes the swapped operand (im, re)
// with the sign pattern (-, +) and a broadcast scalar as operand modifiers (SASS `-R.F32x2.LO_HI.NP`, `R.F32`), and
// a multiplication by +-i folds into the next addition the same way.
struct __align__(8) cf {
  float re, im;
};
__device__ __forceinline__ cf mkf(float r, float i) { cf c; c.re = r; c.im = i; return c; }
__device__ __forceinline__ float2 f2(cf a) { return make_float2(a.re, a.im); }
__device__ __forceinline__ cf fc(float2 a) { return mkf(a.x, a.y); }
__device__ __forceinline__ float2 bc(float s) { return make_float2(s, s); }
#ifndef SPGPE_F32_SCALAR
__device__ __forceinline__ cf operator+(cf a, cf b) { return fc(__fadd2_rn(f2(a), f2(b))); }
__device__ __forceinline__ cf operator-(cf a, cf b) { return fc(__fadd2_rn(f2(a), make_float2(-b.re, -b.im))); }
template <int D>
__device__ __forceinline__ cf mul_if(cf a) { return D > 0 ? mkf(-a.im, a.re) : mkf(a.im, -a.re); }

// a * (hi + lo), real factor.  The small product first: added to an already rounded a * hi it would be rounded away
// again (it is below half an ulp), which leaves a systematic error of lo/hi -- measured as a norm loss of 3.4e-8 per
// application before this order was fixed.
__device__ __forceinline__ cf mul2(cf a, float hi, float lo) {
  return fc(__ffma2_rn(f2(a), bc(hi), __fmul2_rn(f2(a), bc(lo))));
}
// a * (w_hi + w_lo), w = (hr + lr) + i (hi + li): the small products first; four packed instructions
__device__ __forceinline__ cf cmul2(cf a, float hr, float hi, float lr, float li) {
  const float2 x = f2(a), xs = make_float2(a.im, a.re);
  float2 p = __fmul2_rn(x, bc(lr));
  p = __ffma2_rn(xs, make_float2(-li, li), p);
  p = __ffma2_rn(xs, make_float2(-hi, hi), p);
  p = __ffma2_rn(x, bc(hr), p);
  return fc(p);
}
#else  // diagnostic build: the same arithmetic with scalar fp32 instructions
__device__ __forceinline__ cf operator+(cf a, cf b) { return mkf(a.re + b.re, a.im + b.im); }
__device__ __forceinline__ cf operator-(cf a, cf b) { return mkf(a.re - b.re, a.im - b.im); }
template <int D>
__device__ __forceinline__ cf mul_if(cf a) { return D > 0 ? mkf(-a.im, a.re) : mkf(a.im, -a.re); }
__device__ __forceinline__ cf mul2(cf a, float hi, float lo) { return mkf(fmaf(a.re, hi, a.re * lo), fmaf(a.im, hi, a.im * lo)); }
__device__ __forceinline__ cf cmul2(cf a, float hr, float hi, float lr, float li) {
  float re = fmaf(a.re, lr, -(a.im * li));
  float im = fmaf(a.re, li, a.im * lr);
  re = fmaf(-a.im, hi, re);
  im = fmaf(a.im, hr, im);
  re = fmaf(a.re, hr, re);
  im = fmaf(a.re, hi, im);
  return mkf(re, im);
}
#endif
// a * conj(w)
__device__ __forceinline__ cf cmul2c(cf a, float hr, float hi, float lr, float li) {
  return cmul2(a, hr, -hi, lr, -li);
}

// two-float constants of the radix-16 butterfly
#define SPGPE_F_SQRT1_2_HI 0.707106769084930419921875f
#define SPGPE_F_SQRT1_2_LO 1.2101617485882343e-08f
#define SPGPE_F_COS_PI_8_HI 0.92387950420379638671875f
#define SPGPE_F_COS_PI_8_LO 2.830748968563057e-08f
#define SPGPE_F_SIN_PI_8_HI 0.3826834261417388916015625f
#define SPGPE_F_SIN_PI_8_LO 6.2233507236442165e-09f

template <int D>
__device__ __forceinline__ void dft4f(cf& a0, cf& a1, cf& a2, cf& a3) {
  cf s0 = a0 + a2, d0 = a0 - a2, s1 = a1 + a3, d1 = mul_if<D>(a1 - a3);
  a0 = s0 + s1;
  a2 = s0 - s1;
  a1 = d0 + d1;
  a3 = d0 - d1;
}

// multiply by exp(D * 2 pi i m / 16), m compile-time in [0, 16)
template <int D, int m>
__device__ __forceinline__ cf mul_w16f(cf a) {
  constexpr int q = m & 3;
  constexpr int quad = (m >> 2);
  cf r;
  if (q == 0) {
    r = a;
  } else if (q == 2) {  // (1 + D i)/sqrt2
    r = mul2(a + mul_if<D>(a), SPGPE_F_SQRT1_2_HI, SPGPE_F_SQRT1_2_LO);
  } else {
    constexpr float ch = (q == 1) ? SPGPE_F_COS_PI_8_HI : SPGPE_F_SIN_PI_8_HI;
    constexpr float cl = (q == 1) ? SPGPE_F_COS_PI_8_LO : SPGPE_F_SIN_PI_8_LO;
    constexpr float sh = D * ((q == 1) ? SPGPE_F_SIN_PI_8_HI : SPGPE_F_COS_PI_8_HI);
    constexpr float sl = D * ((q == 1) ? SPGPE_F_SIN_PI_8_LO : SPGPE_F_COS_PI_8_LO);
    r = cmul2(a, ch, sh, cl, sl);
  }
  if (quad == 1) r = mul_if<D>(r);
  if (quad == 2) r = mkf(-r.re, -r.im);
  if (quad == 3) r = mul_if<-D>(r);
  return r;
}

template <int D>
__device__ __forceinline__ void dft8f(cf* v) {
  cf e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
  cf o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
  dft4f<D>(e0, e1, e2, e3);
  dft4f<D>(o0, o1, o2, o3);
  o1 = mul_w16f<D, 2>(o1);
  o2 = mul_if<D>(o2);
  o3 = mul_w16f<D, 6>(o3);
  v[0] = e0 + o0; v[4] = e0 - o0;
  v[1] = e1 + o1; v[5] = e1 - o1;
  v[2] = e2 + o2; v[6] = e2 - o2;
  v[3] = e3 + o3; v[7] = e3 - o3;
}

template <int D>
__device__ __forceinline__ void dft16f(cf* v) {
  cf y[4][4];  // y[n2][k1]
#pragma unroll
  for (int n2 = 0; n2 < 4; ++n2) {
    y[n2][0] = v[n2];
    y[n2][1] = v[4 + n2];
    y[n2][2] = v[8 + n2];
    y[n2][3] = v[12 + n2];
    dft4f<D>(y[n2][0], y[n2][1], y[n2][2], y[n2][3]);
  }
  y[1][1] = mul_w16f<D, 1>(y[1][1]);
  y[1][2] = mul_w16f<D, 2>(y[1][2]);
  y[1][3] = mul_w16f<D, 3>(y[1][3]);
  y[2][1] = mul_w16f<D, 2>(y[2][1]);
  y[2][2] = mul_w16f<D, 4>(y[2][2]);
  y[2][3] = mul_w16f<D, 6>(y[2][3]);
  y[3][1] = mul_w16f<D, 3>(y[3][1]);
  y[3][2] = mul_w16f<D, 6>(y[3][2]);
  y[3][3] = mul_w16f<D, 9>(y[3][3]);
#pragma unroll
  for (int k1 = 0; k1 < 4; ++k1) {
    dft4f<D>(y[0][k1], y[1][k1], y[2][k1], y[3][k1]);
    v[k1] = y[0][k1];
    v[k1 + 4] = y[1][k1];
    v[k1 + 8] = y[2][k1];
    v[k1 + 12] = y[3][k1];
  }
}

template <int D, int R>
__device__ __forceinline__ void dft_lastf(cf* v) {
  if (R == 16) {
    dft16f<D>(v);
  } else if (R == 8) {
    dft8f<D>(v);
    dft8f<D>(v + 8);
  } else if (R == 4) {
#pragma unroll
    for (int g = 0; g < 4; ++g) dft4f<D>(v[4 * g], v[4 * g + 1], v[4 * g + 2], v[4 * g + 3]);
  } else {
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      cf s = v[2 * g] + v[2 * g + 1], d = v[2 * g] - v[2 * g + 1];
      v[2 * g] = s;
      v[2 * g + 1] = d;
    }
  }
}

// ---- positions (the formulas of line_fft.cuh; a thread index t here covers both components) ---------------------
// shared-memory slot (float4 units) of point p of a line
template <int N>
__device__ __forceinline__ int slot32(int p) {
  return p + (p >> Plan<N>::PADSHIFT);
}
// radix-16 stage J (1-based): register n <-> position hi*16*M + n*M + lo, t = hi*M + lo, M = N >> 4J
template <int N, int J>
__device__ __forceinline__ int stage_pos32(int t, int n) {
  constexpr int M = N >> (4 * J);
  const int lo = t & (M - 1);
  return ((t - lo) << 4) + lo + n * M;
}
// last stage: register g*RL + s <-> position (q0 + g*GSTEP)*RL + s
template <int N>
__device__ __forceinline__ int last_pos32(int t, int g, int s) {
  typedef Plan<N> P;
  const int q0 = (P::NS == 3) ? (t / P::RL) * 16 + (t % P::RL) : t;
  constexpr int GSTEP = (P::NS == 3) ? P::RL : P::T;
  return (q0 + g * GSTEP) * P::RL + s;
}
// stored position (index along the line in global memory) of register g*RL + s on the k-space side
template <int N>
__device__ __forceinline__ int stored_pos32(int t, int r) {
  typedef Plan<N> P;
  const int g = r / P::RL, s = r % P::RL;
  return (t + g * P::T) + (N / P::RL) * s;
}

__device__ __forceinline__ void sts4(float4* buf, int idx, cf u, cf d) { buf[idx] = make_float4(u.re, u.im, d.re, d.im); }
__device__ __forceinline__ void lds4(const float4* buf, int idx, cf& u, cf& d) {
  const float4 q = buf[idx];
  u = mkf(q.x, q.y);
  d = mkf(q.z, q.w);
}

// Exchange barrier.  Three-stage plans: the exchange in front of the last stage stays inside the RL threads that own
// one block of N/16 points; when those sit in one warp (LAST_WARP, decided by the kernel from its thread mapping) a
// __syncwarp is enough.  Every other exchange spans the line: LINE_WARP says that a whole line sits in one warp
// (two-stage plans).  For two-stage plans the only exchange is the line-wide one and LAST_WARP == LINE_WARP.
template <bool WARP_ONLY>
__device__ __forceinline__ void sync32() {
  if (WARP_ONLY) __syncwarp();
  else __syncthreads();
}

// twiddles of stage J: table entry (k-1)*M + lo = exp(-2 pi i k lo / (16 M)) as (hi.re, hi.im, lo.re, lo.im)
template <int N, int J, int D>
__device__ __forceinline__ void twiddle32(const float4* tw, int t, cf* u, cf* d) {
  constexpr int M = N >> (4 * J);
  const int lo = t & (M - 1);
  const float4* w = tw + tw_offset<N>(J) + lo;
#pragma unroll
  for (int k = 1; k < 16; ++k) {
    const float4 q = w[(k - 1) * M];
    if (D < 0) {
      u[k] = cmul2(u[k], q.x, q.y, q.z, q.w);
      d[k] = cmul2(d[k], q.x, q.y, q.z, q.w);
    } else {
      u[k] = cmul2c(u[k], q.x, q.y, q.z, q.w);
      d[k] = cmul2c(d[k], q.x, q.y, q.z, q.w);
    }
  }
}

// Forward transform of both components up to (not including) the last-stage butterflies: input register n = point
// t + n*T (natural order); on return the registers hold the last stage's inputs.  LINE_WARP: see sync32.
template <int N, int J, bool LINE_WARP, bool LAST_WARP>
__device__ __forceinline__ void fwd_stages32(float4* buf, const float4* tw, int t, cf* u, cf* d) {
  typedef Plan<N> P;
  if constexpr (J < P::NS) {
    dft16f<-1>(u);
    dft16f<-1>(d);
    twiddle32<N, J, -1>(tw, t, u, d);
#pragma unroll
    for (int n = 0; n < 16; ++n) sts4(buf, slot32<N>(stage_pos32<N, J>(t, n)), u[n], d[n]);
    if constexpr (J + 1 < P::NS) {
      sync32<LINE_WARP>();
#pragma unroll
      for (int n = 0; n < 16; ++n) lds4(buf, slot32<N>(stage_pos32<N, J + 1>(t, n)), u[n], d[n]);
    } else {
      sync32<LAST_WARP>();
#pragma unroll
      for (int g = 0; g < P::G; ++g)
#pragma unroll
        for (int s = 0; s < P::RL; ++s) lds4(buf, slot32<N>(last_pos32<N>(t, g, s)), u[g * P::RL + s], d[g * P::RL + s]);
    }
    fwd_stages32<N, J + 1, LINE_WARP, LAST_WARP>(buf, tw, t, u, d);
  }
}
template <int N, bool LINE_WARP, bool LAST_WARP>
__device__ __forceinline__ void line_fwd32(float4* buf, const float4* tw, int t, cf* u, cf* d) {
  fwd_stages32<N, 1, LINE_WARP, LAST_WARP>(buf, tw, t, u, d);
  dft_lastf<-1, Plan<N>::RL>(u);
  dft_lastf<-1, Plan<N>::RL>(d);
}

// Inverse transform (unnormalised), the mirror image.  hook() runs right after the last read of the line buffer.
template <int N, int J, bool LINE_WARP, bool LAST_WARP, typename Hook>
__device__ __forceinline__ void inv_stages32(float4* buf, const float4* tw, int t, cf* u, cf* d, const Hook& hook) {
  typedef Plan<N> P;
  if constexpr (J >= 1) {
    if constexpr (J + 1 < P::NS) {
#pragma unroll
      for (int n = 0; n < 16; ++n) sts4(buf, slot32<N>(stage_pos32<N, J + 1>(t, n)), u[n], d[n]);
      sync32<LINE_WARP>();
    } else {
#pragma unroll
      for (int g = 0; g < P::G; ++g)
#pragma unroll
        for (int s = 0; s < P::RL; ++s) sts4(buf, slot32<N>(last_pos32<N>(t, g, s)), u[g * P::RL + s], d[g * P::RL + s]);
      sync32<LAST_WARP>();
    }
#pragma unroll
    for (int n = 0; n < 16; ++n) lds4(buf, slot32<N>(stage_pos32<N, J>(t, n)), u[n], d[n]);
    if constexpr (J == 1) hook();
    twiddle32<N, J, +1>(tw, t, u, d);
    dft16f<+1>(u);
    dft16f<+1>(d);
    inv_stages32<N, J - 1, LINE_WARP, LAST_WARP>(buf, tw, t, u, d, hook);
  }
}
template <int N, bool LINE_WARP, bool LAST_WARP, typename Hook>
__device__ __forceinline__ void line_inv32(float4* buf, const float4* tw, int t, cf* u, cf* d, const Hook& hook) {
  dft_lastf<+1, Plan<N>::RL>(u);
  dft_lastf<+1, Plan<N>::RL>(d);
  inv_stages32<N, Plan<N>::NS - 1, LINE_WARP, LAST_WARP>(buf, tw, t, u, d, hook);
}

}  // namespace spgpe
