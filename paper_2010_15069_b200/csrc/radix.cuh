// radix.cuh -- small DFTs in registers.  dftR<D>(v): v[k] <- sum_n v[n] exp(D * 2 pi i n k / R),
// D = -1 forward, +1 inverse (unnormalised), natural order in and out.  All indices are compile-time
// so every array lives in registers.
#pragma once
#include "common.cuh"

namespace spgpe {

#define SPGPE_SQRT1_2 0.70710678118654752440
#define SPGPE_COS_PI_8 0.92387953251128675613
#define SPGPE_SIN_PI_8 0.38268343236508977173

template <int D>
__device__ __forceinline__ void dft2(cplx& a0, cplx& a1) {
  cplx s = a0 + a1, d = a0 - a1;
  a0 = s;
  a1 = d;
}

template <int D>
__device__ __forceinline__ void dft4(cplx& a0, cplx& a1, cplx& a2, cplx& a3) {
  cplx s0 = a0 + a2, d0 = a0 - a2, s1 = a1 + a3, d1 = mul_i<D>(a1 - a3);
  a0 = s0 + s1;
  a2 = s0 - s1;
  a1 = d0 + d1;
  a3 = d0 - d1;
}

// multiply by exp(D * 2 pi i m / 16), m compile-time in [0, 16)
template <int D, int m>
__device__ __forceinline__ cplx mul_w16(cplx a) {
  constexpr int q = m & 3;        // position inside the quadrant
  constexpr int quad = (m >> 2);  // multiples of i^D
  cplx r;
  if (q == 0) {
    r = a;
  } else if (q == 2) {  // (1 + D i)/sqrt2
    r = mk(SPGPE_SQRT1_2 * (a.re - D * a.im), SPGPE_SQRT1_2 * (a.im + D * a.re));
  } else {
    constexpr double c = (q == 1) ? SPGPE_COS_PI_8 : SPGPE_SIN_PI_8;
    constexpr double s = D * ((q == 1) ? SPGPE_SIN_PI_8 : SPGPE_COS_PI_8);
    r = mk(fma(c, a.re, -(s * a.im)), fma(c, a.im, s * a.re));
  }
  if (quad == 1) r = mul_i<D>(r);
  if (quad == 2) r = mk(-r.re, -r.im);
  if (quad == 3) r = mul_i<-D>(r);
  return r;
}

template <int D>
__device__ __forceinline__ void dft8(cplx* v) {
  // even / odd split: X[k] = E[k] + W8^k O[k], X[k+4] = E[k] - W8^k O[k]
  cplx e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
  cplx o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
  dft4<D>(e0, e1, e2, e3);
  dft4<D>(o0, o1, o2, o3);
  o1 = mul_w16<D, 2>(o1);
  o2 = mul_i<D>(o2);
  o3 = mul_w16<D, 6>(o3);
  v[0] = e0 + o0; v[4] = e0 - o0;
  v[1] = e1 + o1; v[5] = e1 - o1;
  v[2] = e2 + o2; v[6] = e2 - o2;
  v[3] = e3 + o3; v[7] = e3 - o3;
}

template <int D>
__device__ __forceinline__ void dft16(cplx* v) {
  // n = 4 n1 + n2, k = k1 + 4 k2:  X[k1 + 4 k2] = sum_n2 W16^(n2 k1) W4^(n2 k2) sum_n1 x[4 n1 + n2] W4^(n1 k1)
  cplx y[4][4];  // y[n2][k1]
#pragma unroll
  for (int n2 = 0; n2 < 4; ++n2) {
    y[n2][0] = v[n2];
    y[n2][1] = v[4 + n2];
    y[n2][2] = v[8 + n2];
    y[n2][3] = v[12 + n2];
    dft4<D>(y[n2][0], y[n2][1], y[n2][2], y[n2][3]);
  }
  y[1][1] = mul_w16<D, 1>(y[1][1]);
  y[1][2] = mul_w16<D, 2>(y[1][2]);
  y[1][3] = mul_w16<D, 3>(y[1][3]);
  y[2][1] = mul_w16<D, 2>(y[2][1]);
  y[2][2] = mul_w16<D, 4>(y[2][2]);
  y[2][3] = mul_w16<D, 6>(y[2][3]);
  y[3][1] = mul_w16<D, 3>(y[3][1]);
  y[3][2] = mul_w16<D, 6>(y[3][2]);
  y[3][3] = mul_w16<D, 9>(y[3][3]);
#pragma unroll
  for (int k1 = 0; k1 < 4; ++k1) {
    dft4<D>(y[0][k1], y[1][k1], y[2][k1], y[3][k1]);
    v[k1] = y[0][k1];
    v[k1 + 4] = y[1][k1];
    v[k1 + 8] = y[2][k1];
    v[k1 + 12] = y[3][k1];
  }
}

// last-stage butterflies: G = 16/R groups of R consecutive registers
template <int D, int R>
__device__ __forceinline__ void dft_last(cplx* v) {
  if (R == 16) {
    dft16<D>(v);
  } else if (R == 8) {
    dft8<D>(v);
    dft8<D>(v + 8);
  } else if (R == 4) {
#pragma unroll
    for (int g = 0; g < 4; ++g) dft4<D>(v[4 * g], v[4 * g + 1], v[4 * g + 2], v[4 * g + 3]);
  } else {
#pragma unroll
    for (int g = 0; g < 8; ++g) dft2<D>(v[2 * g], v[2 * g + 1]);
  }
}

}  // namespace spgpe
