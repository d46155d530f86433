// pass_x.cuh -- the row pass: x-direction transforms fused with the real-space half-steps
// (SURVEY.md 8(a) rows a1, a2/a4 (x part), a5, a6; include/spgpe.h).
//
// One CTA handles LINES rows; a team of 2*T threads (T = NX/16) owns one row, thread (t, c) holding 16 points of
// component c.  Lane pairs (c = 0, 1) sit next to each other so that a pair reads/writes one 32-byte point.
//
//   MODE_PRO : psi(x) -> [scale] -> R(tau) -> F_x -> * ex_c(k_x) -> psi^(k_x)          (first half of a step)
//   MODE_MID : psi^(k_x) -> F_x^-1 -> R(tau) R(tau) -> F_x -> * ex_c(k_x) -> psi^(k_x)  (real time, steps n | n+1)
//   MODE_EPI : psi^(k_x) -> F_x^-1 -> R(tau) -> [norm partials] -> psi(x)              (second half of a step)
//   MODE_FWD : src psi(x) -> F_x -> dst psi^(k_x)                                      (energy only)
// The two half-steps of MODE_MID are two evaluations with refreshed densities (R-6); only their scalar phases
// e^{-i a1 tau} e^{-i a2 tau} are merged into one (unit-modulus phases do not change densities).
#pragma once
#include "line_fft.cuh"
#include "su2.cuh"

namespace spgpe {

enum { MODE_PRO = 0, MODE_MID = 1, MODE_EPI = 2, MODE_FWD = 3 };

struct PassXArgs {
  const void* src;       // psi in   [ny][NX][2]
  void* dst;             // psi out (== src for in-place)
  const void* V;         // fields [ny][NX] or NULL
  const void* Om;
  const void* De;
  const double2* tw;     // twiddles of NX
  const double2* exk;    // [2][NX] k_x phase in stored order (MODE_PRO, MODE_MID)
  const double* scale;   // [2] per-component factor applied at load (MODE_PRO, imaginary time) or NULL
  double* partial;       // [gridDim.x][2] sum |psi_c|^2 of this CTA (MODE_EPI with want_norm)
  double tau;            // half-step size dt/2
  HalfCoef hc;
  int imag;
  int want_norm;
};

__device__ __forceinline__ double shfl_xor_d(double x, int m) { return __shfl_xor_sync(0xffffffffu, x, m); }
__device__ __forceinline__ cplx shfl_xor_c(cplx a, int m) { return mk(shfl_xor_d(a.re, m), shfl_xor_d(a.im, m)); }

// Real-space part on the thread's registers v[n] = psi_c(x = t + n*T).  Pair exchange: the c=0 thread takes both
// components of the points n = 0..7, the c=1 thread those of n = 8..15.
template <int DT, int NX, int MODE>
__device__ __forceinline__ void real_space(cplx* v, const PassXArgs& a, size_t rowbase, int t, int c,
                                           double& su, double& sd) {
  typedef Store<DT> St;
  constexpr int T = NX / 16;
  // fields of the thread's 8 points, fetched one point ahead of their use (the loads of point i+1 are in
  // flight while point i is being evaluated)
  const size_t x0 = rowbase + t + (8 * c) * T;
  double Vn = a.V ? St::ldr(a.V, x0) : 0.0;
  double On = a.Om ? St::ldr(a.Om, x0) : 0.0;
  double Dn = a.De ? St::ldr(a.De, x0) : 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    // send what the partner needs, receive the partner's component at my points
    cplx mine = c ? v[8 + i] : v[i];
    cplx send = c ? v[i] : v[8 + i];
    cplx recv = shfl_xor_c(send, 1);
    cplx up = c ? recv : mine;
    cplx dn = c ? mine : recv;
    const double Vv = Vn, Ov = On, Dv = Dn;
    if (i < 7) {
      const size_t x = x0 + (i + 1) * T;
      Vn = a.V ? St::ldr(a.V, x) : 0.0;
      On = a.Om ? St::ldr(a.Om, x) : 0.0;
      Dn = a.De ? St::ldr(a.De, x) : 0.0;
    }
    if (MODE == MODE_MID) {
      double a1 = su2_apply<false>(up, dn, Vv, Ov, Dv, a.tau, a.hc);
      double a2 = su2_apply<false>(up, dn, Vv, Ov, Dv, a.tau, a.hc);
      double pr, pi;
      phase_eval((a1 + a2) * a.tau, pr, pi);
      apply_phase(up, dn, pr, pi);
    } else if (a.imag) {
      double a1 = su2_apply<true>(up, dn, Vv, Ov, Dv, a.tau, a.hc);
      double e = exp(-a1 * a.tau);
      up = mk(up.re * e, up.im * e);
      dn = mk(dn.re * e, dn.im * e);
    } else {
      double a1 = su2_apply<false>(up, dn, Vv, Ov, Dv, a.tau, a.hc);
      double pr, pi;
      phase_eval(a1 * a.tau, pr, pi);
      apply_phase(up, dn, pr, pi);
    }
    if (MODE == MODE_EPI) {
      su += fma(up.re, up.re, up.im * up.im);
      sd += fma(dn.re, dn.re, dn.im * dn.im);
    }
    // give the partner its component back
    cplx keep = c ? dn : up;
    cplx back = shfl_xor_c(c ? up : dn, 1);
    if (c) { v[8 + i] = keep; v[i] = back; }
    else   { v[i] = keep; v[8 + i] = back; }
  }
}

template <int DT, int NX, int LINES, int MODE>
__global__ void __launch_bounds__(LINES * (NX / 8), (LINES * (NX / 8) <= 256) ? 2 : 1)
pass_x_kernel(const PassXArgs a) {
  typedef Plan<NX> P;
  typedef Store<DT> St;
  extern __shared__ double2 smem[];
  constexpr int T = P::T;
  const int tid = threadIdx.x;
  const int c = tid & 1;
  const int t = (tid >> 1) % T;
  const int line = (tid >> 1) / T;
  double2* buf = smem + (size_t)line * (P::PTS * 2);
  const size_t row = (size_t)blockIdx.x * LINES + line;
  const size_t rowbase = row * NX;  // in points
  cplx v[16];

  if (MODE == MODE_PRO || MODE == MODE_FWD) {
#pragma unroll
    for (int n = 0; n < 16; ++n) v[n] = St::ld(a.src, (rowbase + t + n * T) * 2 + c);
    if (MODE == MODE_PRO && a.scale != nullptr) {
      const double s = a.scale[c];
#pragma unroll
      for (int n = 0; n < 16; ++n) v[n] = mk(v[n].re * s, v[n].im * s);
    }
  } else {
#pragma unroll
    for (int g = 0; g < P::G; ++g)
#pragma unroll
      for (int s = 0; s < P::RL; ++s)
        v[g * P::RL + s] = St::ld(a.src, (rowbase + (t + g * T) + (NX / P::RL) * s) * 2 + c);
    line_fft_inv<NX>(buf, a.tw, t, c, v);
  }

  double su = 0.0, sd = 0.0;
  if (MODE != MODE_FWD) real_space<DT, NX, MODE>(v, a, rowbase, t, c, su, sd);

  if (MODE == MODE_EPI) {
#pragma unroll
    for (int n = 0; n < 16; ++n) St::st(a.dst, (rowbase + t + n * T) * 2 + c, v[n]);
    if (a.want_norm) {
      // the c=0 thread of a pair summed points n<8, the c=1 thread n>=8: add over the whole CTA
      __shared__ double red[2][32];
#pragma unroll
      for (int m = 16; m >= 1; m >>= 1) {
        su += shfl_xor_d(su, m);
        sd += shfl_xor_d(sd, m);
      }
      const int w = tid >> 5, nw = (blockDim.x + 31) >> 5;
      if ((tid & 31) == 0) { red[0][w] = su; red[1][w] = sd; }
      __syncthreads();
      if (tid == 0) {
        double s0 = 0.0, s1 = 0.0;
        for (int i = 0; i < nw; ++i) { s0 += red[0][i]; s1 += red[1][i]; }
        a.partial[2 * blockIdx.x] = s0;
        a.partial[2 * blockIdx.x + 1] = s1;
      }
    }
  } else {
    line_fft_fwd<NX>(buf, a.tw, t, c, v);
#pragma unroll
    for (int g = 0; g < P::G; ++g)
#pragma unroll
      for (int s = 0; s < P::RL; ++s) {
        const int pos = (t + g * T) + (NX / P::RL) * s;
        cplx o = v[g * P::RL + s];
        if (MODE != MODE_FWD) {
          double2 e = __ldg(a.exk + c * NX + pos + late_zero(o.re));
          o = cmul(o, mk(e.x, e.y));
        }
        St::st(a.dst, (rowbase + pos) * 2 + c, o);
      }
  }
}

}  // namespace spgpe
