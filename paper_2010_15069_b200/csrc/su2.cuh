// su2.cuh -- per-point 2x2 exponential of the real-space half-step (include/spgpe.h: R(tau);
// paper Eqs. 6-8; closed SU(2) form of BASELINE.json north_star).
//
// H_loc = a 1 + b_x sigma_x + b_z sigma_z,  a = V + ca_u n_up + ca_d n_dn,  b_z = delta/2 + cb_u n_up + cb_d n_dn,
// b_x = Omega/2.  exp(-i tau H_loc) = e^{-i a tau} [C(z) 1 - i tau S(z) (b_x sigma_x + b_z sigma_z)], z = -theta^2,
// theta = |b| tau, with the entire functions C(z) = sum z^k/(2k)! (cos theta = C(-theta^2), cosh theta = C(theta^2))
// and S(z) = sum z^k/(2k+1)! (sin theta/theta, sinh theta/theta).  Imaginary time: e^{-a tau}[C(z) 1 - tau S(z)(b.sigma)],
// z = +theta^2.  Writing sin(theta)/|b| = tau S(z) needs no square root, no division and no |b| -> 0 special case.
//
// Evaluation tiers (the choice is warp-uniform, so there is no divergence):
//   |z| <= 2^-13 : series to degree 3 (first dropped term z^4/8! < 6e-21)
//   |z| <= 1/4   : series to degree 7 (first dropped term z^8/16! < 8e-19)
//   otherwise    : libm sincos / cosh / sinh
#pragma once
#include "common.cuh"

namespace spgpe {

struct HalfCoef {
  double ca_u, ca_d, cb_u, cb_d;  // (g_uu+g_ud)/2, (g_dd+g_ud)/2, (g_uu-g_ud)/2, (g_ud-g_dd)/2
};

#define SPGPE_Z_TINY 0.0001220703125
#define SPGPE_Z_FAST 0.25

// C(z), S(z) to degree 3
__device__ __forceinline__ void cs_series3(double z, double& C, double& S) {
  double c = fma(z, 1.0 / 720.0, 1.0 / 24.0);
  double s = fma(z, 1.0 / 5040.0, 1.0 / 120.0);
  c = fma(c, z, 0.5);
  s = fma(s, z, 1.0 / 6.0);
  C = fma(c, z, 1.0);
  S = fma(s, z, 1.0);
}

// C(z), S(z) to degree 7
__device__ __forceinline__ void cs_series7(double z, double& C, double& S) {
  double c = fma(z, 1.0 / 87178291200.0, 1.0 / 479001600.0);   // 1/14!, 1/12!
  double s = fma(z, 1.0 / 1307674368000.0, 1.0 / 6227020800.0);  // 1/15!, 1/13!
  c = fma(c, z, 1.0 / 3628800.0);    // 1/10!
  s = fma(s, z, 1.0 / 39916800.0);   // 1/11!
  c = fma(c, z, 1.0 / 40320.0);      // 1/8!
  s = fma(s, z, 1.0 / 362880.0);     // 1/9!
  c = fma(c, z, 1.0 / 720.0);        // 1/6!
  s = fma(s, z, 1.0 / 5040.0);       // 1/7!
  c = fma(c, z, 1.0 / 24.0);
  s = fma(s, z, 1.0 / 120.0);
  c = fma(c, z, 0.5);
  s = fma(s, z, 1.0 / 6.0);
  C = fma(c, z, 1.0);
  S = fma(s, z, 1.0);
}

// general argument: z = -theta^2 (real time, IMAG = false) or +theta^2 (imaginary time)
template <bool IMAG>
__device__ __noinline__ void cs_general(double z, double& C, double& S) {
  double th = sqrt(fabs(z));
  if (fabs(z) <= SPGPE_Z_FAST) {
    cs_series7(z, C, S);
  } else if (!IMAG) {
    double sn, cn;
    sincos(th, &sn, &cn);
    C = cn;
    S = sn / th;
  } else {
    C = cosh(th);
    S = sinh(th) / th;
  }
}

// tier of a warp: 0 tiny, 1 fast, 2 general (the largest |z| among the lanes decides)
__device__ __forceinline__ int cs_tier(double absz) {
  if (!__any_sync(0xffffffffu, absz > SPGPE_Z_TINY)) return 0;
  if (!__any_sync(0xffffffffu, absz > SPGPE_Z_FAST)) return 1;
  return 2;
}

template <bool IMAG>
__device__ __forceinline__ void cs_eval(double z, double& C, double& S) {
  const int tier = cs_tier(fabs(z));
  if (tier == 0) cs_series3(z, C, S);
  else if (tier == 1) cs_series7(z, C, S);
  else cs_general<IMAG>(z, C, S);
}

// e^{-i x}: (cos x, -sin x)
static __device__ __noinline__ void phase_general(double x, double& pr, double& pi) {
  double sn, cn;
  sincos(x, &sn, &cn);
  pr = cn;
  pi = -sn;
}
__device__ __forceinline__ void phase_eval(double x, double& pr, double& pi) {
  const double z = -(x * x);
  const int tier = cs_tier(-z);
  if (tier == 2) {
    phase_general(x, pr, pi);
  } else {
    double C, S;
    if (tier == 0) cs_series3(z, C, S);
    else cs_series7(z, C, S);
    pr = C;
    pi = -(x * S);
  }
}

// Apply the traceless part M = C 1 - (i) tau S (b.sigma) to (up, dn) with the densities of (up, dn);
// returns a (the scalar part of H_loc) so that the caller applies e^{-i a tau} / e^{-a tau}.
// hOm = Omega/2 and hDe = delta/2 are passed halved.
template <bool IMAG>
__device__ __forceinline__ double su2_apply(cplx& up, cplx& dn, double V, double hOm, double hDe, double tau,
                                            double tau2, const HalfCoef& hc) {
  const double nu = fma(up.re, up.re, up.im * up.im);
  const double nd = fma(dn.re, dn.re, dn.im * dn.im);
  const double a = fma(hc.ca_u, nu, fma(hc.ca_d, nd, V));
  const double bz = fma(hc.cb_u, nu, fma(hc.cb_d, nd, hDe));
  const double bx = hOm;
  const double th2 = tau2 * fma(bx, bx, bz * bz);
  double C, S;
  cs_eval<IMAG>(IMAG ? th2 : -th2, C, S);
  const double ts = tau * S;
  const double sx = ts * bx, sz = ts * bz;
  // w_up = sz up + sx dn,  w_dn = sx up - sz dn
  const cplx wu = mk(fma(sz, up.re, sx * dn.re), fma(sz, up.im, sx * dn.im));
  const cplx wd = mk(fma(sx, up.re, -(sz * dn.re)), fma(sx, up.im, -(sz * dn.im)));
  if (IMAG) {
    up = mk(fma(C, up.re, -wu.re), fma(C, up.im, -wu.im));
    dn = mk(fma(C, dn.re, -wd.re), fma(C, dn.im, -wd.im));
  } else {  // -i w = (w.im, -w.re)
    up = mk(fma(C, up.re, wu.im), fma(C, up.im, -wu.re));
    dn = mk(fma(C, dn.re, wd.im), fma(C, dn.im, -wd.re));
  }
  return a;
}

__device__ __forceinline__ void apply_phase(cplx& up, cplx& dn, double pr, double pi) {
  up = cmul(up, mk(pr, pi));
  dn = cmul(dn, mk(pr, pi));
}

}  // namespace spgpe
