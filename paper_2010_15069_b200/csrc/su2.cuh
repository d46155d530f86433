// su2.cuh -- per-point 2x2 exponential of the real-space half-step (include/spgpe.h: R(tau);
// paper Eqs. 6-8; closed SU(2) form of BASELINE.json north_star).
//
// H_loc = a 1 + b_x sigma_x + b_z sigma_z,  a = V + ca_u n_up + ca_d n_dn,  b_z = delta/2 + cb_u n_up + cb_d n_dn,
// b_x = Omega/2.  exp(-i tau H_loc) = e^{-i a tau} [C(z) 1 - i tau S(z) (b_x sigma_x + b_z sigma_z)], z = -theta^2,
// theta = |b| tau, with the entire functions C(z) = sum z^k/(2k)! (cos theta = C(-theta^2), cosh theta = C(theta^2))
// and S(z) = sum z^k/(2k+1)! (sin theta/theta, sinh theta/theta).  Imaginary time: e^{-a tau}[C(z) 1 - tau S(z)(b.sigma)],
// z = +theta^2.  Writing sin(theta)/|b| = tau S(z) needs no square root, no division and no |b| -> 0 special case.
//
// Evaluation tiers:
//   |z| <= 2^-20 : series to degree 2 (first dropped term z^3/6! < 1.3e-21)
//   |z| <= 2^-13 : series to degree 3 (first dropped term z^4/8! < 6e-21)
//   |z| <= 1/4   : series to degree 7 (first dropped term z^8/16! < 8e-19)
//   otherwise    : libm sincos / cosh / sinh
// The tier is chosen once per warp and row from rigorous bounds on |z| (pass_x.cuh), so the per-point code is
// straight-line.
#pragma once
#include "common.cuh"

namespace spgpe {

struct HalfCoef {
  double ca_u, ca_d, cb_u, cb_d;  // (g_uu+g_ud)/2, (g_dd+g_ud)/2, (g_uu-g_ud)/2, (g_ud-g_dd)/2
};

#define SPGPE_Z_MICRO 9.5367431640625e-07
#define SPGPE_Z_TINY 0.0001220703125
#define SPGPE_Z_FAST 0.25

// C(z), S(z) to degree 2
__device__ __forceinline__ void cs_series2(double z, double& C, double& S) {
  const double c = fma(z, 1.0 / 24.0, 0.5);
  const double s = fma(z, 1.0 / 120.0, 1.0 / 6.0);
  C = fma(c, z, 1.0);
  S = fma(s, z, 1.0);
}

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

// general argument: z = -theta^2 (real time, IMAG = false) or +theta^2 (imaginary time); returns (C, S)
template <bool IMAG>
__device__ __noinline__ double2 cs_general(double z) {
  double C, S;
  const double th = sqrt(fabs(z));
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
  return make_double2(C, S);
}

// TIER 0: |z| <= SPGPE_Z_MICRO guaranteed by the caller; 1: |z| <= SPGPE_Z_TINY; 2: |z| <= SPGPE_Z_FAST; 3: anything
template <bool IMAG, int TIER>
__device__ __forceinline__ void cs_eval(double z, double& C, double& S) {
  if (TIER == 0) {
    cs_series2(z, C, S);
  } else if (TIER == 1) {
    cs_series3(z, C, S);
  } else if (TIER == 2) {
    cs_series7(z, C, S);
  } else {
    const double2 r = cs_general<IMAG>(z);
    C = r.x;
    S = r.y;
  }
}

// e^{-i x} = (cos x, -sin x); TIER 0-2: x^2 <= SPGPE_Z_FAST guaranteed by the caller (series to degree 7)
static __device__ __noinline__ double2 phase_general(double x) {
  double sn, cn;
  sincos(x, &sn, &cn);
  return make_double2(cn, -sn);
}
template <int TIER>
__device__ __forceinline__ void phase_eval(double x, double& pr, double& pi) {
  if (TIER == 3) {
    const double2 r = phase_general(x);
    pr = r.x;
    pi = r.y;
  } else {
    double C, S;
    cs_series7(-(x * x), C, S);
    pr = C;
    pi = -(x * S);
  }
}

// Per-lane form of the local Hamiltonian.  A lane holds "its" component m (up for the even lane of a pair, down
// for the odd one) and receives the other component o.  In the basis (m, o) the matrix keeps its form with
//   a  = V + cam |m|^2 + cao |o|^2,   b_z = hDs + cbm |m|^2 + cbo |o|^2,   b_x = hO,
// (even lane: cam = ca_u, cao = ca_d, cbm = cb_u, cbo = cb_d, hDs = +delta/2; odd lane: cam = ca_d, cao = ca_u,
// cbm = -cb_d, cbo = -cb_u, hDs = -delta/2, because sigma_z changes sign when the basis order is swapped), so
// no lane ever has to sort (m, o) into (up, down).
struct LaneCoef {
  double cam, cao, cbm, cbo;
  double hs;  // +0.5 or -0.5: factor that turns delta into hDs
};
__device__ __forceinline__ LaneCoef lane_coef(const HalfCoef& hc, int c) {
  LaneCoef l;
  l.cam = c ? hc.ca_d : hc.ca_u;
  l.cao = c ? hc.ca_u : hc.ca_d;
  l.cbm = c ? -hc.cb_d : hc.cb_u;
  l.cbo = c ? -hc.cb_u : hc.cb_d;
  l.hs = c ? -0.5 : 0.5;
  return l;
}

// Apply the traceless part M = C 1 - (i) tau S (b.sigma) to (m, o) with the densities of (m, o); returns a (the
// scalar part of H_loc) so that the caller applies e^{-i a tau} / e^{-a tau}.
// BZ0: g_uu = g_dd = g_ud, so b_z carries no density term (cbm = cbo = 0).
template <bool IMAG, int TIER, bool BZ0>
__device__ __forceinline__ double su2_apply(cplx& m, cplx& o, double V, double hO, double hDs, double tau,
                                            double tau2, const LaneCoef& lc) {
  const double nm = fma(m.re, m.re, m.im * m.im);
  const double no = fma(o.re, o.re, o.im * o.im);
  const double a = fma(lc.cam, nm, fma(lc.cao, no, V));
  const double bz = BZ0 ? hDs : fma(lc.cbm, nm, fma(lc.cbo, no, hDs));
  const double th2 = tau2 * fma(hO, hO, bz * bz);
  double C, S;
  cs_eval<IMAG, TIER>(IMAG ? th2 : -th2, C, S);
  const double ts = tau * S;
  const double sx = ts * hO, sz = ts * bz;
  // w_m = sz m + sx o,  w_o = sx m - sz o
  const cplx wm = mk(fma(sz, m.re, sx * o.re), fma(sz, m.im, sx * o.im));
  const cplx wo = mk(fma(sx, m.re, -(sz * o.re)), fma(sx, m.im, -(sz * o.im)));
  if (IMAG) {
    m = mk(fma(C, m.re, -wm.re), fma(C, m.im, -wm.im));
    o = mk(fma(C, o.re, -wo.re), fma(C, o.im, -wo.im));
  } else {  // -i w = (w.im, -w.re)
    m = mk(fma(C, m.re, wm.im), fma(C, m.im, -wm.re));
    o = mk(fma(C, o.re, wo.im), fma(C, o.im, -wo.re));
  }
  return a;
}

__device__ __forceinline__ void apply_phase(cplx& up, cplx& dn, double pr, double pi) {
  up = cmul(up, mk(pr, pi));
  dn = cmul(dn, mk(pr, pi));
}

// ---- nested second-order split of the real-space part (R-15) -----------
//   R_nested(tau) = D(tau/2) X(tau) D(tau/2),
// D(s): psi_c <- e^{-i s d_c} psi_c with d_m = a + b_z, d_o = a - b_z in the lane's (mine, other) basis (a, b_z as in
// LaneCoef above, densities of the psi that enters D); X(s) = exp(-i s (Omega/2) sigma_x).  Imaginary time: e^{-s d_c},
// cosh / sinh.  FAST: every phase argument x of the warp satisfies x^2 <= SPGPE_Z_FAST (series), else libm.
template <bool IMAG, bool FAST>
__device__ __forceinline__ void nested_diag(cplx& m, cplx& o, double V, double hDs, double s, const LaneCoef& lc) {
  const double nm = fma(m.re, m.re, m.im * m.im);
  const double no = fma(o.re, o.re, o.im * o.im);
  const double a = fma(lc.cam, nm, fma(lc.cao, no, V));
  const double bz = fma(lc.cbm, nm, fma(lc.cbo, no, hDs));
  const double dm = a + bz, dn = a - bz;
  if (IMAG) {
    const double em = exp(-dm * s), eo = exp(-dn * s);
    m = mk(m.re * em, m.im * em);
    o = mk(o.re * eo, o.im * eo);
  } else {
    double pr, pi;
    phase_eval<FAST ? 2 : 3>(dm * s, pr, pi);
    m = cmul(m, mk(pr, pi));
    phase_eval<FAST ? 2 : 3>(dn * s, pr, pi);
    o = cmul(o, mk(pr, pi));
  }
}
template <bool IMAG, bool FAST>
__device__ __forceinline__ void nested_rot(cplx& m, cplx& o, double hO, double s) {
  const double th = hO * s;
  double C, S;
  cs_eval<IMAG, FAST ? 2 : 3>(IMAG ? th * th : -(th * th), C, S);
  const double sn = th * S;  // sin(th) or sinh(th)
  const cplx m0 = m;
  if (IMAG) {
    m = mk(fma(C, m.re, -(sn * o.re)), fma(C, m.im, -(sn * o.im)));
    o = mk(fma(C, o.re, -(sn * m0.re)), fma(C, o.im, -(sn * m0.im)));
  } else {  // -i sn (x + i y) = sn y - i sn x
    m = mk(fma(C, m.re, sn * o.im), fma(C, m.im, -(sn * o.re)));
    o = mk(fma(C, o.re, sn * m0.im), fma(C, o.im, -(sn * m0.re)));
  }
}

}  // namespace spgpe
