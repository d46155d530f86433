// pass_x.cuh -- the row pass: x-direction transforms fused with the real-space half-steps
// (SURVEY.md 8(a) rows a1, a2/a4 (x part), a5, a6; include/spgpe.h).
//
// One CTA handles LINES rows; a team of 2*T threads (T = NX/16) owns one row, thread (t, c) holding 16 points of
// component c.  Lane pairs (c = 0, 1) sit next to each other so that a pair reads/writes one 32-byte point.
//
//   MODE_PRO : psi(x) -> [scale] -> R(tau) -> F_x -> psi^(k_x)                          (first half of a step)
//   MODE_MID : psi^(k_x) -> F_x^-1 -> R(tau) R(tau) -> F_x -> psi^(k_x)                  (real time, steps n | n+1)
//   MODE_EPI : psi^(k_x) -> F_x^-1 -> R(tau) -> [norm partials] -> psi(x)              (second half of a step)
//   MODE_EPI_OBS: MODE_EPI with the observables' partial sums
//   MODE_FWD : src psi(x) -> F_x -> dst psi^(k_x)                                      (energy only)
// The two half-steps of MODE_MID are two evaluations with refreshed densities (R-6); only their scalar phases
// e^{-i a1 tau} e^{-i a2 tau} are merged into one (unit-modulus phases do not change densities).  One exact exception:
// when g_uu = g_dd = g_ud the two half-steps are evaluated as one step of 2 tau (real_space_tier, BZ0).
#pragma once
#include "line_fft.cuh"
#include "su2.cuh"

namespace spgpe {

enum { MODE_PRO = 0, MODE_MID = 1, MODE_EPI = 2, MODE_FWD = 3, MODE_EPI_OBS = 4 };
// MODE_EPI_OBS: MODE_EPI that also sums rho_up^2, rho_dn^2, rho_up rho_dn (spgpe_step_observe); its own instantiation,
// so that the closing pass of every imaginary-time step keeps its register budget
__host__ __device__ constexpr bool mode_is_epi(int m) { return m == MODE_EPI || m == MODE_EPI_OBS; }

struct PassXArgs {
  const void* src;       // psi in   [ny][NX][2]
  void* dst;             // psi out (== src for in-place)
  const void* V;         // fields [ny][NX] or NULL
  const void* Om;
  const void* De;
  const double2* tw;     // twiddles of NX
  const float4* tw32;    // the same twiddles as two-float values (hi.re, hi.im, lo.re, lo.im): fp32 kernels, pass32.cuh
  const double* scale;   // [2] per-component factor applied at load (MODE_PRO, imaginary time) or NULL
  double* partial;       // [ny / LINES][pstride] sums of every row group (MODE_EPI with want_norm, MODE_EPI_OBS)
  double tau;            // half-step size dt/2
  HalfCoef hc;
  int imag;
  int want_norm;
  int ny;                // number of lines (rows x xs)
  int xs;                // 1: a line is a row; 2: a line is every second point of a row (split transform, api.cu)
  int* sched;            // [2] device: work counter (common.cuh, sched_next)
  const double* target;  // [2] device: norm targets (MODE_EPI with want_norm)
  double* scale_out;     // [2] device: rescale factors written by the last CTA (MODE_EPI with want_norm)
  double cell;           // dx dy
  int norm_mode;         // SPGPE_NORM_PER_COMPONENT | SPGPE_NORM_TOTAL
  const double* fmax;    // [3] device: max |V|, max |Omega|, max |delta| over the grid (tier bounds)
  int nest;              // 1: nested second-order split D(tau/2) X(tau) D(tau/2) of the real-space part (su2.cuh)
  int pstride;           // doubles per row group in `partial`: 2 (norms only) or 8 (MODE_EPI_OBS: five sums)
  // annealing (MODE_PRO): noise of event `anneal_event` (0: none) added to the order parameter at load
  long long anneal_event;
  unsigned long long anneal_seed;
  unsigned long long anneal_elems;  // 2 nx ny: elements per event
  double anneal_amp;
  int dbg;               // experiment switches (bit 0: psi rows by bulk copy, 1: field rows by per-thread cp.async instead of bulk copies, 2: early L2 prefetch)
};

// observables of the final state (MODE_EPI_OBS): sums of rho_m^2, rho_o^2, rho_m rho_o over the lane's points
struct ObsSums {
  double mm, oo, mo;
};

__device__ __forceinline__ double shfl_xor_d(double x, int m) { return __shfl_xor_sync(0xffffffffu, x, m); }
__device__ __forceinline__ cplx shfl_xor_c(cplx a, int m) { return mk(shfl_xor_d(a.re, m), shfl_xor_d(a.im, m)); }

// Annealing noise (include/spgpe.h spgpe_set_annealing): element e of event k uses the
// counter q = k * elems + e and the uniforms U(2q), U(2q+1) of the splitmix64 stream of `seed`,
//   U(j) = (mix64(seed + (j+1) * 0x9E3779B97F4A7C15) >> 11) * 2^-53,   xi = sqrt(-2 ln(1 - u1)) e^{2 pi i u2},
// and receives (amp / sqrt 2) xi.
__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
  z ^= z >> 27; z *= 0x94D049BB133111EBULL;
  z ^= z >> 31;
  return z;
}
__device__ __forceinline__ double stream_uniform(unsigned long long seed, unsigned long long j) {
  return (double)(mix64(seed + (j + 1ULL) * 0x9E3779B97F4A7C15ULL) >> 11) * (1.0 / 9007199254740992.0);
}
static __device__ __noinline__ cplx anneal_noise(const PassXArgs& a, unsigned long long elem) {
  const unsigned long long q = (unsigned long long)a.anneal_event * a.anneal_elems + elem;
  const double u1 = stream_uniform(a.anneal_seed, 2ULL * q), u2 = stream_uniform(a.anneal_seed, 2ULL * q + 1ULL);
  const double r = (a.anneal_amp * 0.70710678118654752440) * sqrt(-2.0 * log1p(-u1));
  double sn, cn;
  sincos(6.283185307179586476925286766559 * u2, &sn, &cn);
  return mk(r * cn, r * sn);
}

// Field rows in shared memory: [field][line][x] in working precision, with a gap of 64 bytes in the middle of every
// row.  The two lanes of a pair read different halves of the row (x = t + i T and x = t + (i + 8) T, T = NX/16): without
// the gap the halves are a multiple of 128 bytes apart and the two lanes of every pair hit the same banks (measured:
// every field read took twice its wavefronts, 1.2 M conflict wavefronts per launch at 2048^2, all of the row pass's
// bank conflicts); with it the second half sits 16 banks further and a warp's read is conflict-free.
template <int DT, int NX, int LINES>
struct FieldLayout {
  typedef typename Store<DT>::real real;
  static constexpr int GAP = 64 / (int)sizeof(real);                 // elements
  static constexpr int ROW = NX + GAP;                               // elements of a staged row
  static constexpr int FIELD = LINES * ROW;                          // elements of a staged field
  static constexpr int HALF_BYTES = (NX / 2) * (int)sizeof(real);    // bytes of half a row
  static constexpr int ROW_BYTES = NX * (int)sizeof(real);
  static __device__ __forceinline__ int at(int line, int x) { return line * ROW + x + (x >= NX / 2 ? GAP : 0); }
};

// Copy the three field rows of this CTA's LINES rows into shared memory (FieldLayout); a NULL field is filled with
// zeros.  Every thread of the CTA takes part.  Rows (XS == 1) are contiguous: thread 0 issues two bulk copies per field
// and row (the two halves; completion on `bar`, evict-first in L2: the fields are read once per pass and must not push
// the order parameter out); the strided lines of a split axis take one cp.async per real.
template <int DT, int NX, int LINES, int XS>
__device__ __forceinline__ void stage_fields(void* fbuf, const PassXArgs& a, size_t first_point, int first_line,
                                             int tid, unsigned long long* bar, bool fbulk) {
  typedef typename Store<DT>::real real;
  typedef FieldLayout<DT, NX, LINES> FL;
  constexpr int FIELD_BYTES = LINES * NX * (int)sizeof(real);   // bytes copied per field
  constexpr int NCH = FIELD_BYTES / 16;
  constexpr int PAD_BYTES = FL::FIELD * (int)sizeof(real);      // bytes a staged field occupies
  constexpr int NTHR = LINES * (NX / 8);
  const void* src[3] = {a.V, a.Om, a.De};
  auto zero_fill = [&](int f) {
    char* dst = reinterpret_cast<char*>(fbuf) + f * PAD_BYTES;
    for (int k = tid; k < PAD_BYTES / 16; k += NTHR) *reinterpret_cast<float4*>(dst + k * 16) = make_float4(0.f, 0.f, 0.f, 0.f);
  };
  if constexpr (XS != 1) {  // strided lines: one cp.async per real
    constexpr int S = XS;
#pragma unroll
    for (int f = 0; f < 3; ++f) {
      real* dst = reinterpret_cast<real*>(fbuf) + f * FL::FIELD;
      const real* g = reinterpret_cast<const real*>(src[f]);
      if (g == nullptr) { zero_fill(f); continue; }
      for (int k = tid; k < LINES * NX; k += NTHR) {
        const int l = k / NX, L = first_line + l, pos = k % NX;
        cp_async_real(dst + FL::at(l, pos), g + (size_t)(L / S) * NX * S + (size_t)pos * S + (L % S));
      }
    }
  } else if (!fbulk) {
#pragma unroll
    for (int f = 0; f < 3; ++f) {
      char* dst = reinterpret_cast<char*>(fbuf) + f * PAD_BYTES;
      if (src[f] != nullptr) {
        const char* g = reinterpret_cast<const char*>(src[f]) + first_point * sizeof(real);
#pragma unroll
        for (int k = tid; k < NCH; k += NTHR) {
          const int l = (k * 16) / FL::ROW_BYTES, off = (k * 16) % FL::ROW_BYTES;
          cp_async16(dst + l * (FL::ROW * (int)sizeof(real)) + off + (off >= FL::HALF_BYTES ? 64 : 0), g + k * 16);
        }
      } else {
        zero_fill(f);
      }
    }
  } else {
    if (tid == 0) {
      const unsigned long long policy = l2_policy_evict_first();
      const unsigned n = (src[0] != nullptr) + (src[1] != nullptr) + (src[2] != nullptr);
      fence_proxy_async();
      mbar_expect_tx(bar, n * (unsigned)FIELD_BYTES);  // n == 0: the phase completes at once
#pragma unroll
      for (int f = 0; f < 3; ++f)
        if (src[f] != nullptr) {
          const char* g = reinterpret_cast<const char*>(src[f]) + first_point * sizeof(real);
          char* dst = reinterpret_cast<char*>(fbuf) + f * PAD_BYTES;
#pragma unroll
          for (int l = 0; l < LINES; ++l)
#pragma unroll
            for (int hf = 0; hf < 2; ++hf)
              bulk_load_1d_hint(dst + l * (FL::ROW * (int)sizeof(real)) + hf * (FL::HALF_BYTES + 64),
                                g + l * FL::ROW_BYTES + hf * FL::HALF_BYTES, FL::HALF_BYTES, bar, policy);
        }
    }
#pragma unroll
    for (int f = 0; f < 3; ++f)
      if (src[f] == nullptr) zero_fill(f);
  }
}

// Real-space part.  Register layout on the natural-order side (see twiddle(), flip): the lane of component c at
// thread position t holds in v[i], i < 8, its component at "its" points x = t + (i + 8c) T and in v[8 + i] its
// component at the partner lane's points.  For point i a lane receives the partner's v[8 + i] (the other
// component at its own point), evaluates the half-step(s) in the (mine, other) basis (su2.cuh, LaneCoef) and
// sends the other component back.  Fields come from shared memory (stage_fields, FieldLayout).
// TIER: evaluation tier of su2.cuh, guaranteed by the caller for every point of the warp.
// TIME: 0 real time, 1 imaginary time (both known at compile time: the default kernels), 2 decided by a.imag at run time
template <int DT, int NX, int LINES, int MODE, int TIER, bool BZ0, int TIME>
__device__ __forceinline__ void real_space_tier(cplx* v, const PassXArgs& a, const void* fbuf, int line, int t, int c,
                                                const LaneCoef& lc, double& sm, double& so, ObsSums& ob) {
  typedef Store<DT> St;
  typedef typename St::real real;
  constexpr int T = NX / 16;
  typedef FieldLayout<DT, NX, LINES> FL;
  const real* fV = reinterpret_cast<const real*>(fbuf) + line * FL::ROW + t + c * (8 * T + FL::GAP);
  const real* fO = fV + FL::FIELD;
  const real* fD = fO + FL::FIELD;
  const double tau = a.tau, tau2 = a.tau * a.tau;
  // the other component of the lane's 8 points arrives first (one batch of shuffles), then the points are
  // evaluated without touching the shuffle / shared-memory path, then the other component goes back in one batch
  cplx o[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) o[i] = shfl_xor_c(v[8 + i], 1);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    cplx m = v[i];
    const double Vv = St::lds(fV, i * T);
    const double hO = 0.5 * St::lds(fO, i * T);
    const double hD = lc.hs * St::lds(fD, i * T);
    if (MODE == MODE_MID && BZ0) {
      // all g equal: the traceless part of H_loc holds no density and its scalar part only n_up + n_dn, which the
      // unitary half-step conserves, so R(tau) R(tau) = R(2 tau) exactly (one evaluation; differs from two by rounding)
      const double a1 = su2_apply<false, TIER, BZ0>(m, o[i], Vv, hO, hD, 2.0 * tau, 4.0 * tau2, lc);
      double pr, pi;
      phase_eval<TIER>(a1 * (2.0 * tau), pr, pi);
      apply_phase(m, o[i], pr, pi);
    } else if (MODE == MODE_MID) {
      const double a1 = su2_apply<false, TIER, BZ0>(m, o[i], Vv, hO, hD, tau, tau2, lc);
      const double a2 = su2_apply<false, TIER, BZ0>(m, o[i], Vv, hO, hD, tau, tau2, lc);
      double pr, pi;
      phase_eval<TIER>((a1 + a2) * tau, pr, pi);
      apply_phase(m, o[i], pr, pi);
    } else if (TIME == 2 ? (a.imag != 0) : (TIME == 1)) {
      const double a1 = su2_apply<true, TIER, BZ0>(m, o[i], Vv, hO, hD, tau, tau2, lc);
      const double e = exp(-a1 * tau);
      m = mk(m.re * e, m.im * e);
      o[i] = mk(o[i].re * e, o[i].im * e);
    } else {
      const double a1 = su2_apply<false, TIER, BZ0>(m, o[i], Vv, hO, hD, tau, tau2, lc);
      double pr, pi;
      phase_eval<TIER>(a1 * tau, pr, pi);
      apply_phase(m, o[i], pr, pi);
    }
    if (mode_is_epi(MODE)) {
      const double rm = fma(m.re, m.re, m.im * m.im), ro = fma(o[i].re, o[i].re, o[i].im * o[i].im);
      sm += rm;
      so += ro;
      if (MODE == MODE_EPI_OBS) { ob.mm = fma(rm, rm, ob.mm); ob.oo = fma(ro, ro, ob.oo); ob.mo = fma(rm, ro, ob.mo); }
    }
    v[i] = m;
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) v[8 + i] = shfl_xor_c(o[i], 1);
}

// Tier of the warp for this row, from bounds that hold for every point the warp touches:
//   n_up + n_dn <= NT = max_n |own v[n]|^2 + the partner's maximum (conserved by the real-time half-step),
//   |b_z| <= max|delta|/2 + max(|cbm|, |cbo|) NT,  |b_x| <= max|Omega|/2,  |a| <= max|V| + max(|cam|, |cao|) NT.
// merged: the two half-steps of MODE_MID are evaluated as one step of 2 tau (real_space_tier, BZ0)
template <int MODE>
__device__ __forceinline__ int row_tier(const cplx* v, const PassXArgs& a, const LaneCoef& lc, bool merged) {
  double nmax = 0.0;
#pragma unroll
  for (int n = 0; n < 16; ++n) nmax = fmax(nmax, fma(v[n].re, v[n].re, v[n].im * v[n].im));
  const double NT = nmax + shfl_xor_d(nmax, 1);
  const double bz = fma(fmax(fabs(lc.cbm), fabs(lc.cbo)), NT, 0.5 * a.fmax[2]);
  const double bx = 0.5 * a.fmax[1];
  const double z = (merged ? 4.0 : 1.0) * (a.tau * a.tau) * fma(bx, bx, bz * bz);
  const double x = (MODE == MODE_MID ? 2.0 : 1.0) * a.tau * fma(fmax(fabs(lc.cam), fabs(lc.cao)), NT, a.fmax[0]);
  const bool ph_ok = (x * x <= SPGPE_Z_FAST);
  const bool t0 = ph_ok && (z <= SPGPE_Z_MICRO);  // NaN fails every test and lands in the general tier
  const bool t1 = ph_ok && (z <= SPGPE_Z_TINY);
  const bool t2 = ph_ok && (z <= SPGPE_Z_FAST);
  if (__all_sync(0xffffffffu, t0)) return 0;
  if (__all_sync(0xffffffffu, t1)) return 1;
  if (__all_sync(0xffffffffu, t2)) return 2;
  return 3;
}

// Nested split (su2.cuh): MODE_MID runs D(tau/2) X(tau) D(tau) X(tau) D(tau/2): the trailing D(tau/2) of step n and the
// leading one of step n+1 see the same densities (a diagonal phase does not change them) and are one D(tau).
template <int DT, int NX, int LINES, int MODE, bool FAST>
__device__ __forceinline__ void real_space_nested(cplx* v, const PassXArgs& a, const void* fbuf, int line, int t, int c,
                                                  const LaneCoef& lc, double& sm, double& so, ObsSums& ob) {
  typedef Store<DT> St;
  typedef typename St::real real;
  constexpr int T = NX / 16;
  typedef FieldLayout<DT, NX, LINES> FL;
  const real* fV = reinterpret_cast<const real*>(fbuf) + line * FL::ROW + t + c * (8 * T + FL::GAP);
  const real* fO = fV + FL::FIELD;
  const real* fD = fO + FL::FIELD;
  const double tau = a.tau, th = 0.5 * a.tau;
  cplx o[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) o[i] = shfl_xor_c(v[8 + i], 1);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    cplx m = v[i], oo = o[i];
    const double Vv = St::lds(fV, i * T);
    const double hO = 0.5 * St::lds(fO, i * T);
    const double hD = lc.hs * St::lds(fD, i * T);
    if (a.imag) {
      nested_diag<true, FAST>(m, oo, Vv, hD, th, lc);
      nested_rot<true, FAST>(m, oo, hO, tau);
      nested_diag<true, FAST>(m, oo, Vv, hD, th, lc);
    } else {
      nested_diag<false, FAST>(m, oo, Vv, hD, th, lc);
      nested_rot<false, FAST>(m, oo, hO, tau);
      if (MODE == MODE_MID) {
        nested_diag<false, FAST>(m, oo, Vv, hD, tau, lc);
        nested_rot<false, FAST>(m, oo, hO, tau);
      }
      nested_diag<false, FAST>(m, oo, Vv, hD, th, lc);
    }
    if (mode_is_epi(MODE)) {
      const double rm = fma(m.re, m.re, m.im * m.im), ro = fma(oo.re, oo.re, oo.im * oo.im);
      sm += rm;
      so += ro;
      if (MODE == MODE_EPI_OBS) { ob.mm = fma(rm, rm, ob.mm); ob.oo = fma(ro, ro, ob.oo); ob.mo = fma(rm, ro, ob.mo); }
    }
    v[i] = m;
    o[i] = oo;
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) v[8 + i] = shfl_xor_c(o[i], 1);
}

// every phase argument of the nested split of this warp and row is small enough for the series
__device__ __forceinline__ bool nested_fast(const cplx* v, const PassXArgs& a, const LaneCoef& lc) {
  double nmax = 0.0;
#pragma unroll
  for (int n = 0; n < 16; ++n) nmax = fmax(nmax, fma(v[n].re, v[n].re, v[n].im * v[n].im));
  const double NT = nmax + shfl_xor_d(nmax, 1);
  // |d_c| <= max|V| + max|delta|/2 + (|ca| + |cb|)max NT; the longest diagonal factor is D(tau) (MODE_MID)
  const double d = a.fmax[0] + 0.5 * a.fmax[2] +
                   (fmax(fabs(lc.cam), fabs(lc.cao)) + fmax(fabs(lc.cbm), fabs(lc.cbo))) * NT;
  const double x = a.tau * d, th = 0.5 * a.tau * a.fmax[1];
  const bool ok = (x * x <= SPGPE_Z_FAST) && (th * th <= SPGPE_Z_FAST);  // NaN fails
  return __all_sync(0xffffffffu, ok);
}

template <int DT, int NX, int LINES, int MODE, bool NEST, int TIME>
__device__ __forceinline__ void real_space(cplx* v, const PassXArgs& a, const void* fbuf, int line, int t, int c,
                                           const LaneCoef& lc, double& sm, double& so, ObsSums& ob) {
  if constexpr (NEST) {
    // in imaginary time the densities grow or shrink inside D; the bound above holds for the entering state only,
    // so imaginary time takes the general path (libm exp either way)
    if (!a.imag && nested_fast(v, a, lc)) real_space_nested<DT, NX, LINES, MODE, true>(v, a, fbuf, line, t, c, lc, sm, so, ob);
    else real_space_nested<DT, NX, LINES, MODE, false>(v, a, fbuf, line, t, c, lc, sm, so, ob);
    return;
  }
  const bool bz0 = a.hc.cb_u == 0.0 && a.hc.cb_d == 0.0;
  const int tier = row_tier<MODE>(v, a, lc, bz0 && MODE == MODE_MID);
  if (bz0) {  // all g equal: b_z has no density term
    if (tier == 0) real_space_tier<DT, NX, LINES, MODE, 0, true, TIME>(v, a, fbuf, line, t, c, lc, sm, so, ob);
    else if (tier == 1) real_space_tier<DT, NX, LINES, MODE, 1, true, TIME>(v, a, fbuf, line, t, c, lc, sm, so, ob);
    else if (tier == 2) real_space_tier<DT, NX, LINES, MODE, 2, true, TIME>(v, a, fbuf, line, t, c, lc, sm, so, ob);
    else real_space_tier<DT, NX, LINES, MODE, 3, true, TIME>(v, a, fbuf, line, t, c, lc, sm, so, ob);
  } else {
    if (tier == 0) real_space_tier<DT, NX, LINES, MODE, 0, false, TIME>(v, a, fbuf, line, t, c, lc, sm, so, ob);
    else if (tier == 1) real_space_tier<DT, NX, LINES, MODE, 1, false, TIME>(v, a, fbuf, line, t, c, lc, sm, so, ob);
    else if (tier == 2) real_space_tier<DT, NX, LINES, MODE, 2, false, TIME>(v, a, fbuf, line, t, c, lc, sm, so, ob);
    else real_space_tier<DT, NX, LINES, MODE, 3, false, TIME>(v, a, fbuf, line, t, c, lc, sm, so, ob);
  }
}

// dynamic shared memory of the row pass: LINES padded line buffers, then the twiddle table
template <int NX, int LINES>
struct XSmem {
  static constexpr int EBUF = LINES * Plan<NX>::PTS * 2;                 // double2 elements
  static constexpr size_t BYTES = (size_t)(EBUF + tw_total<NX>()) * 16;
};

// Persistent: CTA b handles the row groups b, b + gridDim.x, ...; while one group is being transformed the next
// one (psi rows and field rows) is requested into L2, so that its loads find the data there.
// NEST: the real-space part is the nested split (PassXArgs::nest; its own instantiation, so that the default kernels
// keep their register budget)
// TIME: see real_space_tier (the nested instantiations keep the run-time switch)
template <int DT, int NX, int LINES, int MODE, int XS, bool NEST, int TIME>
__global__ void __launch_bounds__(LINES * (NX / 8), (LINES * (NX / 8) <= 256) ? 2 : 1)
pass_x_kernel(const PassXArgs a) {
  typedef Plan<NX> P;
  typedef Store<DT> St;
  typedef typename St::real real;
  typedef typename St::elem elem;
  extern __shared__ __align__(128) double2 smem[];
  constexpr int NTHR = LINES * (NX / 8);
  constexpr int T = P::T;
  const int tid = threadIdx.x;
  const int c = tid & 1;
  const int t = (tid >> 1) % T;
  const int line = (tid >> 1) / T;
  double2* buf = smem + (size_t)line * (P::PTS * 2);
  const int ngroups = a.ny / LINES;
  double sm = 0.0, so = 0.0;  // sums of |own component|^2 and |other component|^2 over this lane's points
  ObsSums ob = {0.0, 0.0, 0.0};
  const LaneCoef lc = lane_coef(a.hc, c);
  const int flip = c ? (int)0x80000000 : 0;  // the odd lane keeps its points rotated by 8 (twiddle())
  cplx v[16];
  // twiddle table of NX behind the line buffers, copied once per (persistent) CTA
  double2* twS = smem + XSmem<NX, LINES>::EBUF;
  pdl_launch_dependents();
  copy_table_async(twS, a.tw, tw_total<NX>(), tid, NTHR);  // completes with the first cp_async_wait_all below

  // The psi rows of a group travel global -> shared memory asynchronously into the line buffers, which are idle at
  // that time, one group ahead, so that the transfer runs under the tail of the previous group.  Rows (XS == 1) are
  // contiguous: ONE bulk copy (cp.async.bulk, mbarrier completion) moves the LINES rows of a group and they land in
  // memory order [line][x][c].  The interleaved half rows of a split axis (XS == 2) go through per-thread cp.async,
  // slot (n, tid) holding register n of thread tid.
  elem* stg = reinterpret_cast<elem*>(smem);
  constexpr int S = XS;  // == a.xs
  const bool BULK = (XS == 1) && (a.dbg & 1);
  const bool FBULK = (XS == 1) && !(a.dbg & 2);
  constexpr unsigned GROUP_BYTES = (unsigned)LINES * NX * 2 * (unsigned)sizeof(elem);
  __shared__ __align__(8) unsigned long long full, ffull;  // psi rows landed / field rows landed
  // point index of position 0 of line L: lines are rows (xs = 1) or the even / odd points of a row (xs = 2)
  auto line_base = [&](int L) { return (size_t)(L / S) * NX * S + (size_t)(L % S); };
  auto issue_loads = [&](int grp) {
    const elem* src = reinterpret_cast<const elem*>(a.src);
    if (BULK) {
      if (tid == 0) {
        fence_proxy_async();  // the line buffers were last touched through the generic proxy
        mbar_expect_tx(&full, GROUP_BYTES);
        bulk_load_1d(stg, src + (size_t)grp * LINES * NX * 2, GROUP_BYTES, &full);
      }
    } else {
      const size_t lb = line_base(grp * LINES + line);
      if (MODE == MODE_PRO || MODE == MODE_FWD) {
        // slot n holds point t + n T of BOTH lanes of a pair (one contiguous 32-byte point per pair and copy); the odd
        // lane, which keeps its points rotated by 8, takes register n out of slot (n + 8) mod 16 (staged())
#pragma unroll
        for (int n = 0; n < 16; ++n)
          cp_async_elem(stg + n * NTHR + tid, src + (lb + (size_t)(t + n * T) * S) * 2 + c);
      } else {
#pragma unroll
        for (int g = 0; g < P::G; ++g)
#pragma unroll
          for (int s = 0; s < P::RL; ++s)
            cp_async_elem(stg + (g * P::RL + s) * NTHR + tid,
                          src + (lb + (size_t)((t + g * T) + (NX / P::RL) * s) * S) * 2 + c);
      }
    }
  };
  // register n of this thread out of the staged group
  auto staged = [&](int n) {
    if (BULK) {
      const elem* row = stg + (size_t)line * NX * 2;
      if (MODE == MODE_PRO || MODE == MODE_FWD) return St::cv(row[(t + ((n + 8 * c) & 15) * T) * 2 + c]);
      const int g = n / P::RL, s = n % P::RL;
      return St::cv(row[((t + g * T) + (NX / P::RL) * s) * 2 + c]);
    } else {
      if (MODE == MODE_PRO || MODE == MODE_FWD) return St::cv(stg[((n + 8 * c) & 15) * NTHR + tid]);
      return St::cv(stg[n * NTHR + tid]);
    }
  };
  if (tid == 0) {
    mbar_init(&full, 1);
    mbar_init(&ffull, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // Work distribution: the group of iteration it+1 is in `nxt` (thread 0), fetched with the atomic one iteration
  // ahead so that its latency never sits in front of a barrier; published to the CTA through next_s.  As soon as it is
  // known, the group's psi rows and field rows are requested into L2, a whole period before they are copied.
  int nxt = ngroups;
  __syncthreads();  // the barriers are initialised before anyone waits on them
  pdl_wait();  // psi and the work counter belong to the preceding kernel
  if ((int)blockIdx.x < ngroups) {
    issue_loads(blockIdx.x);
    if (tid == 0) nxt = sched_next(a.sched);
  }
  auto prefetch_group_l2 = [&](int grp) {  // thread 0
    if (S != 1 || grp >= ngroups || !(a.dbg & 4)) return;
    const size_t first = (size_t)grp * LINES * NX;
    prefetch_l2_bulk(reinterpret_cast<const elem*>(a.src) + first * 2, GROUP_BYTES);
    if (MODE != MODE_FWD) {
      constexpr unsigned FB = LINES * NX * (unsigned)sizeof(real);
      if (a.V) prefetch_l2_bulk(reinterpret_cast<const real*>(a.V) + first, FB);
      if (a.Om) prefetch_l2_bulk(reinterpret_cast<const real*>(a.Om) + first, FB);
      if (a.De) prefetch_l2_bulk(reinterpret_cast<const real*>(a.De) + first, FB);
    }
  };

  __shared__ double red[5][32];
  __shared__ int next_s[2];  // group this CTA takes next (written by thread 0, double-buffered over iterations)
  int it = 0;
  TL_DECL(8);
  for (int grp = blockIdx.x; grp < ngroups; ++it) {
    const size_t first_point = (size_t)grp * LINES * NX;  // first point of the CTA's lines (xs = 1)
    const size_t lbase = line_base(grp * LINES + line);
    if (tid == 0) {
      next_s[it & 1] = nxt;  // visible to the CTA behind the next barrier
      prefetch_group_l2(nxt);
    }
    cp_async_wait_all();  // twiddle table (first iteration), staged rows of a split axis
    if (BULK) mbar_wait(&full, it & 1);
#pragma unroll
    for (int n = 0; n < 16; ++n) v[n] = staged(n);
    if (MODE == MODE_PRO && TIME != 0 && a.scale != nullptr) {
      const double s = a.scale[c];
#pragma unroll
      for (int n = 0; n < 16; ++n) v[n] = mk(v[n].re * s, v[n].im * s);
    }
    if (MODE == MODE_PRO && TIME != 0 && a.anneal_event > 0) {
#pragma unroll 1
      for (int n = 0; n < 16; ++n) {
        // register n holds point t + ((n + 8c) mod 16) T of the line (same index as the load above)
        const unsigned long long e = (unsigned long long)(lbase + (size_t)(t + ((n + 8 * c) & 15) * T) * S) * 2ULL + c;
        const cplx z = anneal_noise(a, e);
        // v[n] with a run-time n would leave the registers: select instead
#pragma unroll
        for (int k = 0; k < 16; ++k)
          if (k == n) v[k] = v[k] + z;
      }
    }
    __syncthreads();  // every thread has taken its staged values: the buffers may be overwritten
    TL_MARK(0);
    // The exchange buffer is idle during the real-space part: it holds the field rows meanwhile.  Their copy starts
    // as soon as every warp has done its last read of the line buffers (the loads of the inverse transform's last
    // radix-16 stage), so it runs under that stage's twiddles and butterflies.
    auto fields_hook = [&]() {
      __syncthreads();
      stage_fields<DT, NX, LINES, XS>(smem, a, first_point, grp * LINES, tid, &ffull, FBULK);
    };
    if (MODE == MODE_MID || mode_is_epi(MODE)) line_fft_inv<NX>(buf, twS, t, c, v, flip, fields_hook);
    TL_MARK(1);

    if (MODE != MODE_FWD) {
      if (MODE == MODE_PRO) fields_hook();
      cp_async_wait_all();
      if (FBULK) mbar_wait(&ffull, it & 1);
      // zero fills and cp.async copies are per-thread writes: a barrier makes them visible; bulk copies
      // complete on the mbarrier every thread has just waited on
      if (!FBULK || a.V == nullptr || a.Om == nullptr || a.De == nullptr) __syncthreads();
      TL_MARK(2);
      real_space<DT, NX, LINES, MODE, NEST, TIME>(v, a, smem, line, t, c, lc, sm, so, ob);
      TL_MARK(3);
      if (mode_is_epi(MODE) && (a.want_norm || MODE == MODE_EPI_OBS)) {
        // norm partials of this row group, one slot per group: the sums do not depend on which CTA took the group,
        // so the reduction order (and every imaginary-time result) is the same from run to run.  Each lane summed
        // its own and the other component over its 8 points: sort into (up, down) first.
        double su = c ? so : sm, sd = c ? sm : so;
        sm = 0.0;
        so = 0.0;
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
          su += shfl_xor_d(su, m);
          sd += shfl_xor_d(sd, m);
        }
        if ((tid & 31) == 0) { red[0][tid >> 5] = su; red[1][tid >> 5] = sd; }
        if (MODE == MODE_EPI_OBS) {  // rho_up^2, rho_dn^2, rho_up rho_dn of the group (same sorting, same fixed order)
          double quu = c ? ob.oo : ob.mm, qdd = c ? ob.mm : ob.oo, qud = ob.mo;
          ob.mm = ob.oo = ob.mo = 0.0;
#pragma unroll
          for (int m = 16; m >= 1; m >>= 1) {
            quu += shfl_xor_d(quu, m);
            qdd += shfl_xor_d(qdd, m);
            qud += shfl_xor_d(qud, m);
          }
          if ((tid & 31) == 0) { red[2][tid >> 5] = quu; red[3][tid >> 5] = qdd; red[4][tid >> 5] = qud; }
        }
      }
      __syncthreads();
      if (mode_is_epi(MODE) && (a.want_norm || MODE == MODE_EPI_OBS) && tid == 0) {
        const int nk = MODE == MODE_EPI_OBS ? 5 : 2;
        for (int k = 0; k < nk; ++k) {
          double s0 = 0.0;
          for (int i = 0; i < NTHR / 32; ++i) s0 += red[k][i];
          a.partial[(size_t)a.pstride * grp + k] = s0;
        }
      }
    }

    if (!mode_is_epi(MODE)) {
      fwd_stages<NX, 1>(buf, twS, t, c, v, flip, CtaSync());
      __syncthreads();  // the last exchange has been read by every warp: the line buffers are free
    }
    const int nxt_grp = next_s[it & 1];
    TL_MARK(4);
    if (nxt_grp < ngroups) {  // the line buffers are free: the next group may land
      issue_loads(nxt_grp);
      if (tid == 0) nxt = sched_next(a.sched);  // consumed in the next iteration
    }
    if (mode_is_epi(MODE)) {
      // point m = t + m T is written by both lanes of a pair at once (one full 32-byte point): the odd lane holds it in
      // register (m + 8) mod 16
#pragma unroll
      for (int m = 0; m < 16; ++m) {
        const cplx val = c ? v[(m + 8) & 15] : v[m];
        St::st(a.dst, (lbase + (size_t)(t + m * T) * S) * 2 + c, val);
      }
    } else {
      dft_last<-1, P::RL>(v);
      TL_MARK(5);
      // the k_x phase of the k-space factor is applied by the column pass (one table value per thread there)
#pragma unroll
      for (int g = 0; g < P::G; ++g)
#pragma unroll
        for (int s = 0; s < P::RL; ++s) {
          const int off = g * T + (NX / P::RL) * s;
          St::st(a.dst, (lbase + (size_t)(t + off) * S) * 2 + c, v[g * P::RL + s]);
        }
    }
    TL_MARK(6);
    TL_TILE();
    grp = nxt_grp;
  }
  if (MODE == MODE_MID) TL_DUMP("xmid wait+stage|inv|fields|real|fwd|issue+last|ex+store", 7);
  if (MODE == MODE_PRO) TL_DUMP("xpro wait+stage|inv|fields|real|fwd|issue+last|ex+store", 7);
  if (MODE == MODE_EPI) TL_DUMP("xepi wait+stage|inv|fields|real|fwd|issue+last|ex+store", 7);
  if (mode_is_epi(MODE)) {
    // imaginary time (a6): the CTA that finishes last turns the per-group norm partials into the rescale factors
    // of the next step (fixed summation order), so no separate kernel is needed
    __shared__ int last_s;
    if (tid == 0) last_s = sched_finish(a.sched) ? 1 : 0;
    if (a.want_norm) {
      __syncthreads();
      if (last_s) {
        double x0 = 0.0, x1 = 0.0;
        for (int b = tid; b < ngroups; b += NTHR) {
          x0 += __ldcg(a.partial + (size_t)a.pstride * b);
          x1 += __ldcg(a.partial + (size_t)a.pstride * b + 1);
        }
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
          x0 += shfl_xor_d(x0, m);
          x1 += shfl_xor_d(x1, m);
        }
        if ((tid & 31) == 0) { red[0][tid >> 5] = x0; red[1][tid >> 5] = x1; }
        __syncthreads();
        if (tid == 0) {
          double nu = 0.0, nd = 0.0;
          for (int i = 0; i < NTHR / 32; ++i) { nu += red[0][i]; nd += red[1][i]; }
          nu *= a.cell;
          nd *= a.cell;
          // a component (or state) of zero norm keeps scale 1 and stays zero instead of turning into NaN (0/0)
          if (a.norm_mode == 0) {
            a.scale_out[0] = nu > 0.0 ? sqrt(a.target[0] / nu) : 1.0;
            a.scale_out[1] = nd > 0.0 ? sqrt(a.target[1] / nd) : 1.0;
          } else {
            a.scale_out[0] = a.scale_out[1] = (nu + nd) > 0.0 ? sqrt((a.target[0] + a.target[1]) / (nu + nd)) : 1.0;
          }
        }
      }
    }
  } else {
    if (tid == 0) sched_finish(a.sched);
  }

}

}  // namespace spgpe
