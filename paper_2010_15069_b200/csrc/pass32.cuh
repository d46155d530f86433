// pass32.cuh -- row pass and column pass of the complex64 path with single-precision transforms (fft32.cuh).
// Same passes, modes, stored order and tables as pass_x.cuh / pass_y.cuh; what differs:
//   * a thread holds 16 points of BOTH components, so the real-space part needs no shuffles and a line of N points
//     takes N/16 threads; shared-memory exchanges move one float4 per point;
//   * butterflies, twiddles and the k-space factor are fp32 with two-float factors (fft32.cuh); the per-point 2x2
//     exponential, the norm sums and every table stay fp64 (su2.cuh), converted at the point;
//   * psi rows arrive by one bulk copy per row group, column tiles by TMA, both into the idle line buffers.
// Covers the plain step (real and imaginary time, single-exponential real-space part, unsplit axes); the nested split,
// the observables, annealed opening passes and split axes stay on the fp64-arithmetic kernels (api.cu picks per launch;
// both families read and write the same layout).
#pragma once
#include <cuda.h>

#include "fft32.cuh"
#include "pass_x.cuh"
#include "pass_y.cuh"

namespace spgpe {

// rows per CTA of the fp32 row pass / columns per CTA of the fp32 column pass (threads = lines * N / 16)
template <int N> struct Lines32 {
  static constexpr int X = (N == 4096) ? 2 : (N == 2048) ? 1 : (N == 1024 ? 4 : (N == 512 ? 8 : 16));
  static constexpr int Y = (N >= 1024) ? 2 : (N == 512 ? 4 : (N == 256 ? 2 : 4));
  static constexpr int XCTAS = (N == 4096) ? 1 : 2;  // resident CTAs per SM the row pass is compiled for
};

template <int N, int LINES>
struct Smem32 {
  static constexpr int PTS = N + (N >> Plan<N>::PADSHIFT);          // float4 slots of one padded line buffer
  static constexpr int LOFF = (LINES == 2) ? 4 : (LINES == 4 ? 2 : 0);  // column mapping: keeps a quarter-warp's lines apart
  static constexpr int LSTRIDE_X = PTS;
  static constexpr int LSTRIDE_Y = PTS + LOFF;
  static constexpr int EBUF_X = LINES * LSTRIDE_X;
  static constexpr int EBUF_Y = LINES * LSTRIDE_Y;
  static constexpr size_t BYTES_X = (size_t)(EBUF_X + tw_total<N>()) * 16;
  static constexpr size_t BYTES_Y = (size_t)(EBUF_Y + tw_total<N>()) * 16;
};

// ---- real-space part on one thread's 16 points (both components in the thread) ----------------------------------
// XS = 2: the LINES = 2 lines of the CTA are the even and the odd points of ONE row (split x axis, split.cu): point x of
// line `line` is point 2 x + line of the row, in the staged row as well as in the staged fields.
template <int NX, int LINES, int MODE, int TIER, bool BZ0, int XS>
__device__ __forceinline__ void real_space32_tier(cf* u, cf* d, const PassXArgs& a, const float* fbuf, int line, int t,
                                                  const LaneCoef& lc, double& su, double& sd) {
  constexpr int T = (XS == 1) ? NX / 16 : 2 * (NX / 16);  // distance of a thread's consecutive points in the field rows
  const float* fV = fbuf + (XS == 1 ? line * NX + t : 2 * t + line);
  const float* fO = fV + LINES * NX;
  const float* fD = fO + LINES * NX;
  const double tau = a.tau, tau2 = a.tau * a.tau;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    cplx m = mk((double)u[i].re, (double)u[i].im), o = mk((double)d[i].re, (double)d[i].im);
    const double Vv = (double)fV[i * T];
    const double hO = 0.5 * (double)fO[i * T];
    const double hD = 0.5 * (double)fD[i * T];
    if (MODE == MODE_MID && BZ0) {  // R(tau) R(tau) = R(2 tau) when all g are equal (pass_x.cuh, R-6)
      const double a1 = su2_apply<false, TIER, BZ0>(m, o, Vv, hO, hD, 2.0 * tau, 4.0 * tau2, lc);
      double pr, pi;
      phase_eval<TIER>(a1 * (2.0 * tau), pr, pi);
      apply_phase(m, o, pr, pi);
    } else if (MODE == MODE_MID) {
      const double a1 = su2_apply<false, TIER, BZ0>(m, o, Vv, hO, hD, tau, tau2, lc);
      const double a2 = su2_apply<false, TIER, BZ0>(m, o, Vv, hO, hD, tau, tau2, lc);
      double pr, pi;
      phase_eval<TIER>((a1 + a2) * tau, pr, pi);
      apply_phase(m, o, pr, pi);
    } else if (a.imag) {
      const double a1 = su2_apply<true, TIER, BZ0>(m, o, Vv, hO, hD, tau, tau2, lc);
      const double e = exp(-a1 * tau);
      m = mk(m.re * e, m.im * e);
      o = mk(o.re * e, o.im * e);
    } else {
      const double a1 = su2_apply<false, TIER, BZ0>(m, o, Vv, hO, hD, tau, tau2, lc);
      double pr, pi;
      phase_eval<TIER>(a1 * tau, pr, pi);
      apply_phase(m, o, pr, pi);
    }
    if (MODE == MODE_EPI) {
      su += fma(m.re, m.re, m.im * m.im);
      sd += fma(o.re, o.re, o.im * o.im);
    }
    u[i] = mkf((float)m.re, (float)m.im);
    d[i] = mkf((float)o.re, (float)o.im);
  }
}

template <int NX, int LINES, int MODE, int XS>
__device__ __forceinline__ void real_space32(cf* u, cf* d, const PassXArgs& a, const float* fbuf, int line, int t,
                                             const LaneCoef& lc, double& su, double& sd) {
  // tier of the warp (bounds as in pass_x.cuh, row_tier): n_up + n_dn <= NT at every point of the thread
  float nmax = 0.f;
#pragma unroll
  for (int n = 0; n < 16; ++n)
    nmax = fmaxf(nmax, fmaf(u[n].re, u[n].re, u[n].im * u[n].im) + fmaf(d[n].re, d[n].re, d[n].im * d[n].im));
  const bool bz0 = a.hc.cb_u == 0.0 && a.hc.cb_d == 0.0;
  const bool merged = bz0 && MODE == MODE_MID;
  const double NT = (double)nmax * 1.000001;
  const double bz = fma(fmax(fabs(lc.cbm), fabs(lc.cbo)), NT, 0.5 * a.fmax[2]);
  const double bx = 0.5 * a.fmax[1];
  const double z = (merged ? 4.0 : 1.0) * (a.tau * a.tau) * fma(bx, bx, bz * bz);
  const double x = (MODE == MODE_MID ? 2.0 : 1.0) * a.tau * fma(fmax(fabs(lc.cam), fabs(lc.cao)), NT, a.fmax[0]);
  const bool ph_ok = (x * x <= SPGPE_Z_FAST);
  int tier = 3;
  if (__all_sync(0xffffffffu, ph_ok && z <= SPGPE_Z_FAST)) tier = 2;
  if (__all_sync(0xffffffffu, ph_ok && z <= SPGPE_Z_MICRO)) tier = 0;
  // two series tiers are enough here (degree 2 and degree 7): the fp32 path is not bound by this arithmetic
  if (bz0) {
    if (tier == 0) real_space32_tier<NX, LINES, MODE, 0, true, XS>(u, d, a, fbuf, line, t, lc, su, sd);
    else if (tier == 2) real_space32_tier<NX, LINES, MODE, 2, true, XS>(u, d, a, fbuf, line, t, lc, su, sd);
    else real_space32_tier<NX, LINES, MODE, 3, true, XS>(u, d, a, fbuf, line, t, lc, su, sd);
  } else {
    if (tier == 0) real_space32_tier<NX, LINES, MODE, 0, false, XS>(u, d, a, fbuf, line, t, lc, su, sd);
    else if (tier == 2) real_space32_tier<NX, LINES, MODE, 2, false, XS>(u, d, a, fbuf, line, t, lc, su, sd);
    else real_space32_tier<NX, LINES, MODE, 3, false, XS>(u, d, a, fbuf, line, t, lc, su, sd);
  }
}

// ---- row pass ---------------------------------------------------------------------------------------------------
// MODE_PRO / MODE_MID / MODE_EPI as in pass_x.cuh.  XS = 1: a line is a row.  XS = 2 (LINES = 2): the two lines are the
// even and the odd points of one row of 2 NX points (split x axis).  a.tw32: two-float twiddles of NX.
template <int NX, int LINES, int MODE, int XS>
__global__ void __launch_bounds__(LINES * (NX / 16), (LINES * (NX / 16) <= 128) ? 3 : (LINES * (NX / 16) <= 256) ? 2 : 1) row32_kernel(const PassXArgs a) {
  static_assert(XS == 1 || LINES == 2, "a split row is handled as its two interleaved lines");
  typedef Plan<NX> P;
  typedef Smem32<NX, LINES> SM;
  extern __shared__ __align__(128) float4 smem4[];
  constexpr int T = P::T;
  constexpr int NTHR = LINES * T;
  constexpr bool LINEW = (P::NS == 2);          // a whole line sits in one warp (T <= 16)
  constexpr bool LASTW = LINEW || P::NS == 3;   // the RL threads of a block are consecutive t: one warp
  static_assert(NTHR % 32 == 0 && 32 % (T < 32 ? T : 32) == 0, "lines must not straddle warps");
  const int tid = threadIdx.x;
  // XS == 1: a line (row) per group of T consecutive threads.  XS == 2: the even and the odd points of one row sit in
  // ADJACENT lanes (column-style mapping, line buffers LSTRIDE_Y apart): a lane pair then reads and writes one 32-byte
  // piece of the row (with the two lines in different warps every store was a 16-byte piece at a 32-byte pitch)
  const int t = (XS == 2) ? tid / 2 : tid % T;
  const int line = (XS == 2) ? tid % 2 : tid / T;
  float4* buf = smem4 + (size_t)line * (XS == 2 ? SM::LSTRIDE_Y : SM::LSTRIDE_X);
  float4* twS = smem4 + (XS == 2 ? SM::EBUF_Y : SM::EBUF_X);
  const float4* stg = smem4;                                    // staged rows, dense: [line][x]
  const float* fbuf = reinterpret_cast<const float*>(smem4);    // staged fields: [field][line][x]
  const int ngroups = a.ny / LINES;
  const LaneCoef lc = lane_coef(a.hc, 0);
  constexpr unsigned GROUP_BYTES = (unsigned)LINES * NX * 16u;
  constexpr unsigned FIELD_BYTES = (unsigned)LINES * NX * 4u;
  __shared__ __align__(8) unsigned long long full, ffull;
  __shared__ double red[2][32];
  __shared__ int next_s[2];
  pdl_launch_dependents();
  for (int i = tid; i < tw_total<NX>(); i += NTHR) cp_async16(twS + i, a.tw32 + i);
  if (tid == 0) {
    mbar_init(&full, 1);
    mbar_init(&ffull, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  auto issue_loads = [&](int grp) {  // thread 0
    fence_proxy_async();
    mbar_expect_tx(&full, GROUP_BYTES);
    bulk_load_1d(smem4, reinterpret_cast<const char*>(a.src) + (size_t)grp * GROUP_BYTES, GROUP_BYTES, &full);
  };
  int nxt = ngroups;
  __syncthreads();
  pdl_wait();
  if ((int)blockIdx.x < ngroups && tid == 0) {
    issue_loads(blockIdx.x);
    nxt = sched_next(a.sched);
  }
  cp_async_wait_all();
  double su = 0.0, sd = 0.0;
  cf u[16], d[16];
  int it = 0;
  TL_DECL(8);
  for (int grp = blockIdx.x; grp < ngroups; ++it) {
    if (tid == 0) {
      next_s[it & 1] = nxt;
      // one CTA per SM (512 threads): nothing else covers the next group's load, so it is asked into L2 a whole
      // period ahead (with two CTAs per SM the other CTA covers it and the prefetch only costs, as in pass_x.cuh)
      if (NTHR > 256 && nxt < ngroups) {
        prefetch_l2_bulk(reinterpret_cast<const char*>(a.src) + (size_t)nxt * GROUP_BYTES, GROUP_BYTES);
        if (a.V) prefetch_l2_bulk(reinterpret_cast<const char*>(a.V) + (size_t)nxt * FIELD_BYTES, FIELD_BYTES);
        if (a.Om) prefetch_l2_bulk(reinterpret_cast<const char*>(a.Om) + (size_t)nxt * FIELD_BYTES, FIELD_BYTES);
        if (a.De) prefetch_l2_bulk(reinterpret_cast<const char*>(a.De) + (size_t)nxt * FIELD_BYTES, FIELD_BYTES);
      }
    }
    mbar_wait(&full, it & 1);
    TL_MARK(0);
    {
#pragma unroll
      for (int n = 0; n < 16; ++n) {
        const int x = (MODE == MODE_PRO) ? (t + n * T) : stored_pos32<NX>(t, n);
        lds4(stg, XS == 1 ? line * NX + x : 2 * x + line, u[n], d[n]);
      }
    }
    if (MODE == MODE_PRO && a.scale != nullptr) {
      const double e0 = a.scale[0], e1 = a.scale[1];
#pragma unroll
      for (int n = 0; n < 16; ++n) {
        u[n] = mkf((float)((double)u[n].re * e0), (float)((double)u[n].im * e0));
        d[n] = mkf((float)((double)d[n].re * e1), (float)((double)d[n].im * e1));
      }
    }
    __syncthreads();  // every thread has taken its staged values (twiddles have landed): the buffers may be overwritten
    auto fields_hook = [&]() {
      __syncthreads();  // last read of the line buffers done by every warp
      if (tid == 0) {
        const void* src[3] = {a.V, a.Om, a.De};
        const unsigned long long policy = l2_policy_evict_first();
        const unsigned n = (src[0] != nullptr) + (src[1] != nullptr) + (src[2] != nullptr);
        fence_proxy_async();
        mbar_expect_tx(&ffull, n * FIELD_BYTES);
#pragma unroll
        for (int f = 0; f < 3; ++f)
          if (src[f] != nullptr)
            bulk_load_1d_hint(reinterpret_cast<char*>(smem4) + f * FIELD_BYTES,
                              reinterpret_cast<const char*>(src[f]) + (size_t)grp * FIELD_BYTES, FIELD_BYTES, &ffull, policy);
      }
      const void* src[3] = {a.V, a.Om, a.De};
#pragma unroll
      for (int f = 0; f < 3; ++f)
        if (src[f] == nullptr) {
          float4* z = reinterpret_cast<float4*>(reinterpret_cast<char*>(smem4) + f * FIELD_BYTES);
          for (int k = tid; k < (int)(FIELD_BYTES / 16); k += NTHR) z[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    };
    TL_MARK(1);
    if (MODE == MODE_MID || MODE == MODE_EPI) line_inv32<NX, LINEW, LASTW>(buf, twS, t, u, d, fields_hook);
    else fields_hook();
    TL_MARK(2);
    mbar_wait(&ffull, it & 1);
    TL_MARK(3);
    if (a.V == nullptr || a.Om == nullptr || a.De == nullptr) __syncthreads();  // zero fills are per-thread writes
    real_space32<NX, LINES, MODE, XS>(u, d, a, fbuf, line, t, lc, su, sd);
    TL_MARK(4);
    if (MODE == MODE_EPI && a.want_norm) {
#pragma unroll
      for (int m = 16; m >= 1; m >>= 1) {
        su += __shfl_xor_sync(0xffffffffu, su, m);
        sd += __shfl_xor_sync(0xffffffffu, sd, m);
      }
      if ((tid & 31) == 0) { red[0][tid >> 5] = su; red[1][tid >> 5] = sd; }
      su = 0.0;
      sd = 0.0;
    }
    __syncthreads();  // the field rows have been read: the line buffers belong to the transform again
    if (MODE == MODE_EPI && a.want_norm && tid == 0) {
      double s0 = 0.0, s1 = 0.0;
      for (int i = 0; i < NTHR / 32; ++i) { s0 += red[0][i]; s1 += red[1][i]; }
      a.partial[(size_t)a.pstride * grp] = s0;
      a.partial[(size_t)a.pstride * grp + 1] = s1;
    }
    if (MODE != MODE_EPI) {
      fwd_stages32<NX, 1, LINEW, LASTW>(buf, twS, t, u, d);
      __syncthreads();  // the last exchange has been read by every warp: the line buffers are free
      TL_MARK(5);
    }
    const int nxt_grp = next_s[it & 1];
    if (tid == 0 && nxt_grp < ngroups) {
      issue_loads(nxt_grp);
      nxt = sched_next(a.sched);
    }
    float4* dst = reinterpret_cast<float4*>(a.dst) + (size_t)grp * LINES * NX;  // first point of the group's rows
    if (MODE == MODE_EPI) {
#pragma unroll
      for (int n = 0; n < 16; ++n)
        dst[XS == 1 ? line * NX + (t + n * T) : 2 * (t + n * T) + line] = make_float4(u[n].re, u[n].im, d[n].re, d[n].im);
    } else {
      dft_lastf<-1, P::RL>(u);
      dft_lastf<-1, P::RL>(d);
#pragma unroll
      for (int n = 0; n < 16; ++n) {
        const int x = stored_pos32<NX>(t, n);
        dst[XS == 1 ? line * NX + x : 2 * x + line] = make_float4(u[n].re, u[n].im, d[n].re, d[n].im);
      }
    }
    TL_MARK(6);
    TL_TILE();
    grp = nxt_grp;
  }
  if (MODE == MODE_MID) TL_DUMP("row32 wait|stage|inv|fieldwait|real|fwd|last+store", 7);
  if (MODE == MODE_EPI) {
    __shared__ int last_s;
    if (tid == 0) last_s = sched_finish(a.sched) ? 1 : 0;
    if (a.want_norm) {
      __syncthreads();
      if (last_s) {  // the CTA that finishes last turns the partials into the rescale factors (pass_x.cuh)
        double x0 = 0.0, x1 = 0.0;
        for (int b = tid; b < ngroups; b += NTHR) {
          x0 += __ldcg(a.partial + (size_t)a.pstride * b);
          x1 += __ldcg(a.partial + (size_t)a.pstride * b + 1);
        }
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
          x0 += __shfl_xor_sync(0xffffffffu, x0, m);
          x1 += __shfl_xor_sync(0xffffffffu, x1, m);
        }
        if ((tid & 31) == 0) { red[0][tid >> 5] = x0; red[1][tid >> 5] = x1; }
        __syncthreads();
        if (tid == 0) {
          double nu = 0.0, nd = 0.0;
          for (int i = 0; i < NTHR / 32; ++i) { nu += red[0][i]; nd += red[1][i]; }
          nu *= a.cell;
          nd *= a.cell;
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


// ---- column pass ------------------------------------------------------------------------------------------------
// YMODE_STEP: psi^(k_x, y) -> F_y -> * ex_c(k_x) ey(k_y) -> F_y^-1 -> psi^(k_x, y), in place, LINES adjacent columns per
// CTA, thread index = line + LINES * t.  a.tw32: two-float twiddles of NY; a.eyk32 [NY], a.exk32 [2][nx]: two-float
// phase tables (hi.re, hi.im, lo.re, lo.im); a.tmap32: box [min(NY, 256) rows][LINES points].
// YMODE_FWDONLY / YMODE_INVONLY (split transforms, api.cu): forward transform only, results in stored order / inverse
// transform only, input in stored order.  YMODE_STEP with a.exk32 == NULL applies the k_y factor alone (split x axis).
template <int NY, int LINES, int YMODE>
__global__ void __launch_bounds__(LINES * (NY / 16), (LINES * (NY / 16) <= 256) ? 2 : 1) col32_kernel(const __grid_constant__ PassYArgs a) {
  typedef Plan<NY> P;
  typedef Smem32<NY, LINES> SM;
  extern __shared__ __align__(128) float4 smem4[];
  constexpr int T = P::T;
  constexpr int NTHR = LINES * T;
  constexpr bool LINEW = (P::NS == 2) && (T * LINES <= 32);
  constexpr bool LASTW = (P::NS == 2) ? LINEW : (P::RL * LINES <= 32);
  constexpr int BR = NY < 256 ? NY : 256;
  constexpr unsigned TILE_BYTES = (unsigned)NY * LINES * 16u;
  const int tid = threadIdx.x;
  const int line = tid % LINES;
  const int t = tid / LINES;
  float4* buf = smem4 + (size_t)line * SM::LSTRIDE_Y;
  float4* twS = smem4 + SM::EBUF_Y;
  const float4* stg = smem4;  // the tile lands here, dense: [row][line]
  const int ngroups = a.nx / LINES;
  __shared__ __align__(8) unsigned long long mbar;
  __shared__ int next_s[2];
  pdl_launch_dependents();
  for (int i = tid; i < tw_total<NY>(); i += NTHR) cp_async16(twS + i, a.tw32 + i);
  auto issue_loads = [&](int grp) {  // thread 0
    fence_proxy_async();
    mbar_expect_tx(&mbar, TILE_BYTES);
#pragma unroll
    for (int b = 0; b < NY / BR; ++b)
      tma_load_2d(smem4 + (size_t)b * BR * LINES, &a.tmap32, grp * LINES * 4, b * BR, &mbar);
  };
  if (tid == 0) {
    mbar_init(&mbar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  int nxt = ngroups;
  pdl_wait();
  if (tid == 0 && (int)blockIdx.x < ngroups) {
    issue_loads(blockIdx.x);
    nxt = sched_next(a.sched);
  }
  cp_async_wait_all();
  __syncthreads();
  cf u[16], d[16];
  int it = 0;
  TL_DECL(8);
  for (int grp = blockIdx.x; grp < ngroups; ++it) {
    const size_t col = (size_t)grp * LINES + line;
    if (tid == 0) {
      next_s[it & 1] = nxt;
      if (nxt < ngroups) {
#pragma unroll
        for (int b = 0; b < NY / BR; ++b) tma_prefetch_2d(&a.tmap32, nxt * LINES * 4, b * BR);
      }
    }
    mbar_wait(&mbar, it & 1);
    TL_MARK(0);
#pragma unroll
    for (int n = 0; n < 16; ++n)
      lds4(stg, (YMODE == YMODE_INVONLY ? stored_pos32<NY>(t, n) : t + n * T) * LINES + line, u[n], d[n]);
    __syncthreads();  // every thread has taken its staged values: the buffers may be overwritten
    TL_MARK(1);
    int nxt_grp = ngroups;
    auto hook = [&]() {
      __syncthreads();  // last read of the line buffers done by every warp: the next tile may land
      nxt_grp = next_s[it & 1];
      if (tid == 0 && nxt_grp < ngroups) {
        issue_loads(nxt_grp);
        nxt = sched_next(a.sched);
      }
    };
    if (YMODE == YMODE_FWDONLY) {
      // the line buffers are free behind the last exchange: the next tile's load runs under the last butterflies too
      fwd_stages32<NY, 1, LINEW, LASTW>(buf, twS, t, u, d);
      hook();
      dft_lastf<-1, P::RL>(u);
      dft_lastf<-1, P::RL>(d);
    } else if (YMODE != YMODE_INVONLY) {
      line_fwd32<NY, LINEW, LASTW>(buf, twS, t, u, d);
    }
    TL_MARK(2);
    if (YMODE == YMODE_STEP) {
      const bool has_x = a.exk32 != nullptr;
      const float4 one = make_float4(1.f, 0.f, 0.f, 0.f);
      const float4 xu = has_x ? __ldg(a.exk32 + col) : one, xd = has_x ? __ldg(a.exk32 + (size_t)a.nx + col) : one;
#pragma unroll
      for (int r = 0; r < 16; ++r) {
        const float4 f = __ldg(a.eyk32 + stored_pos32<NY>(t, r));
        u[r] = cmul2(u[r], f.x, f.y, f.z, f.w);
        d[r] = cmul2(d[r], f.x, f.y, f.z, f.w);
        if (has_x) {
          u[r] = cmul2(u[r], xu.x, xu.y, xu.z, xu.w);
          d[r] = cmul2(d[r], xd.x, xd.y, xd.z, xd.w);
        }
      }
    }
    TL_MARK(3);
    float4* dst = reinterpret_cast<float4*>(a.psi) + col;
    if (YMODE == YMODE_FWDONLY) {
#pragma unroll
      for (int n = 0; n < 16; ++n)
        dst[(size_t)stored_pos32<NY>(t, n) * a.nx] = make_float4(u[n].re, u[n].im, d[n].re, d[n].im);
    } else {
      line_inv32<NY, LINEW, LASTW>(buf, twS, t, u, d, hook);
      TL_MARK(4);
#pragma unroll
      for (int n = 0; n < 16; ++n) dst[(size_t)(t + n * T) * a.nx] = make_float4(u[n].re, u[n].im, d[n].re, d[n].im);
    }
    TL_MARK(5);
    TL_TILE();
    grp = nxt_grp;
  }
  TL_DUMP("col32 wait|stage|fwd|phase|inv|store", 6);
  if (tid == 0) sched_finish(a.sched);
}


}  // namespace spgpe
