// tables.cu -- host-side plan queries: twiddle tables and the stored-position -> frequency map of the
// register/shared-memory transform of line_fft.cuh.
#include <math.h>

#include "internal.h"
#include "launch.cuh"
#include "pass32.cuh"

namespace spgpe {

namespace {
struct PlanInfo { int ns, rl, lines_y; };
PlanInfo plan_info(int n) {
  switch (n) {
    case 64: return {Plan<64>::NS, Plan<64>::RL, Lines<64>::Y};
    case 128: return {Plan<128>::NS, Plan<128>::RL, Lines<128>::Y};
    case 256: return {Plan<256>::NS, Plan<256>::RL, Lines<256>::Y};
    case 512: return {Plan<512>::NS, Plan<512>::RL, Lines<512>::Y};
    case 1024: return {Plan<1024>::NS, Plan<1024>::RL, Lines<1024>::Y};
    case 2048: return {Plan<2048>::NS, Plan<2048>::RL, Lines<2048>::Y};
    case 4096: return {Plan<4096>::NS, Plan<4096>::RL, Lines<4096>::Y};
    default: return {0, 0, 0};
  }
}
}  // namespace


int plan_lines_y(int n) { return plan_info(n).lines_y; }
int plan_lines_x(int n) {
  switch (n) {
    case 64: return Lines<64>::X;
    case 128: return Lines<128>::X;
    case 256: return Lines<256>::X;
    case 512: return Lines<512>::X;
    case 1024: return Lines<1024>::X;
    case 2048: return Lines<2048>::X;
    default: return Lines<4096>::X;
  }
}
int plan_lines_x32(int n) {
  switch (n) {
    case 64: return Lines32<64>::X;
    case 128: return Lines32<128>::X;
    case 256: return Lines32<256>::X;
    case 512: return Lines32<512>::X;
    case 1024: return Lines32<1024>::X;
    case 2048: return Lines32<2048>::X;
    default: return Lines32<4096>::X;
  }
}
int plan_lines_y32(int n) {
  switch (n) {
    case 64: return Lines32<64>::Y;
    case 128: return Lines32<128>::Y;
    case 256: return Lines32<256>::Y;
    case 512: return Lines32<512>::Y;
    case 1024: return Lines32<1024>::Y;
    case 2048: return Lines32<2048>::Y;
    default: return Lines32<4096>::Y;
  }
}
int plan_lines_ydb(int n) { return n == 2048 ? Lines<2048>::YDB : (n == 1024 ? Lines<1024>::YDB : 0); }


int plan_tw_total(int n) {
  PlanInfo p = plan_info(n);
  int total = 0;
  for (int j = 1; j < p.ns; ++j) total += 15 * (n >> (4 * j));
  return total;
}

void plan_fill_twiddles(int n, double2* host) {
  PlanInfo p = plan_info(n);
  const long double two_pi = 6.283185307179586476925286766559005768L;
  int off = 0;
  for (int j = 1; j < p.ns; ++j) {
    const int M = n >> (4 * j);
    for (int k = 1; k < 16; ++k)
      for (int lo = 0; lo < M; ++lo) {
        // exp(-2 pi i k lo / (16 M)), angle reduced in integers first
        const int num = (k * lo) % (16 * M);
        const long double ang = -two_pi * (long double)num / (long double)(16 * M);
        host[off + (k - 1) * M + lo] = make_double2((double)cosl(ang), (double)sinl(ang));
      }
    off += 15 * M;
  }
}

// hi = fp32 rounding of the fp64 twiddle, lo = fp32 rounding of the remainder (fft32.cuh)
void plan_fill_twiddles32(int n, float4* host) {
  const int total = plan_tw_total(n);
  double2* tmp = new double2[total > 0 ? total : 1];
  plan_fill_twiddles(n, tmp);
  for (int i = 0; i < total; ++i) {
    const float hr = (float)tmp[i].x, hi = (float)tmp[i].y;
    host[i] = make_float4(hr, hi, (float)(tmp[i].x - (double)hr), (float)(tmp[i].y - (double)hi));
  }
  delete[] tmp;
}

// Frequency index held at stored position pos = (t + g*T) + (n/RL) * s (T = n/16 threads per component, thread t,
// last-stage group g, output s of the last butterfly).  Decimation in frequency: the first stage's output index is
// the least significant digit.  Two-stage plans: the group q = t + g*T is the first stage's output k1, f = k1 + 16 s.
// Three-stage plans (line_fft.cuh): thread t = (hi, lo), hi = t / RL = k1, its groups hold k2 = lo + g*RL,
// f = k1 + 16 k2 + 256 s.
int plan_freq_of_pos(int n, int pos) {
  PlanInfo p = plan_info(n);
  const int groups = n / p.rl;
  const int s = pos / groups;
  const int q = pos % groups;
  if (p.ns == 2) return q + 16 * s;
  const int T = n / 16;
  const int t = q % T, g = q / T;
  const int hi = t / p.rl, lo = t % p.rl;
  return hi + 16 * (lo + g * p.rl) + 256 * s;
}

}  // namespace spgpe
