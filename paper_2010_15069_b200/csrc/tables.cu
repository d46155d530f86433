// tables.cu -- host-side plan queries: twiddle tables and the stored-position -> frequency map of the
// register/shared-memory transform of line_fft.cuh.
#include <math.h>

#include "internal.h"
#include "launch.cuh"

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

// Stored position pos = q + (n/RL) * k_last, q = sum_{j<NS} k_j * (n / (16^j RL));  f = sum_j k_j 16^(j-1).
int plan_freq_of_pos(int n, int pos) {
  PlanInfo p = plan_info(n);
  const int groups = n / p.rl;
  const int klast = pos / groups;
  const int q = pos % groups;
  int f = 0, w = 1;
  for (int j = 1; j < p.ns; ++j) {
    const int weight = (n >> (4 * j)) / p.rl;
    const int kj = (q / weight) % 16;
    f += kj * w;
    w *= 16;
  }
  return f + klast * w;
}

}  // namespace spgpe
