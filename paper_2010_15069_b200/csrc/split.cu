// split.cu -- line lengths above 4096 (one line no longer fits one CTA's registers and shared memory).
//
// An axis of length n = 2 m is transformed as two interleaved sub-lines of length m (even and odd samples) by the
// ordinary pass kernels; this kernel supplies the radix-2 decimation-in-time step that joins them, applies the
// k-space phase of the split axes on the joined spectrum and undoes the join:
//   X[f]     = E[f] + w^f O[f],   X[f + m] = E[f] - w^f O[f],   w = exp(-2 pi i / n),  f = 0..m-1
//   X <- phase * X                                              (k_x phase always, k_y phase of a split y axis)
//   E'[f]    = X[f] + X[f + m],   O'[f]    = conj(w^f) (X[f] - X[f + m])          (unnormalised, like the passes)
// E and O sit interleaved in memory: sub-line p of the x axis occupies the points x = 2 pos + p, sub-line p of the
// y axis the rows y = 2 pos + p, pos = stored position of the sub-transform.  One thread owns the SX x SY block of
// one (pos_x, pos_y) and both components, so the step is local and in place.
// MODE_ENERGY instead accumulates sum (Kx_c + Ky) |X|^2 (spgpe_energy) and writes nothing back.
#include "internal.h"
#include "fft32.cuh"

namespace spgpe {

template <int DT, int SX, int SY, bool ENERGY>
__global__ void __launch_bounds__(256) split_kernel(const SplitArgs a) {
  typedef Store<DT> St;
  const int mx = a.nx / SX, my = a.ny / SY;
  double esum = 0.0;
  for (size_t b = (size_t)blockIdx.x * blockDim.x + threadIdx.x; b < (size_t)mx * my;
       b += (size_t)gridDim.x * blockDim.x) {
    const int px = (int)(b % mx), py = (int)(b / mx);
    cplx u[SY][SX][2];
#pragma unroll
    for (int j = 0; j < SY; ++j)
#pragma unroll
      for (int i = 0; i < SX; ++i) {
        const size_t pt = ((size_t)py * SY + j) * a.nx + (size_t)px * SX + i;
        if (DT == 1) {  // complex64 storage: both components of a point in one 16-byte access
          const float4 q = __ldcs(reinterpret_cast<const float4*>(a.psi) + pt);
          u[j][i][0] = mk((double)q.x, (double)q.y);
          u[j][i][1] = mk((double)q.z, (double)q.w);
        } else {
#pragma unroll
          for (int c = 0; c < 2; ++c) u[j][i][c] = St::ld(a.psi, pt * 2 + c);
        }
      }
    // the tables of a split axis are stored in the order of the join (api.cu, fill_ktables): entry i*m + pos
    const int fx = px, fy = py;
    if (SX == 2) {
      const double2 w = a.wx[px];
#pragma unroll
      for (int j = 0; j < SY; ++j)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          const cplx e = u[j][0][c], o = cmul(u[j][1][c], mk(w.x, w.y));
          u[j][0][c] = e + o;
          u[j][1][c] = e - o;
        }
    }
    if (SY == 2) {
      const double2 w = a.wy[py];
#pragma unroll
      for (int i = 0; i < SX; ++i)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          const cplx e = u[0][i][c], o = cmul(u[1][i][c], mk(w.x, w.y));
          u[0][i][c] = e + o;
          u[1][i][c] = e - o;
        }
    }
    if (ENERGY) {
#pragma unroll
      for (int j = 0; j < SY; ++j)
#pragma unroll
        for (int i = 0; i < SX; ++i)
#pragma unroll
          for (int c = 0; c < 2; ++c) {
            const double k = a.Kx[(size_t)c * a.nx + fx + i * mx] + a.Ky[fy + j * my];
            esum = fma(k, fma(u[j][i][c].re, u[j][i][c].re, u[j][i][c].im * u[j][i][c].im), esum);
          }
      continue;
    }
    {  // k_x phase: entry px + i*mx along a split x axis, stored position (i = 0) along an unsplit one
#pragma unroll
      for (int j = 0; j < SY; ++j)
#pragma unroll
        for (int i = 0; i < SX; ++i)
#pragma unroll
          for (int c = 0; c < 2; ++c) {
            const double2 p = a.phx[(size_t)c * a.nx + fx + i * mx];
            u[j][i][c] = cmul(u[j][i][c], mk(p.x, p.y));
          }
    }
    if (SY == 2) {
#pragma unroll
      for (int j = 0; j < SY; ++j) {
        const double2 p = a.phy[fy + j * my];
#pragma unroll
        for (int i = 0; i < SX; ++i)
#pragma unroll
          for (int c = 0; c < 2; ++c) u[j][i][c] = cmul(u[j][i][c], mk(p.x, p.y));
      }
    }
    if (SY == 2) {
      const double2 w = a.wy[py];
#pragma unroll
      for (int i = 0; i < SX; ++i)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          const cplx s = u[0][i][c] + u[1][i][c], d = u[0][i][c] - u[1][i][c];
          u[0][i][c] = s;
          u[1][i][c] = cmulc(d, mk(w.x, w.y));
        }
    }
    if (SX == 2) {
      const double2 w = a.wx[px];
#pragma unroll
      for (int j = 0; j < SY; ++j)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          const cplx s = u[j][0][c] + u[j][1][c], d = u[j][0][c] - u[j][1][c];
          u[j][0][c] = s;
          u[j][1][c] = cmulc(d, mk(w.x, w.y));
        }
    }
#pragma unroll
    for (int j = 0; j < SY; ++j)
#pragma unroll
      for (int i = 0; i < SX; ++i) {
        const size_t pt = ((size_t)py * SY + j) * a.nx + (size_t)px * SX + i;
        if (DT == 1) {
          reinterpret_cast<float4*>(a.psi)[pt] = make_float4((float)u[j][i][0].re, (float)u[j][i][0].im,
                                                             (float)u[j][i][1].re, (float)u[j][i][1].im);
        } else {
#pragma unroll
          for (int c = 0; c < 2; ++c) St::st(a.psi, pt * 2 + c, u[j][i][c]);
        }
      }
  }
  if (ENERGY) {
    __shared__ double red[8];
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) esum += __shfl_xor_sync(0xffffffffu, esum, m);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = esum;
    __syncthreads();
    if (threadIdx.x == 0) {
      double s = 0.0;
      for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += red[i];
      a.partial[blockIdx.x] = s;
    }
  }
}

// The same join for complex64 storage in the arithmetic of the fp32 transforms (fft32.cuh, R-14): fp32
// butterflies, every fixed factor (join twiddles, k-space phases) as a two-float value.  One thread owns the SX x SY
// block of one (pos_x, pos_y), both components of a point in one 16-byte access.
template <int SX, int SY>
__global__ void __launch_bounds__(256) split32_kernel(const SplitArgs a) {
  const int mx = a.nx / SX, my = a.ny / SY;
  float4* psi = reinterpret_cast<float4*>(a.psi);
  for (size_t b = (size_t)blockIdx.x * blockDim.x + threadIdx.x; b < (size_t)mx * my;
       b += (size_t)gridDim.x * blockDim.x) {
    const int px = (int)(b % mx), py = (int)(b / mx);
    cf u[SY][SX], d[SY][SX];
#pragma unroll
    for (int j = 0; j < SY; ++j)
#pragma unroll
      for (int i = 0; i < SX; ++i) {
        const float4 q = __ldcs(psi + ((size_t)py * SY + j) * a.nx + (size_t)px * SX + i);
        u[j][i] = mkf(q.x, q.y);
        d[j][i] = mkf(q.z, q.w);
      }
    float4 wx = make_float4(1.f, 0.f, 0.f, 0.f), wy = wx;
    if (SX == 2) {
      wx = __ldg(a.wx32 + px);
#pragma unroll
      for (int j = 0; j < SY; ++j) {
        const cf ou = cmul2(u[j][1], wx.x, wx.y, wx.z, wx.w), od = cmul2(d[j][1], wx.x, wx.y, wx.z, wx.w);
        const cf eu = u[j][0], ed = d[j][0];
        u[j][0] = eu + ou; u[j][1] = eu - ou;
        d[j][0] = ed + od; d[j][1] = ed - od;
      }
    }
    if (SY == 2) {
      wy = __ldg(a.wy32 + py);
#pragma unroll
      for (int i = 0; i < SX; ++i) {
        const cf ou = cmul2(u[1][i], wy.x, wy.y, wy.z, wy.w), od = cmul2(d[1][i], wy.x, wy.y, wy.z, wy.w);
        const cf eu = u[0][i], ed = d[0][i];
        u[0][i] = eu + ou; u[1][i] = eu - ou;
        d[0][i] = ed + od; d[1][i] = ed - od;
      }
    }
    // k_x phase (entry px + i*mx; stored position for an unsplit x axis), k_y phase of a split y axis (entry py + j*my)
#pragma unroll
    for (int i = 0; i < SX; ++i) {
      const float4 fu = __ldg(a.phx32 + px + i * mx), fd = __ldg(a.phx32 + (size_t)a.nx + px + i * mx);
#pragma unroll
      for (int j = 0; j < SY; ++j) {
        u[j][i] = cmul2(u[j][i], fu.x, fu.y, fu.z, fu.w);
        d[j][i] = cmul2(d[j][i], fd.x, fd.y, fd.z, fd.w);
      }
    }
    if (SY == 2) {
#pragma unroll
      for (int j = 0; j < SY; ++j) {
        const float4 f = __ldg(a.phy32 + py + j * my);
#pragma unroll
        for (int i = 0; i < SX; ++i) {
          u[j][i] = cmul2(u[j][i], f.x, f.y, f.z, f.w);
          d[j][i] = cmul2(d[j][i], f.x, f.y, f.z, f.w);
        }
      }
#pragma unroll
      for (int i = 0; i < SX; ++i) {
        const cf su = u[0][i] + u[1][i], du = u[0][i] - u[1][i], sd = d[0][i] + d[1][i], dd = d[0][i] - d[1][i];
        u[0][i] = su; u[1][i] = cmul2c(du, wy.x, wy.y, wy.z, wy.w);
        d[0][i] = sd; d[1][i] = cmul2c(dd, wy.x, wy.y, wy.z, wy.w);
      }
    }
    if (SX == 2) {
#pragma unroll
      for (int j = 0; j < SY; ++j) {
        const cf su = u[j][0] + u[j][1], du = u[j][0] - u[j][1], sd = d[j][0] + d[j][1], dd = d[j][0] - d[j][1];
        u[j][0] = su; u[j][1] = cmul2c(du, wx.x, wx.y, wx.z, wx.w);
        d[j][0] = sd; d[j][1] = cmul2c(dd, wx.x, wx.y, wx.z, wx.w);
      }
    }
#pragma unroll
    for (int j = 0; j < SY; ++j)
#pragma unroll
      for (int i = 0; i < SX; ++i)
        psi[((size_t)py * SY + j) * a.nx + (size_t)px * SX + i] = make_float4(u[j][i].re, u[j][i].im, d[j][i].re, d[j][i].im);
  }
}

template <int DT, bool ENERGY>
static cudaError_t launch_split_dt(const SplitArgs& a, int sx, int sy, int nblk, cudaStream_t s) {
  if (sx == 2 && sy == 2) split_kernel<DT, 2, 2, ENERGY><<<nblk, 256, 0, s>>>(a);
  else if (sx == 2) split_kernel<DT, 2, 1, ENERGY><<<nblk, 256, 0, s>>>(a);
  else if (sy == 2) split_kernel<DT, 1, 2, ENERGY><<<nblk, 256, 0, s>>>(a);
  else split_kernel<DT, 1, 1, ENERGY><<<nblk, 256, 0, s>>>(a);
  return cudaGetLastError();
}

// nblk CTAs of 256 threads; with energy != 0 partial[nblk] receives the per-CTA sums
cudaError_t launch_split(int dt, const SplitArgs& a, int sx, int sy, int energy, int nblk, cudaStream_t s) {
  if (dt == 0) return energy ? launch_split_dt<0, true>(a, sx, sy, nblk, s) : launch_split_dt<0, false>(a, sx, sy, nblk, s);
  if (!energy && a.phx32 != nullptr) {  // complex64 storage, step: fp32 arithmetic with two-float factors
    if (sx == 2 && sy == 2) split32_kernel<2, 2><<<nblk, 256, 0, s>>>(a);
    else if (sx == 2) split32_kernel<2, 1><<<nblk, 256, 0, s>>>(a);
    else split32_kernel<1, 2><<<nblk, 256, 0, s>>>(a);
    return cudaGetLastError();
  }
  return energy ? launch_split_dt<1, true>(a, sx, sy, nblk, s) : launch_split_dt<1, false>(a, sx, sy, nblk, s);
}

}  // namespace spgpe
