// pass_y.cuh -- the column pass: y-direction forward transform, k-space phase, inverse transform
// (SURVEY.md 8(a) rows a2/a4 (y part) and a3; include/spgpe.h).  The k-space factor
// exp(-i K_c dt) is separable into ex_c(k_x) ey(k_y), ey(k_y) = exp(-i k_y^2 dt / 2) / (nx ny) (imaginary time: the
// decaying real factors).  Both are applied here: ey from a per-thread table, ex_c(k_x) as ONE value per thread and
// tile, since a thread's 16 points share their column (in the row pass it would take 16 table loads per thread).
//
// One CTA handles LINES adjacent columns; thread index = c + 2*(line + LINES*t), so that a warp-wide access
// covers LINES*32 contiguous bytes in each of 16/LINES rows.
//
//   YMODE_STEP   : psi^(k_x, y) -> F_y -> * ex_c(k_x) ey(k_y) -> F_y^-1 -> psi^(k_x, y)  (in place)
//   YMODE_ENERGY : psi^(k_x, y) -> F_y -> sum (Kx_c(k_x) + Ky(k_y)) |psi^|^2 -> partial[CTA]
//   YMODE_FWDONLY: psi^(k_x, y) -> F_y -> psi^(k_x, k_y) in stored order          (split transforms, api.cu)
//   YMODE_INVONLY: psi^(k_x, k_y) in stored order -> F_y^-1 -> psi^(k_x, y)
//   YMODE_STEP_OBS: YMODE_STEP that also leaves, per CTA, the k-space sums of include/spgpe.h spgpe_step_observe
//                  (sum |psi^_c|^2, sum K_c |psi^_c|^2, sum k_x |psi^_c|^2, taken in front of the k-space factor)
#pragma once
#include <cuda.h>

#include "line_fft.cuh"

namespace spgpe {

enum { YMODE_STEP = 0, YMODE_ENERGY = 1, YMODE_FWDONLY = 2, YMODE_INVONLY = 3, YMODE_STEP_OBS = 4 };

struct PassYArgs {
  void* psi;            // [NY][nx][2]
  const double2* tw;    // twiddles of NY
  const float4* tw32;   // two-float twiddles, k_y phases [NY] and k_x phases [2][nx] of the fp32 kernels (pass32.cuh)
  const float4* eyk32;
  const float4* exk32;
  const double2* eyk;   // [NY] k_y phase in stored order (YMODE_STEP)
  const double2* exk;   // [2][nx] k_x phase in the row pass's stored order (YMODE_STEP), or NULL (none applied here)
  const double* Kx;     // [2][nx] (k_x +- k_L)^2/2 in the row pass's stored order (YMODE_ENERGY)
  const double* Ky;     // [NY] k_y^2/2 in stored order (YMODE_ENERGY)
  double* partial;      // [gridDim.x] sum over this CTA's columns (YMODE_ENERGY); [gridDim.x][6] (YMODE_STEP_OBS)
  const double* kxv;    // [nx] k_x in the row pass's stored order (YMODE_STEP_OBS)
  int nx;
  int* sched;           // [2] device: work counter (common.cuh, sched_next)
  // psi as a 2-D tensor [NY rows][4 nx reals], box = [min(NY, 256) rows][4 LINES reals]: the columns of a group
  CUtensorMap tmap;
  CUtensorMap tmap_db;  // the same tensor with the box of the double-buffered kernel (pass_y_db_kernel)
  CUtensorMap tmap32;   // the same tensor with the tile of col32_kernel (pass32.cuh)
};

template <int NY, int LINES>
struct YLayout {
  // padded points per line buffer; the residue mod 4 keeps a quarter-warp's lines on distinct banks
  static constexpr int BASE = Plan<NY>::PTS;
  static constexpr int WANT = (LINES >= 4) ? 1 : (LINES == 2 ? 2 : 0);
  static constexpr int LINE_PTS = BASE + ((WANT - (BASE & 3)) & 3);
};

// dynamic shared memory of the column pass: LINES padded line buffers, the twiddle table, and (YMODE_STEP, when
// it fits in 227 KB) the k_y phase table
// EYG: the k_y phase table stays in global memory (read through L1/L2) so that two CTAs fit one SM
template <int NY, int LINES, bool EYG = false>
struct YSmem {
  static constexpr int EBUF = LINES * YLayout<NY, LINES>::LINE_PTS * 2;  // double2 elements
  static constexpr int TW = tw_total<NY>();
  static constexpr bool EY_SMEM = !EYG && (size_t)(EBUF + TW + NY) * 16 <= 227u * 1024u;
  static constexpr size_t BYTES = (size_t)(EBUF + TW + (EY_SMEM ? NY : 0)) * 16;
};

// Persistent: CTA b handles the column groups b, b + gridDim.x, ...
template <int DT, int NY, int LINES, int YMODE, bool EYG = false>
__global__ void __launch_bounds__(LINES * (NY / 8), (LINES * (NY / 8) <= 256) ? 2 : 1)
pass_y_kernel(const __grid_constant__ PassYArgs a) {
  typedef Plan<NY> P;
  typedef Store<DT> St;
  typedef YSmem<NY, LINES, EYG> SM;
  extern __shared__ __align__(128) double2 smem[];
  constexpr int T = P::T;
  constexpr int NTHR = LINES * (NY / 8);
  constexpr bool STEP = (YMODE == YMODE_STEP || YMODE == YMODE_STEP_OBS);
  constexpr bool OBS = (YMODE == YMODE_STEP_OBS);
  const int tid = threadIdx.x;
  const int c = tid & 1;
  const int line = (tid >> 1) % LINES;
  const int t = (tid >> 1) / LINES;
  double2* buf = smem + (size_t)line * (YLayout<NY, LINES>::LINE_PTS * 2);
  double2* twS = smem + SM::EBUF;
  const double2* ey = a.eyk;
  double om = 0.0, ot = 0.0, op = 0.0;  // OBS: sums of |z|^2, K_c |z|^2, k_x |z|^2 of this thread's component
  pdl_launch_dependents();
  copy_table_async(twS, a.tw, SM::TW, tid, NTHR);
  if (STEP && SM::EY_SMEM) {
    double2* eyS = twS + SM::TW;
    copy_table_async(eyS, a.eyk, NY, tid, NTHR);
    ey = eyS;
  }
  const size_t nx = (size_t)a.nx;
  const int ngroups = a.nx / LINES;
  const size_t estride = (size_t)T * nx * 2;  // rows of one thread are T*nx points apart
  double e = 0.0;
  cplx v[16];

  // The columns of a group travel global -> shared memory through TMA: NY / BR boxes of BR rows x (LINES columns x
  // 2 components), landing densely ([row][line][c]) in the line buffers while these are idle, issued one group
  // ahead by one thread; completion is signalled on an mbarrier (phase = iteration parity).
  typedef typename St::elem elem;
  constexpr int BR = NY < 256 ? NY : 256;
  constexpr unsigned TILE_BYTES = (unsigned)NY * LINES * 2 * (unsigned)sizeof(elem);
  elem* stg = reinterpret_cast<elem*>(smem);
  __shared__ __align__(8) unsigned long long mbar;
  auto issue_loads = [&](int grp) {  // thread 0 only
    fence_proxy_async();
    mbar_expect_tx(&mbar, TILE_BYTES);
#pragma unroll
    for (int b = 0; b < NY / BR; ++b)
      tma_load_2d(stg + (size_t)b * BR * LINES * 2, &a.tmap, grp * LINES * 4, b * BR, &mbar);
  };
  if (tid == 0) {
    mbar_init(&mbar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // psi and the work counter belong to the preceding kernel.  The tables copied above do not: the twiddles are
  // written at spgpe_create, and the k_y phase table by aux_phase_tables, an ordinary (non-programmatic) launch that
  // has completed before the row pass in front of this kernel could start; this kernel can only become resident
  // after that row pass has started, so the table is complete whenever the prologue runs.
  pdl_wait();
  if (tid == 0 && (int)blockIdx.x < ngroups) issue_loads(blockIdx.x);
  cp_async_wait_all();
  __syncthreads();  // tables and the barrier are visible to every thread

  __shared__ int next_s[2];  // group this CTA takes next (written by thread 0, double-buffered over iterations)
  int it = 0;
  for (int grp = blockIdx.x; grp < ngroups; ++it) {
    const size_t col = (size_t)grp * LINES + line;
    const size_t e0 = ((size_t)t * nx + col) * 2 + c;  // element (row t, column col, component c)
    // k_x phase of this column and component (see pass_y_db_kernel); requested now, used after the forward transform
    double2 exv = make_double2(1.0, 0.0);
    if (STEP && a.exk != nullptr) exv = __ldg(a.exk + (size_t)c * nx + col);
    // the next group is requested now and published before the last barrier of this iteration (latency hidden)
    int nxt_req = 0;
    if (tid == 0) {
      nxt_req = sched_next(a.sched);
      if (nxt_req < ngroups) {
#pragma unroll
        for (int b = 0; b < NY / BR; ++b) tma_prefetch_2d(&a.tmap, nxt_req * LINES * 4, b * BR);
      }
    }
    mbar_wait(&mbar, it & 1);
    if (YMODE == YMODE_INVONLY) {
#pragma unroll
      for (int g = 0; g < P::G; ++g)
#pragma unroll
        for (int s = 0; s < P::RL; ++s)
          v[g * P::RL + s] = St::cv(stg[(((t + g * T) + (NY / P::RL) * s) * LINES + line) * 2 + c]);
    } else {
#pragma unroll
      for (int n = 0; n < 16; ++n) v[n] = St::cv(stg[((t + n * T) * LINES + line) * 2 + c]);
    }
    __syncthreads();  // every thread has taken its staged values: the buffers may be overwritten
    int nxt_grp = ngroups;

    if (YMODE != YMODE_INVONLY) line_fft_fwd<NY>(buf, twS, t, c, v);

    if (OBS) {
      const double kxc = a.Kx[(size_t)c * nx + col], kx1 = a.kxv[col];
      double m0 = 0.0, t0 = 0.0;
#pragma unroll
      for (int g = 0; g < P::G; ++g)
#pragma unroll
        for (int s = 0; s < P::RL; ++s) {
          const cplx z = v[g * P::RL + s];
          const double r = fma(z.re, z.re, z.im * z.im);
          m0 += r;
          t0 = fma(kxc + a.Ky[(t + g * T) + (NY / P::RL) * s], r, t0);
        }
      om += m0;
      ot += t0;
      op = fma(kx1, m0, op);
    }
    if (STEP || YMODE == YMODE_INVONLY) {
      if (STEP) {
#pragma unroll
      for (int g = 0; g < P::G; ++g)
#pragma unroll
        for (int s = 0; s < P::RL; ++s) {
          const int pos = (t + g * T) + (NY / P::RL) * s;
          double2 f = SM::EY_SMEM ? ey[pos] : __ldg(ey + pos + late_zero(v[g * P::RL + s].re));
          v[g * P::RL + s] = cmul(cmul(v[g * P::RL + s], mk(f.x, f.y)), mk(exv.x, exv.y));
        }
      }
      // after the last read of the line buffers the next group's transfer starts under the last butterflies
      auto hook = [&]() {
        if (tid == 0) next_s[it & 1] = nxt_req;
        __syncthreads();
        nxt_grp = next_s[it & 1];
        if (tid == 0 && nxt_grp < ngroups) issue_loads(nxt_grp);
      };
      line_fft_inv<NY>(buf, twS, t, c, v, 0, hook);
#pragma unroll
      for (int n = 0; n < 16; ++n) St::st(a.psi, e0 + n * estride, v[n]);
    } else if (YMODE == YMODE_FWDONLY) {
      if (tid == 0) next_s[it & 1] = nxt_req;
      __syncthreads();
      nxt_grp = next_s[it & 1];
      if (tid == 0 && nxt_grp < ngroups) issue_loads(nxt_grp);
#pragma unroll
      for (int g = 0; g < P::G; ++g)
#pragma unroll
        for (int s = 0; s < P::RL; ++s) {
          const size_t pos = (size_t)((t + g * T) + (NY / P::RL) * s);
          St::st(a.psi, (pos * nx + col) * 2 + c, v[g * P::RL + s]);
        }
    } else {
      if (tid == 0) next_s[it & 1] = nxt_req;
      __syncthreads();
      nxt_grp = next_s[it & 1];
      if (tid == 0 && nxt_grp < ngroups) issue_loads(nxt_grp);
      const double kx = a.Kx[(size_t)c * nx + col];
#pragma unroll
      for (int g = 0; g < P::G; ++g)
#pragma unroll
        for (int s = 0; s < P::RL; ++s) {
          const cplx z = v[g * P::RL + s];
          e = fma(kx + a.Ky[(t + g * T) + (NY / P::RL) * s], fma(z.re, z.re, z.im * z.im), e);
        }
    }
    grp = nxt_grp;
  }
  if (tid == 0) sched_finish(a.sched);

  if (OBS) {
    // component c sits in the lanes of parity c: reduce over the lanes of equal parity, then over the warps
    __shared__ double redo[6][32];
#pragma unroll
    for (int m = 16; m >= 2; m >>= 1) {
      om += __shfl_xor_sync(0xffffffffu, om, m);
      ot += __shfl_xor_sync(0xffffffffu, ot, m);
      op += __shfl_xor_sync(0xffffffffu, op, m);
    }
    const int w = tid >> 5, nw = (blockDim.x + 31) >> 5;
    if ((tid & 31) < 2) { redo[c][w] = om; redo[2 + c][w] = ot; redo[4 + c][w] = op; }
    __syncthreads();
    if (tid < 6) {
      double s0 = 0.0;
      for (int i = 0; i < nw; ++i) s0 += redo[tid][i];
      a.partial[(size_t)blockIdx.x * 6 + tid] = s0;
    }
  }
  if (YMODE == YMODE_ENERGY) {
    __shared__ double red[32];
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) e += __shfl_xor_sync(0xffffffffu, e, m);
    const int w = tid >> 5, nw = (blockDim.x + 31) >> 5;
    if ((tid & 31) == 0) red[w] = e;
    __syncthreads();
    if (tid == 0) {
      double s0 = 0.0;
      for (int i = 0; i < nw; ++i) s0 += red[i];
      a.partial[blockIdx.x] = s0;
    }
  }
}

// ---- double-buffered variant of YMODE_STEP ------------------------------------------------------------------------
// One 256-thread CTA per SM works on tiles of LINES columns with three buffers: the line buffers (exchanges of the
// transforms), a staging buffer (the TMA load of the next tile is issued as soon as the current one has been taken
// out of it, a whole tile period ahead) and an output buffer (the results leave with a TMA store that has a whole
// tile period to drain).  No warp ever issues a global load or store of psi, and the DRAM traffic is spread over the
// whole period instead of coming in bursts between the transforms.  With 256 threads per SM the kernel has registers
// to spare: the k_y phases of a thread's 16 stored positions and its 15 stage-1 twiddles live in registers (loaded
// once from global memory), so shared memory holds only the twiddles of the later stages.
template <int NY, int LINES>
struct YSmemDB {
  static constexpr int EBUF = LINES * YLayout<NY, LINES>::LINE_PTS * 2;  // double2 elements
  static constexpr int STG = NY * LINES * 2;                             // staging / output, in double2 elements (c128)
  static constexpr int TW2 = tw_total<NY>() - tw_offset<NY>(2);          // twiddles of stages >= 2
  static constexpr size_t BYTES = (size_t)(EBUF + 2 * STG + TW2) * 16;
  static constexpr bool FITS = BYTES <= 227u * 1024u;
};

// CTA-wide exchanges, stage-1 twiddles in registers.  A three-stage transform has exactly one CTA-wide barrier (the
// exchange after stage 1); the kernel hangs its own hand-overs on it instead of adding barriers: with mode = 1
// thread 0 runs `after` behind the next barrier, with mode = 2 it runs `before` ahead of it (then mode returns to 0).
template <typename Before, typename After>
struct RegTwSync {
  static constexpr bool REG_TW1 = true;
  double2 tw1[15];  // the thread's stage-1 twiddles
  Before before;
  After after;
  int tid;
  mutable int mode;
  __device__ __forceinline__ RegTwSync(Before b, After a_, int tid_) : before(b), after(a_), tid(tid_), mode(0) {}
  // `before` belongs to thread 0 (which issues the stores it waits for), `after` to the first thread of warp 1, so
  // that the two chores do not pile up on one warp, whose delay the whole CTA would feel at the next barrier
  static constexpr int AFTER_TID = 32;
  __device__ __forceinline__ void sync() const {
    if (mode == 2 && tid == 0) before();
    __syncthreads();
    if (mode == 1 && tid == AFTER_TID) after();
    mode = 0;
  }
  __device__ __forceinline__ void acquire() const {}
  __device__ __forceinline__ void release() const {}
};

template <int DT, int NY, int LINES>
__global__ void __launch_bounds__(LINES * (NY / 8), 1) pass_y_db_kernel(const __grid_constant__ PassYArgs a) {
  typedef Plan<NY> P;
  typedef Store<DT> St;
  typedef typename St::elem elem;
  typedef YSmemDB<NY, LINES> SM;
  static_assert(P::NS == 3, "the double-buffered column pass is built for three-stage plans");
  extern __shared__ __align__(128) double2 smem[];
  constexpr int T = P::T;
  constexpr int NTHR = LINES * (NY / 8);
  constexpr int BR = NY < 256 ? NY : 256;
  constexpr unsigned TILE_BYTES = (unsigned)NY * LINES * 2 * (unsigned)sizeof(elem);
  const int tid = threadIdx.x;
  const int c = tid & 1;
  const int line = (tid >> 1) % LINES;
  const int t = (tid >> 1) / LINES;
  double2* buf = smem + (size_t)line * (YLayout<NY, LINES>::LINE_PTS * 2);
  elem* stg = reinterpret_cast<elem*>(smem + SM::EBUF);            // the next tile arrives here
  elem* out = reinterpret_cast<elem*>(smem + SM::EBUF + SM::STG);  // results leave from here
  double2* tw2S = smem + SM::EBUF + 2 * SM::STG;
  const double2* twS = tw2S - tw_offset<NY>(2);  // table base as line_fft.cuh indexes it; stage 1 is never read
  __shared__ __align__(8) unsigned long long mbar;
  __shared__ int next_s[2];
  pdl_launch_dependents();
  copy_table_async(tw2S, a.tw + tw_offset<NY>(2), SM::TW2, tid, NTHR);
  const int ngroups = a.nx / LINES;
  auto issue_loads = [&](int grp) {  // thread 0 only
    fence_proxy_async();
    mbar_expect_tx(&mbar, TILE_BYTES);
#pragma unroll
    for (int b = 0; b < NY / BR; ++b)
      tma_load_2d(stg + (size_t)b * BR * LINES * 2, &a.tmap_db, grp * LINES * 4, b * BR, &mbar);
  };
  // Work distribution: the tile of iteration it+1 is in `nxt`, fetched (atomic) one iteration ahead by thread 0 so
  // that its latency never sits in front of a barrier; published to the other threads through next_s.  (Held by
  // thread LT, the one that issues the loads.)
  int nxt = 0, it = 0;
  // hand-overs on the transforms' own barriers (thread 0):
  //  forward: behind the barrier every thread has taken its values out of the staging buffer -> load the next tile
  //  inverse: ahead of the barrier the store of the previous tile (issued a period ago) has released the output buffer
  constexpr int LT = 32;  // the thread that loads: first thread of warp 1 (RegTwSync::AFTER_TID)
  auto load_next = [&]() {
    if (nxt < ngroups) {
      issue_loads(nxt);
      nxt = sched_next(a.sched);  // consumed in the next iteration
      if (nxt < ngroups) {        // ... and asked into L2 a whole period before its load
#pragma unroll
        for (int b = 0; b < NY / BR; ++b) tma_prefetch_2d(&a.tmap_db, nxt * LINES * 4, b * BR);
      }
    } else {
      nxt = ngroups;
    }
  };
  auto drain_out = [&]() { if (it > 0) tma_store_wait_read(); };
  // per-thread constants kept in registers for the whole kernel (tables written before any pass kernel started, see
  // pass_y_kernel): the thread's 15 stage-1 twiddles and the k_y phases of its 16 stored positions
  RegTwSync<decltype(drain_out), decltype(load_next)> sy(drain_out, load_next, tid);
#pragma unroll
  for (int k = 1; k < 16; ++k) sy.tw1[k - 1] = __ldg(a.tw + tw_offset<NY>(1) + (k - 1) * (NY >> 4) + t);
  double2 eyr[16];
#pragma unroll
  for (int g = 0; g < P::G; ++g)
#pragma unroll
    for (int s = 0; s < P::RL; ++s) eyr[g * P::RL + s] = __ldg(a.eyk + (t + g * T) + (NY / P::RL) * s);
  // the loading thread initialises the barriers itself: its first expect_tx follows the initialisation in program
  // order (initialised by another warp, the first load could reach an uninitialised barrier and the tile would never
  // be seen as landed); every other thread meets the barriers behind the __syncthreads below
  if (tid == LT) {
    mbar_init(&mbar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  pdl_wait();
  if (tid == LT) {
    if ((int)blockIdx.x < ngroups) issue_loads(blockIdx.x);
    nxt = sched_next(a.sched);
  }
  cp_async_wait_all();
  __syncthreads();
  cplx v[16];
  TL_DECL(8);
  for (int grp = blockIdx.x; grp < ngroups; ++it) {
    // k_x phase of this column and component (applied here and not at the end of the row pass: there it costs
    // sixteen table loads per thread, here one); requested now, used after the forward transform
    double2 exv = make_double2(1.0, 0.0);
    if (a.exk != nullptr) exv = __ldg(a.exk + (size_t)c * a.nx + (size_t)grp * LINES + line);
    if (tid == LT) next_s[it & 1] = nxt;  // visible to everyone behind the forward transform's barrier
    mbar_wait(&mbar, it & 1);
    TL_MARK(0);
#pragma unroll
    for (int n = 0; n < 16; ++n) v[n] = St::cv(stg[((t + n * T) * LINES + line) * 2 + c]);
    TL_MARK(1);
    sy.mode = 1;
    line_fft_fwd<NY>(buf, twS, t, c, v, 0, sy);
    TL_MARK(2);
#pragma unroll
    for (int g = 0; g < P::G; ++g)
#pragma unroll
      for (int s = 0; s < P::RL; ++s) {
        const double2 f = eyr[g * P::RL + s];
        v[g * P::RL + s] = cmul(cmul(v[g * P::RL + s], mk(f.x, f.y)), mk(exv.x, exv.y));
      }
    TL_MARK(3);
    sy.mode = 2;
    line_fft_inv<NY>(buf, twS, t, c, v, 0, NoHook(), sy);
    TL_MARK(4);
    const int nxt_grp = next_s[it & 1];
#pragma unroll
    for (int n = 0; n < 16; ++n) out[((t + n * T) * LINES + line) * 2 + c] = St::el(v[n]);
    fence_proxy_async();  // these generic-proxy writes are read by the TMA store
    __syncthreads();
    TL_MARK(5);
    if (tid == 0) {
#pragma unroll
      for (int b = 0; b < NY / BR; ++b)
        tma_store_2d(&a.tmap_db, grp * LINES * 4, b * BR, out + (size_t)b * BR * LINES * 2);
      tma_store_commit();
    }
    TL_MARK(6);
    TL_TILE();
    grp = nxt_grp;
  }
  TL_DUMP("ydb wait|stage|fwd|ey|inv|out|store", 7);
  if (tid == 0) {
    tma_store_wait_all();
    sched_finish(a.sched);
  }
}

}  // namespace spgpe
