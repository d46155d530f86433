// common.cuh -- complex arithmetic in registers, storage-precision loads/stores, plan constants.
// Part of libspgpe (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// Phase timeline of the pass kernels (diagnostic builds only: nvcc -DSPGPE_TIMELINE).  Thread 0 of CTA 0 sums the
// cycles between successive marks over all its tiles and prints them once per launch.  Compiled out by default.
#ifdef SPGPE_TIMELINE
#include <stdio.h>
#define TL_DECL(n) long long tl_[n] = {}; long long tl_last_ = clock64(); int tl_n_ = 0
#define TL_MARK(i) do { const long long now_ = clock64(); tl_[i] += now_ - tl_last_; tl_last_ = now_; } while (0)
#define TL_TILE() (++tl_n_)
#define TL_DUMP(name, n)                                                                     \
  do {                                                                                       \
    if (blockIdx.x == 0 && threadIdx.x == 0 && tl_n_ > 0) {                                  \
      printf("TL %s tiles %d:", name, tl_n_);                                                \
      for (int i_ = 0; i_ < n; ++i_) printf(" %lld", tl_[i_] / tl_n_);                       \
      printf("\n");                                                                          \
    }                                                                                        \
  } while (0)
#else
#define TL_DECL(n)
#define TL_MARK(i)
#define TL_TILE()
#define TL_DUMP(name, n)
#endif

namespace spgpe {

// What a launcher needs to know about its handle: the device the handle lives on (the current device of the
// calling thread during every entry point, api.cu) and the diagnostic switches read once at spgpe_create.
struct LaunchEnv {
  int device;        // CUDA device ordinal of the handle
  int ctas_per_sm;   // SPGPE_DEBUG_CTAS_PER_SM: cap on resident CTAs per SM of the persistent kernels (0: none)
  int no_ydb;        // SPGPE_DEBUG_NO_YDB=1: column pass on the two-column kernel instead of the double-buffered one
  int xdbg;          // SPGPE_DEBUG_X: experiment switches of the row pass
};

struct cplx {
  double re, im;
};

__device__ __forceinline__ cplx mk(double r, double i) { cplx c; c.re = r; c.im = i; return c; }
__device__ __forceinline__ cplx operator+(cplx a, cplx b) { return mk(a.re + b.re, a.im + b.im); }
__device__ __forceinline__ cplx operator-(cplx a, cplx b) { return mk(a.re - b.re, a.im - b.im); }
// a * b
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return mk(fma(a.re, b.re, -(a.im * b.im)), fma(a.re, b.im, a.im * b.re));
}
// a * conj(b)
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {
  return mk(fma(a.re, b.re, a.im * b.im), fma(a.im, b.re, -(a.re * b.im)));
}
// multiply by +i (D=+1) or -i (D=-1)
template <int D>
__device__ __forceinline__ cplx mul_i(cplx a) {
  return D > 0 ? mk(-a.im, a.re) : mk(a.im, -a.re);
}

// A zero that the compiler cannot see through: g_zero is a __constant__ 0, so (bits of x) & g_zero is 0 but
// carries a data dependency on x.  Added to the index of a table load it pins the load after the producer
// of x; without it ptxas hoists all twiddle / phase-table loads to the top of the kernel and spills.
static __constant__ int g_zero = 0;
__device__ __forceinline__ int late_zero(double x) { return __double2hiint(x) & g_zero; }

// ---- storage precision: C128 = double2 per component, C64 = float2 per component -----------------
// psi streams through the kernels once per pass: its loads bypass L1 allocation (L1::no_allocate) so that the
// twiddle and phase tables, which every thread re-reads, stay resident there.
__device__ __forceinline__ double2 ldg_stream(const double2* p) {
  double2 v;
  asm volatile("ld.global.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ float2 ldg_stream(const float2* p) {
  float2 v;
  asm volatile("ld.global.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
  return v;
}

template <int DT> struct Store;
template <> struct Store<0> {
  typedef double real;
  typedef double2 elem;
  static __device__ __forceinline__ cplx ld(const void* base, size_t idx) {
    double2 v = ldg_stream(reinterpret_cast<const double2*>(base) + idx);
    return mk(v.x, v.y);
  }
  static __device__ __forceinline__ void st(void* base, size_t idx, cplx c) {
    reinterpret_cast<double2*>(base)[idx] = make_double2(c.re, c.im);
  }
  static __device__ __forceinline__ double ldr(const void* base, size_t idx) {
    return __ldg(reinterpret_cast<const double*>(base) + idx);
  }
  static __device__ __forceinline__ double lds(const void* base, int idx) {
    return reinterpret_cast<const double*>(base)[idx];
  }
  static __device__ __forceinline__ cplx cv(double2 e) { return mk(e.x, e.y); }
  static __device__ __forceinline__ double2 el(cplx c) { return make_double2(c.re, c.im); }
};
template <> struct Store<1> {
  typedef float real;
  typedef float2 elem;
  static __device__ __forceinline__ cplx ld(const void* base, size_t idx) {
    float2 v = ldg_stream(reinterpret_cast<const float2*>(base) + idx);
    return mk((double)v.x, (double)v.y);
  }
  static __device__ __forceinline__ void st(void* base, size_t idx, cplx c) {
    reinterpret_cast<float2*>(base)[idx] = make_float2((float)c.re, (float)c.im);
  }
  static __device__ __forceinline__ double ldr(const void* base, size_t idx) {
    return (double)__ldg(reinterpret_cast<const float*>(base) + idx);
  }
  static __device__ __forceinline__ double lds(const void* base, int idx) {
    return (double)reinterpret_cast<const float*>(base)[idx];
  }
  static __device__ __forceinline__ cplx cv(float2 e) { return mk((double)e.x, (double)e.y); }
  static __device__ __forceinline__ float2 el(cplx c) { return make_float2((float)c.re, (float)c.im); }
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// ---- asynchronous copies ------------------------------------------------------------------------------------
// 16-byte global -> shared copy that bypasses registers (LDGSTS); completion through cp_async_wait_all
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
// 8-byte variant (complex64 elements)
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_real(double* smem_dst, const double* gsrc) { cp_async8(smem_dst, gsrc); }
__device__ __forceinline__ void cp_async_real(float* smem_dst, const float* gsrc) { cp_async4(smem_dst, gsrc); }
__device__ __forceinline__ void cp_async_elem(double2* smem_dst, const double2* gsrc) { cp_async16(smem_dst, gsrc); }
__device__ __forceinline__ void cp_async_elem(float2* smem_dst, const float2* gsrc) { cp_async8(smem_dst, gsrc); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
// 1-D bulk copy global -> shared memory (one instruction for a whole row; bytes a multiple of 16, both addresses
// 16-byte aligned), completion on bar
__device__ __forceinline__ void bulk_load_1d(void* smem_dst, const void* gsrc, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(smem_dst)),
               "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
// L2 eviction policy for data that is read once per pass (the fields): evict first, so that the streams do not
// push the order parameter, which the next pass reads again, out of L2
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
  unsigned long long p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// bulk_load_1d with an L2 cache policy
__device__ __forceinline__ void bulk_load_1d_hint(void* smem_dst, const void* gsrc, unsigned bytes,
                                                  unsigned long long* bar, unsigned long long policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(smem_dst)),
      "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}
// ask L2 to fetch `bytes` (multiple of 16) starting at the 16-byte aligned address p; no registers, no scoreboard
__device__ __forceinline__ void prefetch_l2_bulk(const void* p, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// ---- TMA (cp.async.bulk.tensor) and mbarrier, raw PTX ----------------------------------------------------------
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// generic-proxy accesses to shared memory before this fence are ordered before later async-proxy (TMA) accesses
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 2-D tile global -> shared: box of the tensor map at (c0 = inner coordinate, c1 = row), completion on bar
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const void* tmap, int c0, int c1, unsigned long long* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
          smem_u32(smem_dst)),
      "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(bar))
      : "memory");
}

// ---- programmatic dependent launch ----------------------------------------------------------------------------
// The pass kernels are launched with programmatic stream serialization: a kernel may become resident while its
// predecessor drains, runs its prologue (table copies, barrier set-up) and then waits here for the predecessor's
// memory to be complete before it touches psi or the work counters.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// cooperative copy of n double2 entries global -> shared memory with cp.async (no register round trip)
__device__ __forceinline__ void copy_table_async(double2* dst, const double2* src, int n, int tid, int nthreads) {
  for (int i = tid; i < n; i += nthreads) cp_async16(dst + i, src + i);
}

// 2-D tile shared -> global (bulk async group); the shared-memory source may be reused after tma_store_wait_read
__device__ __forceinline__ void tma_store_2d(const void* tmap, int c0, int c1, const void* smem_src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(tmap), "r"(c0),
               "r"(c1), "r"(smem_u32(smem_src))
               : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// ask L2 to fetch the box of the tensor map at (c0, c1): spreads the DRAM reads of the next tile over the time the
// current one is being transformed (the later tma_load_2d then finds the data in L2)
__device__ __forceinline__ void tma_prefetch_2d(const void* tmap, int c0, int c1) {
  asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];" ::"l"(tmap), "r"(c0), "r"(c1) : "memory");
}

// ---- dynamic work distribution of the persistent pass kernels -------------------------------------------------
// sched[0] = number of groups handed out beyond the first gridDim.x, sched[1] = CTAs that have finished.  CTA b
// starts with group b and then takes gridDim.x + atomicAdd(sched[0], 1), so that fast SMs take more groups than
// slow ones.  The last CTA to finish resets both words for the next launch (launches on one stream are serial).
__device__ __forceinline__ int sched_next(int* sched) { return (int)gridDim.x + atomicAdd(&sched[0], 1); }
// returns true in the CTA that finishes last (every other CTA's global writes are visible to it)
__device__ __forceinline__ bool sched_finish(int* sched) {
  __threadfence();
  if (atomicAdd(&sched[1], 1) == (int)gridDim.x - 1) {
    sched[0] = 0;
    sched[1] = 0;
    __threadfence();
    return true;
  }
  return false;
}

// ---- transform plan: N = 16 * 16 * ... * R_LAST, every thread holds 16 points of one component ----
// Stage j (1-based) has radix 16 and stride M_j = N / 16^j; the last stage has radix R_LAST and the
// thread runs G = 16 / R_LAST butterflies on groups q = t + g*T of R_LAST consecutive positions.
template <int N> struct Plan;
#define SPGPE_PLAN(N_, NS_, RL_)                                             \
  template <> struct Plan<N_> {                                              \
    static constexpr int NS = NS_;     /* number of stages */               \
    static constexpr int RL = RL_;     /* radix of the last stage */        \
    static constexpr int T = N_ / 16;  /* threads per component per line */ \
    static constexpr int G = 16 / RL_; /* groups per thread, last stage */  \
    static constexpr int PADSHIFT = (RL_ == 16 ? 4 : RL_ == 4 ? 2 : 3);      \
    static constexpr int PTS = N_ + (N_ >> PADSHIFT); /* padded points */    \
  };
SPGPE_PLAN(64, 2, 4)
SPGPE_PLAN(128, 2, 8)
SPGPE_PLAN(256, 2, 16)
SPGPE_PLAN(512, 3, 2)
SPGPE_PLAN(1024, 3, 4)
SPGPE_PLAN(2048, 3, 8)
SPGPE_PLAN(4096, 3, 16)
#undef SPGPE_PLAN

// stride of radix-16 stage j (1-based, j < NS)
template <int N>
__host__ __device__ constexpr int stage_stride(int j) {
  int m = N;
  for (int i = 0; i < j; ++i) m /= 16;
  return m;
}

// offset of stage j's twiddle block in the per-N twiddle table: block j holds 15 * M_j entries,
// entry (k-1) * M_j + lo = exp(-2 pi i k lo / (16 M_j)), k = 1..15
template <int N>
__host__ __device__ constexpr int tw_offset(int j) {
  int off = 0;
  for (int i = 1; i < j; ++i) off += 15 * stage_stride<N>(i);
  return off;
}
template <int N>
__host__ __device__ constexpr int tw_total() {
  return tw_offset<N>(Plan<N>::NS);
}

}  // namespace spgpe
