// api.cu -- the C ABI of include/spgpe.h: handle, uploads, step orchestration, norm, energy.
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <stdlib.h>

#include <new>
#include <vector>

#include <cuda.h>
#include <cudaTypedefs.h>

#include "../../include/spgpe.h"
#include "internal.h"

using namespace spgpe;

struct spgpe_ctx {
  int nx, ny;
  int sx, sy;  // 2: the axis is transformed as two interleaved sub-lines of length mx / my (split.cu), else 1
  int mx, my;  // line lengths of the pass kernels: nx / sx, ny / sy
  double Lx, Ly;
  spgpe_params p;
  cudaStream_t stream;
  LaunchEnv env;  // device of the handle and the diagnostic switches, read once at spgpe_create
  int dt;  // storage precision
  size_t points, field_bytes, psi_bytes;
  void* psi;
  void* scratch;  // second psi buffer, allocated by the first spgpe_energy
  void *Vbuf, *Ombuf, *Debuf;  // owned storage
  const void *V, *Om, *De;     // NULL = zero field
  double2 *tw_x, *tw_y;
  float4 *tw_x32, *tw_y32, *exk32, *eyk32;  // two-float twiddles and phase tables of the fp32 kernels (complex64 storage)
  int f32_dbg;           // SPGPE_DEBUG_NO_F32: 1 no fp32 kernels, 2 fp32 column pass only, 3 fp32 row pass only
  bool f32_ok;           // complex64 storage: the passes of plain steps run on the fp32 kernels (pass32.cuh)
  double *Kx, *Ky;       // kinetic tables in stored order: Kx[2][nx], Ky[ny]
  double* kxv;           // k_x in stored order [nx] (observables)
  double* kpartial;      // [KPARTIAL_ROWS][6] k-space sums of the observed column pass
  int rs_split;          // SPGPE_RS_EXPONENTIAL | SPGPE_RS_NESTED
  int anneal_every;      // annealing period in imaginary-time steps (0: off)
  double anneal_amp;
  unsigned long long anneal_seed;
  long long imag_steps;  // imaginary-time steps taken since spgpe_set_annealing
  double2 *exk, *eyk;    // phase tables of (tab_dt, tab_imag)
  double tab_dt;
  int tab_imag;
  bool tab_valid;
  double *partial, *scale, *target, *dout;
  CUtensorMap tmap_psi, tmap_scratch, tmap_psi_db, tmap_psi32;  // column-pass tensor maps of psi / the energy scratch buffer
  int* sched;    // [4] work counters of the persistent kernels: row pass [0..1], column pass [2..3]
  double2 *wcx, *wcy;         // split axes: join twiddles
  float4 *wcx32, *wcy32;      // ... as two-float values (fp32 join of complex64 storage)
  int *fpx, *fpy;             // split axes: true frequency of a sub-transform position
  double* fmax;  // [3] max |V|, |Omega|, |delta| (tier bounds of the row pass)
  int partial_cap;
  bool ready;
  long long launches;
  int ygrid;  // CTAs of the last column-pass launch
  int xgrid;  // CTAs of the last row-pass launch (rows of `partial` it wrote)
  HalfCoef hc;
  // per-launch CUDA-event timing (spgpe_profile): pairs of events around every row/column pass launch
  bool prof_on;
  std::vector<cudaEvent_t>* prof_ev;  // [2*i], [2*i+1] = start, stop of launch i
  std::vector<int>* prof_cls;         // class of launch i: 0 row pass, 1 column pass
  size_t prof_used;
};

static cudaError_t prof_begin(spgpe_ctx* h, int cls) {
  if (!h->prof_on) return cudaSuccess;
  if (h->prof_ev->size() < 2 * (h->prof_used + 1)) {
    cudaEvent_t a, b;
    cudaError_t e = cudaEventCreate(&a);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&b);
    if (e != cudaSuccess) return e;
    h->prof_ev->push_back(a);
    h->prof_ev->push_back(b);
    h->prof_cls->push_back(cls);
  }
  (*h->prof_cls)[h->prof_used] = cls;
  return cudaEventRecord((*h->prof_ev)[2 * h->prof_used], h->stream);
}
static cudaError_t prof_end(spgpe_ctx* h) {
  if (!h->prof_on) return cudaSuccess;
  cudaError_t e = cudaEventRecord((*h->prof_ev)[2 * h->prof_used + 1], h->stream);
  h->prof_used++;
  return e;
}

static thread_local char g_cuda_err[256] = "";
static const int KPARTIAL_ROWS = 4096;  // >= CTAs of any column-pass launch

// Every entry point that takes a handle runs with the handle's device current and restores the caller's device on
// return (a handle created on GPU 1 keeps working when the caller has switched to GPU 0 in between).
struct DeviceGuard {
  int prev;
  bool switched;
  cudaError_t err;
  explicit DeviceGuard(int dev) : prev(-1), switched(false), err(cudaSuccess) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) {
      err = cudaSetDevice(dev);
      switched = (err == cudaSuccess);
    }
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};
#define ON_DEVICE(h)                                   \
  DeviceGuard guard__((h)->env.device);                \
  if (guard__.err != cudaSuccess) return cuda_fail(guard__.err)

static int cuda_fail(cudaError_t e) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
  return SPGPE_ERR_CUDA;
}
#define CK(call)                                  \
  do {                                            \
    cudaError_t e__ = (call);                     \
    if (e__ != cudaSuccess) return cuda_fail(e__); \
  } while (0)

// Tensor map of a psi-shaped buffer for the column pass (pass_y.cuh): 2-D [ny rows][4 nx reals], box of
// min(ny, 256) rows x 4 * lines reals.  The driver entry point is looked up at run time (no libcuda link).
static cudaError_t make_col_tmap(const spgpe_ctx* h, void* base, int lines, CUtensorMap* out, int rows = 0) {
  // looked up once per process (the driver entry point is the same for every device); C++11 makes the
  // initialisation of a function-local static thread-safe
  static const PFN_cuTensorMapEncodeTiled_v12000 encode = []() -> PFN_cuTensorMapEncodeTiled_v12000 {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess) return nullptr;
    if (!fn || q != cudaDriverEntryPointSuccess) return nullptr;
    return (PFN_cuTensorMapEncodeTiled_v12000)fn;
  }();
  if (!encode) return cudaErrorNotSupported;
  const size_t rsz = (h->dt == SPGPE_C128) ? 8 : 4;
  // a split y axis is seen as my rows of sy * nx points: row r of that view holds the rows sy * r + p of the grid
  const cuuint64_t gdim[2] = {(cuuint64_t)h->nx * h->sy * 4, (cuuint64_t)h->my};
  const cuuint64_t gstride[1] = {(cuuint64_t)h->nx * h->sy * 4 * rsz};
  if (rows <= 0) rows = h->my < 256 ? h->my : 256;
  const cuuint32_t box[2] = {(cuuint32_t)lines * 4, (cuuint32_t)rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = encode(out, h->dt == SPGPE_C128 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                      base, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                      CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

static bool size_ok(int n) { return n >= 64 && n <= 8192 && (n & (n - 1)) == 0; }
// an axis is split when it is longer than the longest line of the pass kernels (or, for tests, when
// SPGPE_DEBUG_SPLIT_MIN asks for it)
static int split_of(int n, int nmin) { return n >= nmin ? 2 : 1; }
// the three diagnostic environment variables are read here, once per spgpe_create
static int env_int(const char* name) {
  const char* e = getenv(name);
  return e ? atoi(e) : 0;
}

static cudaError_t dispatch_x_raw(spgpe_ctx* h, int mode, const PassXArgs& a) {
  const int nl = h->ny * h->sx;  // lines
  // complex64 storage: the plain passes run on the fp32 kernels; the nested split, the observed closing pass, an
  // annealed opening pass and the transform-only mode stay on the fp64-arithmetic kernels (same layout)
  if (h->f32_ok && h->f32_dbg != 2 && a.tw32 != nullptr && !a.nest && (mode == MODE_PRO || mode == MODE_MID || mode == MODE_EPI) &&
      !(mode == MODE_PRO && a.anneal_event > 0) && (a.xs == 1 || h->mx >= 512)) {
    switch (h->mx) {
      case 64: return launch_row32_64(mode, a, nl, h->stream, h->env, &h->xgrid);
      case 128: return launch_row32_128(mode, a, nl, h->stream, h->env, &h->xgrid);
      case 256: return launch_row32_256(mode, a, nl, h->stream, h->env, &h->xgrid);
      case 512: return launch_row32_512(mode, a, nl, h->stream, h->env, &h->xgrid);
      case 1024: return launch_row32_1024(mode, a, nl, h->stream, h->env, &h->xgrid);
      case 2048: return launch_row32_2048(mode, a, nl, h->stream, h->env, &h->xgrid);
      default: return launch_row32_4096(mode, a, nl, h->stream, h->env, &h->xgrid);
    }
  }
  switch (h->mx) {
    case 64: return launch_pass_x_64(h->dt, mode, a, nl, h->stream, h->env, &h->xgrid);
    case 128: return launch_pass_x_128(h->dt, mode, a, nl, h->stream, h->env, &h->xgrid);
    case 256: return launch_pass_x_256(h->dt, mode, a, nl, h->stream, h->env, &h->xgrid);
    case 512: return launch_pass_x_512(h->dt, mode, a, nl, h->stream, h->env, &h->xgrid);
    case 1024: return launch_pass_x_1024(h->dt, mode, a, nl, h->stream, h->env, &h->xgrid);
    case 2048: return launch_pass_x_2048(h->dt, mode, a, nl, h->stream, h->env, &h->xgrid);
    default: return launch_pass_x_4096(h->dt, mode, a, nl, h->stream, h->env, &h->xgrid);
  }
}
static cudaError_t dispatch_y_raw(spgpe_ctx* h, int ymode, const PassYArgs& a) {
  if (h->f32_ok && h->f32_dbg != 3 && a.tw32 != nullptr && (ymode == YMODE_STEP || ymode == YMODE_FWDONLY || ymode == YMODE_INVONLY)) {
    switch (h->my) {
      case 64: return launch_col32_64(ymode, a, h->stream, h->env, &h->ygrid);
      case 128: return launch_col32_128(ymode, a, h->stream, h->env, &h->ygrid);
      case 256: return launch_col32_256(ymode, a, h->stream, h->env, &h->ygrid);
      case 512: return launch_col32_512(ymode, a, h->stream, h->env, &h->ygrid);
      case 1024: return launch_col32_1024(ymode, a, h->stream, h->env, &h->ygrid);
      case 2048: return launch_col32_2048(ymode, a, h->stream, h->env, &h->ygrid);
      default: return launch_col32_4096(ymode, a, h->stream, h->env, &h->ygrid);
    }
  }
  switch (h->my) {
    case 64: return launch_pass_y_64(h->dt, ymode, a, h->stream, h->env, &h->ygrid);
    case 128: return launch_pass_y_128(h->dt, ymode, a, h->stream, h->env, &h->ygrid);
    case 256: return launch_pass_y_256(h->dt, ymode, a, h->stream, h->env, &h->ygrid);
    case 512: return launch_pass_y_512(h->dt, ymode, a, h->stream, h->env, &h->ygrid);
    case 1024: return launch_pass_y_1024(h->dt, ymode, a, h->stream, h->env, &h->ygrid);
    case 2048: return launch_pass_y_2048(h->dt, ymode, a, h->stream, h->env, &h->ygrid);
    default: return launch_pass_y_4096(h->dt, ymode, a, h->stream, h->env, &h->ygrid);
  }
}

static cudaError_t dispatch_x(spgpe_ctx* h, int mode, const PassXArgs& a) {
  h->launches++;
  cudaError_t e = prof_begin(h, 0);
  if (e != cudaSuccess) return e;
  e = dispatch_x_raw(h, mode, a);
  if (e != cudaSuccess) return e;
  return prof_end(h);
}
static cudaError_t dispatch_y(spgpe_ctx* h, int ymode, const PassYArgs& a) {
  h->launches++;
  cudaError_t e = prof_begin(h, 1);
  if (e != cudaSuccess) return e;
  e = dispatch_y_raw(h, ymode, a);
  if (e != cudaSuccess) return e;
  return prof_end(h);
}

// kinetic tables in the stored order of the transforms (Eq. 5; R-2, R-3, R-9)
static void fill_ktables(const spgpe_ctx* h, std::vector<double>& Kx, std::vector<double>& Ky,
                         std::vector<double>& kxv) {
  const double two_pi = 6.283185307179586476925286766559;
  Kx.resize(2 * (size_t)h->nx);
  Ky.resize(h->ny);
  kxv.resize(h->nx);
  // unsplit axis: entry pos belongs to the frequency stored at pos.  Split axis (two sub-lines of m = n/2 points): entry
  // i*m + pos belongs to the frequency f + i*m of the joined spectrum, f = frequency stored at position pos of a
  // sub-transform -- the order in which the join kernel (split.cu) meets them, so that its table reads are coalesced
  auto freq_of_entry = [](int n, int split, int e) {
    if (split == 1) return plan_freq_of_pos(n, e);
    const int m = n / split;
    return plan_freq_of_pos(m, e % m) + (e / m) * m;
  };
  for (int pos = 0; pos < h->nx; ++pos) {
    const int f = freq_of_entry(h->nx, h->sx, pos);
    const int mt = (f < h->nx / 2) ? f : f - h->nx;
    const double k = two_pi * (double)mt / h->Lx;
    Kx[pos] = 0.5 * (k + h->p.k_L) * (k + h->p.k_L);
    Kx[h->nx + pos] = 0.5 * (k - h->p.k_L) * (k - h->p.k_L);
    kxv[pos] = k;
  }
  for (int pos = 0; pos < h->ny; ++pos) {
    const int f = freq_of_entry(h->ny, h->sy, pos);
    const int mt = (f < h->ny / 2) ? f : f - h->ny;
    const double k = two_pi * (double)mt / h->Ly;
    Ky[pos] = 0.5 * k * k;
  }
}

extern "C" int spgpe_create(spgpe_handle* out, int nx, int ny, double Lx, double Ly, const spgpe_params* p,
                            void* cuda_stream) {
  if (!out || !p || !(Lx > 0.0) || !(Ly > 0.0)) return SPGPE_ERR_INVALID_ARG;
  if (p->dtype != SPGPE_C128 && p->dtype != SPGPE_C64) return SPGPE_ERR_INVALID_ARG;
  if (p->norm_mode != SPGPE_NORM_PER_COMPONENT && p->norm_mode != SPGPE_NORM_TOTAL) return SPGPE_ERR_INVALID_ARG;
  if (!size_ok(nx) || !size_ok(ny)) return SPGPE_ERR_UNSUPPORTED;
  int dev = 0, ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return SPGPE_ERR_NO_DEVICE;
  CK(cudaGetDevice(&dev));
  int major = 0;
  CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  if (major != 10) return SPGPE_ERR_NO_DEVICE;

  spgpe_ctx* h = new (std::nothrow) spgpe_ctx();
  if (!h) return SPGPE_ERR_NO_MEMORY;
  memset(h, 0, sizeof(*h));
  h->nx = nx; h->ny = ny; h->Lx = Lx; h->Ly = Ly; h->p = *p;
  h->env.device = dev;
  h->env.ctas_per_sm = env_int("SPGPE_DEBUG_CTAS_PER_SM");
  h->env.no_ydb = env_int("SPGPE_DEBUG_NO_YDB");
  h->env.xdbg = env_int("SPGPE_DEBUG_X");
  int split_min = env_int("SPGPE_DEBUG_SPLIT_MIN");
  if (split_min < 128) split_min = 8192;
  h->sx = split_of(nx, split_min); h->sy = split_of(ny, split_min); h->mx = nx / h->sx; h->my = ny / h->sy;
  h->stream = (cudaStream_t)cuda_stream;
  h->dt = p->dtype;
  h->points = (size_t)nx * ny;
  const size_t rsz = (h->dt == SPGPE_C128) ? 8 : 4;
  h->field_bytes = h->points * rsz;
  h->psi_bytes = h->points * 4 * rsz;
  h->hc.ca_u = 0.5 * (p->g_uu + p->g_ud);
  h->hc.ca_d = 0.5 * (p->g_dd + p->g_ud);
  h->hc.cb_u = 0.5 * (p->g_uu - p->g_ud);
  h->hc.cb_d = 0.5 * (p->g_ud - p->g_dd);
  h->prof_ev = new (std::nothrow) std::vector<cudaEvent_t>();
  h->prof_cls = new (std::nothrow) std::vector<int>();
  if (!h->prof_ev || !h->prof_cls) {
    delete h->prof_ev;
    delete h->prof_cls;
    delete h;
    return SPGPE_ERR_NO_MEMORY;
  }
  h->partial_cap = 16 * (nx > ny ? nx : ny);  // up to 8 doubles per row group of the row pass (at most 2 ny groups)
  if (h->partial_cap < 4 * 2048) h->partial_cap = 4 * 2048;

  cudaError_t e = cudaSuccess;
  auto alloc = [&](void** ptr, size_t bytes) {
    if (e == cudaSuccess) e = cudaMalloc(ptr, bytes);
  };
  alloc(&h->psi, h->psi_bytes);
  alloc(&h->Vbuf, h->field_bytes);
  alloc(&h->Ombuf, h->field_bytes);
  alloc(&h->Debuf, h->field_bytes);
  const int twx = plan_tw_total(h->mx), twy = plan_tw_total(h->my);
  alloc((void**)&h->tw_x, sizeof(double2) * twx);
  alloc((void**)&h->tw_y, sizeof(double2) * twy);
  alloc((void**)&h->Kx, sizeof(double) * 2 * nx);
  alloc((void**)&h->Ky, sizeof(double) * ny);
  alloc((void**)&h->kxv, sizeof(double) * nx);
  alloc((void**)&h->kpartial, sizeof(double) * 6 * KPARTIAL_ROWS);
  alloc((void**)&h->exk, sizeof(double2) * 2 * nx);
  alloc((void**)&h->eyk, sizeof(double2) * ny);
  alloc((void**)&h->exk32, sizeof(float4) * 2 * nx);
  alloc((void**)&h->eyk32, sizeof(float4) * ny);
  alloc((void**)&h->tw_x32, sizeof(float4) * (twx > 0 ? twx : 1));
  alloc((void**)&h->tw_y32, sizeof(float4) * (twy > 0 ? twy : 1));
  h->f32_dbg = env_int("SPGPE_DEBUG_NO_F32");
  h->f32_ok = h->dt == SPGPE_C64 && h->f32_dbg != 1;
  alloc((void**)&h->partial, sizeof(double) * h->partial_cap);
  alloc((void**)&h->scale, sizeof(double) * 2);
  alloc((void**)&h->target, sizeof(double) * 2);
  alloc((void**)&h->dout, sizeof(double) * 24);
  alloc((void**)&h->sched, sizeof(int) * 4);
  if (e == cudaSuccess) e = cudaMemset(h->sched, 0, sizeof(int) * 4);
  alloc((void**)&h->fmax, sizeof(double) * 3);
  if (e == cudaSuccess) e = cudaMemset(h->fmax, 0, sizeof(double) * 3);
  if (e == cudaSuccess) {
    std::vector<double2> tw(twx > twy ? twx : twy);
    plan_fill_twiddles(h->mx, tw.data());
    e = cudaMemcpy(h->tw_x, tw.data(), sizeof(double2) * twx, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
      plan_fill_twiddles(h->my, tw.data());
      e = cudaMemcpy(h->tw_y, tw.data(), sizeof(double2) * twy, cudaMemcpyHostToDevice);
    }
    std::vector<float4> tw32(twx > twy ? twx : twy);
    if (e == cudaSuccess) {
      plan_fill_twiddles32(h->mx, tw32.data());
      e = cudaMemcpy(h->tw_x32, tw32.data(), sizeof(float4) * twx, cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess) {
      plan_fill_twiddles32(h->my, tw32.data());
      e = cudaMemcpy(h->tw_y32, tw32.data(), sizeof(float4) * twy, cudaMemcpyHostToDevice);
    }
  }
  if (e == cudaSuccess) {
    std::vector<double> Kx, Ky, kxv;
    fill_ktables(h, Kx, Ky, kxv);
    e = cudaMemcpy(h->Kx, Kx.data(), sizeof(double) * Kx.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(h->Ky, Ky.data(), sizeof(double) * Ky.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(h->kxv, kxv.data(), sizeof(double) * kxv.size(), cudaMemcpyHostToDevice);
  }
  // join tables of the split axes
  for (int ax = 0; ax < 2 && e == cudaSuccess; ++ax) {
    const int sp = ax ? h->sy : h->sx, n = ax ? ny : nx, m = n / sp;
    if (sp == 1) continue;
    std::vector<int> fp(m);
    std::vector<double2> wc(m);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int pos = 0; pos < m; ++pos) {
      fp[pos] = plan_freq_of_pos(m, pos);
      const long double ang = -two_pi * (long double)fp[pos] / (long double)n;
      wc[pos] = make_double2((double)cosl(ang), (double)sinl(ang));
    }
    int** dfp = ax ? &h->fpy : &h->fpx;
    double2** dwc = ax ? &h->wcy : &h->wcx;
    alloc((void**)dfp, sizeof(int) * m);
    alloc((void**)dwc, sizeof(double2) * m);
    if (e == cudaSuccess) e = cudaMemcpy(*dfp, fp.data(), sizeof(int) * m, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(*dwc, wc.data(), sizeof(double2) * m, cudaMemcpyHostToDevice);
    std::vector<float4> wc32(m);
    for (int pos = 0; pos < m; ++pos) {
      const float hr = (float)wc[pos].x, hi = (float)wc[pos].y;
      wc32[pos] = make_float4(hr, hi, (float)(wc[pos].x - (double)hr), (float)(wc[pos].y - (double)hi));
    }
    float4** dwc32 = ax ? &h->wcy32 : &h->wcx32;
    alloc((void**)dwc32, sizeof(float4) * m);
    if (e == cudaSuccess) e = cudaMemcpy(*dwc32, wc32.data(), sizeof(float4) * m, cudaMemcpyHostToDevice);
  }
  if (e == cudaSuccess) e = make_col_tmap(h, h->psi, plan_lines_y(h->my), &h->tmap_psi);
  if (e == cudaSuccess && h->f32_ok) e = make_col_tmap(h, h->psi, plan_lines_y32(h->my), &h->tmap_psi32);
  if (e == cudaSuccess && plan_lines_ydb(h->my) > 0) e = make_col_tmap(h, h->psi, plan_lines_ydb(h->my), &h->tmap_psi_db);
  if (e != cudaSuccess) {
    spgpe_destroy(h);
    return e == cudaErrorMemoryAllocation ? SPGPE_ERR_NO_MEMORY : cuda_fail(e);
  }
  *out = h;
  return SPGPE_OK;
}

extern "C" int spgpe_destroy(spgpe_handle h) {
  if (!h) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  cudaStreamSynchronize(h->stream);
  void* ptrs[] = {h->psi, h->scratch, h->Vbuf, h->Ombuf, h->Debuf, h->tw_x, h->tw_y, h->Kx, h->Ky, h->kxv, h->kpartial,
                  h->exk, h->eyk, h->exk32, h->eyk32, h->tw_x32, h->tw_y32, h->partial, h->scale, h->target, h->dout, h->fmax, h->sched, h->wcx, h->wcy, h->wcx32, h->wcy32, h->fpx, h->fpy};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  if (h->prof_ev) {
    for (cudaEvent_t ev : *h->prof_ev) cudaEventDestroy(ev);
    delete h->prof_ev;
    delete h->prof_cls;
  }
  delete h;
  return SPGPE_OK;
}

static int set_field(spgpe_handle h, const void* src, void* buf, const void** slot, cudaMemcpyKind kind) {
  if (!h) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  const int which = (buf == h->Vbuf) ? 0 : (buf == h->Ombuf ? 1 : 2);
  if (!src) {
    *slot = nullptr;
    CK(aux_absmax(h->dt, nullptr, 0, h->fmax + which, h->stream));
    return SPGPE_OK;
  }
  CK(cudaMemcpyAsync(buf, src, h->field_bytes, kind, h->stream));
  if (kind == cudaMemcpyHostToDevice) CK(cudaStreamSynchronize(h->stream));
  *slot = buf;
  h->launches++;
  CK(aux_absmax(h->dt, buf, h->points, h->fmax + which, h->stream));
  return SPGPE_OK;
}
extern "C" int spgpe_set_potential(spgpe_handle h, const void* d) {
  return h ? set_field(h, d, h->Vbuf, &h->V, cudaMemcpyDeviceToDevice) : SPGPE_ERR_INVALID_ARG;
}
extern "C" int spgpe_set_raman(spgpe_handle h, const void* d) {
  return h ? set_field(h, d, h->Ombuf, &h->Om, cudaMemcpyDeviceToDevice) : SPGPE_ERR_INVALID_ARG;
}
extern "C" int spgpe_set_zeeman(spgpe_handle h, const void* d) {
  return h ? set_field(h, d, h->Debuf, &h->De, cudaMemcpyDeviceToDevice) : SPGPE_ERR_INVALID_ARG;
}
extern "C" int spgpe_set_potential_host(spgpe_handle h, const void* p) {
  return h ? set_field(h, p, h->Vbuf, &h->V, cudaMemcpyHostToDevice) : SPGPE_ERR_INVALID_ARG;
}
extern "C" int spgpe_set_raman_host(spgpe_handle h, const void* p) {
  return h ? set_field(h, p, h->Ombuf, &h->Om, cudaMemcpyHostToDevice) : SPGPE_ERR_INVALID_ARG;
}
extern "C" int spgpe_set_zeeman_host(spgpe_handle h, const void* p) {
  return h ? set_field(h, p, h->Debuf, &h->De, cudaMemcpyHostToDevice) : SPGPE_ERR_INVALID_ARG;
}

static int norms_to(spgpe_handle h, double* d_out2) {
  const int nblk = 1024;
  h->launches += 2;
  CK(aux_norm_partials(h->dt, h->psi, h->points, h->partial, nblk, h->stream));
  CK(aux_sum_partials(h->partial, nblk, 2, (h->Lx / h->nx) * (h->Ly / h->ny), d_out2, h->stream));
  return SPGPE_OK;
}

static int set_psi_common(spgpe_handle h, const void* src, cudaMemcpyKind kind) {
  if (!h || !src) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  CK(cudaMemcpyAsync(h->psi, src, h->psi_bytes, kind, h->stream));
  if (kind == cudaMemcpyHostToDevice) CK(cudaStreamSynchronize(h->stream));
  h->ready = true;
  return norms_to(h, h->target);  // R-7: targets are the norms of the state handed in
}
extern "C" int spgpe_set_psi(spgpe_handle h, const void* d) { return set_psi_common(h, d, cudaMemcpyDeviceToDevice); }
extern "C" int spgpe_set_psi_host(spgpe_handle h, const void* p) { return set_psi_common(h, p, cudaMemcpyHostToDevice); }

extern "C" int spgpe_get_psi(spgpe_handle h, void* d) {
  if (!h || !d) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  if (!h->ready) return SPGPE_ERR_NOT_READY;
  CK(cudaMemcpyAsync(d, h->psi, h->psi_bytes, cudaMemcpyDeviceToDevice, h->stream));
  return SPGPE_OK;
}
extern "C" int spgpe_get_psi_host(spgpe_handle h, void* p) {
  if (!h || !p) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  if (!h->ready) return SPGPE_ERR_NOT_READY;
  CK(cudaMemcpyAsync(p, h->psi, h->psi_bytes, cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return SPGPE_OK;
}
extern "C" int spgpe_set_norm_targets(spgpe_handle h, double n_up, double n_dn) {
  if (!h || !(n_up > 0.0) || !(n_dn > 0.0)) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  h->launches++;
  CK(aux_set_targets(h->target, n_up, n_dn, h->stream));
  return SPGPE_OK;
}

static int ensure_tables(spgpe_handle h, double dt, int imag) {
  if (h->tab_valid && h->tab_dt == dt && h->tab_imag == imag) return SPGPE_OK;
  h->launches++;
  CK(aux_phase_tables(h->Kx, h->Ky, h->nx, h->ny, dt, imag, h->exk, h->eyk, h->exk32, h->eyk32, h->stream));
  h->tab_dt = dt; h->tab_imag = imag; h->tab_valid = true;
  return SPGPE_OK;
}

static SplitArgs split_args(spgpe_ctx* h, void* psi) {
  SplitArgs sa;
  memset(&sa, 0, sizeof(sa));
  sa.psi = psi; sa.nx = h->nx; sa.ny = h->ny; sa.fx = h->fpx; sa.fy = h->fpy; sa.wx = h->wcx; sa.wy = h->wcy;
  sa.phx = h->exk; sa.phy = h->eyk; sa.Kx = h->Kx; sa.Ky = h->Ky; sa.partial = h->partial;
  if (h->f32_ok && h->f32_dbg == 0) { sa.wx32 = h->wcx32; sa.wy32 = h->wcy32; sa.phx32 = h->exk32; sa.phy32 = h->eyk32; }
  return sa;
}

// y transform, k-space phase, inverse y transform (between two row passes).  Unsplit: one column pass.  With a
// split axis the join kernel (split.cu) applies the phases of the split axes on the joined spectrum.
static cudaError_t kspace_part(spgpe_ctx* h, const PassYArgs& ya) {
  cudaError_t e;
  if (h->sx == 1 && h->sy == 1) return dispatch_y(h, YMODE_STEP, ya);
  const SplitArgs sa = split_args(h, h->psi);
  if (h->sy == 1) {  // only x is split: join along x (any y), then the ordinary column pass
    h->launches++;
    if ((e = launch_split(h->dt, sa, 2, 1, 0, 1184, h->stream)) != cudaSuccess) return e;
    return dispatch_y(h, YMODE_STEP, ya);
  }
  if ((e = dispatch_y(h, YMODE_FWDONLY, ya)) != cudaSuccess) return e;
  h->launches++;
  if ((e = launch_split(h->dt, sa, h->sx, 2, 0, 1184, h->stream)) != cudaSuccess) return e;
  return dispatch_y(h, YMODE_INVONLY, ya);
}

// n Strang steps; obs != NULL: the last step's column pass and closing row pass also leave the sums of
// spgpe_step_observe, which are finished into h->dout[8..19] (device)
static int step_impl(spgpe_handle h, int n, double dt, int imag, bool obs) {
  if (!h || n < 0 || !(dt == dt) || isinf(dt)) return SPGPE_ERR_INVALID_ARG;
  imag = imag ? 1 : 0;
  if (imag && !(dt > 0.0)) return SPGPE_ERR_INVALID_ARG;  // imaginary time: dt = d tau > 0 (spgpe.h)
  if (!h->ready) return SPGPE_ERR_NOT_READY;
  if (obs && (n < 1 || h->sx != 1 || h->sy != 1)) return n < 1 ? SPGPE_ERR_INVALID_ARG : SPGPE_ERR_UNSUPPORTED;
  if (n == 0) return SPGPE_OK;
  ON_DEVICE(h);
  int rc = ensure_tables(h, dt, imag);
  if (rc) return rc;
  PassXArgs xa;
  memset(&xa, 0, sizeof(xa));
  xa.src = h->psi; xa.dst = h->psi; xa.V = h->V; xa.Om = h->Om; xa.De = h->De;
  xa.tw = h->tw_x; xa.tw32 = h->tw_x32; xa.scale = nullptr; xa.partial = h->partial;
  xa.tau = 0.5 * dt; xa.hc = h->hc; xa.imag = imag; xa.want_norm = imag; xa.ny = h->ny * h->sx; xa.xs = h->sx;
  xa.fmax = h->fmax; xa.sched = h->sched; xa.dbg = h->env.xdbg;
  xa.target = h->target; xa.scale_out = h->scale; xa.cell = (h->Lx / h->nx) * (h->Ly / h->ny); xa.norm_mode = h->p.norm_mode;
  xa.nest = h->rs_split == SPGPE_RS_NESTED; xa.pstride = 2;
  xa.anneal_seed = h->anneal_seed; xa.anneal_amp = h->anneal_amp; xa.anneal_elems = 2ULL * h->points;
  PassYArgs ya;
  memset(&ya, 0, sizeof(ya));
  ya.psi = h->psi; ya.tw = h->tw_y; ya.eyk = h->eyk; ya.nx = h->nx * h->sy;
  ya.tw32 = h->tw_y32; ya.eyk32 = h->eyk32; ya.tmap32 = h->tmap_psi32;
  ya.exk32 = (h->sx == 1 && h->sy == 1) ? h->exk32 : nullptr;
  // the k_x phase rides on the column pass unless a split axis sends the k-space phases to the join kernel
  ya.exk = (h->sx == 1 && h->sy == 1) ? h->exk : nullptr; ya.sched = h->sched + 2; ya.tmap = h->tmap_psi; ya.tmap_db = h->tmap_psi_db;
  // the observed column pass (last step only): k-space sums per CTA into kpartial
  auto last_kspace = [&]() -> cudaError_t {
    if (!obs) return kspace_part(h, ya);
    PassYArgs yo = ya;
    yo.Kx = h->Kx; yo.Ky = h->Ky; yo.kxv = h->kxv; yo.partial = h->kpartial;
    return dispatch_y(h, YMODE_STEP_OBS, yo);
  };
  if (!imag) {
    CK(dispatch_x(h, MODE_PRO, xa));
    for (int s = 1; s <= n; ++s) {
      if (s < n) CK(kspace_part(h, ya));
      else CK(last_kspace());
      if (s == n && obs) xa.pstride = 8;
      CK(dispatch_x(h, s < n ? MODE_MID : (obs ? MODE_EPI_OBS : MODE_EPI), xa));
    }
  } else {
    for (int s = 0; s < n; ++s) {
      const long long j = h->imag_steps + s;  // index of this step in the annealing schedule
      xa.anneal_event = (h->anneal_every > 0 && j > 0 && j % h->anneal_every == 0) ? j / h->anneal_every : 0;
      xa.scale = (s > 0) ? h->scale : nullptr;  // rescale of the previous step, applied at load
      CK(dispatch_x(h, MODE_PRO, xa));
      if (s + 1 < n) CK(kspace_part(h, ya));
      else CK(last_kspace());
      const bool last_obs = obs && s + 1 == n;
      if (last_obs) xa.pstride = 8;
      CK(dispatch_x(h, last_obs ? MODE_EPI_OBS : MODE_EPI, xa));  // also writes the rescale factors (last CTA)
    }
    h->imag_steps += n;
    h->launches++;
    CK(aux_apply_scale(h->dt, h->psi, h->points, h->scale, h->stream));
  }
  if (obs) {
    if (h->ygrid > KPARTIAL_ROWS) return SPGPE_ERR_UNSUPPORTED;
    h->launches += 2;
    CK(aux_obs_finish(h->partial, h->ny * h->sx / plan_lines_x(h->mx), 8, xa.cell, imag ? h->scale : nullptr,
                      h->dout + 8, h->stream));
    CK(aux_sum_partials(h->kpartial, h->ygrid, 6, xa.cell / ((double)h->nx * (double)h->ny), h->dout + 14, h->stream));
  }
  return SPGPE_OK;
}

extern "C" int spgpe_step(spgpe_handle h, int n, double dt, int imag) { return step_impl(h, n, dt, imag, false); }

extern "C" int spgpe_step_observe(spgpe_handle h, int n, double dt, int imag, double out[12]) {
  if (!out) return SPGPE_ERR_INVALID_ARG;
  int rc = step_impl(h, n, dt, imag, true);
  if (rc) return rc;
  ON_DEVICE(h);
  CK(cudaMemcpyAsync(out, h->dout + 8, 12 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return SPGPE_OK;
}

extern "C" int spgpe_set_real_space_split(spgpe_handle h, int mode) {
  if (!h || (mode != SPGPE_RS_EXPONENTIAL && mode != SPGPE_RS_NESTED)) return SPGPE_ERR_INVALID_ARG;
  h->rs_split = mode;
  return SPGPE_OK;
}

extern "C" int spgpe_set_annealing(spgpe_handle h, int every, double amp, unsigned long long seed) {
  if (!h || every < 0 || !(amp >= 0.0) || isinf(amp)) return SPGPE_ERR_INVALID_ARG;
  h->anneal_every = every;
  h->anneal_amp = amp;
  h->anneal_seed = seed;
  h->imag_steps = 0;
  return SPGPE_OK;
}

extern "C" int spgpe_norm(spgpe_handle h, double out[2]) {
  if (!h || !out) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  if (!h->ready) return SPGPE_ERR_NOT_READY;
  int rc = norms_to(h, h->dout);
  if (rc) return rc;
  CK(cudaMemcpyAsync(out, h->dout, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return SPGPE_OK;
}

extern "C" int spgpe_energy(spgpe_handle h, double out[5]) {
  if (!h || !out) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  if (!h->ready) return SPGPE_ERR_NOT_READY;
  if (!h->scratch) {
    CK(cudaMalloc(&h->scratch, h->psi_bytes));
    CK(make_col_tmap(h, h->scratch, plan_lines_y(h->my), &h->tmap_scratch));
  }
  const double w = (h->Lx / h->nx) * (h->Ly / h->ny);
  const int nblk = 1024;
  h->launches += 4;
  CK(aux_energy_partials(h->dt, h->psi, h->V, h->Om, h->De, h->points, h->p.g_uu, h->p.g_dd, h->p.g_ud,
                         h->partial, nblk, h->stream));
  CK(aux_sum_partials(h->partial, nblk, 3, w, h->dout + 2, h->stream));
  PassXArgs xa;
  memset(&xa, 0, sizeof(xa));
  xa.src = h->psi; xa.dst = h->scratch; xa.tw = h->tw_x; xa.ny = h->ny * h->sx; xa.xs = h->sx; xa.sched = h->sched; xa.fmax = h->fmax;
  CK(dispatch_x(h, MODE_FWD, xa));
  PassYArgs ya;
  memset(&ya, 0, sizeof(ya));
  ya.psi = h->scratch; ya.tw = h->tw_y; ya.Kx = h->Kx; ya.Ky = h->Ky; ya.partial = h->partial; ya.nx = h->nx * h->sy; ya.sched = h->sched + 2; ya.tmap = h->tmap_scratch;
  int kin_blocks;
  if (h->sx == 1 && h->sy == 1) {
    CK(dispatch_y(h, YMODE_ENERGY, ya));
    kin_blocks = h->ygrid;
  } else {  // full forward transform into the scratch buffer, then the join kernel sums K |psi^|^2
    CK(dispatch_y(h, YMODE_FWDONLY, ya));
    h->launches++;
    kin_blocks = 1024;
    CK(launch_split(h->dt, split_args(h, h->scratch), h->sx, h->sy, 1, kin_blocks, h->stream));
  }
  CK(aux_sum_partials(h->partial, kin_blocks, 1, w / ((double)h->nx * (double)h->ny), h->dout + 1,
                      h->stream));
  double tmp[5];
  CK(cudaMemcpyAsync(tmp + 1, h->dout + 1, 4 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  out[1] = tmp[1]; out[2] = tmp[2]; out[3] = tmp[3]; out[4] = tmp[4];
  out[0] = out[1] + out[2] + out[3] + out[4];
  return SPGPE_OK;
}

extern "C" int spgpe_synchronize(spgpe_handle h) {
  if (!h) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  CK(cudaStreamSynchronize(h->stream));
  return SPGPE_OK;
}
extern "C" int spgpe_profile(spgpe_handle h, int enable) {
  if (!h) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  CK(cudaStreamSynchronize(h->stream));
  h->prof_on = enable != 0;
  h->prof_used = 0;
  return SPGPE_OK;
}
extern "C" int spgpe_profile_read(spgpe_handle h, double ms[2], long long count[2]) {
  if (!h || !ms || !count) return SPGPE_ERR_INVALID_ARG;
  ON_DEVICE(h);
  CK(cudaStreamSynchronize(h->stream));
  ms[0] = ms[1] = 0.0;
  count[0] = count[1] = 0;
  for (size_t i = 0; i < h->prof_used; ++i) {
    float t = 0.f;
    CK(cudaEventElapsedTime(&t, (*h->prof_ev)[2 * i], (*h->prof_ev)[2 * i + 1]));
    const int c = (*h->prof_cls)[i];
    ms[c] += (double)t;
    count[c]++;
  }
  h->prof_used = 0;
  return SPGPE_OK;
}
extern "C" long long spgpe_launch_count(spgpe_handle h) { return h ? h->launches : -1; }

extern "C" const char* spgpe_strerror(int code) {
  switch (code) {
    case SPGPE_OK: return "ok";
    case SPGPE_ERR_INVALID_ARG: return "invalid argument";
    case SPGPE_ERR_UNSUPPORTED: return "unsupported grid size (nx, ny must be powers of two in [64, 8192])";
    case SPGPE_ERR_NOT_READY: return "no order parameter set (call spgpe_set_psi first)";
    case SPGPE_ERR_CUDA: return "CUDA error (see spgpe_last_cuda_error)";
    case SPGPE_ERR_NO_DEVICE: return "no sm_100 CUDA device";
    case SPGPE_ERR_NO_MEMORY: return "out of host or device memory";
    case SPGPE_ERR_TOO_LARGE: return "size beyond the fixed maximum of the no-allocation entry point (nx, ny <= 8192)";
    default: return "unknown error code";
  }
}
extern "C" const char* spgpe_last_cuda_error(void) { return g_cuda_err; }

extern "C" int spgpe_probe_dfma(void* cuda_stream, double* tflops) {
  if (!tflops) return SPGPE_ERR_INVALID_ARG;
  CK(aux_probe_dfma((cudaStream_t)cuda_stream, tflops));
  return SPGPE_OK;
}
extern "C" int spgpe_probe_ffma(void* cuda_stream, double* tflops) {
  if (!tflops) return SPGPE_ERR_INVALID_ARG;
  CK(aux_probe_ffma((cudaStream_t)cuda_stream, tflops));
  return SPGPE_OK;
}
extern "C" int spgpe_probe_copy(void* cuda_stream, long long bytes, double* gbs) {
  if (!gbs || bytes <= 0) return SPGPE_ERR_INVALID_ARG;
  CK(aux_probe_copy((cudaStream_t)cuda_stream, bytes, gbs));
  return SPGPE_OK;
}
