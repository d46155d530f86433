/*
 * spgpe.h -- C ABI of libspgpe: the Strang time-splitting spectral step for the quasi-2D
 * two-component (pseudospinor) Gross-Pitaevskii equation of arXiv 2010.15069, on one NVIDIA
 * B200 (sm_100a).  Every step of the path runs in the library's own CUDA kernels; there is no
 * cuFFT, no CPU fallback and no host synchronisation inside spgpe_step.
 *
 * Citations: "P:Lnnn" = line of the paper text; "R-n" = reading n in DESIGN.md
 * section "Readings of the paper".
 *
 * Model (Eqs. 4-8, sign convention R-1):  i d/dt Psi = H Psi,  Psi = (psi_up, psi_dn),
 *   H = K + V(r) + (delta(r)/2) sigma_z + (Omega(r)/2) sigma_x + diag(g_uu n_up + g_ud n_dn, g_dd n_dn + g_ud n_up),
 *   K_up = ((k_x + k_L)^2 + k_y^2)/2,  K_dn = ((k_x - k_L)^2 + k_y^2)/2   (Eq. 5, R-2, R-3),  n_c = |psi_c|^2.
 * One step of size dt (Eq. 9, operator order R-4):
 *   Psi <- R(dt/2) F^-1 exp(-i K dt) F R(dt/2) Psi,
 * R(tau) = per-point 2x2 exponential exp(-i tau H_loc) in closed SU(2) form with the densities of the
 * Psi entering it (R-5, R-6).  Imaginary time replaces exp(-i . ) by exp(- . ) and
 * renormalises after every step (R-7).
 *
 * Layout.  Grid nx x ny, box [-Lx/2, Lx/2) x [-Ly/2, Ly/2) (R-9), x fastest:
 *   psi   : complex [ny][nx][2], component 0 = up, 1 = down, interleaved per point; one element is
 *           (re, im) of the working precision: 2 doubles (SPGPE_C128) or 2 floats (SPGPE_C64).
 *   fields: real [ny][nx] of the working precision (double or float); V, Omega, delta.
 * All sizes are in elements of that layout; nothing is padded.
 *
 * Pointers.  Arguments named d_* are DEVICE pointers, h_* are HOST pointers.  All arrays are owned by
 * the caller; set_* calls copy into library-owned storage (the caller's buffer may be reused once the
 * stream has passed that point), get_* calls copy out.  The handle owns psi, the three fields, the
 * tables and the reduction scratch.
 *
 * Errors.  Every call returns SPGPE_OK (0) or a negative code; nothing is printed, nothing aborts.
 * spgpe_step only enqueues work on the handle's stream; asynchronous kernel errors surface at the next
 * synchronising call (spgpe_norm, spgpe_energy, spgpe_get_psi_host, spgpe_synchronize).
 * NaN/Inf are propagated, not trapped.
 */
#ifndef SPGPE_H
#define SPGPE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spgpe_ctx* spgpe_handle; /* opaque */

enum { SPGPE_C128 = 0, SPGPE_C64 = 1 }; /* storage precision of psi and fields; arithmetic: DESIGN.md R-14 */
enum { SPGPE_NORM_PER_COMPONENT = 0, SPGPE_NORM_TOTAL = 1 }; /* R-7 */
enum { SPGPE_RS_EXPONENTIAL = 0, SPGPE_RS_NESTED = 1 };      /* form of the real-space part R(tau), R-5 / R-15 */

enum {
  SPGPE_OK = 0,
  SPGPE_ERR_INVALID_ARG = -1, /* NULL handle/pointer, non-positive size, unknown enum */
  SPGPE_ERR_UNSUPPORTED = -2, /* nx or ny not a power of two in [64, 8192] */
  SPGPE_ERR_NOT_READY = -3,   /* step/norm/energy/get before set_psi */
  SPGPE_ERR_CUDA = -4,        /* a CUDA call failed; spgpe_last_cuda_error() gives its text */
  SPGPE_ERR_NO_DEVICE = -5,   /* no CUDA device / not an sm_100 device */
  SPGPE_ERR_NO_MEMORY = -6,   /* host or device allocation failed in spgpe_create */
  SPGPE_ERR_TOO_LARGE = -7    /* spgpe_norm_noalloc: nx or ny beyond its fixed maximum of 8192 */
};

typedef struct {
  int dtype;               /* SPGPE_C128 | SPGPE_C64 */
  double g_uu, g_dd, g_ud; /* Eq. 7 */
  double k_L;              /* signed recoil wavenumber along x, Eq. 5, R-2; 0 disables the shift */
  int norm_mode;           /* imaginary-time renormalisation rule, R-7 */
} spgpe_params;

/* Create a solver for an nx x ny grid on the box of full widths Lx, Ly.  cuda_stream is a cudaStream_t
 * (NULL = the default stream); all work of the handle is enqueued on it.  Fields start as zero.  The handle lives on
 * the CUDA device that is current in the calling thread; later calls may come from any thread (one at a time per
 * handle) with any device current. */
int spgpe_create(spgpe_handle* out, int nx, int ny, double Lx, double Ly, const spgpe_params* p,
                 void* cuda_stream);
int spgpe_destroy(spgpe_handle h);

/* Fields of Eqs. 6 and 8: trap V(r), Raman coupling Omega(r) (real, R-11), Zeeman
 * detuning delta(r).  real [ny][nx]; NULL = zero everywhere. */
int spgpe_set_potential(spgpe_handle h, const void* d_V);
int spgpe_set_raman(spgpe_handle h, const void* d_Omega);
int spgpe_set_zeeman(spgpe_handle h, const void* d_delta);
int spgpe_set_potential_host(spgpe_handle h, const void* h_V);
int spgpe_set_raman_host(spgpe_handle h, const void* h_Omega);
int spgpe_set_zeeman_host(spgpe_handle h, const void* h_delta);

/* Order parameter in / out ("initial order parameter in, final order parameter available").
 * set_psi also captures the imaginary-time norm targets N_up, N_dn of the given state (R-7). */
int spgpe_set_psi(spgpe_handle h, const void* d_psi);
int spgpe_get_psi(spgpe_handle h, void* d_psi);
int spgpe_set_psi_host(spgpe_handle h, const void* h_psi); /* synchronous w.r.t. the host buffer */
int spgpe_get_psi_host(spgpe_handle h, void* h_psi);       /* synchronises the stream */
int spgpe_set_norm_targets(spgpe_handle h, double n_up, double n_dn);

/* n Strang steps of size dt.  imag != 0: imaginary time with dt = d tau > 0 and a
 * renormalisation after every step.  dt may be negative in real time; NaN or infinite dt, and dt <= 0 in imaginary
 * time, return SPGPE_ERR_INVALID_ARG.  A component whose norm is zero keeps scale 1 (it stays zero).  Asynchronous.
 * step(n) then step(m) equals step(n+m) to rounding.
 * Stream capture: the call only enqueues kernels on the handle's stream (no allocation, no synchronisation, no host
 * read-back; the imaginary-time rescale factors travel through device memory), so a caller may record it into a CUDA
 * graph (cudaStreamBeginCapture on that stream) and replay the graph; every replay advances the state by n steps,
 * bit-identical with the plain call (tests/test_gpu_graph.py).  Two conditions: the k-space tables of (dt, imag) are
 * built by the first call that uses them, so one plain call with the same (dt, imag) precedes the capture; and an
 * annealed schedule (spgpe_set_annealing) fixes its event indices at capture time and must not be replayed.
 * spgpe_profile must be off during a capture. */
int spgpe_step(spgpe_handle h, int n, double dt, int imag);

/* Form of the real-space part R(tau) used by later steps (host-side switch, no device work):
 *   SPGPE_RS_EXPONENTIAL (default): one 2x2 exponential of the whole local matrix, densities frozen at entry (R-5);
 *     second order in dt when Omega = 0 or all g are equal, first order otherwise.
 *   SPGPE_RS_NESTED: the paper's remark that the real-space operators "do not necessarily commute and should be split
 *     to second-order", read as (R-15)  R(tau) = D(tau/2) X(tau) D(tau/2),  D(s) = exp(-i s diag(d_up, d_dn)),
 *     d_up = V + g_uu n_up + g_ud n_dn + delta/2, d_dn = V + g_dd n_dn + g_ud n_up - delta/2 with the densities of the
 *     psi entering D, X(s) = exp(-i s (Omega/2) sigma_x); imaginary time with the decaying counterparts.  Second order
 *     for every parameter set and exactly reversible in real time.  No extra memory traffic. */
int spgpe_set_real_space_split(spgpe_handle h, int mode);

/* Annealing of imaginary-time runs ("we periodically 'annealed' the system with Gaussian noise"; the paper
 * states neither period nor amplitude: R-16).  Counting the imaginary-time steps taken since this call as j = 0, 1, ...,
 * the order parameter that enters step j receives complex Gaussian noise when every > 0, j > 0 and j % every == 0
 * (event k = j / every); the renormalisation at the end of that step restores the norms.  every = 0 switches it off.
 * The noise is a counter-based stream, the same for any launch geometry: element e = (iy*nx + ix)*2 + c of event k uses
 * q = k * (2 nx ny) + e and the uniforms U(2q), U(2q+1),
 *   U(j) = (mix64(seed + (j+1) * 0x9E3779B97F4A7C15) >> 11) * 2^-53          (output j of splitmix64),
 *   mix64(z): z ^= z >> 30; z *= 0xBF58476D1CE4E5B9; z ^= z >> 27; z *= 0x94D049BB133111EB; z ^= z >> 31,
 *   psi_e += (amp / sqrt 2) sqrt(-2 ln(1 - U(2q))) exp(2 pi i U(2q+1))       (<|noise|^2> = amp^2),
 * generated in fp64 inside the row pass (no extra sweep over psi).  amp >= 0. */
int spgpe_set_annealing(spgpe_handle h, int every, double amp, unsigned long long seed);

/* spgpe_step(n, dt, imag), n >= 1, with the observables accumulated inside the passes of the LAST step (no extra
 * sweep over psi); synchronises.  h_out (host, 12 doubles):
 *   [0..5]  of the final state: N_up, N_dn, I_uu = dx dy sum rho_up^2, I_dd, I_ud = dx dy sum rho_up rho_dn and the
 *           phase-separation parameter of Eq. 14 (system-averaged reading R-17)
 *           s = 1 - <rho_up rho_dn> / sqrt(<rho_up^2> <rho_dn^2>) = 1 - I_ud / sqrt(I_uu I_dd),  rho_c = |psi_c|^2;
 *   [6..11] of the order parameter in the middle of the last step (after its first half-step, in front of the k-space
 *           factor), from its transform psi^: M_c = (dx dy / nx ny) sum_k |psi^_c|^2 (= its N_c), kinetic energy
 *           T_c = (dx dy / nx ny) sum_k K_c |psi^_c|^2 (R-8) and x momentum P_c = (dx dy / nx ny) sum_k k_x |psi^_c|^2,
 *           in the order M_up, M_dn, T_up, T_dn, P_up, P_dn.
 * Grids with an axis longer than 4096 return SPGPE_ERR_UNSUPPORTED. */
int spgpe_step_observe(spgpe_handle h, int n, double dt, int imag, double h_out[12]);

/* N_c = dx dy sum_r |psi_c|^2 (R-8); out = {N_up, N_dn}; synchronises. */
int spgpe_norm(spgpe_handle h, double out[2]);
/* The same norms N_c = dx dy sum_r |psi_c|^2 (R-8) WITHOUT a handle and without any allocation, for callers that
 * cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
 *   d_psi : DEVICE pointer, complex [ny][nx][2] of `dtype` (SPGPE_C128 | SPGPE_C64), caller-owned, read only;
 *   d_out : DEVICE pointer to 2 doubles {N_up, N_dn}, caller-owned, written asynchronously on `cuda_stream`
 *           (a cudaStream_t, NULL = the default stream) of the CURRENT device; the call does not synchronise.
 * Limit: 1 <= nx, ny <= 8192 (no power-of-two requirement); anything larger returns SPGPE_ERR_TOO_LARGE and touches
 * nothing.  The reduction's scratch (1024 x 2 partial sums, 16 KiB) is a fixed device array inside the library that
 * every GPU loading the library holds until the process exits; its address is looked up once per device on the first
 * call there (make that call outside a graph capture).  All calls on a device share that array: calls that overlap on
 * the GPU (two streams, two host threads) race on it -- keep them on one stream or order them with events.  No slot of
 * it has to be cleared between calls (each call overwrites every slot before reading it).  Calls no cudaMalloc,
 * cudaFree or allocating library routine.  Same summation order as spgpe_norm (bit-identical results). */
int spgpe_norm_noalloc(const void* d_psi, int dtype, int nx, int ny, double Lx, double Ly, double* d_out,
                       void* cuda_stream);
/* Energy functional implied by Eqs. 4-8 (R-8), totals not per particle:
 * out = {total, kinetic, potential+Zeeman, interaction, Raman}; synchronises. */
int spgpe_energy(spgpe_handle h, double out[5]);

int spgpe_synchronize(spgpe_handle h);
/* Number of kernels the handle has launched so far (bench.py's gpu_launches claim). */
long long spgpe_launch_count(spgpe_handle h);
/* Per-launch timing with CUDA events on the handle's stream (measurement only; bench.py's roofline).
 * spgpe_profile(h, 1) synchronises and starts recording an event pair around every row-pass and column-pass
 * launch of later spgpe_step calls; spgpe_profile_read synchronises, returns the summed durations in
 * milliseconds and the launch counts per class (0 = row pass, 1 = column pass) and resets the record;
 * spgpe_profile(h, 0) stops.  Host arrays. */
int spgpe_profile(spgpe_handle h, int enable);
int spgpe_profile_read(spgpe_handle h, double h_ms[2], long long h_count[2]);
const char* spgpe_strerror(int code);
const char* spgpe_last_cuda_error(void);

/* Measurement helpers (not part of the method): peak probes used for bench.py's roofline denominators.
 * spgpe_probe_dfma / spgpe_probe_ffma: sustained fp64 / fp32 FMA rate of the device in TFLOP/s (2 flops per FMA).
 * spgpe_probe_copy: device-to-device copy bandwidth in GB/s (read + write bytes) over `bytes` bytes. */
int spgpe_probe_dfma(void* cuda_stream, double* tflops);
int spgpe_probe_ffma(void* cuda_stream, double* tflops);
int spgpe_probe_copy(void* cuda_stream, long long bytes, double* gbs);

#ifdef __cplusplus
}
#endif
#endif /* SPGPE_H */
