/*
 * spgpe_oracle.c -- CPU ORACLE for the Strang time-splitting spectral step of the
 * quasi-2D two-component Gross-Pitaevskii equation (arXiv 2010.15069).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant with the CUDA path under
 * paper_2010_15069_b200/csrc/.  Plain C, fp64 throughout, no blocking, fusion or
 * reordering beyond what the cited passages state; OpenMP only distributes
 * independent lines / points over threads (no arithmetic is reordered by it,
 * except the order of the partial sums in norm / energy).
 *
 * Citations: "P:Lnnn" = line of /root/reference/PAPER.md; "R-n" = reading n of
 * DESIGN.md section "Readings of the paper" (same numbering as SURVEY.md 8(c)).
 *
 * Parity pins (tests/test_oracle_*.py): every function below is pinned by at least one
 * check that does not come from this file: naive-DFT and numpy.fft equality, exact
 * plane-wave solution, Rabi closed form, scipy.linalg.expm for the SU(2) factor,
 * Eq. 11 band minima, Gaussian ground-state energy, decay rate e^{-tau} of the first
 * excited state, norm / energy conservation, reversibility, order of convergence;
 * the operator order of orc_step against a numpy.fft / scipy expm composition; the nested
 * split against per-point expm factors and its order 2 of convergence; the annealing noise
 * against an independent numpy evaluation of the same counter stream and its moments; the
 * observables against closed forms on uniform / separated states and numpy sums.
 * Nothing here is "parity unpinned".
 *
 * Layout (same as the C ABI of include/spgpe.h): psi[iy][ix][c] complex128, c = 0 (up),
 * 1 (down), x fastest, i.e. double index ((iy*nx + ix)*2 + c)*2 + {0: re, 1: im}.
 * Fields V, Omega, delta: double [iy][ix]; a NULL pointer means zero.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int nx, ny;              /* grid */
    double Lx, Ly;           /* full box widths: x in [-Lx/2, Lx/2) (R-9) */
    double g_uu, g_dd, g_ud; /* Eq. 7 */
    double k_L;              /* signed recoil wavenumber, Eq. 5, R-2 */
    int norm_mode;           /* 0: per component (BASELINE.json), 1: total, R-7 */
    int naive_max;           /* per-axis length up to which the O(N^2) DFT is used (default 32) */
    int rs_split;            /* real-space part: 0 = one 2x2 exponential (north_star, R-5),
                                1 = nested second-order split D(tau/2) X(tau) D(tau/2) (R-15) */
} orc_params;

static const double ORC_PI = 3.14159265358979323846264338327950288;

int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- grids (R-9): k_m = 2*pi*mt/L, mt = m for m < n/2, m - n otherwise;
 * the Nyquist index n/2 maps to -pi/dx.  FFT-native order. ---- */
void orc_kgrid(int n, double L, double *k) {
    for (int m = 0; m < n; ++m) {
        int mt = (m < n / 2) ? m : m - n;
        k[m] = 2.0 * ORC_PI * (double)mt / L;
    }
}
void orc_xgrid(int n, double L, double *x) {
    for (int j = 0; j < n; ++j) x[j] = -0.5 * L + (L / n) * (double)j;
}

/* ---- DFT: forward X_m = sum_j x_j e^{-2 pi i jm/N} (sign = -1),
 * inverse with e^{+...} (sign = +1); the 1/N of the inverse is applied by the caller.
 * a: interleaved (re, im), length n; out-of-place naive sum, angle reduced mod n in integers. */
void orc_dft_naive(const double *in, double *out, int n, int sign) {
    for (int m = 0; m < n; ++m) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < n; ++j) {
            long long jm = ((long long)j * (long long)m) % n;
            double ang = (double)sign * 2.0 * ORC_PI * (double)jm / (double)n;
            double c = cos(ang), s = sin(ang);
            double xr = in[2 * j], xi = in[2 * j + 1];
            sr += xr * c - xi * s;
            si += xr * s + xi * c;
        }
        out[2 * m] = sr;
        out[2 * m + 1] = si;
    }
}

/* Iterative radix-2 decimation-in-time FFT, in place, n a power of two.
 * tw: table of n/2 twiddles e^{sign * 2 pi i j / n}, j < n/2, each from cos/sin in double. */
static void fft_radix2_tw(double *a, int n, const double *tw) {
    /* bit reversal */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = a[2 * i], ti = a[2 * i + 1];
            a[2 * i] = a[2 * j];
            a[2 * i + 1] = a[2 * j + 1];
            a[2 * j] = tr;
            a[2 * j + 1] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int i = 0; i < n; i += len) {
            for (int j = 0; j < half; ++j) {
                double wr = tw[2 * (j * step)], wi = tw[2 * (j * step) + 1];
                double ur = a[2 * (i + j)], ui = a[2 * (i + j) + 1];
                double xr = a[2 * (i + j + half)], xi = a[2 * (i + j + half) + 1];
                double vr = xr * wr - xi * wi, vi = xr * wi + xi * wr;
                a[2 * (i + j)] = ur + vr;
                a[2 * (i + j) + 1] = ui + vi;
                a[2 * (i + j + half)] = ur - vr;
                a[2 * (i + j + half) + 1] = ui - vi;
            }
        }
    }
}

static void make_twiddles(double *tw, int n, int sign) {
    for (int j = 0; j < n / 2; ++j) {
        double ang = (double)sign * 2.0 * ORC_PI * (double)j / (double)n;
        tw[2 * j] = cos(ang);
        tw[2 * j + 1] = sin(ang);
    }
}

void orc_fft_radix2(double *a, int n, int sign) {
    double *tw = (double *)malloc(sizeof(double) * (size_t)(n > 1 ? n : 2));
    make_twiddles(tw, n, sign);
    fft_radix2_tw(a, n, tw);
    free(tw);
}

/* 1-D transform of `count` lines of one component of psi.  Line l starts at element offset
 * l*line_stride, consecutive points are elem_stride elements apart (elements = complex numbers
 * of the [iy][ix][c] array).  Naive DFT for n <= naive_max, radix-2 above. */
static void transform_lines(double *psi, int n, int count, size_t line_stride, size_t elem_stride,
                            size_t offset, int sign, int naive_max) {
    int use_naive = (n <= naive_max) || (n & (n - 1));
    double *tw = NULL;
    if (!use_naive) {
        tw = (double *)malloc(sizeof(double) * (size_t)n);
        make_twiddles(tw, n, sign);
    }
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 2 * (size_t)n);
        double *out = (double *)malloc(sizeof(double) * 2 * (size_t)n);
#pragma omp for schedule(static)
        for (int l = 0; l < count; ++l) {
            double *base = psi + 2 * (offset + (size_t)l * line_stride);
            for (int j = 0; j < n; ++j) {
                buf[2 * j] = base[2 * (size_t)j * elem_stride];
                buf[2 * j + 1] = base[2 * (size_t)j * elem_stride + 1];
            }
            double *res = buf;
            if (use_naive) {
                orc_dft_naive(buf, out, n, sign);
                res = out;
            } else {
                fft_radix2_tw(buf, n, tw);
            }
            for (int j = 0; j < n; ++j) {
                base[2 * (size_t)j * elem_stride] = res[2 * j];
                base[2 * (size_t)j * elem_stride + 1] = res[2 * j + 1];
            }
        }
        free(buf);
        free(out);
    }
    free(tw);
}

/* 2-D DFT of both components in place: all rows (x), then all columns (y).
 * sign = -1 forward (no scaling), +1 inverse (scaled by 1/(nx*ny)). */
void orc_fft2(double *psi, const orc_params *p, int sign) {
    const int nx = p->nx, ny = p->ny;
    for (int c = 0; c < 2; ++c) {
        /* rows: line iy starts at (iy*nx)*2 + c, points 2 elements apart */
        transform_lines(psi, nx, ny, (size_t)nx * 2, 2, (size_t)c, sign, p->naive_max);
        /* columns: line ix starts at ix*2 + c, points nx*2 elements apart */
        transform_lines(psi, ny, nx, 2, (size_t)nx * 2, (size_t)c, sign, p->naive_max);
    }
    if (sign > 0) {
        const double s = 1.0 / ((double)nx * (double)ny);
        const size_t n = (size_t)nx * ny * 4;
#pragma omp parallel for schedule(static)
        for (size_t i = 0; i < n; ++i) psi[i] *= s;
    }
}

/* ---- closed SU(2) form of the local 2x2 factor (BASELINE.json north_star;
 * operators of Eqs. 6-8; sign convention R-1: U = exp(-i H tau), imaginary time exp(-H tau)).
 * H_loc = a*1 + b_x sigma_x + b_z sigma_z.
 * real:  U = e^{-i a tau} [cos(theta) 1 - i sin(theta)/|b| (b_x sigma_x + b_z sigma_z)], theta = |b| tau
 * imag:  U = e^{-a tau}   [cosh(theta) 1 -  sinh(theta)/|b| (b_x sigma_x + b_z sigma_z)]
 * sin(theta)/|b| = tau*sinc: for |theta| < 1e-8 use tau (1 -+ theta^2/6); test on |theta| so tau < 0 works.
 * U (row-major 2x2 complex): U[0..1] = U_uu, U[2..3] = U_ud, U[4..5] = U_du, U[6..7] = U_dd. */
void orc_su2(double a, double bx, double bz, double tau, int imag, double *U) {
    double b = sqrt(bx * bx + bz * bz);
    double theta = b * tau;
    double c, s_over_b;
    if (!imag) {
        c = cos(theta);
        s_over_b = (fabs(theta) < 1e-8) ? tau * (1.0 - theta * theta / 6.0) : sin(theta) / b;
        /* M = c*1 - i s_over_b (bx sx + bz sz) */
        double m_uu_r = c, m_uu_i = -s_over_b * bz;
        double m_dd_r = c, m_dd_i = +s_over_b * bz;
        double m_od_r = 0.0, m_od_i = -s_over_b * bx;
        double pr = cos(a * tau), pi = -sin(a * tau); /* e^{-i a tau} */
        U[0] = pr * m_uu_r - pi * m_uu_i; U[1] = pr * m_uu_i + pi * m_uu_r;
        U[2] = pr * m_od_r - pi * m_od_i; U[3] = pr * m_od_i + pi * m_od_r;
        U[4] = U[2];                      U[5] = U[3];
        U[6] = pr * m_dd_r - pi * m_dd_i; U[7] = pr * m_dd_i + pi * m_dd_r;
    } else {
        c = cosh(theta);
        s_over_b = (fabs(theta) < 1e-8) ? tau * (1.0 + theta * theta / 6.0) : sinh(theta) / b;
        double e = exp(-a * tau);
        U[0] = e * (c - s_over_b * bz); U[1] = 0.0;
        U[2] = e * (-s_over_b * bx);    U[3] = 0.0;
        U[4] = U[2];                    U[5] = 0.0;
        U[6] = e * (c + s_over_b * bz); U[7] = 0.0;
    }
}

/* ---- real-space half-step R(tau) (Eqs. 6-8).
 * Densities are those of the psi that ENTERS the call (R-6).
 * d_up = V + g_uu n_up + g_ud n_dn + delta/2;  d_dn = V + g_dd n_dn + g_ud n_up - delta/2
 * a = (d_up + d_dn)/2, b_z = (d_up - d_dn)/2, b_x = Omega/2. */
void orc_half_nested(double *psi, const double *V, const double *Om, const double *de, const orc_params *p,
                     double tau, int imag);
void orc_half(double *psi, const double *V, const double *Om, const double *de, const orc_params *p,
              double tau, int imag) {
    const size_t P = (size_t)p->nx * p->ny;
    if (p->rs_split == 1) {
        orc_half_nested(psi, V, Om, de, p, tau, imag);
        return;
    }
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < P; ++i) {
        double ur = psi[4 * i], ui = psi[4 * i + 1], dr = psi[4 * i + 2], di = psi[4 * i + 3];
        double n_up = ur * ur + ui * ui, n_dn = dr * dr + di * di;
        double v = V ? V[i] : 0.0, om = Om ? Om[i] : 0.0, dl = de ? de[i] : 0.0;
        double d_up = v + p->g_uu * n_up + p->g_ud * n_dn + 0.5 * dl;
        double d_dn = v + p->g_dd * n_dn + p->g_ud * n_up - 0.5 * dl;
        double a = 0.5 * (d_up + d_dn), bz = 0.5 * (d_up - d_dn), bx = 0.5 * om;
        double U[8];
        orc_su2(a, bx, bz, tau, imag, U);
        psi[4 * i]     = U[0] * ur - U[1] * ui + U[2] * dr - U[3] * di;
        psi[4 * i + 1] = U[0] * ui + U[1] * ur + U[2] * di + U[3] * dr;
        psi[4 * i + 2] = U[4] * ur - U[5] * ui + U[6] * dr - U[7] * di;
        psi[4 * i + 3] = U[4] * ui + U[5] * ur + U[6] * di + U[7] * dr;
    }
}

/* ---- nested second-order real-space split (the real-space operators U^(2,3,4)
 * "do not necessarily commute and should be split to second-order"; reading R-15 of DESIGN.md):
 *   R_nested(tau) = D(tau/2) X(tau) D(tau/2)
 * D(s): the diagonal factors U^(2) U^(3) and the detuning: psi_c <- e^{-i s d_c} psi_c with
 *       d_up = V + g_uu n_up + g_ud n_dn + delta/2, d_dn = V + g_dd n_dn + g_ud n_up - delta/2 (Eqs. 6-7),
 *       densities of the psi that enters D (a diagonal phase does not change them); imaginary time e^{-s d_c}.
 * X(s): the Raman factor U^(4) = exp(-i s (Omega/2) sigma_x) (Eq. 8): with th = s Omega/2,
 *       psi_up <- cos(th) psi_up - i sin(th) psi_dn, psi_dn <- -i sin(th) psi_up + cos(th) psi_dn;
 *       imaginary time: cosh(th), -sinh(th).
 * The second D uses the densities after X (refreshed), which is what makes the product symmetric. */
static void nested_diag(double *q, double v, double dl, const orc_params *p, double s, int imag) {
    double n_up = q[0] * q[0] + q[1] * q[1], n_dn = q[2] * q[2] + q[3] * q[3];
    double d_up = v + p->g_uu * n_up + p->g_ud * n_dn + 0.5 * dl;
    double d_dn = v + p->g_dd * n_dn + p->g_ud * n_up - 0.5 * dl;
    if (!imag) {
        double cu = cos(d_up * s), su = -sin(d_up * s), cd = cos(d_dn * s), sd = -sin(d_dn * s);
        double ur = q[0], ui = q[1], dr = q[2], di = q[3];
        q[0] = ur * cu - ui * su; q[1] = ur * su + ui * cu;
        q[2] = dr * cd - di * sd; q[3] = dr * sd + di * cd;
    } else {
        double eu = exp(-d_up * s), ed = exp(-d_dn * s);
        q[0] *= eu; q[1] *= eu; q[2] *= ed; q[3] *= ed;
    }
}
void orc_half_nested(double *psi, const double *V, const double *Om, const double *de, const orc_params *p,
                     double tau, int imag) {
    const size_t P = (size_t)p->nx * p->ny;
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < P; ++i) {
        double *q = psi + 4 * i;
        double v = V ? V[i] : 0.0, om = Om ? Om[i] : 0.0, dl = de ? de[i] : 0.0;
        nested_diag(q, v, dl, p, 0.5 * tau, imag);
        double th = 0.5 * om * tau;
        double ur = q[0], ui = q[1], dr = q[2], di = q[3];
        if (!imag) {
            double c = cos(th), s = sin(th);
            /* -i s (a + i b) = s b - i s a */
            q[0] = c * ur + s * di; q[1] = c * ui - s * dr;
            q[2] = c * dr + s * ui; q[3] = c * di - s * ur;
        } else {
            double c = cosh(th), s = sinh(th);
            q[0] = c * ur - s * dr; q[1] = c * ui - s * di;
            q[2] = c * dr - s * ur; q[3] = c * di - s * ui;
        }
        nested_diag(q, v, dl, p, 0.5 * tau, imag);
    }
}

/* kinetic energies in k space (Eq. 5 P:L111 with the readings R-1, R-2, R-3):
 * K_up = ((k_x + k_L)^2 + k_y^2)/2, K_dn = ((k_x - k_L)^2 + k_y^2)/2.
 * Kx_up, Kx_dn: nx values ((k_x +- k_L)^2/2); Ky: ny values (k_y^2/2). */
void orc_kinetic_tables(const orc_params *p, double *Kx_up, double *Kx_dn, double *Ky) {
    double *kx = (double *)malloc(sizeof(double) * (size_t)p->nx);
    double *ky = (double *)malloc(sizeof(double) * (size_t)p->ny);
    orc_kgrid(p->nx, p->Lx, kx);
    orc_kgrid(p->ny, p->Ly, ky);
    for (int m = 0; m < p->nx; ++m) {
        Kx_up[m] = 0.5 * (kx[m] + p->k_L) * (kx[m] + p->k_L);
        Kx_dn[m] = 0.5 * (kx[m] - p->k_L) * (kx[m] - p->k_L);
    }
    for (int m = 0; m < p->ny; ++m) Ky[m] = 0.5 * ky[m] * ky[m];
    free(kx);
    free(ky);
}

/* ---- kinetic step: 2-D DFT of each component, multiply by
 * e^{-i K_c dt} (imaginary time e^{-K_c dt}), inverse 2-D DFT. */
void orc_kinetic(double *psi, const orc_params *p, double dt, int imag) {
    const int nx = p->nx, ny = p->ny;
    double *Kxu = (double *)malloc(sizeof(double) * (size_t)nx);
    double *Kxd = (double *)malloc(sizeof(double) * (size_t)nx);
    double *Ky = (double *)malloc(sizeof(double) * (size_t)ny);
    orc_kinetic_tables(p, Kxu, Kxd, Ky);
    orc_fft2(psi, p, -1);
#pragma omp parallel for schedule(static)
    for (int iy = 0; iy < ny; ++iy) {
        for (int ix = 0; ix < nx; ++ix) {
            size_t i = (size_t)iy * nx + ix;
            for (int c = 0; c < 2; ++c) {
                double K = (c == 0 ? Kxu[ix] : Kxd[ix]) + Ky[iy];
                double re = psi[4 * i + 2 * c], im = psi[4 * i + 2 * c + 1];
                if (!imag) {
                    double cr = cos(K * dt), ci = -sin(K * dt);
                    psi[4 * i + 2 * c] = re * cr - im * ci;
                    psi[4 * i + 2 * c + 1] = re * ci + im * cr;
                } else {
                    double e = exp(-K * dt);
                    psi[4 * i + 2 * c] = re * e;
                    psi[4 * i + 2 * c + 1] = im * e;
                }
            }
        }
    }
    orc_fft2(psi, p, +1);
    free(Kxu);
    free(Kxd);
    free(Ky);
}

/* ---- norms (R-8): N_c = dx dy sum_r |psi_c|^2 */
void orc_norm(const double *psi, const orc_params *p, double *out) {
    const size_t P = (size_t)p->nx * p->ny;
    double su = 0.0, sd = 0.0;
#pragma omp parallel for reduction(+ : su, sd) schedule(static)
    for (size_t i = 0; i < P; ++i) {
        su += psi[4 * i] * psi[4 * i] + psi[4 * i + 1] * psi[4 * i + 1];
        sd += psi[4 * i + 2] * psi[4 * i + 2] + psi[4 * i + 3] * psi[4 * i + 3];
    }
    const double w = (p->Lx / p->nx) * (p->Ly / p->ny);
    out[0] = w * su;
    out[1] = w * sd;
}

/* ---- n Strang steps (operator order R-4; P:L138 for the renormalisation):
 * half(dt/2) -> kinetic(dt) -> half(dt/2) -> if imag: norms and rescale to targets (R-7). */
/* a6 (R-7): rescale to the target norms, per component or in total */
static void renormalise(double *psi, const orc_params *p, const double *targets) {
    const size_t P = (size_t)p->nx * p->ny;
    double nn[2], su, sd;
    orc_norm(psi, p, nn);
    if (p->norm_mode == 0) {
        su = sqrt(targets[0] / nn[0]);
        sd = sqrt(targets[1] / nn[1]);
    } else {
        su = sd = sqrt((targets[0] + targets[1]) / (nn[0] + nn[1]));
    }
#pragma omp parallel for schedule(static)
    for (size_t i = 0; i < P; ++i) {
        psi[4 * i] *= su;
        psi[4 * i + 1] *= su;
        psi[4 * i + 2] *= sd;
        psi[4 * i + 3] *= sd;
    }
}
void orc_step(double *psi, const double *V, const double *Om, const double *de, const orc_params *p,
              int n, double dt, int imag, const double *targets) {
    for (int s = 0; s < n; ++s) {
        orc_half(psi, V, Om, de, p, 0.5 * dt, imag);
        orc_kinetic(psi, p, dt, imag);
        orc_half(psi, V, Om, de, p, 0.5 * dt, imag);
        if (imag) renormalise(psi, p, targets);
    }
}

/* ---- energy (R-8): out = {total, kinetic, potential+Zeeman, interaction, Raman}
 * kinetic = (dx dy/(nx ny)) sum_k [K_up |psi^_up|^2 + K_dn |psi^_dn|^2]
 * pot+Z   = dx dy sum_r [V (n_up + n_dn) + (delta/2)(n_up - n_dn)]
 * inter   = dx dy sum_r [(g_uu/2) n_up^2 + (g_dd/2) n_dn^2 + g_ud n_up n_dn]
 * Raman   = dx dy sum_r Omega Re(conj(psi_up) psi_dn)            (totals, not per particle) */
void orc_energy(const double *psi, const double *V, const double *Om, const double *de, const orc_params *p,
                double *out) {
    const int nx = p->nx, ny = p->ny;
    const size_t P = (size_t)nx * ny;
    const double w = (p->Lx / nx) * (p->Ly / ny);
    double ep = 0.0, ei = 0.0, er = 0.0, ek = 0.0;
#pragma omp parallel for reduction(+ : ep, ei, er) schedule(static)
    for (size_t i = 0; i < P; ++i) {
        double ur = psi[4 * i], ui = psi[4 * i + 1], dr = psi[4 * i + 2], di = psi[4 * i + 3];
        double n_up = ur * ur + ui * ui, n_dn = dr * dr + di * di;
        double v = V ? V[i] : 0.0, om = Om ? Om[i] : 0.0, dl = de ? de[i] : 0.0;
        ep += v * (n_up + n_dn) + 0.5 * dl * (n_up - n_dn);
        ei += 0.5 * p->g_uu * n_up * n_up + 0.5 * p->g_dd * n_dn * n_dn + p->g_ud * n_up * n_dn;
        er += om * (ur * dr + ui * di);
    }
    double *hat = (double *)malloc(sizeof(double) * 4 * P);
    memcpy(hat, psi, sizeof(double) * 4 * P);
    orc_fft2(hat, p, -1);
    double *Kxu = (double *)malloc(sizeof(double) * (size_t)nx);
    double *Kxd = (double *)malloc(sizeof(double) * (size_t)nx);
    double *Ky = (double *)malloc(sizeof(double) * (size_t)ny);
    orc_kinetic_tables(p, Kxu, Kxd, Ky);
#pragma omp parallel for reduction(+ : ek) schedule(static)
    for (int iy = 0; iy < ny; ++iy) {
        for (int ix = 0; ix < nx; ++ix) {
            size_t i = (size_t)iy * nx + ix;
            double n_up = hat[4 * i] * hat[4 * i] + hat[4 * i + 1] * hat[4 * i + 1];
            double n_dn = hat[4 * i + 2] * hat[4 * i + 2] + hat[4 * i + 3] * hat[4 * i + 3];
            ek += (Kxu[ix] + Ky[iy]) * n_up + (Kxd[ix] + Ky[iy]) * n_dn;
        }
    }
    free(hat);
    free(Kxu);
    free(Kxd);
    free(Ky);
    out[1] = w * ek / ((double)nx * (double)ny);
    out[2] = w * ep;
    out[3] = w * ei;
    out[4] = w * er;
    out[0] = out[1] + out[2] + out[3] + out[4];
}

/* ---- annealing noise ("we periodically 'annealed' the system with Gaussian noise to
 * more quickly find the ground state"; the paper gives neither amplitude nor period: reading R-16 of DESIGN.md).
 * Counter-based generator (its own implementation here; the CUDA path implements the same definition):
 *   U(j)  = (mix64(seed + (j+1) * 0x9E3779B97F4A7C15) >> 11) * 2^-53      (splitmix64 output j, 53-bit uniform in [0,1))
 *   mix64(z): z ^= z >> 30; z *= 0xBF58476D1CE4E5B9; z ^= z >> 27; z *= 0x94D049BB133111EB; z ^= z >> 31
 * Element e = (iy*nx + ix)*2 + c of annealing event k >= 1 uses the counter q = k * (2 nx ny) + e and the pair
 * u1 = U(2q), u2 = U(2q+1):  r = sqrt(-2 ln(1 - u1)),  xi = r (cos 2 pi u2 + i sin 2 pi u2)   (Box-Muller),
 *   psi_e <- psi_e + (amp / sqrt 2) xi        (re and im each N(0, amp^2 / 2), so <|noise|^2> = amp^2). */
static unsigned long long orc_mix64(unsigned long long z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}
static double orc_uniform(unsigned long long seed, unsigned long long j) {
    unsigned long long z = orc_mix64(seed + (j + 1ULL) * 0x9E3779B97F4A7C15ULL);
    return (double)(z >> 11) * (1.0 / 9007199254740992.0);
}
void orc_anneal_noise(double *psi, const orc_params *p, unsigned long long seed, long long event, double amp) {
    const size_t E = (size_t)p->nx * p->ny * 2;
    const double a = amp / sqrt(2.0);
#pragma omp parallel for schedule(static)
    for (size_t e = 0; e < E; ++e) {
        unsigned long long q = (unsigned long long)event * (unsigned long long)E + (unsigned long long)e;
        double u1 = orc_uniform(seed, 2ULL * q), u2 = orc_uniform(seed, 2ULL * q + 1ULL);
        double r = sqrt(-2.0 * log1p(-u1));
        double ang = 2.0 * ORC_PI * u2;
        psi[2 * e] += a * r * cos(ang);
        psi[2 * e + 1] += a * r * sin(ang);
    }
}

/* n imaginary-time steps with annealing: j = first_step + s is the index of the step since the schedule began;
 * when every > 0, j > 0 and j % every == 0 the noise of event j / every is added to the order parameter that enters
 * step j (the renormalisation at the end of that step restores the norms). */
void orc_step_anneal(double *psi, const double *V, const double *Om, const double *de, const orc_params *p,
                     int n, double dt, const double *targets, long long first_step, int every, double amp,
                     unsigned long long seed) {
    for (int s = 0; s < n; ++s) {
        long long j = first_step + s;
        if (every > 0 && j > 0 && j % every == 0) orc_anneal_noise(psi, p, seed, j / every, amp);
        orc_step(psi, V, Om, de, p, 1, dt, 1, targets);
    }
}

/* ---- observables.
 * Real space (out_r[6]): N_up, N_dn (R-8), I_uu = dx dy sum rho_up^2, I_dd = dx dy sum rho_dn^2,
 * I_ud = dx dy sum rho_up rho_dn, and the phase-separation parameter of Eq. 14 (the printed equation carries
 * both a sum over r and system averages: reading R-17, the system-averaged form)
 *   s = 1 - <rho_up rho_dn> / sqrt(<rho_up^2> <rho_dn^2>) = 1 - I_ud / sqrt(I_uu I_dd),  rho_c = |psi_c|^2.
 * k space (out_k[6]) of a TRANSFORMED order parameter hat = F psi (unnormalised forward DFT), per component c:
 *   M_c = (dx dy/(nx ny)) sum_k |hat_c|^2 (= N_c, Parseval), T_c = (dx dy/(nx ny)) sum_k K_c(k) |hat_c|^2 (kinetic
 *   energy, R-8), P_c = (dx dy/(nx ny)) sum_k k_x |hat_c|^2 (x momentum); order: M_up, M_dn, T_up, T_dn, P_up, P_dn. */
void orc_observables(const double *psi, const orc_params *p, double *out_r) {
    const size_t P = (size_t)p->nx * p->ny;
    const double w = (p->Lx / p->nx) * (p->Ly / p->ny);
    double nu = 0.0, nd = 0.0, uu = 0.0, dd = 0.0, ud = 0.0;
#pragma omp parallel for reduction(+ : nu, nd, uu, dd, ud) schedule(static)
    for (size_t i = 0; i < P; ++i) {
        double ru = psi[4 * i] * psi[4 * i] + psi[4 * i + 1] * psi[4 * i + 1];
        double rd = psi[4 * i + 2] * psi[4 * i + 2] + psi[4 * i + 3] * psi[4 * i + 3];
        nu += ru; nd += rd; uu += ru * ru; dd += rd * rd; ud += ru * rd;
    }
    out_r[0] = w * nu; out_r[1] = w * nd; out_r[2] = w * uu; out_r[3] = w * dd; out_r[4] = w * ud;
    out_r[5] = 1.0 - ud / sqrt(uu * dd);
}
void orc_kspace_observables(const double *hat, const orc_params *p, double *out_k) {
    const int nx = p->nx, ny = p->ny;
    const double w = (p->Lx / nx) * (p->Ly / ny) / ((double)nx * (double)ny);
    double *Kxu = (double *)malloc(sizeof(double) * (size_t)nx);
    double *Kxd = (double *)malloc(sizeof(double) * (size_t)nx);
    double *Ky = (double *)malloc(sizeof(double) * (size_t)ny);
    double *kx = (double *)malloc(sizeof(double) * (size_t)nx);
    orc_kinetic_tables(p, Kxu, Kxd, Ky);
    orc_kgrid(nx, p->Lx, kx);
    double mu = 0.0, md = 0.0, tu = 0.0, td = 0.0, pu = 0.0, pd = 0.0;
#pragma omp parallel for reduction(+ : mu, md, tu, td, pu, pd) schedule(static)
    for (int iy = 0; iy < ny; ++iy) {
        for (int ix = 0; ix < nx; ++ix) {
            size_t i = (size_t)iy * nx + ix;
            double ru = hat[4 * i] * hat[4 * i] + hat[4 * i + 1] * hat[4 * i + 1];
            double rd = hat[4 * i + 2] * hat[4 * i + 2] + hat[4 * i + 3] * hat[4 * i + 3];
            mu += ru; md += rd;
            tu += (Kxu[ix] + Ky[iy]) * ru; td += (Kxd[ix] + Ky[iy]) * rd;
            pu += kx[ix] * ru; pd += kx[ix] * rd;
        }
    }
    free(Kxu); free(Kxd); free(Ky); free(kx);
    out_k[0] = w * mu; out_k[1] = w * md; out_k[2] = w * tu; out_k[3] = w * td; out_k[4] = w * pu; out_k[5] = w * pd;
}

/* n Strang steps with the observables of the fused call spgpe_step_observe (include/spgpe.h): the k-space sums are
 * those of the order parameter in the middle of the LAST step (after its first half-step and the forward transform;
 * the k-space phase has unit modulus in real time, so before or after it is the same; in imaginary time: before it),
 * the real-space ones those of the final state (after the renormalisation in imaginary time). */
void orc_step_observe(double *psi, const double *V, const double *Om, const double *de, const orc_params *p,
                      int n, double dt, int imag, const double *targets, double *out_r, double *out_k) {
    const size_t P = (size_t)p->nx * p->ny;
    if (n > 1) orc_step(psi, V, Om, de, p, n - 1, dt, imag, targets);
    if (n >= 1) {
        double *hat = (double *)malloc(sizeof(double) * 4 * P);
        orc_half(psi, V, Om, de, p, 0.5 * dt, imag);
        memcpy(hat, psi, sizeof(double) * 4 * P);
        orc_fft2(hat, p, -1);
        orc_kspace_observables(hat, p, out_k);
        free(hat);
        orc_kinetic(psi, p, dt, imag);
        orc_half(psi, V, Om, de, p, 0.5 * dt, imag);
        if (imag) renormalise(psi, p, targets);
    }
    orc_observables(psi, p, out_r);
}
