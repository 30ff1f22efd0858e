/*
 * gpe_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation of the symmetric split-step
 * Fourier propagation of the 2-D Gross-Pitaevskii equation (Eqs. 2-4;
 * imaginary time PAPER.md:112-116; cavity potentials PAPER.md:170-188, Eqs. 10-15).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this file.  It shares no code, header, table or helper with the CUDA
 * path under paper_2404_14401_b200/csrc/ and neither includes the other.
 *
 * Arithmetic: REAL is double (the oracle proper, complex128).  Compiling with
 * -DREAL=float gives the same statements in complex64; that build is used only to
 * measure the fp32 round-off floor of the *method* (SURVEY.md 8(c) R1), never as an oracle.
 * Transcendentals (phases, twiddles, tables) are always evaluated in double and rounded.
 *
 * Conventions:
 *   hbar = m = 1.  Grid x_i = -Lx/2 + i*Lx/nx, i = 0..nx-1 (periodic, end point excluded),
 *   likewise y_j.  psi stored [batch][nx][ny], y fastest.  Integral = sum * dx * dy.
 *   Forward FFT unnormalised with kernel exp(-i(kx x + ky y)); inverse carries 1/(nx*ny).
 *   k_x[p] = 2*pi*p/Lx for p < nx/2, 2*pi*(p-nx)/Lx otherwise (likewise k_y).
 *
 * One step n -> n+1 of member b (sigma = i in real time, 1 in imaginary time):
 *   1. A_n = schedule(n).  Theta_n = sum cos(kc x)cos(kc y)|psi|^2 dx dy.
 *      eta_n = eta (mode 0) or sqrt(|A_n| u) (mode 1).
 *      alpha_n = N_at eta_n Theta_n / (Delta + i kappa)          [PAPER.md:183, Eq. 14]
 *      real time with a probe: alpha_n += Omega_c exp(i (Delta_p t_n + phi)) / (Delta + i kappa),
 *      t_n = n dt (Eq. 17; with cav_u0 its denominator carries the dispersive
 *      shift of the next line, Delta~_n + i kappa)
 *      with cav_u0 = U_0 (full cavity model): Delta above is replaced by
 *      Delta~_n = Delta - N_at U_0 B_n, B_n = sum cos^2(kc x)|psi|^2 dx dy   [PAPER.md:188, Eq. 15]
 *      and V_n gains the cavity lattice D_n cos^2(kc x), D_n = U_0 |alpha_n|^2 [PAPER.md:177, Eq. 12]
 *      C_n = 2 eta_n Re(alpha_n)                                 [PAPER.md:179, Eq. 13]
 *   2. V_n = V_static + A_n cos^2(k_l * (x or y)) + C_n cos(kc x)cos(kc y)   [Eqs. 9-13]
 *   3. psi <- psi * exp(-sigma (V_n + g|psi|^2) dt/2)            [PAPER.md:67,71]
 *   4. psi^ = FFT2(psi); psi^ <- psi^ * exp(-sigma (kx^2+ky^2) dt/2); psi = IFFT2(psi^)
 *   5. psi <- psi * exp(-sigma (V_n + g|psi|^2) dt/2), |psi|^2 from the psi entering
 *      this line ("most up-to-date wave function")
 *   6. imaginary time only: psi <- psi / sqrt(sum |psi|^2 dx dy)  [PAPER.md:116]
 * With ordering = 1 (T/2 V T/2, the form the paper prints, Eqs. 3-4) steps 3-5 become:
 * half of step 4 (dt/4 in its exponent), steps 1-2 evaluated on the psi at that point, one full
 * potential factor exp(-sigma (V_n + g|psi|^2) dt), half of step 4 again.
 *
 * Pins: tests/test_oracle_*.py (direct DFT, numpy.fft, Parseval, shift theorem, exact
 * composition of kinetic steps, free Gaussian expansion, Jacobi-Anger/Bessel, the Gaussian
 * recurrence closed form in a harmonic trap, E -> (wx+wy)/2, Thomas-Fermi, norm
 * conservation, time reversal, Kapitza-Dirac coupled-mode ODE, energy conservation with the
 * cavity, convergence order, batch == single).  Nothing in Figs. 2-6 of the paper is
 * available (image placeholders), so parity against the paper's plots is "unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef REAL
#define REAL double
#endif
typedef REAL real_t;
typedef REAL _Complex cplx_t;

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    int nx, ny, batch;
    double Lx, Ly;
    const double *v_static;   /* [nx*ny] or [batch][nx*ny]; NULL = 0 */
    int v_static_batched;
    const double *g;          /* [batch] */
    int lattice_axis;         /* -1 none, 0: cos^2(k x), 1: cos^2(k y) */
    double lattice_k;
    int sched_len;            /* piecewise-linear amplitude over step index */
    const double *sched_step; /* [sched_len] non-decreasing */
    const double *sched_amp;  /* [sched_len] or [batch][sched_len] */
    int sched_batched;
    int cavity_on;
    double cavity_k;
    int eta_mode;             /* 0: eta given, 1: eta_n = sqrt(|A_n| u) */
    const double *eta_or_u;   /* [batch] */
    const double *n_atoms;    /* [batch] */
    const double *delta;      /* [batch] */
    const double *kappa;      /* [batch] */
    /* on-axis cavity probe (Eq. 17), real time only; NULL = none */
    const double *probe_omega; /* [batch] Omega_c */
    const double *probe_delta; /* [batch] Delta_p */
    const double *probe_phi;   /* [batch] phi */
    /* full cavity model (Eqs. 12 and 15): U_0 per member; NULL = off */
    const double *cav_u0;      /* [batch] */
    /* 1: the schedule amplitude of step n is sampled at the middle of the step, A((n + 1/2) dt),
     * instead of its start (reading Q4) */
    int sched_midpoint;
    /* 0: V/2 T V/2 (steps 3-5 above, north_star); 1: T/2 V T/2, the ordering the paper prints
     * (Eqs. 3-4; reading Q1): half a kinetic step,
     * the scalars of step 1 from the psi that ENTERS the potential factor, one full potential
     * factor exp(-sigma (V_n + g|psi|^2) dt) with |psi|^2 of that same psi, half a kinetic step,
     * then step 6 */
    int ordering;
} oracle_params;

/* ------------------------------------------------------------------ FFT */

/* Direct O(N^2) DFT, used for N <= 16 and as a cross-check.  sign = -1 forward, +1 inverse
 * (no normalisation here). */
static void dft_direct(cplx_t *a, int n, int sign)
{
    cplx_t *out = (cplx_t *)malloc(sizeof(cplx_t) * (size_t)n);
    for (int k = 0; k < n; ++k) {
        double _Complex acc = 0.0;
        for (int j = 0; j < n; ++j) {
            double ang = sign * 2.0 * M_PI * (double)(((long)j * k) % n) / (double)n;
            acc += (double _Complex)a[j] * cexp(I * ang);
        }
        out[k] = (cplx_t)acc;
    }
    memcpy(a, out, sizeof(cplx_t) * (size_t)n);
    free(out);
}

/* Iterative radix-2 decimation-in-time FFT with bit reversal.  n power of two. */
static void fft_radix2(cplx_t *a, int n, int sign)
{
    int logn = 0;
    while ((1 << logn) < n) ++logn;
    for (int i = 0; i < n; ++i) {
        int r = 0;
        for (int b = 0; b < logn; ++b)
            if (i & (1 << b)) r |= 1 << (logn - 1 - b);
        if (r > i) { cplx_t t = a[i]; a[i] = a[r]; a[r] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        for (int start = 0; start < n; start += len) {
            for (int j = 0; j < half; ++j) {
                double ang = sign * 2.0 * M_PI * (double)j / (double)len;
                cplx_t w = (cplx_t)cexp(I * ang);
                cplx_t u = a[start + j];
                cplx_t v = a[start + j + half] * w;
                a[start + j] = u + v;
                a[start + j + half] = u - v;
            }
        }
    }
}

/* Lengths that are not powers of two ("non-optimal grid sizes") take the
 * plain definition of the transform, dft_direct: O(n^2), no factorisation to get wrong. */
static void fft_1d(cplx_t *a, int n, int sign, int force_direct)
{
    if (n <= 16 || force_direct || (n & (n - 1)) != 0) dft_direct(a, n, sign);
    else fft_radix2(a, n, sign);
}

/* 2-D transform of one [nx][ny] grid: rows (along y) then columns (along x).
 * sign=-1: forward unnormalised; sign=+1: inverse including 1/(nx*ny). */
static void fft2_grid(cplx_t *psi, int nx, int ny, int sign, int force_direct)
{
#pragma omp parallel for schedule(static)
    for (int i = 0; i < nx; ++i) fft_1d(psi + (size_t)i * ny, ny, sign, force_direct);
#pragma omp parallel
    {
        cplx_t *col = (cplx_t *)malloc(sizeof(cplx_t) * (size_t)nx);
#pragma omp for schedule(static)
        for (int j = 0; j < ny; ++j) {
            for (int i = 0; i < nx; ++i) col[i] = psi[(size_t)i * ny + j];
            fft_1d(col, nx, sign, force_direct);
            for (int i = 0; i < nx; ++i) psi[(size_t)i * ny + j] = col[i];
        }
        free(col);
    }
    if (sign > 0) {
        real_t s = (real_t)(1.0 / ((double)nx * (double)ny));
#pragma omp parallel for schedule(static)
        for (long q = 0; q < (long)nx * ny; ++q) psi[q] *= s;
    }
}

/* exported for the FFT pins */
void oracle_fft2(cplx_t *psi, int nx, int ny, int sign, int force_direct)
{
    fft2_grid(psi, nx, ny, sign, force_direct);
}
void oracle_fft1(cplx_t *a, int n, int sign, int force_direct)
{
    fft_1d(a, n, sign, force_direct);
}

/* ------------------------------------------------------------------ grid helpers */

static double coord(int i, int n, double L) { return -0.5 * L + (double)i * L / (double)n; }
static double wavenumber(int p, int n, double L)
{
    return 2.0 * M_PI * (double)(p < n / 2 ? p : p - n) / L;
}

/* piecewise-linear schedule at step index n: the last knot with
 * step <= n starts the segment; before the first knot the first amplitude holds, after
 * the last knot the last amplitude holds. */
double oracle_schedule(const oracle_params *P, int b, double n)
{
    if (P->sched_len <= 0) return 0.0;
    const double *amp = P->sched_amp + (P->sched_batched ? (size_t)b * P->sched_len : 0);
    const double *st = P->sched_step;
    int L = P->sched_len;
    if (n < st[0]) return amp[0];
    int i = 0;
    for (int q = 0; q < L; ++q) if (st[q] <= n) i = q;
    if (i == L - 1) return amp[L - 1];
    double t = (n - st[i]) / (st[i + 1] - st[i]);
    return amp[i] + t * (amp[i + 1] - amp[i]);
}

static double v_static_at(const oracle_params *P, int b, size_t q)
{
    if (!P->v_static) return 0.0;
    return P->v_static[(P->v_static_batched ? (size_t)b * P->nx * P->ny : 0) + q];
}

/* cos^2(k_l r) along the lattice axis and the cavity mode cos(kc x)cos(kc y); the 1-D
 * cosines are tabulated once per call (plain hoisting of a per-point cos, nothing else). */
typedef struct { double *lat_x, *lat_y, *cav_x, *cav_y; } axis_tables;

static axis_tables make_tables(const oracle_params *P)
{
    axis_tables T;
    T.lat_x = (double *)malloc(sizeof(double) * P->nx); T.cav_x = (double *)malloc(sizeof(double) * P->nx);
    T.lat_y = (double *)malloc(sizeof(double) * P->ny); T.cav_y = (double *)malloc(sizeof(double) * P->ny);
    for (int i = 0; i < P->nx; ++i) {
        double x = coord(i, P->nx, P->Lx), c = cos(P->lattice_k * x);
        T.lat_x[i] = P->lattice_axis == 0 ? c * c : 0.0;
        T.cav_x[i] = cos(P->cavity_k * x);
    }
    for (int j = 0; j < P->ny; ++j) {
        double y = coord(j, P->ny, P->Ly), c = cos(P->lattice_k * y);
        T.lat_y[j] = P->lattice_axis == 1 ? c * c : 0.0;
        T.cav_y[j] = cos(P->cavity_k * y);
    }
    return T;
}
static void free_tables(axis_tables *T) { free(T->lat_x); free(T->lat_y); free(T->cav_x); free(T->cav_y); }

/* lattice shape: exactly one of lat_x / lat_y is non-zero (or none) */
#define LATTICE_SHAPE(T, i, j) ((T)->lat_x[i] + (T)->lat_y[j])
#define CAVITY_MODE(T, i, j) ((T)->cav_x[i] * (T)->cav_y[j])

static double sum_norm(const oracle_params *P, const cplx_t *psi)
{
    double s = 0.0;
    long n = (long)P->nx * P->ny;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (long q = 0; q < n; ++q) {
        double re = creal(psi[q]), im = cimag(psi[q]);
        s += re * re + im * im;
    }
    return s * (P->Lx / P->nx) * (P->Ly / P->ny);
}

static double sum_theta(const oracle_params *P, const axis_tables *T, const cplx_t *psi)
{
    double s = 0.0;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (int i = 0; i < P->nx; ++i)
        for (int j = 0; j < P->ny; ++j) {
            cplx_t z = psi[(size_t)i * P->ny + j];
            double re = creal(z), im = cimag(z);
            s += CAVITY_MODE(T, i, j) * (re * re + im * im);
        }
    return s * (P->Lx / P->nx) * (P->Ly / P->ny);
}

static double sum_bunch(const oracle_params *P, const axis_tables *T, const cplx_t *psi)
{
    double s = 0.0;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (int i = 0; i < P->nx; ++i)
        for (int j = 0; j < P->ny; ++j) {
            cplx_t z = psi[(size_t)i * P->ny + j];
            double re = creal(z), im = cimag(z);
            s += T->cav_x[i] * T->cav_x[i] * (re * re + im * im);
        }
    return s * (P->Lx / P->nx) * (P->Ly / P->ny);
}

/* step 1 of the header: per-step scalars of member b at step index n from the current psi */
/* t < 0: no probe (imaginary time, observables) */
static void cavity_scalars(const oracle_params *P, int b, double A, double theta, double bunch, double t,
                           double *eta, double _Complex *alpha, double *C, double *Dc)
{
    *eta = 0.0; *alpha = 0.0; *C = 0.0; *Dc = 0.0;
    if (!P->cavity_on) return;
    *eta = P->eta_mode == 0 ? P->eta_or_u[b] : sqrt(fabs(A) * P->eta_or_u[b]);
    double D = P->delta[b];
    if (P->cav_u0) D -= P->n_atoms[b] * P->cav_u0[b] * bunch;          /* Eq. 15 */
    *alpha = P->n_atoms[b] * (*eta) * theta / (D + I * P->kappa[b]);
    if (t >= 0.0 && P->probe_omega && P->probe_omega[b] != 0.0)
        *alpha += P->probe_omega[b] * cexp(I * (P->probe_delta[b] * t + P->probe_phi[b])) / (D + I * P->kappa[b]);
    if (P->cav_u0) *Dc = P->cav_u0[b] * (creal(*alpha) * creal(*alpha) + cimag(*alpha) * cimag(*alpha));  /* Eq. 12 */
    *C = 2.0 * (*eta) * creal(*alpha);
}

/* steps 3 / 5 of the header */
static void potential_half_step(const oracle_params *P, const axis_tables *T, int b, cplx_t *psi, double A, double C,
                                double Dc, double dt, int imag_time)
{
    double g = P->g ? P->g[b] : 0.0;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < P->nx; ++i)
        for (int j = 0; j < P->ny; ++j) {
            size_t q = (size_t)i * P->ny + j;
            double re = creal(psi[q]), im = cimag(psi[q]);
            double V = v_static_at(P, b, q) + A * LATTICE_SHAPE(T, i, j);
            if (P->cavity_on) V += C * CAVITY_MODE(T, i, j) + Dc * T->cav_x[i] * T->cav_x[i];
            double W = (V + g * (re * re + im * im)) * dt * 0.5;
            cplx_t f = imag_time ? (cplx_t)exp(-W) : (cplx_t)cexp(-I * W);
            psi[q] = psi[q] * f;
        }
}

/* step 4 of the header */
static void kinetic_step(const oracle_params *P, cplx_t *psi, double dt, int imag_time)
{
    fft2_grid(psi, P->nx, P->ny, -1, 0);
#pragma omp parallel for schedule(static)
    for (int p = 0; p < P->nx; ++p)
        for (int q = 0; q < P->ny; ++q) {
            double kx = wavenumber(p, P->nx, P->Lx), ky = wavenumber(q, P->ny, P->Ly);
            double W = (kx * kx + ky * ky) * dt * 0.5;
            cplx_t f = imag_time ? (cplx_t)exp(-W) : (cplx_t)cexp(-I * W);
            psi[(size_t)p * P->ny + q] *= f;
        }
    fft2_grid(psi, P->nx, P->ny, +1, 0);
}

#define ORACLE_NREC 6

/* Evolve all members n_steps steps in place.  step0 = index of the first step (time origin
 * of the schedule).  records (may be NULL): [n_rec][batch][6] = {step, norm, theta,
 * re_alpha, im_alpha, A} written after every step whose index (step0+s+1) is a multiple of
 * record_every, from the psi at that moment and the schedule at that index. */
int oracle_evolve(const oracle_params *P, cplx_t *psi, double dt, long n_steps, int imag_time,
                  long step0, long record_every, double *records)
{
    size_t npts = (size_t)P->nx * P->ny;
    long nrec = 0;
    axis_tables T = make_tables(P);
    for (long s = 0; s < n_steps; ++s) {
        long n = step0 + s;
        for (int b = 0; b < P->batch; ++b) {
            cplx_t *w = psi + (size_t)b * npts;
            double A = oracle_schedule(P, b, (double)n + (P->sched_midpoint ? 0.5 : 0.0));
            double theta = P->cavity_on ? sum_theta(P, &T, w) : 0.0;
            double bunch = (P->cavity_on && P->cav_u0) ? sum_bunch(P, &T, w) : 0.0;
            double eta, C, Dc; double _Complex alpha;
            if (P->ordering == 1) {
                /* T/2 V T/2: kinetic_step(dt') multiplies by exp(-sigma k^2 dt'/2), so dt' = dt/2 is
                 * half a kinetic step; potential_half_step(dt') multiplies by exp(-sigma (V + g|psi|^2) dt'/2),
                 * so dt' = 2 dt is the full potential factor */
                kinetic_step(P, w, 0.5 * dt, imag_time);
                theta = P->cavity_on ? sum_theta(P, &T, w) : 0.0;
                bunch = (P->cavity_on && P->cav_u0) ? sum_bunch(P, &T, w) : 0.0;
                cavity_scalars(P, b, A, theta, bunch, imag_time ? -1.0 : (double)n * dt, &eta, &alpha, &C, &Dc);
                potential_half_step(P, &T, b, w, A, C, Dc, 2.0 * dt, imag_time);
                kinetic_step(P, w, 0.5 * dt, imag_time);
            } else {
            cavity_scalars(P, b, A, theta, bunch, imag_time ? -1.0 : (double)n * dt, &eta, &alpha, &C, &Dc);
            potential_half_step(P, &T, b, w, A, C, Dc, dt, imag_time);
            kinetic_step(P, w, dt, imag_time);
            potential_half_step(P, &T, b, w, A, C, Dc, dt, imag_time);
            }
            if (imag_time) {
                real_t inv = (real_t)(1.0 / sqrt(sum_norm(P, w)));
#pragma omp parallel for schedule(static)
                for (long q = 0; q < (long)npts; ++q) w[q] *= inv;
            }
        }
        if (records && record_every > 0 && ((n + 1) % record_every) == 0) {
            for (int b = 0; b < P->batch; ++b) {
                cplx_t *w = psi + (size_t)b * npts;
                double A = oracle_schedule(P, b, (double)(n + 1) + (P->sched_midpoint ? 0.5 : 0.0));
                double theta = P->cavity_on ? sum_theta(P, &T, w) : 0.0;
                double bunch = (P->cavity_on && P->cav_u0) ? sum_bunch(P, &T, w) : 0.0;
                double eta, C, Dc; double _Complex alpha;
                cavity_scalars(P, b, A, theta, bunch, imag_time ? -1.0 : (double)(n + 1) * dt, &eta, &alpha, &C, &Dc);
                double *r = records + ((size_t)nrec * P->batch + b) * ORACLE_NREC;
                r[0] = (double)(n + 1); r[1] = sum_norm(P, w); r[2] = theta;
                r[3] = creal(alpha); r[4] = cimag(alpha); r[5] = A;
            }
            ++nrec;
        }
    }
    free_tables(&T);
    return 0;
}

/* Observables of member-wise psi at step index n (for A_n):
 * out[b][8] = {norm, e_kin, e_pot, e_int, e_cav, theta, re_alpha, im_alpha}
 * density (may be NULL): |psi|^2 ; kdensity (may be NULL): |psi^|^2 / sum |psi^|^2. */
int oracle_observables(const oracle_params *P, const cplx_t *psi, long n, double *out,
                       double *density, double *kdensity)
{
    size_t npts = (size_t)P->nx * P->ny;
    double dxdy = (P->Lx / P->nx) * (P->Ly / P->ny);
    cplx_t *hat = (cplx_t *)malloc(sizeof(cplx_t) * npts);
    axis_tables T = make_tables(P);
    for (int b = 0; b < P->batch; ++b) {
        const cplx_t *w = psi + (size_t)b * npts;
        double A = oracle_schedule(P, b, (double)n + (P->sched_midpoint ? 0.5 : 0.0));
        double g = P->g ? P->g[b] : 0.0;
        double norm = sum_norm(P, w);
        double theta = P->cavity_on ? sum_theta(P, &T, w) : 0.0;
        double bunch = (P->cavity_on && P->cav_u0) ? sum_bunch(P, &T, w) : 0.0;
        double eta, C, Dc; double _Complex alpha;
        cavity_scalars(P, b, A, theta, bunch, -1.0, &eta, &alpha, &C, &Dc);
        double epot = 0.0, eint = 0.0;
        for (int i = 0; i < P->nx; ++i)
            for (int j = 0; j < P->ny; ++j) {
                size_t q = (size_t)i * P->ny + j;
                double re = creal(w[q]), im = cimag(w[q]);
                double d = re * re + im * im;
                epot += (v_static_at(P, b, q) + A * LATTICE_SHAPE(&T, i, j)) * d;
                eint += 0.5 * g * d * d;
                if (density) density[(size_t)b * npts + q] = d;
            }
        epot *= dxdy; eint *= dxdy;
        memcpy(hat, w, sizeof(cplx_t) * npts);
        fft2_grid(hat, P->nx, P->ny, -1, 0);
        double ksum = 0.0, k2sum = 0.0;
        for (int p = 0; p < P->nx; ++p)
            for (int q = 0; q < P->ny; ++q) {
                cplx_t z = hat[(size_t)p * P->ny + q];
                double d = creal(z) * creal(z) + cimag(z) * cimag(z);
                double kx = wavenumber(p, P->nx, P->Lx), ky = wavenumber(q, P->ny, P->Ly);
                ksum += d; k2sum += (kx * kx + ky * ky) * d;
            }
        if (kdensity)
            for (size_t q = 0; q < npts; ++q) {
                double d = creal(hat[q]) * creal(hat[q]) + cimag(hat[q]) * cimag(hat[q]);
                kdensity[(size_t)b * npts + q] = d / ksum;
            }
        double ekin = 0.5 * k2sum / ksum * norm;
        double ecav = 0.0;
        if (P->cavity_on) {
            double D = P->delta[b] - (P->cav_u0 ? P->n_atoms[b] * P->cav_u0[b] * bunch : 0.0), K = P->kappa[b];
            ecav = P->n_atoms[b] * eta * eta * theta * theta * D / (D * D + K * K);
        }
        double *o = out + (size_t)b * 8;
        o[0] = norm; o[1] = ekin; o[2] = epot; o[3] = eint; o[4] = ecav;
        o[5] = theta; o[6] = creal(alpha); o[7] = cimag(alpha);
    }
    free(hat); free_tables(&T);
    return 0;
}

/* Momentum-order populations: for m = -m_max..m_max,
 * out[b][m+m_max] = sum over |k_axis - 2 m k_l| < k_l (all k on the other axis) of
 * |psi^|^2 / sum |psi^|^2. */
int oracle_populations(const oracle_params *P, const cplx_t *psi, int axis, double k_l, int m_max,
                       double *out)
{
    size_t npts = (size_t)P->nx * P->ny;
    cplx_t *hat = (cplx_t *)malloc(sizeof(cplx_t) * npts);
    for (int b = 0; b < P->batch; ++b) {
        memcpy(hat, psi + (size_t)b * npts, sizeof(cplx_t) * npts);
        fft2_grid(hat, P->nx, P->ny, -1, 0);
        double tot = 0.0;
        double *o = out + (size_t)b * (2 * m_max + 1);
        for (int m = 0; m < 2 * m_max + 1; ++m) o[m] = 0.0;
        for (int p = 0; p < P->nx; ++p)
            for (int q = 0; q < P->ny; ++q) {
                cplx_t z = hat[(size_t)p * P->ny + q];
                double d = creal(z) * creal(z) + cimag(z) * cimag(z);
                tot += d;
                double k = axis == 0 ? wavenumber(p, P->nx, P->Lx) : wavenumber(q, P->ny, P->Ly);
                for (int m = -m_max; m <= m_max; ++m)
                    if (fabs(k - 2.0 * m * k_l) < k_l) o[m + m_max] += d;
            }
        for (int m = 0; m < 2 * m_max + 1; ++m) o[m] /= tot;
    }
    free(hat);
    return 0;
}

int oracle_real_bytes(void) { return (int)sizeof(real_t); }

/* The two factors of the step exported on their own, for the pins that test one factor at a
 * time (Jacobi-Anger for the potential factor, exact composition / free expansion for the
 * kinetic factor).  A and C are evaluated as in step 1 of the header at step index n. */
int oracle_potential_half_step(const oracle_params *P, cplx_t *psi, double dt, int imag_time, long n)
{
    size_t npts = (size_t)P->nx * P->ny;
    axis_tables T = make_tables(P);
    for (int b = 0; b < P->batch; ++b) {
        cplx_t *w = psi + (size_t)b * npts;
        double A = oracle_schedule(P, b, (double)n + (P->sched_midpoint ? 0.5 : 0.0));
        double theta = P->cavity_on ? sum_theta(P, &T, w) : 0.0;
        double bunch = (P->cavity_on && P->cav_u0) ? sum_bunch(P, &T, w) : 0.0;
        double eta, C, Dc; double _Complex alpha;
        cavity_scalars(P, b, A, theta, bunch, -1.0, &eta, &alpha, &C, &Dc);
        potential_half_step(P, &T, b, w, A, C, Dc, dt, imag_time);
    }
    free_tables(&T);
    return 0;
}

int oracle_kinetic_step(const oracle_params *P, cplx_t *psi, double dt, int imag_time)
{
    size_t npts = (size_t)P->nx * P->ny;
    for (int b = 0; b < P->batch; ++b) kinetic_step(P, psi + (size_t)b * npts, dt, imag_time);
    return 0;
}
