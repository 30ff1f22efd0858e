/*
 * gpe3_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation of the symmetric split-step Fourier
 * propagation of the Gross-Pitaevskii equation on a THREE-dimensional grid: the paper's method
 * (Eq. 1 is written for psi(r, t) in any dimension; Eqs. 2-4 the
 * split-step; PAPER.md:112-116 imaginary time) carried to the first item of its outlook
 * ("extending the method to three dimensions"), second half.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may load this file.  It shares
 * no code, header, table or helper with the CUDA path under paper_2404_14401_b200/csrc/, nor with the
 * 2-D oracle gpe_oracle.c (which one of its pins compares it with).
 *
 * Arithmetic: REAL is double (the oracle proper).  -DREAL=float gives the same statements in
 * complex64: the fp32 round-off floor of the method, never used as an oracle.
 *
 * Conventions (those of the 2-D path): hbar = m = 1.  x_i = -Lx/2 + i Lx/nx
 * (periodic, end point excluded), likewise y_j, z_l.  psi stored [nz][nx][ny], y fastest, z slowest.
 * Integral = sum * dx dy dz.  Forward transform unnormalised with kernel exp(-i k.r), the inverse
 * carries 1/(nx ny nz).  k_x[p] = 2 pi p / Lx for 2 p < nx, 2 pi (p - nx)/Lx otherwise.
 *
 * One step (sigma = i in real time, 1 in imaginary time), V = v_static + vx[i] + vy[j] + vz[l]:
 *   1. psi <- psi * exp(-sigma (V + g|psi|^2) dt/2)                      [PAPER.md:67,71]
 *   2. psi^ = FFT3(psi); psi^ <- psi^ * exp(-sigma (kx^2+ky^2+kz^2) dt/2); psi = IFFT3(psi^)
 *   3. psi <- psi * exp(-sigma (V + g|psi|^2) dt/2), |psi|^2 of the psi entering this line
 *      ("most up-to-date wave function")
 *   4. imaginary time only: psi <- psi / sqrt(sum |psi|^2 dx dy dz)      [PAPER.md:116]
 *
 * Pins: tests/test_oracle_3d.py (numpy.fft.fftn, the plain 3-D DFT sum on a tiny grid, the
 * Gaussian recurrence closed form in an anisotropic harmonic trap, free expansion of a Gaussian,
 * E -> (wx+wy+wz)/2, nz = 1 equals the 2-D oracle, separability for g = 0, norm conservation and
 * time reversal, convergence order 2).
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
    int nx, ny, nz;
    double Lx, Ly, Lz;
    const double *v_static;   /* [nz][nx][ny] or NULL */
    const double *vx, *vy, *vz; /* separable part: [nx], [ny], [nz], each may be NULL */
    double g;
} oracle3_params;

/* ------------------------------------------------------------------ 1-D transforms */

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

/* recursive radix-2 decimation in time (Cooley-Tukey as printed in any textbook): X[k] = E[k] + w^k O[k],
 * X[k + n/2] = E[k] - w^k O[k].  n a power of two; other lengths take the definition. */
static void fft_rec(cplx_t *a, cplx_t *tmp, int n, int sign)
{
    if (n <= 8 || (n & 1)) { dft_direct(a, n, sign); return; }
    int h = n / 2;
    for (int j = 0; j < h; ++j) { tmp[j] = a[2 * j]; tmp[h + j] = a[2 * j + 1]; }
    memcpy(a, tmp, sizeof(cplx_t) * (size_t)n);
    fft_rec(a, tmp, h, sign);
    fft_rec(a + h, tmp, h, sign);
    for (int k = 0; k < h; ++k) {
        double ang = sign * 2.0 * M_PI * (double)k / (double)n;
        cplx_t w = (cplx_t)cexp(I * ang);
        cplx_t e = a[k], o = a[h + k] * w;
        a[k] = e + o;
        a[h + k] = e - o;
    }
}

/* transform along one axis of a [n0][n1][n2] array (axis 0, 1 or 2): every line is copied out, transformed, copied back */
static void fft_axis(cplx_t *psi, int n0, int n1, int n2, int axis, int sign)
{
    const int dims[3] = {n0, n1, n2};
    const long strides[3] = {(long)n1 * n2, n2, 1};
    const int n = dims[axis];
    const int a = (axis + 1) % 3, b = (axis + 2) % 3;
#pragma omp parallel
    {
        cplx_t *line = (cplx_t *)malloc(sizeof(cplx_t) * (size_t)n);
        cplx_t *tmp = (cplx_t *)malloc(sizeof(cplx_t) * (size_t)n);
#pragma omp for collapse(2) schedule(static)
        for (int p = 0; p < dims[a]; ++p)
            for (int q = 0; q < dims[b]; ++q) {
                cplx_t *base = psi + p * strides[a] + q * strides[b];
                for (int i = 0; i < n; ++i) line[i] = base[i * strides[axis]];
                fft_rec(line, tmp, n, sign);
                for (int i = 0; i < n; ++i) base[i * strides[axis]] = line[i];
            }
        free(line); free(tmp);
    }
}

/* sign = -1: forward, unnormalised; sign = +1: inverse including 1/(nx ny nz) */
static void fft3_grid(cplx_t *psi, int nz, int nx, int ny, int sign)
{
    fft_axis(psi, nz, nx, ny, 2, sign);
    fft_axis(psi, nz, nx, ny, 1, sign);
    fft_axis(psi, nz, nx, ny, 0, sign);
    if (sign > 0) {
        real_t s = (real_t)(1.0 / ((double)nx * (double)ny * (double)nz));
        long n = (long)nx * ny * nz;
#pragma omp parallel for schedule(static)
        for (long q = 0; q < n; ++q) psi[q] *= s;
    }
}

void oracle3_fft3(cplx_t *psi, int nz, int nx, int ny, int sign) { fft3_grid(psi, nz, nx, ny, sign); }

/* ------------------------------------------------------------------ the step */

static double coord(int i, int n, double L) { return -0.5 * L + (double)i * L / (double)n; }
/* 2 p < n is p < n/2 for the even sizes of the method and also takes k = 0 on an axis of length 1 */
static double wavenumber(int p, int n, double L) { return 2.0 * M_PI * (double)(2 * p < n ? p : p - n) / L; }

static double potential_at(const oracle3_params *P, int l, int i, int j)
{
    double V = 0.0;
    if (P->v_static) V += P->v_static[((size_t)l * P->nx + i) * P->ny + j];
    if (P->vx) V += P->vx[i];
    if (P->vy) V += P->vy[j];
    if (P->vz) V += P->vz[l];
    return V;
}

static double sum_norm(const oracle3_params *P, const cplx_t *psi)
{
    double s = 0.0;
    long n = (long)P->nx * P->ny * P->nz;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (long q = 0; q < n; ++q) {
        double re = creal(psi[q]), im = cimag(psi[q]);
        s += re * re + im * im;
    }
    return s * (P->Lx / P->nx) * (P->Ly / P->ny) * (P->Lz / P->nz);
}

/* steps 1 / 3 of the header */
static void potential_half_step(const oracle3_params *P, cplx_t *psi, double dt, int imag_time)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int l = 0; l < P->nz; ++l)
        for (int i = 0; i < P->nx; ++i)
            for (int j = 0; j < P->ny; ++j) {
                size_t q = ((size_t)l * P->nx + i) * P->ny + j;
                double re = creal(psi[q]), im = cimag(psi[q]);
                double W = (potential_at(P, l, i, j) + P->g * (re * re + im * im)) * dt * 0.5;
                cplx_t f = imag_time ? (cplx_t)exp(-W) : (cplx_t)cexp(-I * W);
                psi[q] = psi[q] * f;
            }
}

/* step 2 of the header */
static void kinetic_step(const oracle3_params *P, cplx_t *psi, double dt, int imag_time)
{
    fft3_grid(psi, P->nz, P->nx, P->ny, -1);
#pragma omp parallel for collapse(2) schedule(static)
    for (int r = 0; r < P->nz; ++r)
        for (int p = 0; p < P->nx; ++p)
            for (int q = 0; q < P->ny; ++q) {
                double kz = wavenumber(r, P->nz, P->Lz), kx = wavenumber(p, P->nx, P->Lx), ky = wavenumber(q, P->ny, P->Ly);
                double W = (kx * kx + ky * ky + kz * kz) * dt * 0.5;
                cplx_t f = imag_time ? (cplx_t)exp(-W) : (cplx_t)cexp(-I * W);
                psi[((size_t)r * P->nx + p) * P->ny + q] *= f;
            }
    fft3_grid(psi, P->nz, P->nx, P->ny, +1);
}

#define ORACLE3_NREC 3

/* Evolve n_steps steps in place.  records (may be NULL): [n_rec][3] = {step, norm, norm_pre} written after every
 * step whose index (step0 + s + 1) is a multiple of record_every: norm = sum |psi|^2 dx dy dz of the psi at that
 * moment, norm_pre = the same sum taken BEFORE line 4 of the header (equal to norm in real time; in imaginary time
 * -log(norm_pre) / (2 dt) estimates the chemical potential). */
int oracle3_evolve(const oracle3_params *P, cplx_t *psi, double dt, long n_steps, int imag_time, long step0,
                   long record_every, double *records)
{
    long nrec = 0;
    long npts = (long)P->nx * P->ny * P->nz;
    for (long s = 0; s < n_steps; ++s) {
        long n = step0 + s;
        potential_half_step(P, psi, dt, imag_time);
        kinetic_step(P, psi, dt, imag_time);
        potential_half_step(P, psi, dt, imag_time);
        double pre = sum_norm(P, psi);
        if (imag_time) {
            real_t inv = (real_t)(1.0 / sqrt(pre));
#pragma omp parallel for schedule(static)
            for (long q = 0; q < npts; ++q) psi[q] *= inv;
        }
        if (records && record_every > 0 && ((n + 1) % record_every) == 0) {
            double *r = records + (size_t)nrec * ORACLE3_NREC;
            r[0] = (double)(n + 1); r[1] = sum_norm(P, psi); r[2] = pre;
            ++nrec;
        }
    }
    return 0;
}

/* out[8] = {norm, e_kin, e_pot, e_int, <x^2>, <y^2>, <z^2>, 0}:
 *   e_kin = (1/2) sum |k|^2 |psi^|^2 / sum |psi^|^2 * norm,  e_pot = sum V |psi|^2 dV,  e_int = (g/2) sum |psi|^4 dV,
 *   <x^2> = sum x^2 |psi|^2 dV (not divided by the norm). */
int oracle3_observables(const oracle3_params *P, const cplx_t *psi, double *out)
{
    long npts = (long)P->nx * P->ny * P->nz;
    double dV = (P->Lx / P->nx) * (P->Ly / P->ny) * (P->Lz / P->nz);
    double norm = sum_norm(P, psi), epot = 0.0, eint = 0.0, x2 = 0.0, y2 = 0.0, z2 = 0.0;
    for (int l = 0; l < P->nz; ++l)
        for (int i = 0; i < P->nx; ++i)
            for (int j = 0; j < P->ny; ++j) {
                size_t q = ((size_t)l * P->nx + i) * P->ny + j;
                double re = creal(psi[q]), im = cimag(psi[q]), d = re * re + im * im;
                double x = coord(i, P->nx, P->Lx), y = coord(j, P->ny, P->Ly), z = coord(l, P->nz, P->Lz);
                epot += potential_at(P, l, i, j) * d;
                eint += 0.5 * P->g * d * d;
                x2 += x * x * d; y2 += y * y * d; z2 += z * z * d;
            }
    cplx_t *hat = (cplx_t *)malloc(sizeof(cplx_t) * (size_t)npts);
    memcpy(hat, psi, sizeof(cplx_t) * (size_t)npts);
    fft3_grid(hat, P->nz, P->nx, P->ny, -1);
    double ksum = 0.0, k2sum = 0.0;
    for (int r = 0; r < P->nz; ++r)
        for (int p = 0; p < P->nx; ++p)
            for (int q = 0; q < P->ny; ++q) {
                cplx_t z = hat[((size_t)r * P->nx + p) * P->ny + q];
                double d = creal(z) * creal(z) + cimag(z) * cimag(z);
                double kz = wavenumber(r, P->nz, P->Lz), kx = wavenumber(p, P->nx, P->Lx), ky = wavenumber(q, P->ny, P->Ly);
                ksum += d; k2sum += (kx * kx + ky * ky + kz * kz) * d;
            }
    free(hat);
    out[0] = norm; out[1] = 0.5 * k2sum / ksum * norm; out[2] = epot * dV; out[3] = eint * dV;
    out[4] = x2 * dV; out[5] = y2 * dV; out[6] = z2 * dV; out[7] = 0.0;
    return 0;
}

int oracle3_real_bytes(void) { return (int)sizeof(real_t); }

/* the two factors on their own, for pins that test one factor at a time */
int oracle3_potential_half_step(const oracle3_params *P, cplx_t *psi, double dt, int imag_time)
{
    potential_half_step(P, psi, dt, imag_time);
    return 0;
}
int oracle3_kinetic_step(const oracle3_params *P, cplx_t *psi, double dt, int imag_time)
{
    kinetic_step(P, psi, dt, imag_time);
    return 0;
}
