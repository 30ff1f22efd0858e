// gpe_api.cu -- the C ABI of include/gpe.h: plan, tables, launch sequencing, observables.
// Host logic only, plus the small non-FFT kernels (prologue reduction, final rescale,
// observables).  The FFT passes live in gpe_kernels.cuh (one TU per dtype and size).
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <functional>
#include <string>
#include <vector>

#include "../../include/gpe.h"
#include "gpe_dispatch.h"
#include "gpe_kernels.cuh"
#include "gpe_mixed.cuh"

using namespace gpe;

namespace {

constexpr int kMaxCpm = 2048;   // partial-sum slots per member (one per row in the mixed-radix family)
constexpr int kReduceCtas = 1024;  // CTAs per member of the prologue reduction
constexpr int kStepsPerGraph = 8;  // split-steps per CUDA graph launch
constexpr double kPi = 3.14159265358979323846;

thread_local std::string g_create_error;

}  // namespace

struct gpe_plan {
    int nx = 0, ny = 0, batch = 0;
    double Lx = 0, Ly = 0;
    gpe_dtype dtype = GPE_C64;
    cudaStream_t stream = nullptr;
    bool pot_set = false;
    long step = 0;
    std::string err;
    int device = 0;            // the device the plan was created on; every call checks it is current
    // test hooks, read ONCE at gpe_plan_create from the environment (tests/test_gpu_parity.py):
    // GPE_NO_PAIR = one-number-per-element kernels for complex64 too, GPE_NO_MERGE = separate half-steps
    bool no_pair = false, no_merge = false, no_fuse = false;   // GPE_NO_FUSE: never the 2-pass form
    bool no_chip = false;      // GPE_NO_CHIP: never the one-launch cluster kernel of gpe_chip.cuh
    int chip_ok = -1;          // -1 not asked yet; 1 a cluster of that shape fits this device
    bool mixed = false;        // nx or ny is not a power of two: the mixed-radix family (gpe_mixed.cuh)
    MixPlan plx = {}, ply = {};

    // device tables (typed by dtype)
    void *tw_x = nullptr, *tw_y = nullptr;
    void *tw1_x = nullptr, *tw1_y = nullptr;
    void *tw_hy = nullptr, *tw1_hy = nullptr;  // length ny/2 (paired row passes)
    void *tw1e_x = nullptr, *tw1e_y = nullptr; // first-stage twiddles for eight points per thread (cluster kernel)
    void *ytab2 = nullptr;
    void *kin_x = nullptr, *kin_y = nullptr, *kin_y2 = nullptr;
    double kin_dt = 0.0;
    int kin_mode = -1;
    void *vx = nullptr, *vy = nullptr, *latx = nullptr, *laty = nullptr, *cavx = nullptr, *cavy = nullptr;
    void *ytab = nullptr;
    void *g = nullptr;
    void *v2d = nullptr;
    size_t v2d_elems = 0;
    int flags = 0;

    // device scalars
    MemberState *st = nullptr;
    double2 *partials = nullptr;
    double *partials_b = nullptr;   // third sum (full cavity model)
    double *partials_k = nullptr;   // k-space partial sums of pass B (T/2 V T/2 in imaginary time, merged kinetic halves)
    double *d_u0 = nullptr;         // [batch] U0 of Eqs. 12, 15; nullptr = three-term model
    std::vector<double> h_u0;
    unsigned int *counters = nullptr;
    int *nonfinite = nullptr;
    double *d_sched_step = nullptr, *d_sched_amp = nullptr;
    double *d_eta = nullptr, *d_natoms = nullptr, *d_delta = nullptr, *d_kappa = nullptr;
    double *d_probe_omega = nullptr, *d_probe_delta = nullptr, *d_probe_phi = nullptr;   // nullptr = no probe

    // host copies of the descriptor
    int lattice_axis = -1, sched_len = 0, sched_batched = 0, cavity_on = 0, eta_mode = 0, sched_midpoint = 0;
    int ordering = 0;          // 0: V/2 T V/2, 1: T/2 V T/2 (gpe.h)
    // T/2 V T/2: second set of kinetic tables, for half a kinetic step (dt/2)
    void *kinh_x = nullptr, *kinh_y = nullptr, *kinh_y2 = nullptr;
    double kinh_dt = 0.0;
    int kinh_mode = -1;
    double lattice_k = 0, cavity_k = 0;
    std::vector<double> h_sched_step, h_sched_amp, h_eta, h_natoms, h_delta, h_kappa, h_g;

    // per-call parameters on the device + cached CUDA graph of kStepsPerGraph steps
    CallParams *d_call = nullptr;
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t g_exec = nullptr;
    const void *g_psi = nullptr;
    double g_dt = 0.0;
    int g_mode = -1;
    int g_fused = -1;          // the cached graph holds (B, CA) pairs of the 2-pass form
    long g_epoch = -1;
    long epoch = 0;  // bumped whenever device tables / flags may have changed

    // observables workspace
    void *scratch = nullptr;     // complex [batch][nx][ny]
    double *obs_dev = nullptr;   // [batch][8]
    double *pop_dev = nullptr;
    int pop_len = 0;
    double *obsA_dev = nullptr;  // [batch]
};

namespace {

size_t real_bytes(const gpe_plan *p) { return p->dtype == GPE_C64 ? 4 : 8; }

gpe_status fail(gpe_plan *p, gpe_status s, const std::string &msg) {
    if (p) p->err = msg; else g_create_error = msg;
    return s;
}
gpe_status cuda_fail(gpe_plan *p, cudaError_t e, const char *what) {
    cudaGetLastError();   // clear the (non-sticky) error so that a later launch check does not report it again
    return fail(p, e == cudaErrorMemoryAllocation ? GPE_ENOMEM : GPE_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define GPE_CUDA(p, call)                                              \
    do {                                                               \
        cudaError_t e__ = (call);                                      \
        if (e__ != cudaSuccess) return cuda_fail((p), e__, #call);     \
    } while (0)

// every call must run with the plan's device current: device pointers, the kernels' shared-memory
// opt-in (cudaFuncSetAttribute is per device) and the plan's buffers all belong to it
gpe_status check_device(gpe_plan *p) {
    int dev = -1;
    GPE_CUDA(p, cudaGetDevice(&dev));
    if (dev != p->device) return fail(p, GPE_EINVAL, "the plan was created on device " + std::to_string(p->device) +
                                                      " but device " + std::to_string(dev) + " is current");
    return GPE_OK;
}
#define GPE_CHECK_DEVICE(p)                                            \
    do {                                                               \
        gpe_status s__ = check_device(p);                              \
        if (s__ != GPE_OK) return s__;                                 \
    } while (0)

bool pow2_in_range(int n) { return n >= 64 && n <= 2048 && (n & (n - 1)) == 0; }
// even, no prime factor above 5
bool smooth_even_in_range(int n) {
    if (n < 64 || n > 2048 || (n & 1)) return false;
    for (int f : {2, 3, 5}) while (n % f == 0) n /= f;
    return n == 1;
}
// radices of the Stockham stages: 8 while it divides, then 5, 4 (only when 8 no longer divides), 3, 2
MixPlan make_mix_plan(int n) {
    MixPlan pl = {};
    for (int r : {8, 5, 4, 3, 2})
        while (n % r == 0 && pl.nr < 12) { pl.radix[pl.nr++] = r; n /= r; }
    return pl;
}

double coord(int i, int n, double L) { return -0.5 * L + (double)i * L / (double)n; }
double wavenumber(int q, int n, double L) { return 2.0 * kPi * (double)(q < n / 2 ? q : q - n) / L; }

// upload a double host vector as T (float/double) into a device buffer (allocating if needed)
template <typename T>
gpe_status upload_real(gpe_plan *p, void **dev, const std::vector<double> &h) {
    if (!*dev) GPE_CUDA(p, cudaMalloc(dev, sizeof(T) * h.size()));
    std::vector<T> t(h.size());
    for (size_t i = 0; i < h.size(); ++i) t[i] = (T)h[i];
    GPE_CUDA(p, cudaMemcpyAsync(*dev, t.data(), sizeof(T) * t.size(), cudaMemcpyHostToDevice, p->stream));
    GPE_CUDA(p, cudaStreamSynchronize(p->stream));
    return GPE_OK;
}
template <typename T>
gpe_status upload_cplx(gpe_plan *p, void **dev, const std::vector<double> &re, const std::vector<double> &im) {
    if (!*dev) GPE_CUDA(p, cudaMalloc(dev, 2 * sizeof(T) * re.size()));
    std::vector<T> t(2 * re.size());
    for (size_t i = 0; i < re.size(); ++i) { t[2 * i] = (T)re[i]; t[2 * i + 1] = (T)im[i]; }
    GPE_CUDA(p, cudaMemcpyAsync(*dev, t.data(), sizeof(T) * t.size(), cudaMemcpyHostToDevice, p->stream));
    GPE_CUDA(p, cudaStreamSynchronize(p->stream));
    return GPE_OK;
}
gpe_status upload_f64(gpe_plan *p, double **dev, const std::vector<double> &h) {
    if (*dev) { cudaFree(*dev); *dev = nullptr; }
    if (h.empty()) return GPE_OK;
    GPE_CUDA(p, cudaMalloc((void **)dev, sizeof(double) * h.size()));
    GPE_CUDA(p, cudaMemcpyAsync(*dev, h.data(), sizeof(double) * h.size(), cudaMemcpyHostToDevice, p->stream));
    GPE_CUDA(p, cudaStreamSynchronize(p->stream));
    return GPE_OK;
}

template <typename T> gpe_status make_twiddles(gpe_plan *p) {
    for (int ax = 0; ax < 2; ++ax) {
        int n = ax == 0 ? p->nx : p->ny;
        std::vector<double> re(n), im(n);
        for (int m = 0; m < n; ++m) {
            double ang = -2.0 * kPi * (double)m / (double)n;
            re[m] = cos(ang); im[m] = sin(ang);
        }
        gpe_status s = upload_cplx<T>(p, ax == 0 ? &p->tw_x : &p->tw_y, re, im);
        if (s != GPE_OK) return s;
        const int m1 = n / 16;
        for (int k = 0; k < 16; ++k)
            for (int j = 0; j < m1; ++j) {
                double a1 = -2.0 * kPi * (double)((long)k * j % n) / (double)n;
                re[k * m1 + j] = cos(a1); im[k * m1 + j] = sin(a1);
            }
        s = upload_cplx<T>(p, ax == 0 ? &p->tw1_x : &p->tw1_y, re, im);
        if (s != GPE_OK) return s;
        const int m8 = n / 8;   // the same table for eight points per thread (gpe_chip.cuh)
        for (int k = 0; k < 8; ++k)
            for (int j = 0; j < m8; ++j) {
                double a1 = -2.0 * kPi * (double)((long)k * j % n) / (double)n;
                re[k * m8 + j] = cos(a1); im[k * m8 + j] = sin(a1);
            }
        s = upload_cplx<T>(p, ax == 0 ? &p->tw1e_x : &p->tw1e_y, re, im);
        if (s != GPE_OK) return s;
    }
    {   // the same two tables for length ny/2 (gpe_pair.cuh, passes A and C)
        const int n = p->ny / 2, m1 = n / 16;
        std::vector<double> re(n), im(n);
        for (int m = 0; m < n; ++m) {
            double ang = -2.0 * kPi * (double)m / (double)n;
            re[m] = cos(ang); im[m] = sin(ang);
        }
        gpe_status s = upload_cplx<T>(p, &p->tw_hy, re, im);
        if (s != GPE_OK) return s;
        for (int k = 0; k < 16; ++k)
            for (int j = 0; j < m1; ++j) {
                double a1 = -2.0 * kPi * (double)((long)k * j % n) / (double)n;
                re[k * m1 + j] = cos(a1); im[k * m1 + j] = sin(a1);
            }
        s = upload_cplx<T>(p, &p->tw1_hy, re, im);
        if (s != GPE_OK) return s;
    }
    return GPE_OK;
}

// kinetic tables for (dt, mode) (row a3); 1/(nx ny) of the inverse transform folded into x.
// Written by a kernel on the plan's stream (fp64 arithmetic, rounded to T once), so that gpe_evolve
// never synchronises with the host (include/gpe.h: "only ENQUEUES").  One thread per table entry.
//   imaginary time: kin_x[q] = exp(-kx^2 dt/2)/P, kin_y[q] = exp(-ky^2 dt/2)                  (real tables)
//   real time:      kin_x[q] = (exp(-i kx^2 dt/2) - 1)/P, kin_y[q] = exp(-i ky^2 dt/2) - 1    (complex),
//                   exp(-i w) - 1 = -2 sin^2(w/2) - i sin w  (see sincosm1_t in gpe_kernels.cuh)
//                   kin_y2 = the y table in split layout per column pair for the paired pass B
template <typename T>
__global__ void k_make_kinetic(T *kin_x, T *kin_y, T *kin_y2, int nx, int ny, double Lx, double Ly, double dt, int imag) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    const double invP = 1.0 / ((double)nx * (double)ny);
    for (int ax = 0; ax < 2; ++ax) {
        const int n = ax == 0 ? nx : ny;
        if (q >= n) continue;
        const double L = ax == 0 ? Lx : Ly, sc = ax == 0 ? invP : 1.0;
        const double k = 2.0 * kPi * (double)(q < n / 2 ? q : q - n) / L, w = k * k * dt * 0.5;
        T *dst = ax == 0 ? kin_x : kin_y;
        if (imag) {
            dst[q] = (T)(exp(-w) * sc);
        } else {
            const double sh = sin(0.5 * w);
            const double re = -2.0 * sh * sh * sc, im = -sin(w) * sc;
            dst[2 * q] = (T)re; dst[2 * q + 1] = (T)im;
            if (ax == 1) {
                const int c = q >> 1, l = q & 1;
                kin_y2[8 * c + l] = (T)(1.0 + re); kin_y2[8 * c + 2 + l] = (T)im;
                kin_y2[8 * c + 4 + l] = (T)(re * invP); kin_y2[8 * c + 6 + l] = (T)(im * invP);
            }
        }
    }
}
// The buffers are allocated once (gpe_plan_create / gpe_set_potential) at their largest (complex) size.
template <typename T> gpe_status make_kinetic_into(gpe_plan *p, void *kx, void *ky, void *ky2, double dt, int mode) {
    const int n = p->nx > p->ny ? p->nx : p->ny;
    k_make_kinetic<T><<<(n + 127) / 128, 128, 0, p->stream>>>((T *)kx, (T *)ky, (T *)ky2, p->nx, p->ny, p->Lx, p->Ly, dt,
                                                              mode == GPE_IMAG_TIME ? 1 : 0);
    GPE_CUDA(p, cudaGetLastError());
    return GPE_OK;
}
template <typename T> gpe_status make_kinetic(gpe_plan *p, double dt, int mode) {
    if (p->kin_mode == mode && p->kin_dt == dt) return GPE_OK;
    gpe_status s = make_kinetic_into<T>(p, p->kin_x, p->kin_y, p->kin_y2, dt, mode);
    if (s != GPE_OK) return s;
    p->kin_mode = mode;
    p->kin_dt = dt;
    return GPE_OK;
}

// T/2 V T/2: tables of half a kinetic step (dt/2) in kinh_* (allocated by gpe_set_potential when
// ordering = 1), those of a whole one (dt) in kin_*.
template <typename T> gpe_status make_kinetic_pair(gpe_plan *p, double dt, int mode) {
    if (!(p->kinh_mode == mode && p->kinh_dt == 0.5 * dt)) {
        gpe_status s = make_kinetic_into<T>(p, p->kinh_x, p->kinh_y, p->kinh_y2, 0.5 * dt, mode);
        if (s != GPE_OK) return s;
        p->kinh_mode = mode;
        p->kinh_dt = 0.5 * dt;
    }
    return make_kinetic<T>(p, dt, mode);
}

// ------------------------------------------------------------------ small kernels
// Prologue of gpe_evolve: sums of the wavefunction as handed in by the caller (row a0 needs
// Theta_0).  grid = (kReduceCtas, batch).
template <typename T>
__global__ void __launch_bounds__(256) k_reduce(const cx<T> *psi, int nx, int ny, const T *cavx,
                                                const T *cavy, int cavity_on, FinalizeParams fin) {
    __shared__ double red[96];
    const int b = blockIdx.y;
    const cx<T> *w = psi + (size_t)b * nx * ny;
    double sn = 0.0, st = 0.0, sb = 0.0;
    for (int i = blockIdx.x; i < nx; i += gridDim.x) {
        double rn = 0.0, rt = 0.0;
        for (int j = threadIdx.x; j < ny; j += blockDim.x) {
            cx<T> z = w[(size_t)i * ny + j];
            double d = (double)z.x * (double)z.x + (double)z.y * (double)z.y;
            rn += d;
            if (cavity_on) rt += d * (double)cavy[j];
        }
        sn += rn;
        if (cavity_on) st += rt * (double)cavx[i];
        if (fin.cav_u0) sb += rn * ((double)cavx[i] * (double)cavx[i]);
    }
    block_reduce_and_finalize(fin, b, blockIdx.x, sn, st, sb, red);
}

// Epilogue of an imaginary-time gpe_evolve: apply the pending lazy scale (row a7).
template <typename T>
__global__ void __launch_bounds__(256) k_rescale(cx<T> *psi, size_t npts, MemberState *st) {
    const int b = blockIdx.y;
    const T s = (T)st[b].scale;
    cx<T> *w = psi + (size_t)b * npts;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < npts; q += (size_t)gridDim.x * blockDim.x) {
        cx<T> z = w[q];
        z.x *= s; z.y *= s;
        w[q] = z;
    }
}
// Epilogue of a real-time gpe_evolve on the paired passes: the second potential half-step of the
// last step, left pending by pass C (MemberState::pend), rows a5 of SURVEY.md 8(a).
template <typename T>
__global__ void __launch_bounds__(256) k_pending_halfstep(cx<T> *psi, int nx, int ny, int flags, const T *v2d,
                                                          const T *vx, const T *vy, const T *latx, const T *laty,
                                                          const T *cavx, const T *cavy, const T *g, T half_dt,
                                                          const MemberState *st) {
    const int b = blockIdx.y;
    if (!st[b].pend) return;
    const T A = (T)st[b].A_pend, Cc = (T)st[b].C_pend, Dc = (T)st[b].D_pend, gg = (flags & F_HAS_G) ? g[b] : T(0);
    const size_t npts = (size_t)nx * ny;
    cx<T> *w = psi + (size_t)b * npts;
    const T *v2 = (flags & F_HAS_V2D) ? v2d + ((flags & F_V2D_BATCHED) ? (size_t)b * npts : 0) : nullptr;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < npts; q += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(q / ny), j = (int)(q % ny);
        T V = T(0);
        if (flags & F_HAS_SEP) V += vx[i] + vy[j];
        if (flags & F_LAT_X) V += A * latx[i];
        if (flags & F_LAT_Y) V += A * laty[j];
        if (flags & F_CAVITY) V += Cc * cavx[i] * cavy[j];
        if (flags & F_CAV_FULL) V += Dc * cavx[i] * cavx[i];
        if (v2) V += v2[q];
        cx<T> z = w[q];
        const T ang = (V + gg * (z.x * z.x + z.y * z.y)) * half_dt;
        T sn, cm1;
        sincosm1_t(-ang, &sn, &cm1);
        const T ox = fma(z.x, cm1, fma(-z.y, sn, z.x)), oy = fma(z.x, sn, fma(z.y, cm1, z.y));
        z.x = ox; z.y = oy;
        w[q] = z;
    }
}
__global__ void k_clear_pend(MemberState *st, int batch) {
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < batch) st[b].pend = 0;
}
__global__ void k_reset_scale(MemberState *st, int batch) {
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < batch) st[b].scale = 1.0;
}

__device__ inline void block_atomic_add(double v, double *dst, double *red) {
    v = warp_sum(v);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) red[w] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int i = 0; i < (int)((blockDim.x + 31) >> 5); ++i) a += red[i];
        atomicAdd(dst, a);
    }
}

// real-space observables: out[b][0..3] += {sum d, sum (Vs + A lat) d, sum d^2, sum cos cos d}
template <typename T>
__global__ void __launch_bounds__(256) k_obs_real(const cx<T> *psi, int nx, int ny, int flags, const T *v2d,
                                                  const T *vx, const T *vy, const T *latx, const T *laty,
                                                  const T *cavx, const T *cavy, const double *A, double *out,
                                                  T *density) {
    __shared__ double red[32];
    const int b = blockIdx.y;
    const size_t npts = (size_t)nx * ny;
    const cx<T> *w = psi + (size_t)b * npts;
    const T *v2 = (flags & F_HAS_V2D) ? v2d + ((flags & F_V2D_BATCHED) ? (size_t)b * npts : 0) : nullptr;
    const double Ab = A[b];
    double sn = 0, sp = 0, s4 = 0, st = 0, sb = 0;
    for (int i = blockIdx.x; i < nx; i += gridDim.x)
        for (int j = threadIdx.x; j < ny; j += blockDim.x) {
            size_t q = (size_t)i * ny + j;
            cx<T> z = w[q];
            T dT = z.x * z.x + z.y * z.y;
            if (density) density[(size_t)b * npts + q] = dT;
            double d = (double)z.x * (double)z.x + (double)z.y * (double)z.y;
            double V = 0.0;
            if (flags & F_HAS_SEP) V += (double)vx[i] + (double)vy[j];
            if (flags & F_LAT_X) V += Ab * (double)latx[i];
            if (flags & F_LAT_Y) V += Ab * (double)laty[j];
            if (v2) V += (double)v2[q];
            sn += d; sp += V * d; s4 += d * d;
            if (flags & F_CAVITY) st += (double)cavx[i] * (double)cavy[j] * d;
            if (flags & F_CAV_FULL) sb += (double)cavx[i] * (double)cavx[i] * d;
        }
    block_atomic_add(sn, out + b * 8 + 0, red);
    block_atomic_add(sp, out + b * 8 + 1, red);
    block_atomic_add(s4, out + b * 8 + 2, red);
    block_atomic_add(st, out + b * 8 + 3, red);
    if (flags & F_CAV_FULL) block_atomic_add(sb, out + b * 8 + 6, red);
}

// k-space sums: out[b][4] += sum |psi^|^2, out[b][5] += sum k^2 |psi^|^2
template <typename T>
__global__ void __launch_bounds__(256) k_obs_k(const cx<T> *hat, int nx, int ny, double Lx, double Ly, double *out) {
    __shared__ double red[32];
    const int b = blockIdx.y;
    const cx<T> *w = hat + (size_t)b * nx * ny;
    double s0 = 0, s2 = 0;
    for (int i = blockIdx.x; i < nx; i += gridDim.x) {
        double kx = 2.0 * kPi * (double)(i < nx / 2 ? i : i - nx) / Lx;
        for (int j = threadIdx.x; j < ny; j += blockDim.x) {
            double ky = 2.0 * kPi * (double)(j < ny / 2 ? j : j - ny) / Ly;
            cx<T> z = w[(size_t)i * ny + j];
            double d = (double)z.x * (double)z.x + (double)z.y * (double)z.y;
            s0 += d; s2 += (kx * kx + ky * ky) * d;
        }
    }
    block_atomic_add(s0, out + b * 8 + 4, red);
    block_atomic_add(s2, out + b * 8 + 5, red);
}

template <typename T>
__global__ void __launch_bounds__(256) k_kdensity(const cx<T> *hat, size_t npts, const double *out, T *kd) {
    const int b = blockIdx.y;
    const double inv = 1.0 / out[b * 8 + 4];
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < npts; q += (size_t)gridDim.x * blockDim.x) {
        cx<T> z = hat[(size_t)b * npts + q];
        kd[(size_t)b * npts + q] = (T)(((double)z.x * (double)z.x + (double)z.y * (double)z.y) * inv);
    }
}

// momentum-order windows: pop[b][m + m_max] += |psi^|^2 for |k - 2 m k_l| < k_l
template <typename T>
__global__ void __launch_bounds__(256) k_populations(const cx<T> *hat, int nx, int ny, double Lx, double Ly, int axis,
                                                     double k_l, int m_max, double *pop) {
    extern __shared__ double spop[];
    const int b = blockIdx.y, nm = 2 * m_max + 1;
    for (int m = threadIdx.x; m < nm; m += blockDim.x) spop[m] = 0.0;
    __syncthreads();
    const cx<T> *w = hat + (size_t)b * nx * ny;
    for (int i = blockIdx.x; i < nx; i += gridDim.x) {
        double kx = 2.0 * kPi * (double)(i < nx / 2 ? i : i - nx) / Lx;
        for (int j = threadIdx.x; j < ny; j += blockDim.x) {
            double ky = 2.0 * kPi * (double)(j < ny / 2 ? j : j - ny) / Ly;
            double k = axis == 0 ? kx : ky;
            cx<T> z = w[(size_t)i * ny + j];
            double d = (double)z.x * (double)z.x + (double)z.y * (double)z.y;
            for (int m = -m_max; m <= m_max; ++m)
                if (fabs(k - 2.0 * m * k_l) < k_l) atomicAdd(&spop[m + m_max], d);
        }
    }
    __syncthreads();
    for (int m = threadIdx.x; m < nm; m += blockDim.x) atomicAdd(&pop[(size_t)b * nm + m], spop[m]);
}

// ------------------------------------------------------------------ roofline denominators (gpe_measure_roofs)
// in-place read + write of a buffer with 128-bit accesses by persistent CTAs: the traffic pattern of one
// fused pass (every byte read once and written once), nothing else
__global__ void __launch_bounds__(256) k_roof_rw(float4 *buf, size_t n4, float add) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n4; q += (size_t)gridDim.x * blockDim.x) {
        float4 v = __ldcg(buf + q);
        v.x += add; v.y += add; v.z += add; v.w += add;
        buf[q] = v;
    }
}
// dependent-free fused multiply-add chains, 8 independent accumulators per thread: the plain-ALU peak
template <typename T> __global__ void __launch_bounds__(256) k_roof_fma(T *out, T a, T b, int iters) {
    T acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = (T)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i] = acc[i] * a + b;
    }
    T sum = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) sum += acc[i];
    if (sum == (T)123456789) out[blockIdx.x * blockDim.x + threadIdx.x] = sum;   // never true: keeps the chains alive
}

// ------------------------------------------------------------------ typed implementations
template <typename T> StepArgs<T, cx<T>> base_args(gpe_plan *p, const void *src, void *dst) {
    StepArgs<T, cx<T>> a;
    memset(&a, 0, sizeof(a));
    a.src = (const cx<T> *)src;
    a.dst = (cx<T> *)dst;
    a.nx = p->nx; a.ny = p->ny; a.batch = p->batch; a.flags = p->flags;
    a.v2d = (const T *)p->v2d;
    a.vx = (const T *)p->vx; a.vy = (const T *)p->vy;
    a.latx = (const T *)p->latx; a.laty = (const T *)p->laty;
    a.cavx = (const T *)p->cavx; a.cavy = (const T *)p->cavy;
    a.ytab = (const T *)p->ytab;
    a.g = (const T *)p->g;
    a.tw_x = (const cx<T> *)p->tw_x; a.tw_y = (const cx<T> *)p->tw_y;
    a.tw1_x = (const cx<T> *)p->tw1_x; a.tw1_y = (const cx<T> *)p->tw1_y;
    a.tw1e_x = (const cx<T> *)p->tw1e_x; a.tw1e_y = (const cx<T> *)p->tw1e_y;
    a.tw_hy = (const cx<T> *)p->tw_hy; a.tw1_hy = (const cx<T> *)p->tw1_hy;
    a.ytab2 = (const T *)p->ytab2;
    a.kin_xc = (const cx<T> *)p->kin_x; a.kin_yc = (const cx<T> *)p->kin_y;
    a.kin_xr = (const T *)p->kin_x; a.kin_yr = (const T *)p->kin_y;
    a.kin_y2 = (const T *)p->kin_y2;
    a.inv_p = (T)(1.0 / ((double)p->nx * (double)p->ny));
    FinalizeParams &f = a.fin;
    f.partials_b = p->partials_b; f.cav_u0 = p->d_u0;
    f.partials_k = p->partials_k; f.knorm = 0; f.cpmk = 0; f.kscale = (double)p->nx * (double)p->ny;
    f.st = p->st; f.partials = p->partials; f.counters = p->counters; f.nonfinite = p->nonfinite;
    f.sched_len = p->sched_len; f.sched_step = p->d_sched_step; f.sched_amp = p->d_sched_amp;
    f.sched_batched = p->sched_batched;
    f.sched_mid = p->sched_midpoint ? 0.5 : 0.0;
    f.cavity_on = p->cavity_on; f.eta_mode = p->eta_mode;
    f.eta_or_u = p->d_eta; f.n_atoms = p->d_natoms; f.delta = p->d_delta; f.kappa = p->d_kappa;
    f.probe_omega = p->d_probe_omega; f.probe_delta = p->d_probe_delta; f.probe_phi = p->d_probe_phi;
    f.probe_dt = 0.0;   // set by a real-time gpe_evolve
    f.dxdy = (p->Lx / p->nx) * (p->Ly / p->ny);
    f.batch = p->batch;
    f.call = p->d_call;
    return a;
}

// per-pass timing (gpe_profile_passes): events bracket ONE pass per step, round-robin, so the
// host stays ahead of the device and no launch gap is measured.
struct PassProfile {
    std::vector<cudaEvent_t> e0, e1;
    std::vector<int> which;
};

gpe_status ensure_scratch(gpe_plan *p);

template <typename T>
gpe_status evolve_impl(gpe_plan *p, void *psi, double dt, long n_steps, gpe_mode mode, long record_every,
                       double *records, PassProfile *prof = nullptr) {
    const bool imag = mode == GPE_IMAG_TIME;
    const bool tvt = p->ordering == 1;
    gpe_status s = tvt ? make_kinetic_pair<T>(p, dt, (int)mode) : make_kinetic<T>(p, dt, (int)mode);
    if (s != GPE_OK) return s;
    const Ops<T> *oy = get_ops<T>(p->ny), *ox = get_ops<T>(p->nx);
    StepArgs<T, cx<T>> a = base_args<T>(p, psi, psi);
    a.half_dt = (T)(0.5 * dt);
    a.fin.probe_dt = imag ? 0.0 : dt;
    // prologue: Theta_0, A_0, C_0 from the wavefunction as given (row a0)
    {
        FinalizeParams f = a.fin;
        f.cpm = kReduceCtas < p->nx ? kReduceCtas : p->nx;
        f.normalise = 0; f.advance = 0; f.step0 = p->step;
        f.record_every = records ? record_every : 0;
        f.rec_first = record_every > 0 ? p->step / record_every : 0;
        f.records = records;
        dim3 grid(f.cpm, p->batch);
        k_reduce<T><<<grid, 256, 0, p->stream>>>((const cx<T> *)psi, p->nx, p->ny, (const T *)p->cavx,
                                                 (const T *)p->cavy, p->cavity_on, f);
        GPE_CUDA(p, cudaGetLastError());
    }
    if (p->mixed) {
        // sizes that are not powers of two: the mixed-radix passes of gpe_mixed.cuh, three
        // launches per step, natural layout, separate half-steps
        if (tvt || prof) return fail(p, GPE_EUNSUPPORTED, "ordering = 1 and per-pass profiling need power-of-two sizes");
        a.fin.cpm = p->nx;   // one row per CTA in pass C
        a.fin.normalise = imag ? 1 : 0;
        a.fin.advance = 1;
        a.fin.prepared = p->d_u0 ? 0 : 1;
        a.fin.merged = 0;
        a.fin.record_every = 0; a.fin.rec_first = 0; a.fin.records = nullptr;
        for (long n = 0; n < n_steps; ++n) {
            GPE_CUDA(p, LaunchMix<T>::row_fwd(a, p->ply, imag, p->stream));
            GPE_CUDA(p, LaunchMix<T>::col(a, p->plx, imag, 0, p->stream));
            GPE_CUDA(p, LaunchMix<T>::row_inv(a, p->ply, imag, p->stream));
        }
        if (imag) {
            dim3 grid(256, p->batch);
            k_rescale<T><<<grid, 256, 0, p->stream>>>((cx<T> *)psi, (size_t)p->nx * p->ny, p->st);
            GPE_CUDA(p, cudaGetLastError());
            k_reset_scale<<<(p->batch + 127) / 128, 128, 0, p->stream>>>(p->st, p->batch);
            GPE_CUDA(p, cudaGetLastError());
        }
        p->step += n_steps;
        return GPE_OK;
    }
    // complex64 hot path: paired passes (gpe_pair.cuh) when built for both axis lengths
    const bool paired = oy->p_row_fwd && ox->p_col && !p->no_pair;
    a.fin.cpm = p->nx / (paired ? oy->p_rows_per_cta : oy->rows_per_cta);
    a.fin.normalise = imag ? 1 : 0;
    a.fin.advance = 1;
    a.fin.prepared = p->d_u0 ? 0 : 1;   // pass B prepares the coefficients of the next step (prepare_member);
                                        // with the dispersive shift they depend on the sums
    // real time: pass C leaves its half-step to the next pass A (one multiply
    // by exp(-i (V_n + V_{n+1} + 2 g |psi|^2) dt/2) instead of two; |psi|^2, hence Theta, is unchanged)
    a.fin.merged = (!imag && !p->no_merge) ? 1 : 0;
    a.fin.record_every = 0; a.fin.rec_first = 0; a.fin.records = nullptr;  // step kernels read *call
    // four-row-interleaved intermediate array (gpe_types.h): psi -> scratch -> scratch -> psi
    const bool oop = paired && p->nx >= GPE_IL4_MIN_N && p->ny >= GPE_IL4_MIN_N && p->batch == 1;
    if (oop && (s = ensure_scratch(p)) != GPE_OK) return s;
    auto pass_a = [&](const StepArgs<T, cx<T>> &u, cudaStream_t st) -> cudaError_t {
        return paired ? oy->p_row_fwd(u, imag, st) : oy->row_fwd(u, imag, st);
    };
    auto pass_b = [&](const StepArgs<T, cx<T>> &u, cudaStream_t st) -> cudaError_t {
        return paired ? ox->p_col(u, imag, st) : ox->col(u, imag, 0, st);
    };
    auto pass_c = [&](const StepArgs<T, cx<T>> &u, cudaStream_t st) -> cudaError_t {
        return paired ? oy->p_row_inv(u, imag, st) : oy->row_inv(u, imag, st);
    };
    auto one_step = [&](cudaStream_t st, int w, cudaEvent_t e0, cudaEvent_t e1) -> gpe_status {
        if (w == 0) GPE_CUDA(p, cudaEventRecord(e0, st));
        if (oop) a.dst = (cx<T> *)p->scratch;
        GPE_CUDA(p, pass_a(a, st));
        if (oop) a.src = (const cx<T> *)p->scratch;
        if (w == 0) GPE_CUDA(p, cudaEventRecord(e1, st));
        if (w == 1) GPE_CUDA(p, cudaEventRecord(e0, st));
        GPE_CUDA(p, pass_b(a, st));
        if (w == 1) GPE_CUDA(p, cudaEventRecord(e1, st));
        if (w == 2) GPE_CUDA(p, cudaEventRecord(e0, st));
        if (oop) a.dst = (cx<T> *)psi;
        GPE_CUDA(p, pass_c(a, st));
        if (oop) a.src = (const cx<T> *)psi;
        if (w == 2) GPE_CUDA(p, cudaEventRecord(e1, st));
        return GPE_OK;
    };
    if (tvt) {
        // T/2 V T/2 (gpe.h `ordering`, Eqs. 3-4).  A "unit" is the three passes with the
        // potential factors of pass A and pass C given separately (0 = none: the multiply is exact).
        if (prof) return fail(p, GPE_EUNSUPPORTED, "per-pass profiling is for the V/2 T V/2 ordering");
        StepArgs<T, cx<T>> ah = a;   // the same passes on the tables of half a kinetic step
        ah.kin_xc = (const cx<T> *)p->kinh_x; ah.kin_yc = (const cx<T> *)p->kinh_y;
        ah.kin_xr = (const T *)p->kinh_x; ah.kin_yr = (const T *)p->kinh_y;
        ah.kin_y2 = (const T *)p->kinh_y2;
        auto unit_on = [&](StepArgs<T, cx<T>> u, T hdt_a, T hdt_c, cudaStream_t st) -> gpe_status {
            u.src = (const cx<T> *)psi; u.dst = (cx<T> *)psi;
            u.half_dt = hdt_a;
            if (oop) u.dst = (cx<T> *)p->scratch;
            GPE_CUDA(p, pass_a(u, st));
            if (oop) u.src = (const cx<T> *)p->scratch;
            GPE_CUDA(p, pass_b(u, st));
            u.half_dt = hdt_c;
            if (oop) u.dst = (cx<T> *)psi;
            GPE_CUDA(p, pass_c(u, st));
            return GPE_OK;
        };
        auto unit = [&](StepArgs<T, cx<T>> u, T hdt_a, T hdt_c) -> gpe_status { return unit_on(u, hdt_a, hdt_c, p->stream); };
        // The units of a chunk except its last are identical launches (all per-step state is on the device):
        // kStepsPerGraph of them are captured once into a CUDA graph and replayed.  `plain` launches one on a stream;
        // `kind` (2: real time, 3: imaginary time) keys the cached graph beside psi, dt, mode and the potential's epoch.
        auto replay_plain = [&](long count, int kind, const std::function<gpe_status(cudaStream_t)> &plain) -> gpe_status {
            long done_u = 0;
            if (count >= 2 * kStepsPerGraph + 1) {
                if (!(p->g_exec && p->g_psi == psi && p->g_dt == dt && p->g_mode == (int)mode && p->g_epoch == p->epoch && p->g_fused == kind)) {
                    if (p->g_exec) { cudaGraphExecDestroy(p->g_exec); p->g_exec = nullptr; }
                    if (!p->cap_stream) GPE_CUDA(p, cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking));
                    gpe_status s1 = plain(p->stream);   // one-time function attributes outside the capture
                    if (s1 != GPE_OK) return s1;
                    done_u = 1;
                    GPE_CUDA(p, cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeThreadLocal));
                    gpe_status cs = GPE_OK;
                    for (int q = 0; q < kStepsPerGraph && cs == GPE_OK; ++q) cs = plain(p->cap_stream);
                    cudaGraph_t graph = nullptr;
                    cudaError_t ce = cudaStreamEndCapture(p->cap_stream, &graph);
                    if (cs != GPE_OK) { if (graph) cudaGraphDestroy(graph); return cs; }
                    if (ce != cudaSuccess) return cuda_fail(p, ce, "cudaStreamEndCapture");
                    ce = cudaGraphInstantiate(&p->g_exec, graph, 0);
                    cudaGraphDestroy(graph);
                    if (ce != cudaSuccess) { p->g_exec = nullptr; return cuda_fail(p, ce, "cudaGraphInstantiate"); }
                    p->g_psi = psi; p->g_dt = dt; p->g_mode = (int)mode; p->g_epoch = p->epoch; p->g_fused = kind;
                }
                for (; done_u + kStepsPerGraph <= count; done_u += kStepsPerGraph) GPE_CUDA(p, cudaGraphLaunch(p->g_exec, p->stream));
            }
            for (; done_u < count; ++done_u) {
                gpe_status s1 = plain(p->stream);
                if (s1 != GPE_OK) return s1;
            }
            return GPE_OK;
        };
        // half a kinetic step, then the scalars of step `stepnow` from the psi it leaves (no advance)
        auto half_kinetic = [&](long stepnow, int real_tvt) -> gpe_status {
            StepArgs<T, cx<T>> u = ah;
            u.fin.advance = 0; u.fin.step0 = stepnow; u.fin.normalise = 0; u.fin.prepared = 0;
            u.fin.merged = real_tvt; u.fin.tvt = real_tvt;
            u.fin.record_every = records ? record_every : 0;
            u.fin.rec_first = record_every > 0 ? p->step / record_every : 0;
            u.fin.records = records;
            return unit(u, (T)0, (T)0);
        };
        if (!imag) {
            // T/2 (V T)^(c-1) V T/2 per chunk of c steps: adjacent kinetic halves merge, the full
            // potential factor is the merged multiply of pass A with both halves on the coefficients
            // of the psi that enters it (finalize_member, f.tvt).  A chunk ends where a record is due,
            // because only there is the stored psi the psi_{n+1} the record is taken from.
            for (long done = 0; done < n_steps;) {
                const long stepnow = p->step + done;
                long chunk = n_steps - done;
                if (records && record_every > 0) {
                    const long to_rec = record_every - (stepnow % record_every);
                    if (to_rec < chunk) chunk = to_rec;
                }
                if ((s = half_kinetic(stepnow, 1)) != GPE_OK) return s;
                {
                    StepArgs<T, cx<T>> u = a;
                    u.fin = a.fin; u.fin.merged = 1; u.fin.tvt = 1;
                    s = replay_plain(chunk - 1, 2, [&](cudaStream_t st) { return unit_on(u, (T)(0.5 * dt), (T)(0.5 * dt), st); });
                    if (s != GPE_OK) return s;
                    u = ah;
                    u.fin = a.fin; u.fin.merged = 1; u.fin.tvt = 1;
                    if ((s = unit(u, (T)(0.5 * dt), (T)(0.5 * dt))) != GPE_OK) return s;
                }
                k_clear_pend<<<(p->batch + 127) / 128, 128, 0, p->stream>>>(p->st, p->batch);
                GPE_CUDA(p, cudaGetLastError());
                done += chunk;
            }
        } else {
            // T/2 (V T N')^(c-1) V T/2 N per chunk of c steps.  The renormalisation N' between the kinetic halves of
            // consecutive steps is a scalar, so the halves merge into ONE pass B on the dt/2 tables applied twice,
            // which takes the norm of the wavefunction at the step boundary as a k-space sum in between (Parseval;
            // k_col_p KNORM); the last block of pass C turns it into the lazy scale and divides Theta by it.  The
            // first half of a chunk is the kinetic-only unit, its last step ends with T/2 and the real-space norm;
            // a chunk ends where a record is due (the record is taken from psi_{n+1} itself).
            const int cpmk = paired ? p->ny / 2 / ox->p_colpairs_per_cta : p->ny / ox->cols_per_cta;
            for (long done = 0; done < n_steps;) {
                const long stepnow = p->step + done;
                long chunk = n_steps - done;
                if (records && record_every > 0) {
                    const long to_rec = record_every - (stepnow % record_every);
                    if (to_rec < chunk) chunk = to_rec;
                }
                if ((s = half_kinetic(stepnow, 0)) != GPE_OK) return s;
                {
                    StepArgs<T, cx<T>> u = ah;
                    u.fin = a.fin; u.fin.merged = 0; u.fin.tvt = 0; u.fin.prepared = 0;
                    StepArgs<T, cx<T>> uk = u;
                    uk.fin.knorm = 1; uk.fin.cpmk = cpmk;
                    s = replay_plain(chunk - 1, 3, [&](cudaStream_t st) { return unit_on(uk, (T)dt, (T)0, st); });
                    if (s != GPE_OK) return s;
                    if ((s = unit(u, (T)dt, (T)0)) != GPE_OK) return s;
                }
                done += chunk;
            }
            dim3 grid(256, p->batch);
            k_rescale<T><<<grid, 256, 0, p->stream>>>((cx<T> *)psi, (size_t)p->nx * p->ny, p->st);
            GPE_CUDA(p, cudaGetLastError());
            k_reset_scale<<<(p->batch + 127) / 128, 128, 0, p->stream>>>(p->st, p->batch);
            GPE_CUDA(p, cudaGetLastError());
        }
        p->step += n_steps;
        return GPE_OK;
    }
    // Small square grids (64^2 .. 256^2): every step of the call inside ONE cluster kernel (gpe_chip.cuh).
    // Measured on B200 (us per step, cluster kernel against the multi-launch passes): 64^2 7.3 / 11.6, 128^2 7.8 / 11.0,
    // 256^2 complex64 10.3 / 11.5 (cavity: 10.7 / 15.1); 256^2 complex128 is fp64-bound on the cluster's 16 SMs
    // (17.0 against 15.2 in the 2-pass form on all SMs, but 17.0 against 23.9 with the cavity term): there the
    // cluster kernel runs only when the 2-pass form is not available.
    const bool fusable = !p->no_fuse && !(p->flags & F_CAVITY) && (imag ? !(p->flags & F_HAS_G) : !p->no_merge) && !p->d_u0;
    const bool chip_wins = p->nx < 256 || sizeof(T) == 4 || !fusable;
    bool chip_done = false;
    if (!prof && !p->no_chip && !p->no_pair && p->nx == p->ny && oy->chip && chip_wins) {
        if (p->chip_ok < 0) p->chip_ok = oy->chip_available() ? 1 : 0;
        if (p->chip_ok == 1) {
            a.src = (const cx<T> *)psi; a.dst = (cx<T> *)psi;
            GPE_CUDA(p, oy->chip(a, imag, n_steps, p->stream));
            chip_done = true;
        }
    }
    // 2-pass form ("fused pass structure"): A B (CA B)^(n-1) C, with CA = pass C of one step and
    // pass A of the next in one kernel (k_row_ca_p / k_row_ca).  Allowed when the potential factor between two
    // kinetic steps needs no global scalar of the array it multiplies: real time without the cavity term
    // (merged half-steps), or imaginary time with g = 0 and no cavity term (a linear step: the per-step
    // renormalisation commutes with it; the plain pass C that ends every call makes the final norm exact).
    const bool fused = !chip_done && !prof && !p->no_fuse && n_steps >= 2 && !(p->flags & F_CAVITY) &&
                       (imag ? !(p->flags & F_HAS_G) : a.fin.merged == 1) && a.fin.prepared == 1 &&
                       (paired ? oy->p_row_ca != nullptr : oy->row_ca != nullptr);
    if (fused) {
        auto pass_ca = [&](const StepArgs<T, cx<T>> &u, cudaStream_t st) -> cudaError_t {
            return paired ? oy->p_row_ca(u, imag, st) : oy->row_ca(u, imag, st);
        };
        cx<T> *mid = oop ? (cx<T> *)p->scratch : (cx<T> *)psi;
        a.src = (const cx<T> *)psi; a.dst = mid;
        GPE_CUDA(p, pass_a(a, p->stream));
        a.src = mid;
        auto pairs = [&](cudaStream_t st, int count) -> gpe_status {
            for (int u = 0; u < count; ++u) {
                GPE_CUDA(p, pass_b(a, st));
                GPE_CUDA(p, pass_ca(a, st));
            }
            return GPE_OK;
        };
        long done = 0;
        const long npairs = n_steps - 1;
        if (npairs >= 2 * kStepsPerGraph + 1) {
            if (!(p->g_exec && p->g_psi == psi && p->g_dt == dt && p->g_mode == (int)mode && p->g_epoch == p->epoch && p->g_fused == 1)) {
                if (p->g_exec) { cudaGraphExecDestroy(p->g_exec); p->g_exec = nullptr; }
                if (!p->cap_stream) GPE_CUDA(p, cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking));
                if ((s = pairs(p->stream, 1)) != GPE_OK) return s;   // one-time function attributes outside the capture
                done = 1;
                GPE_CUDA(p, cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeThreadLocal));
                const gpe_status cs = pairs(p->cap_stream, kStepsPerGraph);
                cudaGraph_t graph = nullptr;
                cudaError_t ce = cudaStreamEndCapture(p->cap_stream, &graph);
                if (cs != GPE_OK) { if (graph) cudaGraphDestroy(graph); return cs; }
                if (ce != cudaSuccess) return cuda_fail(p, ce, "cudaStreamEndCapture");
                ce = cudaGraphInstantiate(&p->g_exec, graph, 0);
                cudaGraphDestroy(graph);
                if (ce != cudaSuccess) { p->g_exec = nullptr; return cuda_fail(p, ce, "cudaGraphInstantiate"); }
                p->g_psi = psi; p->g_dt = dt; p->g_mode = (int)mode; p->g_epoch = p->epoch; p->g_fused = 1;
            }
            for (; done + kStepsPerGraph <= npairs; done += kStepsPerGraph) GPE_CUDA(p, cudaGraphLaunch(p->g_exec, p->stream));
        }
        if ((s = pairs(p->stream, (int)(npairs - done))) != GPE_OK) return s;
        GPE_CUDA(p, pass_b(a, p->stream));
        a.dst = (cx<T> *)psi;
        GPE_CUDA(p, pass_c(a, p->stream));
        a.src = (const cx<T> *)psi;
    }
    long n = (fused || chip_done) ? n_steps : 0;
    if (n == 0 && !prof && n_steps >= 2 * kStepsPerGraph) {
        // The arguments of the three passes do not depend on the step (all per-step state is on the
        // device), so kStepsPerGraph steps are captured once into a CUDA graph and replayed: one
        // host call per 3 * kStepsPerGraph kernels instead of one per kernel.
        if (!(p->g_exec && p->g_psi == psi && p->g_dt == dt && p->g_mode == (int)mode && p->g_epoch == p->epoch && p->g_fused == 0)) {
            if (p->g_exec) { cudaGraphExecDestroy(p->g_exec); p->g_exec = nullptr; }
            if (!p->cap_stream) GPE_CUDA(p, cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking));
            // first launches outside the capture: one-time function attributes are not stream work
            if ((s = one_step(p->stream, -1, nullptr, nullptr)) != GPE_OK) return s;
            n = 1;
            GPE_CUDA(p, cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeThreadLocal));
            gpe_status cs = GPE_OK;
            for (int u = 0; u < kStepsPerGraph && cs == GPE_OK; ++u) cs = one_step(p->cap_stream, -1, nullptr, nullptr);
            cudaGraph_t graph = nullptr;
            cudaError_t ce = cudaStreamEndCapture(p->cap_stream, &graph);
            if (cs != GPE_OK) { if (graph) cudaGraphDestroy(graph); return cs; }
            if (ce != cudaSuccess) return cuda_fail(p, ce, "cudaStreamEndCapture");
            ce = cudaGraphInstantiate(&p->g_exec, graph, 0);
            cudaGraphDestroy(graph);
            if (ce != cudaSuccess) { p->g_exec = nullptr; return cuda_fail(p, ce, "cudaGraphInstantiate"); }
            p->g_psi = psi; p->g_dt = dt; p->g_mode = (int)mode; p->g_epoch = p->epoch; p->g_fused = 0;
        }
        for (; n + kStepsPerGraph <= n_steps; n += kStepsPerGraph) GPE_CUDA(p, cudaGraphLaunch(p->g_exec, p->stream));
    }
    for (; n < n_steps; ++n) {
        const int w = prof ? (int)(n % 3) : -1;
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        if (prof) {
            GPE_CUDA(p, cudaEventCreate(&e0));
            GPE_CUDA(p, cudaEventCreate(&e1));
            prof->e0.push_back(e0); prof->e1.push_back(e1); prof->which.push_back(w);
        }
        if ((s = one_step(p->stream, w, e0, e1)) != GPE_OK) return s;
    }
    if (a.fin.merged) {
        dim3 grid(592, p->batch);
        k_pending_halfstep<T><<<grid, 256, 0, p->stream>>>((cx<T> *)psi, p->nx, p->ny, p->flags, (const T *)p->v2d,
            (const T *)p->vx, (const T *)p->vy, (const T *)p->latx, (const T *)p->laty, (const T *)p->cavx,
            (const T *)p->cavy, (const T *)p->g, a.half_dt, p->st);
        GPE_CUDA(p, cudaGetLastError());
        k_clear_pend<<<(p->batch + 127) / 128, 128, 0, p->stream>>>(p->st, p->batch);
        GPE_CUDA(p, cudaGetLastError());
    }
    if (imag) {
        dim3 grid(256, p->batch);
        k_rescale<T><<<grid, 256, 0, p->stream>>>((cx<T> *)psi, (size_t)p->nx * p->ny, p->st);
        GPE_CUDA(p, cudaGetLastError());
        k_reset_scale<<<(p->batch + 127) / 128, 128, 0, p->stream>>>(p->st, p->batch);
        GPE_CUDA(p, cudaGetLastError());
    }
    p->step += n_steps;
    return GPE_OK;
}

gpe_status ensure_scratch(gpe_plan *p) {
    if (!p->scratch)
        GPE_CUDA(p, cudaMalloc(&p->scratch, 2 * real_bytes(p) * (size_t)p->batch * p->nx * p->ny));
    return GPE_OK;
}

// psi^ of every member into the plan's scratch buffer (natural FFT order)
template <typename T> gpe_status fft_to_scratch(gpe_plan *p, const void *psi) {
    gpe_status s = ensure_scratch(p);
    if (s != GPE_OK) return s;
    const Ops<T> *oy = get_ops<T>(p->ny), *ox = get_ops<T>(p->nx);
    StepArgs<T, cx<T>> a = base_args<T>(p, psi, p->scratch);
    a.flags |= F_NO_POT;
    if (p->mixed) {
        GPE_CUDA(p, LaunchMix<T>::row_fwd(a, p->ply, false, p->stream));
        a.src = (const cx<T> *)p->scratch;
        GPE_CUDA(p, LaunchMix<T>::col(a, p->plx, false, 1, p->stream));
        return GPE_OK;
    }
    GPE_CUDA(p, oy->row_fwd(a, false, p->stream));
    a.src = (const cx<T> *)p->scratch;
    GPE_CUDA(p, ox->col(a, false, 1, p->stream));
    return GPE_OK;
}

double host_schedule(const gpe_plan *p, int b, double n) {
    if (p->sched_len <= 0) return 0.0;
    const double *amp = p->h_sched_amp.data() + (p->sched_batched ? (size_t)b * p->sched_len : 0);
    const double *st = p->h_sched_step.data();
    int L = p->sched_len;
    if (n < st[0]) return amp[0];
    int i = 0;
    for (int q = 0; q < L; ++q)
        if (st[q] <= n) i = q;
    if (i == L - 1) return amp[L - 1];
    double t = (n - st[i]) / (st[i + 1] - st[i]);
    return amp[i] + t * (amp[i + 1] - amp[i]);
}

template <typename T>
gpe_status observables_impl(gpe_plan *p, const void *psi, gpe_obs *out, void *density, void *kdensity) {
    const int B = p->batch;
    const size_t npts = (size_t)p->nx * p->ny;
    if (!p->obs_dev) GPE_CUDA(p, cudaMalloc((void **)&p->obs_dev, sizeof(double) * 8 * B));
    if (!p->obsA_dev) GPE_CUDA(p, cudaMalloc((void **)&p->obsA_dev, sizeof(double) * B));
    std::vector<double> A(B);
    for (int b = 0; b < B; ++b) A[b] = host_schedule(p, b, (double)p->step + (p->sched_midpoint ? 0.5 : 0.0));
    GPE_CUDA(p, cudaMemcpyAsync(p->obsA_dev, A.data(), sizeof(double) * B, cudaMemcpyHostToDevice, p->stream));
    GPE_CUDA(p, cudaMemsetAsync(p->obs_dev, 0, sizeof(double) * 8 * B, p->stream));
    dim3 grid(p->nx < 256 ? p->nx : 256, B);
    k_obs_real<T><<<grid, 256, 0, p->stream>>>((const cx<T> *)psi, p->nx, p->ny, p->flags, (const T *)p->v2d,
                                               (const T *)p->vx, (const T *)p->vy, (const T *)p->latx,
                                               (const T *)p->laty, (const T *)p->cavx, (const T *)p->cavy,
                                               p->obsA_dev, p->obs_dev, (T *)density);
    GPE_CUDA(p, cudaGetLastError());
    gpe_status s = fft_to_scratch<T>(p, psi);
    if (s != GPE_OK) return s;
    k_obs_k<T><<<grid, 256, 0, p->stream>>>((const cx<T> *)p->scratch, p->nx, p->ny, p->Lx, p->Ly, p->obs_dev);
    GPE_CUDA(p, cudaGetLastError());
    if (kdensity) {
        dim3 g2(256, B);
        k_kdensity<T><<<g2, 256, 0, p->stream>>>((const cx<T> *)p->scratch, npts, p->obs_dev, (T *)kdensity);
        GPE_CUDA(p, cudaGetLastError());
    }
    std::vector<double> h(8 * B);
    int nonfinite = 0;
    GPE_CUDA(p, cudaMemcpyAsync(h.data(), p->obs_dev, sizeof(double) * 8 * B, cudaMemcpyDeviceToHost, p->stream));
    GPE_CUDA(p, cudaMemcpyAsync(&nonfinite, p->nonfinite, sizeof(int), cudaMemcpyDeviceToHost, p->stream));
    GPE_CUDA(p, cudaStreamSynchronize(p->stream));
    const double dxdy = (p->Lx / p->nx) * (p->Ly / p->ny);
    for (int b = 0; b < B; ++b) {
        const double *r = &h[8 * b];
        gpe_obs &o = out[b];
        o.norm = r[0] * dxdy;
        o.e_pot = r[1] * dxdy;
        o.e_int = 0.5 * (p->h_g.empty() ? 0.0 : p->h_g[b]) * r[2] * dxdy;
        o.theta = p->cavity_on ? r[3] * dxdy : 0.0;
        o.e_kin = 0.5 * r[5] / r[4] * o.norm;
        o.e_cav = 0.0; o.re_alpha = 0.0; o.im_alpha = 0.0;
        if (p->cavity_on) {
            double eta = p->eta_mode == 0 ? p->h_eta[b] : sqrt(fabs(A[b]) * p->h_eta[b]);
            double D = p->h_delta[b] - (p->h_u0.empty() ? 0.0 : p->h_natoms[b] * p->h_u0[b] * r[6] * dxdy);   // Eq. 15
            double K = p->h_kappa[b], den = D * D + K * K;
            double num = p->h_natoms[b] * eta * o.theta;
            o.re_alpha = num * D / den;
            o.im_alpha = -num * K / den;
            o.e_cav = p->h_natoms[b] * eta * eta * o.theta * o.theta * D / den;
        }
    }
    if (nonfinite) {   // reported once: the flag is cleared so that a later, valid run is not blamed for it
        GPE_CUDA(p, cudaMemsetAsync(p->nonfinite, 0, sizeof(int), p->stream));
        return fail(p, GPE_ENONFINITE, "a non-finite norm was seen during an earlier gpe_evolve (out_host is filled)");
    }
    return GPE_OK;
}

template <typename T>
gpe_status populations_impl(gpe_plan *p, const void *psi, int axis, double k_l, int m_max, double *out) {
    const int B = p->batch, nm = 2 * m_max + 1;
    if (!p->obs_dev) GPE_CUDA(p, cudaMalloc((void **)&p->obs_dev, sizeof(double) * 8 * B));
    if (p->pop_len < nm * B) {
        if (p->pop_dev) cudaFree(p->pop_dev);
        p->pop_dev = nullptr;
        GPE_CUDA(p, cudaMalloc((void **)&p->pop_dev, sizeof(double) * nm * B));
        p->pop_len = nm * B;
    }
    GPE_CUDA(p, cudaMemsetAsync(p->obs_dev, 0, sizeof(double) * 8 * B, p->stream));
    GPE_CUDA(p, cudaMemsetAsync(p->pop_dev, 0, sizeof(double) * nm * B, p->stream));
    gpe_status s = fft_to_scratch<T>(p, psi);
    if (s != GPE_OK) return s;
    dim3 grid(p->nx < 256 ? p->nx : 256, B);
    k_obs_k<T><<<grid, 256, 0, p->stream>>>((const cx<T> *)p->scratch, p->nx, p->ny, p->Lx, p->Ly, p->obs_dev);
    GPE_CUDA(p, cudaGetLastError());
    k_populations<T><<<grid, 256, sizeof(double) * nm, p->stream>>>((const cx<T> *)p->scratch, p->nx, p->ny, p->Lx,
                                                                   p->Ly, axis, k_l, m_max, p->pop_dev);
    GPE_CUDA(p, cudaGetLastError());
    std::vector<double> h(8 * B);
    GPE_CUDA(p, cudaMemcpyAsync(h.data(), p->obs_dev, sizeof(double) * 8 * B, cudaMemcpyDeviceToHost, p->stream));
    GPE_CUDA(p, cudaMemcpyAsync(out, p->pop_dev, sizeof(double) * nm * B, cudaMemcpyDeviceToHost, p->stream));
    GPE_CUDA(p, cudaStreamSynchronize(p->stream));
    for (int b = 0; b < B; ++b)
        for (int m = 0; m < nm; ++m) out[(size_t)b * nm + m] /= h[8 * b + 4];
    return GPE_OK;
}

template <typename T> gpe_status set_potential_impl(gpe_plan *p, const gpe_potential_desc *d) {
    const int nx = p->nx, ny = p->ny, B = p->batch;
    int flags = 0;
    gpe_status s;
    std::vector<double> hx(nx, 0.0), hy(ny, 0.0);
    if (d->vx || d->vy) {
        flags |= F_HAS_SEP;
        if (d->vx) hx.assign(d->vx, d->vx + nx);
        if (d->vy) hy.assign(d->vy, d->vy + ny);
    }
    if ((s = upload_real<T>(p, &p->vx, hx)) != GPE_OK) return s;
    if ((s = upload_real<T>(p, &p->vy, hy)) != GPE_OK) return s;
    std::vector<double> lx(nx, 0.0), ly(ny, 0.0), cxv(nx, 0.0), cyv(ny, 0.0);
    if (d->lattice_axis == 0) {
        flags |= F_LAT_X;
        for (int i = 0; i < nx; ++i) { double c = cos(d->lattice_k * coord(i, nx, p->Lx)); lx[i] = c * c; }
    } else if (d->lattice_axis == 1) {
        flags |= F_LAT_Y;
        for (int j = 0; j < ny; ++j) { double c = cos(d->lattice_k * coord(j, ny, p->Ly)); ly[j] = c * c; }
    }
    if (d->cavity_on) {
        flags |= F_CAVITY;
        if (d->cav_u0) flags |= F_CAV_FULL;
        for (int i = 0; i < nx; ++i) cxv[i] = cos(d->cavity_k * coord(i, nx, p->Lx));
        for (int j = 0; j < ny; ++j) cyv[j] = cos(d->cavity_k * coord(j, ny, p->Ly));
    }
    if ((s = upload_real<T>(p, &p->latx, lx)) != GPE_OK) return s;
    if ((s = upload_real<T>(p, &p->laty, ly)) != GPE_OK) return s;
    if ((s = upload_real<T>(p, &p->cavx, cxv)) != GPE_OK) return s;
    if ((s = upload_real<T>(p, &p->cavy, cyv)) != GPE_OK) return s;
    {   // packed per-y table for the fused passes (zeros where a term is switched off)
        std::vector<double> yt(4 * (size_t)ny, 0.0);
        for (int j = 0; j < ny; ++j) { yt[4 * j] = hy[j]; yt[4 * j + 1] = ly[j]; yt[4 * j + 2] = cyv[j]; }
        if ((s = upload_real<T>(p, &p->ytab, yt)) != GPE_OK) return s;
        // the same for the paired row passes: points n and n + ny/2 side by side
        const int h = ny / 2;
        std::vector<double> y2(8 * (size_t)h, 0.0);
        for (int n = 0; n < h; ++n) {
            y2[8 * n] = hy[n]; y2[8 * n + 1] = hy[n + h]; y2[8 * n + 2] = ly[n]; y2[8 * n + 3] = ly[n + h];
            y2[8 * n + 4] = cyv[n]; y2[8 * n + 5] = cyv[n + h];
        }
        if ((s = upload_real<T>(p, &p->ytab2, y2)) != GPE_OK) return s;
    }
    p->h_g.assign(B, 0.0);
    if (d->g) {
        p->h_g.assign(d->g, d->g + B);
        for (int b = 0; b < B; ++b) if (p->h_g[b] != 0.0) flags |= F_HAS_G;
    }
    if ((s = upload_real<T>(p, &p->g, p->h_g)) != GPE_OK) return s;
    if (d->v_static) {
        flags |= F_HAS_V2D;
        if (d->v_static_batched) flags |= F_V2D_BATCHED;
        size_t elems = (size_t)nx * ny * (d->v_static_batched ? B : 1);
        if (p->v2d && p->v2d_elems != elems) { cudaFree(p->v2d); p->v2d = nullptr; }
        if (!p->v2d) GPE_CUDA(p, cudaMalloc(&p->v2d, sizeof(T) * elems));
        p->v2d_elems = elems;
        GPE_CUDA(p, cudaMemcpyAsync(p->v2d, d->v_static, sizeof(T) * elems, cudaMemcpyDeviceToDevice, p->stream));
    }
    p->flags = flags;
    return GPE_OK;
}

}  // namespace

// ------------------------------------------------------------------ C ABI
extern "C" {

const char *gpe_version(void) { return "libgpe 0.2 sm_100a"; }

int gpe_abi_version(void) { return GPE_ABI_VERSION; }
size_t gpe_sizeof_potential_desc(void) { return sizeof(gpe_potential_desc); }

const char *gpe_last_error(const gpe_plan *p) { return p ? p->err.c_str() : g_create_error.c_str(); }

gpe_status gpe_plan_create(gpe_plan **out, int nx, int ny, double Lx, double Ly, gpe_dtype dtype, int batch) {
    if (!out) return fail(nullptr, GPE_EINVAL, "out is NULL");
    if (nx <= 0 || ny <= 0 || batch < 1 || !(Lx > 0) || !(Ly > 0) || !std::isfinite(Lx) || !std::isfinite(Ly))
        return fail(nullptr, GPE_EINVAL, "nx, ny, batch must be positive and Lx, Ly finite and > 0");
    if (dtype != GPE_C64 && dtype != GPE_C128) return fail(nullptr, GPE_EINVAL, "unknown dtype");
    if (!smooth_even_in_range(nx) || !smooth_even_in_range(ny))
        return fail(nullptr, GPE_EUNSUPPORTED, "nx and ny must be even numbers in [64, 2048] with no prime factor above 5 "
                                                "(powers of two run the fast kernels)");
    gpe_plan *p = new (std::nothrow) gpe_plan();
    if (!p) return fail(nullptr, GPE_ENOMEM, "out of host memory");
    p->nx = nx; p->ny = ny; p->batch = batch; p->Lx = Lx; p->Ly = Ly; p->dtype = dtype;
    p->mixed = !pow2_in_range(nx) || !pow2_in_range(ny);
    p->plx = make_mix_plan(nx); p->ply = make_mix_plan(ny);
    gpe_status s = GPE_OK;
    auto body = [&]() -> gpe_status {
        int dev_count = 0;
        GPE_CUDA(p, cudaGetDeviceCount(&dev_count));
        if (dev_count <= 0) return fail(p, GPE_ECUDA, "no CUDA device");
        GPE_CUDA(p, cudaGetDevice(&p->device));
        p->no_pair = getenv("GPE_NO_PAIR") != nullptr;     // test hooks, read once (see struct gpe_plan)
        p->no_merge = getenv("GPE_NO_MERGE") != nullptr;
        p->no_fuse = getenv("GPE_NO_FUSE") != nullptr;
        p->no_chip = getenv("GPE_NO_CHIP") != nullptr;
        // kinetic tables at their largest (complex) size: gpe_evolve fills them with a kernel and never
        // allocates (an allocation may synchronise the device)
        const size_t rb = dtype == GPE_C64 ? 4 : 8;
        GPE_CUDA(p, cudaMalloc(&p->kin_x, 2 * rb * (size_t)nx));
        GPE_CUDA(p, cudaMalloc(&p->kin_y, 2 * rb * (size_t)ny));
        GPE_CUDA(p, cudaMalloc(&p->kin_y2, 4 * rb * (size_t)ny));
        // out-of-place intermediate array of the paired complex64 passes at 2048^2 (gpe_types.h)
        if (dtype == GPE_C64 && nx >= GPE_IL4_MIN_N && ny >= GPE_IL4_MIN_N && batch == 1 && !p->no_pair)
            GPE_CUDA(p, cudaMalloc(&p->scratch, 2 * rb * (size_t)batch * nx * ny));
        GPE_CUDA(p, cudaMalloc((void **)&p->st, sizeof(MemberState) * batch));
        GPE_CUDA(p, cudaMemset(p->st, 0, sizeof(MemberState) * batch));
        GPE_CUDA(p, cudaMalloc((void **)&p->partials, sizeof(double2) * (size_t)batch * kMaxCpm));
        GPE_CUDA(p, cudaMalloc((void **)&p->partials_b, sizeof(double) * (size_t)batch * kMaxCpm));
        GPE_CUDA(p, cudaMalloc((void **)&p->partials_k, sizeof(double) * (size_t)batch * kMaxCpm));
        GPE_CUDA(p, cudaMalloc((void **)&p->counters, sizeof(unsigned int) * batch));
        GPE_CUDA(p, cudaMemset(p->counters, 0, sizeof(unsigned int) * batch));
        GPE_CUDA(p, cudaMalloc((void **)&p->d_call, sizeof(CallParams)));
        GPE_CUDA(p, cudaMemset(p->d_call, 0, sizeof(CallParams)));
        GPE_CUDA(p, cudaMalloc((void **)&p->nonfinite, sizeof(int)));
        GPE_CUDA(p, cudaMemset(p->nonfinite, 0, sizeof(int)));
        return dtype == GPE_C64 ? make_twiddles<float>(p) : make_twiddles<double>(p);
    };
    s = body();
    if (s != GPE_OK) {
        g_create_error = p->err;
        gpe_plan_destroy(p);
        return s;
    }
    *out = p;
    return GPE_OK;
}

gpe_status gpe_plan_set_stream(gpe_plan *p, void *cuda_stream) {
    if (!p) return GPE_EINVAL;
    p->stream = (cudaStream_t)cuda_stream;
    return GPE_OK;
}

gpe_status gpe_plan_destroy(gpe_plan *p) {
    if (!p) return GPE_OK;
    cudaStreamSynchronize(p->stream);
    if (p->g_exec) cudaGraphExecDestroy(p->g_exec);
    if (p->cap_stream) cudaStreamDestroy(p->cap_stream);
    void *bufs[] = {p->d_call, p->tw_x, p->tw_y, p->tw1_x, p->tw1_y, p->tw1e_x, p->tw1e_y, p->tw_hy, p->tw1_hy, p->ytab2, p->kin_x, p->kin_y, p->kin_y2, p->kinh_x, p->kinh_y, p->kinh_y2, p->vx, p->vy, p->latx, p->laty, p->cavx, p->cavy,
                    p->ytab, p->g, p->v2d, p->st, p->partials, p->partials_b, p->partials_k, p->d_u0, p->counters, p->nonfinite, p->d_sched_step,
                    p->d_sched_amp, p->d_eta, p->d_natoms, p->d_delta, p->d_kappa, p->d_probe_omega, p->d_probe_delta,
                    p->d_probe_phi, p->scratch, p->obs_dev,
                    p->pop_dev, p->obsA_dev};
    for (void *b : bufs)
        if (b) cudaFree(b);
    delete p;
    return GPE_OK;
}

gpe_status gpe_set_potential(gpe_plan *p, const gpe_potential_desc *d) {
    if (!p) return GPE_EINVAL;
    if (!d) return fail(p, GPE_EINVAL, "descriptor is NULL");
    GPE_CHECK_DEVICE(p);
    const int B = p->batch;
    if (d->lattice_axis < -1 || d->lattice_axis > 1) return fail(p, GPE_EINVAL, "lattice_axis must be -1, 0 or 1");
    if (d->sched_len < 0 || (d->sched_len > 0 && (!d->sched_step || !d->sched_amp)))
        return fail(p, GPE_EINVAL, "schedule arrays missing");
    for (int i = 0; i < d->sched_len; ++i) {
        if (!std::isfinite(d->sched_step[i])) return fail(p, GPE_EINVAL, "sched_step not finite");
        if (i > 0 && d->sched_step[i] < d->sched_step[i - 1])
            return fail(p, GPE_EINVAL, "sched_step must be non-decreasing");
    }
    if (d->cav_u0 && !d->cavity_on) return fail(p, GPE_EINVAL, "cav_u0 needs cavity_on");
    if ((d->probe_omega || d->probe_delta || d->probe_phi) && (!d->cavity_on || !d->probe_omega))
        return fail(p, GPE_EINVAL, "the probe needs cavity_on and probe_omega");
    if (d->cavity_on && (!d->eta_or_u || !d->delta || !d->kappa))
        return fail(p, GPE_EINVAL, "cavity_on needs eta_or_u, delta and kappa");
    if (d->cavity_on && d->eta_mode != 0 && d->eta_mode != 1) return fail(p, GPE_EINVAL, "eta_mode must be 0 or 1");
    if (d->cavity_on)
        for (int b = 0; b < B; ++b)
            if (d->delta[b] == 0.0 && d->kappa[b] == 0.0) return fail(p, GPE_EINVAL, "Delta + i kappa is zero");
    if (d->v_static && ((uintptr_t)d->v_static % real_bytes(p)) != 0) return fail(p, GPE_EINVAL, "v_static misaligned");

    if (d->ordering != 0 && d->ordering != 1) return fail(p, GPE_EINVAL, "ordering must be 0 (V/2 T V/2) or 1 (T/2 V T/2)");
    // ---- every check has passed: from here on the plan is rewritten.  A failure below (a CUDA error
    // during an upload) leaves it WITHOUT a potential (GPE_ESTATE on the next gpe_evolve) rather than
    // with a mixture of the old and the new descriptor.
    p->pot_set = false;
    p->epoch++;
    p->lattice_axis = d->lattice_axis; p->lattice_k = d->lattice_k;
    p->sched_len = d->sched_len; p->sched_batched = d->sched_len > 0 ? (d->sched_batched ? 1 : 0) : 0;
    p->cavity_on = d->cavity_on ? 1 : 0; p->cavity_k = d->cavity_k; p->eta_mode = d->eta_mode;
    p->sched_midpoint = d->sched_midpoint ? 1 : 0;
    p->ordering = d->ordering;
    if (p->ordering == 1 && !p->kinh_x) {   // second set of kinetic tables (dt/2), filled by gpe_evolve
        const size_t rb = real_bytes(p);
        GPE_CUDA(p, cudaMalloc(&p->kinh_x, 2 * rb * (size_t)p->nx));
        GPE_CUDA(p, cudaMalloc(&p->kinh_y, 2 * rb * (size_t)p->ny));
        GPE_CUDA(p, cudaMalloc(&p->kinh_y2, 4 * rb * (size_t)p->ny));
    }
    p->h_sched_step.clear(); p->h_sched_amp.clear();
    if (d->sched_len > 0) {
        p->h_sched_step.assign(d->sched_step, d->sched_step + d->sched_len);
        size_t na = (size_t)d->sched_len * (p->sched_batched ? B : 1);
        p->h_sched_amp.assign(d->sched_amp, d->sched_amp + na);
    }
    p->h_eta.assign(B, 0.0); p->h_natoms.assign(B, 1.0); p->h_delta.assign(B, -1.0); p->h_kappa.assign(B, 1.0);
    if (d->cavity_on) {
        p->h_eta.assign(d->eta_or_u, d->eta_or_u + B);
        if (d->n_atoms) p->h_natoms.assign(d->n_atoms, d->n_atoms + B);
        p->h_delta.assign(d->delta, d->delta + B);
        p->h_kappa.assign(d->kappa, d->kappa + B);
    }
    gpe_status s;
    if ((s = upload_f64(p, &p->d_sched_step, p->h_sched_step)) != GPE_OK) return s;
    if ((s = upload_f64(p, &p->d_sched_amp, p->h_sched_amp)) != GPE_OK) return s;
    if ((s = upload_f64(p, &p->d_eta, p->h_eta)) != GPE_OK) return s;
    if ((s = upload_f64(p, &p->d_natoms, p->h_natoms)) != GPE_OK) return s;
    if ((s = upload_f64(p, &p->d_delta, p->h_delta)) != GPE_OK) return s;
    if ((s = upload_f64(p, &p->d_kappa, p->h_kappa)) != GPE_OK) return s;
    {   // on-axis probe (upload_f64 frees and leaves nullptr for an empty vector = no probe)
        std::vector<double> om, de, ph;
        if (d->probe_omega) {
            om.assign(d->probe_omega, d->probe_omega + B);
            de.assign(B, 0.0); ph.assign(B, 0.0);
            if (d->probe_delta) de.assign(d->probe_delta, d->probe_delta + B);
            if (d->probe_phi) ph.assign(d->probe_phi, d->probe_phi + B);
        }
        p->h_u0.clear();
        if (d->cav_u0) p->h_u0.assign(d->cav_u0, d->cav_u0 + B);
        if ((s = upload_f64(p, &p->d_u0, p->h_u0)) != GPE_OK) return s;
        if ((s = upload_f64(p, &p->d_probe_omega, om)) != GPE_OK) return s;
        if ((s = upload_f64(p, &p->d_probe_delta, de)) != GPE_OK) return s;
        if ((s = upload_f64(p, &p->d_probe_phi, ph)) != GPE_OK) return s;
    }
    s = p->dtype == GPE_C64 ? set_potential_impl<float>(p, d) : set_potential_impl<double>(p, d);
    if (s != GPE_OK) return s;
    p->pot_set = true;
    p->epoch++;
    return GPE_OK;
}

gpe_status gpe_evolve(gpe_plan *p, void *psi, double dt, long n_steps, gpe_mode mode, long record_every,
                      double *records) {
    if (!p) return GPE_EINVAL;
    if (!p->pot_set) return fail(p, GPE_ESTATE, "gpe_evolve before gpe_set_potential");
    GPE_CHECK_DEVICE(p);
    if (!psi || ((uintptr_t)psi % 16) != 0) return fail(p, GPE_EINVAL, "psi is NULL or not 16-byte aligned");
    if (mode != GPE_REAL_TIME && mode != GPE_IMAG_TIME) return fail(p, GPE_EINVAL, "unknown mode");
    if (!std::isfinite(dt) || dt == 0.0 || (mode == GPE_IMAG_TIME && dt < 0.0))
        return fail(p, GPE_EINVAL, "dt must be finite, non-zero, and > 0 in imaginary time");
    if (n_steps < 0 || record_every < 0) return fail(p, GPE_EINVAL, "n_steps and record_every must be >= 0");
    if (record_every > 0 && !records) return fail(p, GPE_EINVAL, "record_every > 0 needs a records buffer");
    if (n_steps == 0) return GPE_OK;
    return p->dtype == GPE_C64 ? evolve_impl<float>(p, psi, dt, n_steps, mode, record_every, records)
                               : evolve_impl<double>(p, psi, dt, n_steps, mode, record_every, records);
}

gpe_status gpe_fft2_forward(gpe_plan *p, const void *src, void *dst) {
    if (!p) return GPE_EINVAL;
    if (!src || !dst || ((uintptr_t)src % 16) != 0 || ((uintptr_t)dst % 16) != 0)
        return fail(p, GPE_EINVAL, "src/dst NULL or misaligned");
    GPE_CHECK_DEVICE(p);
    void *keep = p->scratch;
    p->scratch = dst;
    gpe_status s = p->dtype == GPE_C64 ? fft_to_scratch<float>(p, src) : fft_to_scratch<double>(p, src);
    p->scratch = keep;
    return s;
}

gpe_status gpe_profile_passes(gpe_plan *p, void *psi, double dt, long n_steps, gpe_mode mode, double *ms_out) {
    if (!p) return GPE_EINVAL;
    if (!p->pot_set) return fail(p, GPE_ESTATE, "gpe_profile_passes before gpe_set_potential");
    GPE_CHECK_DEVICE(p);
    if (!psi || !ms_out || ((uintptr_t)psi % 16) != 0) return fail(p, GPE_EINVAL, "psi/ms_out NULL or misaligned");
    if (!std::isfinite(dt) || dt == 0.0 || (mode == GPE_IMAG_TIME && dt < 0.0) || n_steps < 3 || n_steps > 30000)
        return fail(p, GPE_EINVAL, "dt invalid or n_steps outside [3, 30000]");
    PassProfile prof;
    gpe_status s = p->dtype == GPE_C64 ? evolve_impl<float>(p, psi, dt, n_steps, mode, 0, nullptr, &prof)
                                       : evolve_impl<double>(p, psi, dt, n_steps, mode, 0, nullptr, &prof);
    cudaError_t e = cudaStreamSynchronize(p->stream);
    double sum[3] = {0, 0, 0};
    long cnt[3] = {0, 0, 0};
    for (size_t i = 0; i < prof.e0.size(); ++i) {
        float ms = 0.f;
        if (s == GPE_OK && e == cudaSuccess && cudaEventElapsedTime(&ms, prof.e0[i], prof.e1[i]) == cudaSuccess) {
            sum[prof.which[i]] += ms;
            cnt[prof.which[i]] += 1;
        }
        cudaEventDestroy(prof.e0[i]);
        cudaEventDestroy(prof.e1[i]);
    }
    if (s != GPE_OK) return s;
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaStreamSynchronize");
    for (int k = 0; k < 3; ++k) ms_out[k] = cnt[k] ? sum[k] / (double)cnt[k] : 0.0;
    return GPE_OK;
}

gpe_status gpe_observables(gpe_plan *p, const void *psi, gpe_obs *out, void *density, void *kdensity) {
    if (!p) return GPE_EINVAL;
    if (!p->pot_set) return fail(p, GPE_ESTATE, "gpe_observables before gpe_set_potential");
    GPE_CHECK_DEVICE(p);
    if (!psi || !out || ((uintptr_t)psi % 16) != 0) return fail(p, GPE_EINVAL, "psi/out NULL or psi misaligned");
    return p->dtype == GPE_C64 ? observables_impl<float>(p, psi, out, density, kdensity)
                               : observables_impl<double>(p, psi, out, density, kdensity);
}

gpe_status gpe_populations(gpe_plan *p, const void *psi, int axis, double k_l, int m_max, double *out) {
    if (!p) return GPE_EINVAL;
    if (!psi || !out || ((uintptr_t)psi % 16) != 0) return fail(p, GPE_EINVAL, "psi/out NULL or psi misaligned");
    if ((axis != 0 && axis != 1) || !(k_l > 0) || m_max < 0 || m_max > 64)
        return fail(p, GPE_EINVAL, "axis in {0,1}, k_l > 0, 0 <= m_max <= 64");
    GPE_CHECK_DEVICE(p);
    return p->dtype == GPE_C64 ? populations_impl<float>(p, psi, axis, k_l, m_max, out)
                               : populations_impl<double>(p, psi, axis, k_l, m_max, out);
}

gpe_status gpe_measure_roofs(void *cuda_stream, double *out) {
    if (!out) return GPE_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        g_create_error = "no CUDA device";
        return GPE_ECUDA;
    }
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return GPE_ECUDA;
    gpe_status rc = GPE_OK;
    void *buf = nullptr;
    const size_t sizes[3] = {32u << 20, 64u << 20, 1024u << 20};
    if (cudaMalloc(&buf, sizes[2]) != cudaSuccess) { cudaGetLastError(); cudaEventDestroy(e0); cudaEventDestroy(e1); g_create_error = "cudaMalloc failed"; return GPE_ENOMEM; }
    cudaMemsetAsync(buf, 0, sizes[2], st);
    for (int k = 0; k < 3; ++k) {
        const size_t n4 = sizes[k] / 16;
        const int reps = k < 2 ? 200 : 10;
        double best = 0.0;
        for (int trial = 0; trial < 3; ++trial) {
            for (int w = 0; w < 3; ++w) k_roof_rw<<<nsm * 8, 256, 0, st>>>((float4 *)buf, n4, 0.f);
            cudaEventRecord(e0, st);
            for (int r = 0; r < reps; ++r) k_roof_rw<<<nsm * 8, 256, 0, st>>>((float4 *)buf, n4, 0.f);
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = GPE_ECUDA; break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            const double gbs = 2.0 * (double)sizes[k] * reps / (ms * 1e-3) / 1e9;
            if (gbs > best) best = gbs;
        }
        out[k] = best;
    }
    for (int k = 0; k < 2 && rc == GPE_OK; ++k) {
        const int iters = 4096, blocks = nsm * 8;
        double best = 0.0;
        for (int trial = 0; trial < 3; ++trial) {
            if (k == 0) k_roof_fma<float><<<blocks, 256, 0, st>>>((float *)buf, 1.0000001f, 1e-9f, 64);
            else k_roof_fma<double><<<blocks, 256, 0, st>>>((double *)buf, 1.0000001, 1e-9, 64);
            cudaEventRecord(e0, st);
            if (k == 0) k_roof_fma<float><<<blocks, 256, 0, st>>>((float *)buf, 1.0000001f, 1e-9f, iters);
            else k_roof_fma<double><<<blocks, 256, 0, st>>>((double *)buf, 1.0000001, 1e-9, iters);
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = GPE_ECUDA; break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            const double tf = 2.0 * 32.0 * iters * 256.0 * blocks / (ms * 1e-3) / 1e12;
            if (tf > best) best = tf;
        }
        out[3 + k] = best;
    }
    if (cudaGetLastError() != cudaSuccess) rc = GPE_ECUDA;
    cudaFree(buf);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return rc;
}

gpe_status gpe_get_step(const gpe_plan *p, long *step) {
    if (!p || !step) return GPE_EINVAL;
    *step = p->step;
    return GPE_OK;
}

gpe_status gpe_set_step(gpe_plan *p, long step) {
    if (!p) return GPE_EINVAL;
    // the record index floor(n / record_every) - floor(n0 / record_every) - 1 and the T/2 V T/2 chunking are
    // written for n >= 0 (C division truncates); shift the schedule knots instead of the counter
    if (step < 0) return fail(p, GPE_EINVAL, "the step counter must be >= 0");
    p->step = step;
    return GPE_OK;
}

}  // extern "C"
