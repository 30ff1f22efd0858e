// gpe3_api.cu -- host side of the 3-D entry points of include/gpe.h (gpe3_*): plan, potential, evolve, observables.
// SURVEY.md 8(f) row f4 (second half); the kernels and the pass structure are in gpe3_kernels.cuh.
#include <cmath>
#include <cstdint>
#include <new>
#include <string>
#include <vector>

#include "../../include/gpe.h"
#include "gpe3_kernels.cuh"

using namespace gpe;

namespace {
constexpr double kPi = 3.14159265358979323846;
thread_local std::string g_create_error3;
constexpr int kObsCtas = 1184;   // 148 SMs x 8 CTAs of 256 threads (k3_observe)
__global__ void k3_reset_scale(State3 *st) { st->scale = 1.0; }
}  // namespace

struct gpe3_plan {
    int nx = 0, ny = 0, nz = 0;
    double Lx = 0, Ly = 0, Lz = 0;
    gpe_dtype dtype = GPE_C64;
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    bool has_potential = false;
    double g = 0.0;
    void *tw[3] = {}, *tw1[3] = {};      // per axis (0: x, 1: y, 2: z)
    void *kin[3] = {}, *k2[3] = {};      // kinetic factor tables (for kin_dt / kin_mode) and k^2
    double kin_dt = 0.0;
    int kin_mode = -1;
    void *v3d = nullptr, *vsep[3] = {};  // potential in the plan's real type
    bool has_v3d = false;
    State3 *st = nullptr;
    double *partials = nullptr, *part6 = nullptr, *measure = nullptr;   // measure: [3] on the device
    unsigned int *counter = nullptr;
    int *nonfinite = nullptr;
    long long step = 0;
    // CUDA graph of kGraphSteps plain steps (small grids) and what its kernel arguments were captured for
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t g_exec = nullptr;
    void *g_psi = nullptr;
    double g_dt = 0.0;
    int g_imag = -1;
};

namespace {

gpe_status fail3(gpe3_plan *p, gpe_status s, const std::string &msg) {
    if (p) p->err = msg; else g_create_error3 = msg;
    return s;
}
gpe_status cuda_fail3(gpe3_plan *p, cudaError_t e, const char *what) {
    cudaGetLastError();
    return fail3(p, e == cudaErrorMemoryAllocation ? GPE_ENOMEM : GPE_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define GPE3_CUDA(p, call)                                              \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) return cuda_fail3((p), e_, #call);       \
    } while (0)

gpe_status check_device3(gpe3_plan *p) {
    int dev = -1;
    GPE3_CUDA(p, cudaGetDevice(&dev));
    if (dev != p->device) return fail3(p, GPE_ESTATE, "the plan was created on another device than the current one");
    return GPE_OK;
}

size_t real_bytes3(const gpe3_plan *p) { return p->dtype == GPE_C64 ? 4 : 8; }
bool size_ok3(int n) { return n == 64 || n == 128 || n == 256 || n == 512 || n == 1024; }
int axis_len(const gpe3_plan *p, int ax) { return ax == 0 ? p->nx : ax == 1 ? p->ny : p->nz; }
double axis_box(const gpe3_plan *p, int ax) { return ax == 0 ? p->Lx : ax == 1 ? p->Ly : p->Lz; }

template <typename T> gpe_status upload3(gpe3_plan *p, void **dev, const std::vector<double> &v) {
    if (!*dev) GPE3_CUDA(p, cudaMalloc(dev, sizeof(T) * v.size()));
    std::vector<T> t(v.size());
    for (size_t i = 0; i < v.size(); ++i) t[i] = (T)v[i];
    GPE3_CUDA(p, cudaMemcpyAsync(*dev, t.data(), sizeof(T) * t.size(), cudaMemcpyHostToDevice, p->stream));
    GPE3_CUDA(p, cudaStreamSynchronize(p->stream));   // t goes out of scope
    return GPE_OK;
}

// twiddles of one axis as gpe_fft.cuh wants them: tw[m] = exp(-2 pi i m / n), tw1[k * (n/16) + j] = exp(-2 pi i k j / n)
template <typename T> gpe_status make_twiddles3(gpe3_plan *p) {
    for (int ax = 0; ax < 3; ++ax) {
        const int n = axis_len(p, ax), m1 = n / 16;
        std::vector<double> a(2 * (size_t)n), b(2 * (size_t)n);
        for (int m = 0; m < n; ++m) {
            const double ang = -2.0 * kPi * (double)m / (double)n;
            a[2 * m] = cos(ang); a[2 * m + 1] = sin(ang);
        }
        for (int k = 0; k < 16; ++k)
            for (int j = 0; j < m1; ++j) {
                const double ang = -2.0 * kPi * (double)((long)k * j % n) / (double)n;
                b[2 * (k * m1 + j)] = cos(ang); b[2 * (k * m1 + j) + 1] = sin(ang);
            }
        gpe_status s = upload3<T>(p, &p->tw[ax], a);
        if (s != GPE_OK) return s;
        if ((s = upload3<T>(p, &p->tw1[ax], b)) != GPE_OK) return s;
        GPE3_CUDA(p, cudaMalloc(&p->kin[ax], 2 * sizeof(T) * (size_t)n));
        GPE3_CUDA(p, cudaMalloc(&p->k2[ax], sizeof(T) * (size_t)n));
        k3_make_tables<T><<<(n + 127) / 128, 128, 0, p->stream>>>((T *)nullptr, (T *)p->k2[ax], n, axis_box(p, ax), 0.0, 0);
        GPE3_CUDA(p, cudaGetLastError());
    }
    return GPE_OK;
}

template <typename T> gpe_status make_kinetic3(gpe3_plan *p, double dt, int mode) {
    if (p->kin_mode == mode && p->kin_dt == dt) return GPE_OK;
    for (int ax = 0; ax < 3; ++ax) {
        const int n = axis_len(p, ax);
        k3_make_tables<T><<<(n + 127) / 128, 128, 0, p->stream>>>((T *)p->kin[ax], (T *)nullptr, n, axis_box(p, ax), dt,
                                                                  mode == GPE_IMAG_TIME ? 1 : 0);
        GPE3_CUDA(p, cudaGetLastError());
    }
    p->kin_mode = mode;
    p->kin_dt = dt;
    return GPE_OK;
}

template <typename T> Args3<T> base_args(gpe3_plan *p, void *psi) {
    Args3<T> a = {};
    a.psi = (cx<T> *)psi;
    a.nx = p->nx; a.ny = p->ny; a.nz = p->nz;
    a.v3d = p->has_v3d ? (const T *)p->v3d : nullptr;
    a.vx = (const T *)p->vsep[0]; a.vy = (const T *)p->vsep[1]; a.vz = (const T *)p->vsep[2];
    a.g = (T)p->g;
    a.fac = T(1);
    a.st = p->st;
    a.partials = p->partials; a.counter = p->counter; a.nonfinite = p->nonfinite;
    a.dV = (p->Lx / p->nx) * (p->Ly / p->ny) * (p->Lz / p->nz);
    return a;
}
template <typename T> void set_axis(gpe3_plan *p, Args3<T> &a, int ax, bool measure) {
    a.kin = (const T *)(measure ? p->k2[ax] : p->kin[ax]);
    a.inv_n = (T)(1.0 / (double)axis_len(p, ax));
    a.tw = (const cx<T> *)p->tw[ax];
    a.tw1 = (const cx<T> *)p->tw1[ax];
    a.final_axis = ax == 2;
    if (ax == 0) { a.line_stride = p->ny; a.slab_stride = (long)p->nx * p->ny; }
    if (ax == 2) { a.line_stride = (long)p->nx * p->ny; a.slab_stride = 0; }
}
// the pass along axis ax (1: rows; 0, 2: columns)
template <typename T> cudaError_t run_axis(gpe3_plan *p, const Args3<T> &a, int ax, bool imag, int mode, cudaStream_t st, unsigned *nctas = nullptr) {
    const Ops3<T> *o = get_ops3<T>(axis_len(p, ax));
    if (ax == 1) return o->row(a, imag, mode, st);
    if (ax == 0) return o->col(a, imag, mode, p->ny, (unsigned)p->nz, nctas, st);
    return o->col(a, imag, mode, (long)p->nx * p->ny, 1u, nctas, st);
}

// one step on stream st.  fac: 1 or 2 (merged real-time halves); sums: reduce the norm at the end; step_index < 0:
// a step replayed from the graph (no record, the device step counter just advances)
template <typename T>
gpe_status step3(gpe3_plan *p, const Args3<T> &base, bool imag, T fac, int sums, long long step_index, double *record, cudaStream_t st) {
    Args3<T> a = base;
    a.step_index = step_index;
    a.pot = 1;
    a.fac = fac;
    set_axis<T>(p, a, 1, false);
    GPE3_CUDA(p, run_axis<T>(p, a, 1, imag, 0, st));
    a.pot = 0;
    // the x pass walks the array backwards: it starts on the slabs the row pass wrote last, which are still in L2
    // (256^3 complex64 real time: 249 -> 246 us per step; reversing other passes, or alternate steps, measured the same)
    a.rev = 1;
    set_axis<T>(p, a, 0, false);
    GPE3_CUDA(p, run_axis<T>(p, a, 0, imag, 0, st));
    set_axis<T>(p, a, 2, false);
    a.rev = 0;
    a.pot = imag ? 1 : 0;
    a.sums = sums;
    a.record = record;
    unsigned int nparts = 0;
    GPE3_CUDA(p, run_axis<T>(p, a, 2, imag, 0, st, &nparts));
    if (sums) {
        const bool pdl = (long)p->nx * p->ny * p->nz <= GPE3_PDL_MAX;
        GPE3_CUDA(p, imag ? launch_pdl(k3_finalize<true>, dim3(1), dim3(256), 0, st, pdl, p->st, (const double *)p->partials, nparts, a.dV, step_index, record, p->nonfinite)
                          : launch_pdl(k3_finalize<false>, dim3(1), dim3(256), 0, st, pdl, p->st, (const double *)p->partials, nparts, a.dV, step_index, record, p->nonfinite));
    }
    return GPE_OK;
}

// Small grids are bound by the host's launch rate (64^3: three 3-us kernels per step against ~7 us of host time per
// launch): kGraphSteps plain steps -- no record, not the first or last step of a real-time call -- are captured once
// into a CUDA graph and replayed.  The graph is keyed by everything its kernel arguments hold.
constexpr int kGraphSteps = 8;
template <typename T> gpe_status graph3(gpe3_plan *p, const Args3<T> &base, bool imag, double dt) {
    if (p->g_exec && p->g_psi == (void *)base.psi && p->g_dt == dt && p->g_imag == (int)imag) return GPE_OK;
    if (p->g_exec) { cudaGraphExecDestroy(p->g_exec); p->g_exec = nullptr; }
    if (!p->cap_stream) GPE3_CUDA(p, cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking));
    GPE3_CUDA(p, cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeThreadLocal));
    gpe_status s = GPE_OK;
    for (int q = 0; q < kGraphSteps && s == GPE_OK; ++q) s = step3<T>(p, base, imag, imag ? T(1) : T(2), imag ? 1 : 0, -1, nullptr, p->cap_stream);
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(p->cap_stream, &g);
    if (s != GPE_OK) { if (g) cudaGraphDestroy(g); return s; }
    if (e != cudaSuccess) return cuda_fail3(p, e, "cudaStreamEndCapture");
    e = cudaGraphInstantiate(&p->g_exec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { p->g_exec = nullptr; return cuda_fail3(p, e, "cudaGraphInstantiate"); }
    p->g_psi = (void *)base.psi; p->g_dt = dt; p->g_imag = (int)imag;
    return GPE_OK;
}

template <typename T>
gpe_status evolve3(gpe3_plan *p, void *psi, double dt, long long n_steps, int mode, long long record_every, double *records) {
    const bool imag = mode == GPE_IMAG_TIME;
    gpe_status s = make_kinetic3<T>(p, dt, mode);
    if (s != GPE_OK) return s;
    Args3<T> base = base_args<T>(p, psi);
    base.half_dt = (T)(0.5 * dt);
    const bool use_graph = (long)p->nx * p->ny * p->nz <= GPE3_PDL_MAX && n_steps >= 2 * kGraphSteps;
    const bool recording = records && record_every > 0;
    long long nrec = 0;
    for (long long q = 0; q < n_steps;) {
        const long long n = p->step + q;
        // a chunk of plain steps: no record falls on indices n+1 .. n+kGraphSteps, and in real time neither the first
        // step of the call (fac = 1) nor the last (it reduces the norm) is inside
        const bool no_rec = !recording || (n + kGraphSteps) / record_every == n / record_every;
        // (q >= 1 in both modes: the first step of a call is launched directly, so that one-time function attributes --
        // not stream work -- are set outside the capture)
        if (use_graph && no_rec && q >= 1 && q + kGraphSteps <= n_steps - (imag ? 0 : 1)) {
            if ((s = graph3<T>(p, base, imag, dt)) != GPE_OK) return s;
            GPE3_CUDA(p, cudaGraphLaunch(p->g_exec, p->stream));
            q += kGraphSteps;
            continue;
        }
        const bool rec = recording && ((n + 1) % record_every) == 0;
        s = step3<T>(p, base, imag, (imag || q == 0) ? T(1) : T(2), (imag || rec || q == n_steps - 1) ? 1 : 0, n,
                     rec ? records + 3 * (nrec++) : nullptr, p->stream);
        if (s != GPE_OK) return s;
        ++q;
    }
    if (n_steps > 0) {
        if (imag) {
            k3_point<T, 1><<<kObsCtas, 256, 0, p->stream>>>(base);
            GPE3_CUDA(p, cudaGetLastError());
            k3_reset_scale<<<1, 1, 0, p->stream>>>(p->st);
        } else {
            k3_point<T, 0><<<kObsCtas, 256, 0, p->stream>>>(base);
        }
        GPE3_CUDA(p, cudaGetLastError());
    }
    p->step += n_steps;
    return GPE_OK;
}

template <typename T> gpe_status observables3(gpe3_plan *p, const void *psi, double *out) {
    Args3<T> a = base_args<T>(p, const_cast<void *>(psi));
    k3_observe<T><<<kObsCtas, 256, 0, p->stream>>>(a, p->Lx, p->Ly, p->Lz, p->part6);
    GPE3_CUDA(p, cudaGetLastError());
    for (int ax = 0; ax < 3; ++ax) {
        Args3<T> m = a;
        set_axis<T>(p, m, ax, true);
        m.measure_out = p->measure + ax;
        GPE3_CUDA(p, run_axis<T>(p, m, ax, false, 1, p->stream));
    }
    std::vector<double> h6((size_t)kObsCtas * 6);
    double k2sum[3];
    GPE3_CUDA(p, cudaMemcpyAsync(h6.data(), p->part6, sizeof(double) * h6.size(), cudaMemcpyDeviceToHost, p->stream));
    GPE3_CUDA(p, cudaMemcpyAsync(k2sum, p->measure, sizeof(k2sum), cudaMemcpyDeviceToHost, p->stream));
    GPE3_CUDA(p, cudaStreamSynchronize(p->stream));
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int c = 0; c < kObsCtas; ++c)
        for (int m = 0; m < 6; ++m) s[m] += h6[(size_t)c * 6 + m];
    const double dV = a.dV;
    // e_kin = (1/2) sum_k |k|^2 |psi^|^2 dV / P, and by Parseval over the two other axes
    // sum_k k_a^2 |psi^|^2 = (P / n_a) sum_(other coordinates) sum_(k_a) k_a^2 |F_a psi|^2
    double ekin = 0.0;
    for (int ax = 0; ax < 3; ++ax) ekin += 0.5 * k2sum[ax] / (double)axis_len(p, ax) * dV;
    out[0] = s[0] * dV; out[1] = ekin; out[2] = s[1] * dV; out[3] = s[2] * dV;
    out[4] = s[3] * dV; out[5] = s[4] * dV; out[6] = s[5] * dV; out[7] = 0.0;
    return GPE_OK;
}

}  // namespace

extern "C" {

const char *gpe3_last_error(const gpe3_plan *p) { return p ? p->err.c_str() : g_create_error3.c_str(); }

gpe_status gpe3_plan_destroy(gpe3_plan *p) {
    if (!p) return GPE_OK;
    cudaStreamSynchronize(p->stream);
    if (p->g_exec) cudaGraphExecDestroy(p->g_exec);
    if (p->cap_stream) cudaStreamDestroy(p->cap_stream);
    void *bufs[] = {p->tw[0], p->tw[1], p->tw[2], p->tw1[0], p->tw1[1], p->tw1[2], p->kin[0], p->kin[1], p->kin[2],
                    p->k2[0], p->k2[1], p->k2[2], p->v3d, p->vsep[0], p->vsep[1], p->vsep[2], p->st, p->partials,
                    p->part6, p->measure, p->counter, p->nonfinite};
    for (void *b : bufs)
        if (b) cudaFree(b);
    delete p;
    return GPE_OK;
}

gpe_status gpe3_plan_create(gpe3_plan **out, int nx, int ny, int nz, double Lx, double Ly, double Lz, gpe_dtype dtype) {
    if (!out) return fail3(nullptr, GPE_EINVAL, "out is NULL");
    if (!(Lx > 0) || !(Ly > 0) || !(Lz > 0) || !std::isfinite(Lx) || !std::isfinite(Ly) || !std::isfinite(Lz))
        return fail3(nullptr, GPE_EINVAL, "Lx, Ly, Lz must be finite and > 0");
    if (dtype != GPE_C64 && dtype != GPE_C128) return fail3(nullptr, GPE_EINVAL, "unknown dtype");
    if (!size_ok3(nx) || !size_ok3(ny) || !size_ok3(nz))
        return fail3(nullptr, GPE_EUNSUPPORTED, "the 3-D path takes nx, ny, nz in {64, 128, 256, 512, 1024}");
    gpe3_plan *p = new (std::nothrow) gpe3_plan;
    if (!p) return fail3(nullptr, GPE_ENOMEM, "host allocation failed");
    p->nx = nx; p->ny = ny; p->nz = nz; p->Lx = Lx; p->Ly = Ly; p->Lz = Lz; p->dtype = dtype;
    auto body = [&]() -> gpe_status {
        GPE3_CUDA(p, cudaGetDevice(&p->device));
        // one partial per CTA of any pass: at most one CTA per line of a face of the grid
        size_t face = (size_t)nx * ny;
        if ((size_t)ny * nz > face) face = (size_t)ny * nz;
        if ((size_t)nz * nx > face) face = (size_t)nz * nx;
        const size_t nparts = face + 64;
        GPE3_CUDA(p, cudaMalloc(&p->st, sizeof(State3)));
        GPE3_CUDA(p, cudaMalloc(&p->partials, sizeof(double) * nparts));
        GPE3_CUDA(p, cudaMalloc(&p->part6, sizeof(double) * 6 * kObsCtas));
        GPE3_CUDA(p, cudaMalloc(&p->measure, sizeof(double) * 4));
        GPE3_CUDA(p, cudaMalloc(&p->counter, sizeof(unsigned int)));
        GPE3_CUDA(p, cudaMalloc(&p->nonfinite, sizeof(int)));
        GPE3_CUDA(p, cudaMemsetAsync(p->counter, 0, sizeof(unsigned int), p->stream));
        GPE3_CUDA(p, cudaMemsetAsync(p->nonfinite, 0, sizeof(int), p->stream));
        const State3 st0 = {1.0, 0.0, 0.0, 0};
        GPE3_CUDA(p, cudaMemcpyAsync(p->st, &st0, sizeof(st0), cudaMemcpyHostToDevice, p->stream));
        GPE3_CUDA(p, cudaStreamSynchronize(p->stream));
        return dtype == GPE_C64 ? make_twiddles3<float>(p) : make_twiddles3<double>(p);
    };
    gpe_status s = body();
    if (s != GPE_OK) {
        g_create_error3 = p->err;
        gpe3_plan_destroy(p);
        return s;
    }
    *out = p;
    return GPE_OK;
}

gpe_status gpe3_plan_set_stream(gpe3_plan *p, void *cuda_stream) {
    if (!p) return GPE_EINVAL;
    p->stream = (cudaStream_t)cuda_stream;
    return GPE_OK;
}

gpe_status gpe3_set_potential(gpe3_plan *p, const void *v_static_dev, const double *vx, const double *vy, const double *vz, double g) {
    if (!p) return GPE_EINVAL;
    gpe_status s = check_device3(p);
    if (s != GPE_OK) return s;
    if (!std::isfinite(g)) return fail3(p, GPE_EINVAL, "g is not finite");
    if (v_static_dev && ((uintptr_t)v_static_dev % real_bytes3(p)) != 0) return fail3(p, GPE_EINVAL, "v_static misaligned");
    const double *sep[3] = {vx, vy, vz};
    for (int ax = 0; ax < 3; ++ax)
        if (sep[ax])
            for (int i = 0; i < axis_len(p, ax); ++i)
                if (!std::isfinite(sep[ax][i])) return fail3(p, GPE_EINVAL, "vx / vy / vz holds a non-finite value");
    p->has_potential = false;
    if (p->g_exec) { cudaGraphExecDestroy(p->g_exec); p->g_exec = nullptr; }   // g, v3d are kernel arguments
    for (int ax = 0; ax < 3; ++ax) {
        std::vector<double> v((size_t)axis_len(p, ax), 0.0);
        if (sep[ax]) v.assign(sep[ax], sep[ax] + axis_len(p, ax));
        s = p->dtype == GPE_C64 ? upload3<float>(p, &p->vsep[ax], v) : upload3<double>(p, &p->vsep[ax], v);
        if (s != GPE_OK) return s;
    }
    const size_t bytes = real_bytes3(p) * (size_t)p->nx * p->ny * p->nz;
    if (v_static_dev) {
        if (!p->v3d) GPE3_CUDA(p, cudaMalloc(&p->v3d, bytes));
        GPE3_CUDA(p, cudaMemcpyAsync(p->v3d, v_static_dev, bytes, cudaMemcpyDeviceToDevice, p->stream));
        GPE3_CUDA(p, cudaStreamSynchronize(p->stream));
    }
    p->has_v3d = v_static_dev != nullptr;
    p->g = g;
    p->has_potential = true;
    return GPE_OK;
}

gpe_status gpe3_evolve(gpe3_plan *p, void *psi_dev, double dt, long long n_steps, gpe_mode mode, long long record_every,
                       double *records_dev) {
    if (!p) return GPE_EINVAL;
    gpe_status s = check_device3(p);
    if (s != GPE_OK) return s;
    if (!p->has_potential) return fail3(p, GPE_ESTATE, "gpe3_evolve before gpe3_set_potential");
    if (!psi_dev || ((uintptr_t)psi_dev % 16) != 0) return fail3(p, GPE_EINVAL, "psi_dev is NULL or not 16-byte aligned");
    if (mode != GPE_REAL_TIME && mode != GPE_IMAG_TIME) return fail3(p, GPE_EINVAL, "unknown mode");
    if (!std::isfinite(dt) || dt == 0.0 || (mode == GPE_IMAG_TIME && dt < 0.0))
        return fail3(p, GPE_EINVAL, "dt must be finite and non-zero, and > 0 in imaginary time");
    if (n_steps < 0 || record_every < 0) return fail3(p, GPE_EINVAL, "n_steps and record_every must be >= 0");
    if (records_dev && ((uintptr_t)records_dev % 8) != 0) return fail3(p, GPE_EINVAL, "records_dev misaligned");
    return p->dtype == GPE_C64 ? evolve3<float>(p, psi_dev, dt, n_steps, mode, record_every, records_dev)
                               : evolve3<double>(p, psi_dev, dt, n_steps, mode, record_every, records_dev);
}

gpe_status gpe3_observables(gpe3_plan *p, const void *psi_dev, double *out_host) {
    if (!p) return GPE_EINVAL;
    gpe_status s = check_device3(p);
    if (s != GPE_OK) return s;
    if (!p->has_potential) return fail3(p, GPE_ESTATE, "gpe3_observables before gpe3_set_potential");
    if (!psi_dev || !out_host || ((uintptr_t)psi_dev % 16) != 0) return fail3(p, GPE_EINVAL, "psi_dev / out_host is NULL or psi_dev misaligned");
    return p->dtype == GPE_C64 ? observables3<float>(p, psi_dev, out_host) : observables3<double>(p, psi_dev, out_host);
}

gpe_status gpe3_synchronize(gpe3_plan *p) {
    if (!p) return GPE_EINVAL;
    gpe_status s = check_device3(p);
    if (s != GPE_OK) return s;
    int flag = 0;
    GPE3_CUDA(p, cudaMemcpyAsync(&flag, p->nonfinite, sizeof(int), cudaMemcpyDeviceToHost, p->stream));
    GPE3_CUDA(p, cudaStreamSynchronize(p->stream));
    if (flag) {
        GPE3_CUDA(p, cudaMemsetAsync(p->nonfinite, 0, sizeof(int), p->stream));
        return fail3(p, GPE_ENONFINITE, "the norm became non-finite (or zero) during an earlier gpe3_evolve");
    }
    return GPE_OK;
}

gpe_status gpe3_get_step(const gpe3_plan *p, long long *step) {
    if (!p || !step) return GPE_EINVAL;
    *step = p->step;
    return GPE_OK;
}
gpe_status gpe3_set_step(gpe3_plan *p, long long step) {
    if (!p) return GPE_EINVAL;
    if (step < 0) return fail3(p, GPE_EINVAL, "step must be >= 0");
    p->step = step;
    return GPE_OK;
}

}  // extern "C"
