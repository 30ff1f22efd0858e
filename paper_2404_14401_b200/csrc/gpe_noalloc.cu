// gpe_noalloc.cu -- gpe_norm_theta_noalloc: the fused norm / cavity-overlap reduction (
// PAPER.md:116 renormalisation, Eq. 14 overlap) as ONE entry point that allocates nothing.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
// forbid it): no plan, no cudaMalloc / cudaFree / allocating library routine.  It is a variant of the prologue
// reduction k_reduce of gpe_api.cu (per-CTA partial sums in scratch memory, the last CTA of a member adds them in a
// fixed order), with that scratch in a file-scope static __device__ array instead of the plan's buffers:
//   g_noalloc_scratch: kSlots double2 partial sums + kMaxBatch counters = 65 792 bytes, held by every GPU that loads
//   the library until the process exits.
// Limits (GPE_EUNSUPPORTED beyond them): batch <= 64, 1 <= nx, ny <= 4096.
// The array is shared by every call and keeps the last call's contents: the counters are cleared on the caller's
// stream at the start of every call, the partial sums are all rewritten before they are read.  Two calls that overlap
// on the GPU (different streams, or concurrent host threads) RACE on it -- serialise them.
// In host code the array's name is only a stand-in: its device address is taken once per device with
// cudaGetSymbolAddress (that device current) and handed to the kernel as a pointer.
#include <cstdint>
#include <mutex>
#include <string>

#include "../../include/gpe.h"

namespace {

constexpr int kMaxBatch = 64;     // members per call
constexpr int kSlots = 4096;      // partial-sum slots shared by the members of a call
constexpr int kMaxN = 4096;       // largest nx, ny (the per-CTA cos table is ny doubles of shared memory)
constexpr int kThreads = 256;
constexpr int kMaxDevices = 64;

// [0, kSlots): per-CTA partial sums (sum |psi|^2, sum cos cos |psi|^2); the last kMaxBatch * 4 bytes: one counter per member
static __device__ __align__(256) double2 g_noalloc_scratch[kSlots + kMaxBatch * sizeof(unsigned int) / sizeof(double2)];

thread_local std::string g_error;
std::mutex g_mutex;
double2 *g_scratch_ptr[kMaxDevices] = {};   // device address of g_noalloc_scratch, per device ordinal

gpe_status fail(gpe_status s, const std::string &msg) {
    g_error = msg;
    return s;
}

__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// sum over the CTA (fixed order); the result is valid in thread 0
__device__ __forceinline__ void cta_sum2(double &a, double &b, double *red) {
    a = warp_sum_d(a);
    b = warp_sum_d(b);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) { red[w] = a; red[32 + w] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = 0.0; b = 0.0;
        for (int q = 0; q < kThreads / 32; ++q) { a += red[q]; b += red[32 + q]; }
    }
}

// grid = (cpm, batch).  psi: [batch][nx][ny] interleaved (re, im), T = float | double.
// out[b] = {sum |psi|^2 dx dy, sum cos(k x_i) cos(k y_j) |psi|^2 dx dy}, x_i = -Lx/2 + i Lx/nx (include/gpe.h).
template <typename T>
__global__ void __launch_bounds__(kThreads) k_norm_theta_noalloc(const T *__restrict__ psi, int nx, int ny, double Lx, double Ly,
                                                                 double k, double2 *scratch, double2 *out) {
    extern __shared__ double cy[];          // cos(k y_j)
    __shared__ double red[64];
    __shared__ int is_last;
    const int b = blockIdx.y, cpm = gridDim.x;
    double2 *part = scratch + (size_t)b * cpm;
    unsigned int *counter = reinterpret_cast<unsigned int *>(scratch + kSlots) + b;
    for (int j = threadIdx.x; j < ny; j += kThreads) cy[j] = cos(k * (-0.5 * Ly + (double)j * Ly / (double)ny));
    __syncthreads();
    const T *w = psi + 2 * (size_t)b * nx * ny;
    double sn = 0.0, st = 0.0;
    for (int i = blockIdx.x; i < nx; i += cpm) {
        const T *row = w + 2 * (size_t)i * ny;
        double rn = 0.0, rt = 0.0;
        for (int j = threadIdx.x; j < ny; j += kThreads) {
            const double re = (double)row[2 * j], im = (double)row[2 * j + 1];
            const double d = re * re + im * im;
            rn += d;
            rt += d * cy[j];
        }
        sn += rn;
        st += rt * cos(k * (-0.5 * Lx + (double)i * Lx / (double)nx));
    }
    cta_sum2(sn, st, red);
    if (threadIdx.x == 0) {
        part[blockIdx.x] = make_double2(sn, st);
        __threadfence();
        is_last = (atomicAdd(counter, 1u) == (unsigned int)(cpm - 1));
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double a = 0.0, c = 0.0;
    for (int q = threadIdx.x; q < cpm; q += kThreads) {
        const double2 p = __ldcg(part + q);
        a += p.x; c += p.y;
    }
    cta_sum2(a, c, red);
    if (threadIdx.x == 0) {
        const double dxdy = (Lx / (double)nx) * (Ly / (double)ny);
        out[b] = make_double2(a * dxdy, c * dxdy);
        *counter = 0u;
    }
}

// device address of the scratch array on the CURRENT device (taken once per device)
gpe_status scratch_address(double2 **ptr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(GPE_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e)); }
    if (dev < 0 || dev >= kMaxDevices) return fail(GPE_EUNSUPPORTED, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(GPE_ECUDA, std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(e));
        }
        g_scratch_ptr[dev] = static_cast<double2 *>(p);
    }
    *ptr = g_scratch_ptr[dev];
    return GPE_OK;
}

}  // namespace

extern "C" {

const char *gpe_noalloc_last_error(void) { return g_error.c_str(); }

gpe_status gpe_norm_theta_noalloc(const void *psi_dev, int nx, int ny, double Lx, double Ly, gpe_dtype dtype, int batch,
                                  double cavity_k, double *out_dev, void *cuda_stream) {
    if (!psi_dev || !out_dev) return fail(GPE_EINVAL, "psi_dev / out_dev is NULL");
    if (dtype != GPE_C64 && dtype != GPE_C128) return fail(GPE_EINVAL, "unknown dtype");
    if (((uintptr_t)psi_dev % (dtype == GPE_C64 ? 8 : 16)) != 0 || ((uintptr_t)out_dev % 16) != 0)
        return fail(GPE_EINVAL, "psi_dev must be aligned to one complex number, out_dev to 16 bytes");
    if (nx < 1 || ny < 1 || batch < 1 || !(Lx > 0) || !(Ly > 0) || !(Lx < 1e300) || !(Ly < 1e300) || !(cavity_k == cavity_k))
        return fail(GPE_EINVAL, "nx, ny, batch must be positive, Lx, Ly finite and > 0, cavity_k not NaN");
    if (batch > kMaxBatch || nx > kMaxN || ny > kMaxN)
        return fail(GPE_EUNSUPPORTED, "gpe_norm_theta_noalloc works in a fixed 65 792-byte device array: batch <= 64 and nx, ny <= 4096 "
                                      "(got batch " + std::to_string(batch) + ", " + std::to_string(nx) + " x " + std::to_string(ny) + ")");
    double2 *scratch = nullptr;
    gpe_status s = scratch_address(&scratch);
    if (s != GPE_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the counters must start at zero whatever an earlier (possibly failed) call left behind
    cudaError_t e = cudaMemsetAsync(scratch + kSlots, 0, kMaxBatch * sizeof(unsigned int), st);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(GPE_ECUDA, std::string("cudaMemsetAsync: ") + cudaGetErrorString(e)); }
    int cpm = kSlots / batch;            // >= 64 CTAs per member
    if (cpm > nx) cpm = nx;
    const dim3 grid((unsigned)cpm, (unsigned)batch);
    const size_t smem = sizeof(double) * (size_t)ny;   // <= 32 KB
    if (dtype == GPE_C64)
        k_norm_theta_noalloc<float><<<grid, kThreads, smem, st>>>((const float *)psi_dev, nx, ny, Lx, Ly, cavity_k, scratch, (double2 *)out_dev);
    else
        k_norm_theta_noalloc<double><<<grid, kThreads, smem, st>>>((const double *)psi_dev, nx, ny, Lx, Ly, cavity_k, scratch, (double2 *)out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GPE_ECUDA, std::string("k_norm_theta_noalloc launch: ") + cudaGetErrorString(e));
    return GPE_OK;
}

}  // extern "C"
