// gpe_kernels.cuh -- the three fused passes of one split-step:
//   pass A (rows):    load psi [x lazy scale] -> potential half-step a1 -> FFT along y -> store
//   pass B (columns): load -> FFT along x -> kinetic factor a3 -> inverse FFT along x -> store
//   pass C (rows):    load -> inverse FFT along y -> potential half-step a5 -> partial sums of
//                     |psi|^2 and cos cos |psi|^2 (a6) -> store; the last block reduces the
//                     partials in a fixed order and writes the scalars of the next step
//                     (a0: A_{n+1}, C_{n+1}; a7: scale; a8: record) -- no host round trip.
// PAPER.md:62-76 (Eqs. 2-4), :116 (renormalisation), :183-186 (Eq. 14).
#pragma once
#include "gpe_fft.cuh"
#include "gpe_types.h"

namespace gpe {

// ---------------------------------------------------------------- launch geometry
template <int N> struct RowGeom {
    static constexpr int TPF = N / 16;
    static constexpr int RPC = (256 / TPF) < 1 ? 1 : (256 / TPF);  // rows per CTA
    static constexpr int THREADS = RPC * TPF;                      // 256
};
template <typename T, int N> struct ColGeom {
    static constexpr int TPF = N / 16;
    static constexpr int WMIN = sizeof(T) == 4 ? 4 : 2;            // >= 32-byte row segments
    static constexpr int W0 = 256 / TPF;
    static constexpr int W = W0 < WMIN ? WMIN : W0;                // columns per CTA
    static constexpr int THREADS = W * TPF;
};

// ---------------------------------------------------------------- scalar update (rows a0, a7, a8)
__device__ inline double schedule_at(const FinalizeParams &f, int b, double n) {
    if (f.sched_len <= 0) return 0.0;
    const double *amp = f.sched_amp + (f.sched_batched ? (size_t)b * f.sched_len : 0);
    const double *st = f.sched_step;
    int L = f.sched_len;
    if (n < st[0]) return amp[0];
    int i = 0;
    for (int q = 0; q < L; ++q)
        if (st[q] <= n) i = q;
    if (i == L - 1) return amp[L - 1];
    double t = (n - st[i]) / (st[i + 1] - st[i]);
    return amp[i] + t * (amp[i + 1] - amp[i]);
}

// Called by one thread of the last block of member b with the raw sums over the stored psi.
__device__ inline void finalize_member(const FinalizeParams &f, int b, double sum_n, double sum_t) {
    MemberState &s = f.st[b];
    double norm = sum_n * f.dxdy, theta = sum_t * f.dxdy;
    if (!(norm == norm) || norm > 1e300 || norm < 0.0 || (f.normalise && !(norm > 0.0))) *f.nonfinite = 1;
    long long n1;
    if (f.advance) n1 = s.step + 1; else n1 = f.step0;
    double scale = 1.0;
    if (f.normalise) {
        scale = 1.0 / sqrt(norm);
        theta = theta / norm;
        norm = 1.0;
    }
    double A = schedule_at(f, b, (double)n1);
    double eta = 0.0, re_a = 0.0, im_a = 0.0, C = 0.0;
    if (f.cavity_on) {
        eta = f.eta_mode == 0 ? f.eta_or_u[b] : sqrt(fabs(A) * f.eta_or_u[b]);
        double D = f.delta[b], K = f.kappa[b], num = f.n_atoms[b] * eta * theta;
        double den = D * D + K * K;               // num / (D + iK) = num (D - iK) / (D^2 + K^2)
        re_a = num * D / den;
        im_a = -num * K / den;
        C = 2.0 * eta * re_a;
    }
    s.scale = scale; s.A = A; s.C = C; s.norm = norm; s.theta = theta;
    s.re_alpha = re_a; s.im_alpha = im_a; s.step = n1;
    if (f.advance && f.records && f.record_every > 0 && (n1 % f.record_every) == 0) {
        long long idx = n1 / f.record_every - f.rec_first - 1;
        double *r = f.records + ((size_t)idx * f.batch + b) * 6;
        r[0] = (double)n1; r[1] = norm; r[2] = theta; r[3] = re_a; r[4] = im_a; r[5] = A;
    }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Block-level sum of (sn, st), one partial per CTA, last CTA of the member finalises.
// `red` is shared scratch of at least 2*32 doubles.  All threads of the CTA must call this.
__device__ inline void block_reduce_and_finalize(const FinalizeParams &f, int b, int cta_in_member,
                                                 double sn, double st, double *red) {
    sn = warp_sum(sn);
    st = warp_sum(st);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) { red[w] = sn; red[32 + w] = st; }
    __syncthreads();
    __shared__ int is_last;
    if (threadIdx.x == 0) {
        double a = 0.0, c = 0.0;
        for (int i = 0; i < nw; ++i) { a += red[i]; c += red[32 + i]; }
        f.partials[(size_t)b * f.cpm + cta_in_member] = make_double2(a, c);
        __threadfence();
        unsigned int old = atomicAdd(&f.counters[b], 1u);
        is_last = (old == (unsigned int)(f.cpm - 1));
    }
    __syncthreads();
    if (is_last && w == 0) {
        __threadfence();
        const volatile double2 *p = f.partials + (size_t)b * f.cpm;
        double a = 0.0, c = 0.0;
        for (int i = lane; i < f.cpm; i += 32) { a += p[i].x; c += p[i].y; }
        a = warp_sum(a);
        c = warp_sum(c);
        if (lane == 0) {
            finalize_member(f, b, a, c);
            f.counters[b] = 0u;
        }
    }
}

// ---------------------------------------------------------------- potential factor (rows a1, a5)
// psi <- psi * exp(-s (V + g|psi|^2) dt/2); returns |psi|^2 after the multiply.
__device__ __forceinline__ float exp_t(float x) { return expf(x); }
__device__ __forceinline__ double exp_t(double x) { return exp(x); }
__device__ __forceinline__ void sincos_t(float x, float *s, float *c) { sincosf(x, s, c); }
__device__ __forceinline__ void sincos_t(double x, double *s, double *c) { sincos(x, s, c); }

// (cos w - 1, sin w).  Real-time phase factors are applied as z + z*(cos w - 1 + i sin w):
// for the small angles of a split-step (w ~ 1e-4..1e-2) cos w sits a few ulps below 1, and
// RN(z * cos w) is then biased low by ~2e-8 per multiply (the product always lands at the same
// fractional position between two floats) -- measured as a norm drift of -2e-7 per step in
// complex64.  The "minus one" form has no such bias and is also cheaper than sincosf.
__device__ __forceinline__ void sincosm1_t(float w, float *s, float *cm1) {
    if (fabsf(w) <= 0.5f) {
        const float w2 = w * w;
        float ps = fmaf(w2, 2.7557319e-6f, -1.9841270e-4f);
        ps = fmaf(w2, ps, 8.3333333e-3f);
        ps = fmaf(w2, ps, -1.6666667e-1f);
        *s = fmaf(w * w2, ps, w);
        float pc = fmaf(w2, 2.4801587e-5f, -1.3888889e-3f);
        pc = fmaf(w2, pc, 4.1666667e-2f);
        pc = fmaf(w2, pc, -0.5f);
        *cm1 = w2 * pc;
    } else {
        float sh, ch;
        sincosf(0.5f * w, &sh, &ch);
        *s = 2.0f * sh * ch;
        *cm1 = -2.0f * sh * sh;
    }
}
__device__ __forceinline__ void sincosm1_t(double w, double *s, double *cm1) {
    double sh, ch;
    sincos(0.5 * w, &sh, &ch);
    *s = 2.0 * sh * ch;
    *cm1 = -2.0 * sh * sh;
}

template <typename T, bool IMAG>
__device__ __forceinline__ T potential_factor(cx<T> &z, T V, T g, T half_dt) {
    T d = z.x * z.x + z.y * z.y;
    T w = (V + g * d) * half_dt;
    if constexpr (IMAG) {
        T e = exp_t(-w);
        z.x *= e; z.y *= e;
        return d * e * e;
    } else {
        T s, cm1;
        sincosm1_t(-w, &s, &cm1);
        const T tx = fma(z.x, cm1, -(z.y * s)), ty = fma(z.x, s, z.y * cm1);
        z.x += tx; z.y += ty;
        return d;
    }
}

template <typename T, typename C> struct RowPot {
    T vrow, crow, A, g, half_dt;
    const T *v2d_row, *vy, *laty, *cavy;
    int flags;
    __device__ __forceinline__ void init(const StepArgs<T, C> &a, int b, int i, T A_, T C_) {
        flags = a.flags;
        A = A_;
        vrow = T(0);
        if (flags & F_HAS_SEP) vrow += a.vx[i];
        if (flags & F_LAT_X) vrow += A_ * a.latx[i];
        crow = (flags & F_CAVITY) ? C_ * a.cavx[i] : T(0);
        g = (flags & F_HAS_G) ? a.g[b] : T(0);
        half_dt = a.half_dt;
        v2d_row = nullptr;
        if (flags & F_HAS_V2D)
            v2d_row = a.v2d + ((flags & F_V2D_BATCHED) ? (size_t)b * a.nx * a.ny : 0) + (size_t)i * a.ny;
        vy = a.vy; laty = a.laty; cavy = a.cavy;
    }
    __device__ __forceinline__ T at(int y) const {
        T V = vrow;
        if (flags & F_HAS_SEP) V += vy[y];
        if (flags & F_LAT_Y) V += A * laty[y];
        if (flags & F_CAVITY) V += crow * cavy[y];
        if (flags & F_HAS_V2D) V += v2d_row[y];
        return V;
    }
};

// ---------------------------------------------------------------- pass A
template <typename T, int NY, bool IMAG>
__global__ void __launch_bounds__(RowGeom<NY>::THREADS) k_row_fwd(const StepArgs<T, cx<T>> a) {
    using C = cx<T>;
    using F = Fft1D<NY, 1, T>;
    using G = RowGeom<NY>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    const long row = (long)blockIdx.x * G::RPC + r;
    const int b = (int)(row / a.nx), i = (int)(row % a.nx);
    C *sm = smem + r * F::SLOTS;
    const C *src = a.src + row * NY;
    C *dst = a.dst + row * NY;
    C v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = src[j + F::M1 * k];
    if (!(a.flags & F_NO_POT)) {
        const MemberState &ms = a.fin.st[b];
        const T scale = (T)ms.scale;
        RowPot<T, C> P;
        P.init(a, b, i, (T)ms.A, (T)ms.C);
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            v[k].x *= scale; v[k].y *= scale;
            potential_factor<T, IMAG>(v[k], P.at(j + F::M1 * k), P.g, P.half_dt);
        }
    }
    F::fwd(v, sm, j, a.tw_y);
#pragma unroll
    for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
        for (int rr = 0; rr < F::RL; ++rr) dst[F::nat(j, ii, rr)] = v[ii * F::RL + rr];
}

// ---------------------------------------------------------------- pass B
// MODE 0: forward, kinetic factor, inverse (the step).  MODE 1: forward only, natural order
// (observables).
template <typename T, int NX, bool IMAG, int MODE>
__global__ void __launch_bounds__(ColGeom<T, NX>::THREADS) k_col(const StepArgs<T, cx<T>> a) {
    using C = cx<T>;
    using G = ColGeom<T, NX>;
    using F = Fft1D<NX, G::W, T>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    const int c = threadIdx.x % G::W, j = threadIdx.x / G::W;
    const int col = blockIdx.x * G::W + c;
    const int b = blockIdx.y;
    const size_t ny = a.ny;
    const C *src = a.src + (size_t)b * NX * ny + col;
    C *dst = a.dst + (size_t)b * NX * ny + col;
    C *sm = smem + c;
    C v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = src[(size_t)(j + F::M1 * k) * ny];
    F::fwd(v, sm, j, a.tw_x);
    if constexpr (MODE == 1) {
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) dst[(size_t)F::nat(j, ii, rr) * ny] = v[ii * F::RL + rr];
        return;
    } else {
        if constexpr (IMAG) {
            const T ey = a.kin_yr[col];
#pragma unroll
            for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
                for (int rr = 0; rr < F::RL; ++rr) {
                    T f = a.kin_xr[F::nat(j, ii, rr)] * ey;
                    v[ii * F::RL + rr].x *= f;
                    v[ii * F::RL + rr].y *= f;
                }
        } else {
            // kinetic factor (1+a)(1+b)/P with a, b = exp(-i k^2 dt/2) - 1 of the two axes, applied
            // as v/P + v*g, g = a' + b' + a'b (a' = a/P from the x table, b' = b/P): see
            // sincosm1_t for why the "minus one" form is used.
            const C bq = a.kin_yc[col];
            const T invp = a.inv_p, cb = T(1) + bq.x;
            const C bp = mk<T>(bq.x * invp, bq.y * invp);
#pragma unroll
            for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
                for (int rr = 0; rr < F::RL; ++rr) {
                    const C ap = a.kin_xc[F::nat(j, ii, rr)];
                    const T gx = fma(ap.x, cb, fma(-ap.y, bq.y, bp.x));
                    const T gy = fma(ap.x, bq.y, fma(ap.y, cb, bp.y));
                    C &z = v[ii * F::RL + rr];
                    const T ox = fma(z.x, gx, fma(-z.y, gy, z.x * invp));
                    const T oy = fma(z.x, gy, fma(z.y, gx, z.y * invp));
                    z.x = ox; z.y = oy;
                }
        }
        F::inv(v, sm, j, a.tw_x);
#pragma unroll
        for (int k = 0; k < 16; ++k) dst[(size_t)(j + F::M1 * k) * ny] = v[k];
    }
}

// ---------------------------------------------------------------- pass C
template <typename T, int NY, bool IMAG>
__global__ void __launch_bounds__(RowGeom<NY>::THREADS) k_row_inv(const StepArgs<T, cx<T>> a) {
    using C = cx<T>;
    using F = Fft1D<NY, 1, T>;
    using G = RowGeom<NY>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    __shared__ double red[64];
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    const long row = (long)blockIdx.x * G::RPC + r;
    const int b = (int)(row / a.nx), i = (int)(row % a.nx);
    C *sm = smem + r * F::SLOTS;
    const C *src = a.src + row * NY;
    C *dst = a.dst + row * NY;
    C v[16];
#pragma unroll
    for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
        for (int rr = 0; rr < F::RL; ++rr) v[ii * F::RL + rr] = src[F::nat(j, ii, rr)];
    F::inv(v, sm, j, a.tw_y);
    const MemberState &ms = a.fin.st[b];
    RowPot<T, C> P;
    P.init(a, b, i, (T)ms.A, (T)ms.C);
    T sn = T(0), st = T(0);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const int y = j + F::M1 * k;
        T d = potential_factor<T, IMAG>(v[k], P.at(y), P.g, P.half_dt);
        sn += d;
        if (a.flags & F_CAVITY) st += d * a.cavy[y];
        dst[y] = v[k];
    }
    double dn = (double)sn, dt_ = (a.flags & F_CAVITY) ? (double)st * (double)a.cavx[i] : 0.0;
    // all rows of a CTA belong to one member (nx is a multiple of RPC)
    const int cta_in_member = (int)(blockIdx.x % (unsigned)(a.nx / G::RPC));
    block_reduce_and_finalize(a.fin, b, cta_in_member, dn, dt_, red);
}

// ---------------------------------------------------------------- launchers (one per T, N)
template <typename T, int N> struct Launch {
    using C = cx<T>;
    using A = StepArgs<T, C>;
    static size_t row_smem() { return sizeof(C) * RowGeom<N>::RPC * Fft1D<N, 1, T>::SLOTS; }
    static size_t col_smem() { return sizeof(C) * ColGeom<T, N>::W * Fft1D<N, 1, T>::SLOTS; }

    template <typename K> static cudaError_t prep(K kern, size_t smem) {
        if (smem > 48 * 1024)
            return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        return cudaSuccess;
    }
    // ny == N
    static cudaError_t row_fwd(const A &a, bool imag, cudaStream_t s) {
        dim3 grid((unsigned)((long)a.batch * a.nx / RowGeom<N>::RPC)), block(RowGeom<N>::THREADS);
        cudaError_t e;
        if (imag) {
            if ((e = prep(k_row_fwd<T, N, true>, row_smem())) != cudaSuccess) return e;
            k_row_fwd<T, N, true><<<grid, block, row_smem(), s>>>(a);
        } else {
            if ((e = prep(k_row_fwd<T, N, false>, row_smem())) != cudaSuccess) return e;
            k_row_fwd<T, N, false><<<grid, block, row_smem(), s>>>(a);
        }
        return cudaGetLastError();
    }
    static cudaError_t row_inv(const A &a, bool imag, cudaStream_t s) {
        dim3 grid((unsigned)((long)a.batch * a.nx / RowGeom<N>::RPC)), block(RowGeom<N>::THREADS);
        cudaError_t e;
        if (imag) {
            if ((e = prep(k_row_inv<T, N, true>, row_smem())) != cudaSuccess) return e;
            k_row_inv<T, N, true><<<grid, block, row_smem(), s>>>(a);
        } else {
            if ((e = prep(k_row_inv<T, N, false>, row_smem())) != cudaSuccess) return e;
            k_row_inv<T, N, false><<<grid, block, row_smem(), s>>>(a);
        }
        return cudaGetLastError();
    }
    // nx == N
    static cudaError_t col(const A &a, bool imag, int mode, cudaStream_t s) {
        dim3 grid((unsigned)(a.ny / ColGeom<T, N>::W), (unsigned)a.batch), block(ColGeom<T, N>::THREADS);
        cudaError_t e;
        if (mode == 1) {
            if ((e = prep(k_col<T, N, false, 1>, col_smem())) != cudaSuccess) return e;
            k_col<T, N, false, 1><<<grid, block, col_smem(), s>>>(a);
        } else if (imag) {
            if ((e = prep(k_col<T, N, true, 0>, col_smem())) != cudaSuccess) return e;
            k_col<T, N, true, 0><<<grid, block, col_smem(), s>>>(a);
        } else {
            if ((e = prep(k_col<T, N, false, 0>, col_smem())) != cudaSuccess) return e;
            k_col<T, N, false, 0><<<grid, block, col_smem(), s>>>(a);
        }
        return cudaGetLastError();
    }
    static int rows_per_cta() { return RowGeom<N>::RPC; }
};

}  // namespace gpe
