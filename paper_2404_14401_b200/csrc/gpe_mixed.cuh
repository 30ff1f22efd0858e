// gpe_mixed.cuh -- the three fused passes for grid sizes that are NOT powers of two
// ("we do not record qualitative deviations from the observed trend for
// non-optimal grid sizes"): nx, ny even with no prime factor above 5, 64 <= n <= 2048.
//
// Transform: mixed-radix Stockham autosort in shared memory (radices 8, 5, 4, 3, 2 chosen on the host), two
// ping-pong buffers, natural order in and out, so the three passes keep psi in its natural layout:
//   stage with radix r, p = product of the radices before it, t = N / r butterflies:
//     butterfly i:  k = i mod p,  j = (i - k) r + k,
//     u[q] = x[i + q t] * exp(SIGN 2 pi i k q / (p r)),  U = DFT_r(u),  y[j + q p] = U[q]     (q < r)
// Every thread loops over butterflies; W independent transforms (the columns of a tile) are interleaved
// element by element.  The potential factor, kinetic factor, sums and the last-block finalisation are those
// of gpe_kernels.cuh, one point at a time (PAPER.md:62-76 Eqs. 2-4, :116, :183-188 Eqs. 14-15); the two
// potential half-steps of consecutive real-time steps are NOT merged here.  This family is for coverage of
// the sizes, not for the roofline: a power of two is always the faster choice (as the paper says of cuFFT).
#pragma once
#include "gpe_kernels.cuh"

namespace gpe {

struct MixPlan {
    int nr;          // number of stages
    int radix[12];   // their radices, product = N
};

template <typename T> __device__ __forceinline__ cx<T> mx_add(cx<T> a, cx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <typename T> __device__ __forceinline__ cx<T> mx_sub(cx<T> a, cx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
template <typename T> __device__ __forceinline__ cx<T> mx_mul(cx<T> a, cx<T> w) { return mk<T>(fma(a.x, w.x, -(a.y * w.y)), fma(a.x, w.y, a.y * w.x)); }
// a * (SG i): a quarter turn in the direction of the transform
template <int SG, typename T> __device__ __forceinline__ cx<T> mx_rot(cx<T> a) { return SG > 0 ? mk<T>(-a.y, a.x) : mk<T>(a.y, -a.x); }

// U[q] = sum_t u[t] exp(SG 2 pi i t q / R), in place
template <int R, int SG, typename T> __device__ __forceinline__ void mx_dft(cx<T> *u) {
    using C = cx<T>;
    if constexpr (R == 2) {
        const C a = u[0];
        u[0] = mx_add<T>(a, u[1]); u[1] = mx_sub<T>(a, u[1]);
    } else if constexpr (R == 3) {
        const T h = T(0.86602540378443864676);   // sin(pi/3)
        const C t1 = mx_add<T>(u[1], u[2]);
        const C m = mk<T>(u[0].x - T(0.5) * t1.x, u[0].y - T(0.5) * t1.y);
        const C d = mx_sub<T>(u[1], u[2]);
        const C s = mx_rot<SG, T>(mk<T>(h * d.x, h * d.y));     // SG i sin(2 pi/3) (u1 - u2)
        u[0] = mx_add<T>(u[0], t1); u[1] = mx_add<T>(m, s); u[2] = mx_sub<T>(m, s);
    } else if constexpr (R == 4) {
        const C a = mx_add<T>(u[0], u[2]), b = mx_sub<T>(u[0], u[2]);
        const C c = mx_add<T>(u[1], u[3]), d = mx_rot<SG, T>(mx_sub<T>(u[1], u[3]));
        u[0] = mx_add<T>(a, c); u[2] = mx_sub<T>(a, c); u[1] = mx_add<T>(b, d); u[3] = mx_sub<T>(b, d);
    } else if constexpr (R == 5) {
        const T c1 = T(0.30901699437494742410), c2 = T(-0.80901699437494742410);   // cos(2 pi/5), cos(4 pi/5)
        const T s1 = T(0.95105651629515357212), s2 = T(0.58778525229247312917);    // sin(2 pi/5), sin(4 pi/5)
        const C a1 = mx_add<T>(u[1], u[4]), a2 = mx_add<T>(u[2], u[3]);
        const C b1 = mx_sub<T>(u[1], u[4]), b2 = mx_sub<T>(u[2], u[3]);
        const C r1 = mk<T>(u[0].x + c1 * a1.x + c2 * a2.x, u[0].y + c1 * a1.y + c2 * a2.y);
        const C r2 = mk<T>(u[0].x + c2 * a1.x + c1 * a2.x, u[0].y + c2 * a1.y + c1 * a2.y);
        const C i1 = mx_rot<SG, T>(mk<T>(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y));
        const C i2 = mx_rot<SG, T>(mk<T>(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y));
        u[0] = mk<T>(u[0].x + a1.x + a2.x, u[0].y + a1.y + a2.y);
        u[1] = mx_add<T>(r1, i1); u[4] = mx_sub<T>(r1, i1);
        u[2] = mx_add<T>(r2, i2); u[3] = mx_sub<T>(r2, i2);
    } else {   // R == 8: two DFT_4 of the even and odd inputs, then exp(SG 2 pi i q / 8)
        static_assert(R == 8, "radices 2, 3, 4, 5, 8");
        const T h = T(0.70710678118654752440);
        C e[4] = {u[0], u[2], u[4], u[6]}, o[4] = {u[1], u[3], u[5], u[7]};
        mx_dft<4, SG, T>(e); mx_dft<4, SG, T>(o);
        const C r1 = mx_rot<SG, T>(o[1]), r3 = mx_rot<SG, T>(o[3]);
        o[1] = mk<T>(h * (o[1].x + r1.x), h * (o[1].y + r1.y));      // o1 (1 + SG i) / sqrt 2
        o[2] = mx_rot<SG, T>(o[2]);                                  // o2 (SG i)
        o[3] = mk<T>(h * (r3.x - o[3].x), h * (r3.y - o[3].y));      // o3 (-1 + SG i) / sqrt 2
#pragma unroll
        for (int q = 0; q < 4; ++q) { u[q] = mx_add<T>(e[q], o[q]); u[q + 4] = mx_sub<T>(e[q], o[q]); }
    }
}

// one stage over W interleaved transforms of length N: x -> y
template <int R, int SG, typename T>
__device__ __forceinline__ void mx_stage(const cx<T> *x, cx<T> *y, int N, int W, int p, const cx<T> *__restrict__ tw) {
    using C = cx<T>;
    const int t = N / R, step = N / (p * R);
    for (int w = threadIdx.x; w < t * W; w += blockDim.x) {
        const int i = w / W, c = w - i * W;
        const int k = i % p, j = (i - k) * R + k;
        C u[R];
#pragma unroll
        for (int q = 0; q < R; ++q) u[q] = x[(size_t)(i + q * t) * W + c];
        if (k != 0) {
#pragma unroll
            for (int q = 1; q < R; ++q) {
                C wq = tw[k * q * step];                  // exp(-2 pi i k q / (p R)); k q step < N
                if (SG > 0) wq.y = -wq.y;
                u[q] = mx_mul<T>(u[q], wq);
            }
        }
        mx_dft<R, SG, T>(u);
#pragma unroll
        for (int q = 0; q < R; ++q) y[(size_t)(j + q * p) * W + c] = u[q];
    }
}

// the whole transform; on return `x` points at the buffer that holds the result (natural order), `y` at the other.
// All threads of the CTA must call it; it ends with a barrier.
template <int SG, typename T>
__device__ __forceinline__ void mx_fft(cx<T> *&x, cx<T> *&y, int N, int W, const MixPlan &pl, const cx<T> *__restrict__ tw) {
    int p = 1;
    __syncthreads();
    for (int s = 0; s < pl.nr; ++s) {
        const int r = pl.radix[s];
        switch (r) {
        case 2: mx_stage<2, SG, T>(x, y, N, W, p, tw); break;
        case 3: mx_stage<3, SG, T>(x, y, N, W, p, tw); break;
        case 4: mx_stage<4, SG, T>(x, y, N, W, p, tw); break;
        case 5: mx_stage<5, SG, T>(x, y, N, W, p, tw); break;
        default: mx_stage<8, SG, T>(x, y, N, W, p, tw); break;
        }
        __syncthreads();
        cx<T> *sw = x; x = y; y = sw;
        p *= r;
    }
}

// ---------------------------------------------------------------- the point-wise factor (rows a1 / a5)
// psi <- psi * exp(-s (V + g|psi|^2) dt/2), V assembled as in potential_step16 (gpe_kernels.cuh)
template <typename T, bool IMAG>
__device__ __forceinline__ cx<T> mx_potential(cx<T> z, const StepArgs<T, cx<T>> &a, int b, int i, int n, T scale, T A, T Cc, T Dc) {
    const int flags = a.flags;
    T V = T(0);
    if (flags & F_HAS_SEP) V += a.vx[i] + a.vy[n];
    if (flags & F_LAT_X) V += A * a.latx[i];
    if (flags & F_LAT_Y) V += A * a.laty[n];
    if (flags & F_CAVITY) V += Cc * a.cavx[i] * a.cavy[n];
    if (flags & F_CAV_FULL) V += Dc * a.cavx[i] * a.cavx[i];
    if (flags & F_HAS_V2D) V += a.v2d[((flags & F_V2D_BATCHED) ? (size_t)b * a.nx * a.ny : 0) + (size_t)i * a.ny + n];
    if constexpr (IMAG) { z.x *= scale; z.y *= scale; }
    const T g = (flags & F_HAS_G) ? a.g[b] : T(0);
    const T w = (V + g * (z.x * z.x + z.y * z.y)) * a.half_dt;
    if constexpr (IMAG) {
        const T e = exp_t(-w);
        z.x *= e; z.y *= e;
    } else {
        T sn, cm1;
        sincosm1_t(-w, &sn, &cm1);
        const T ox = fma(z.x, cm1, fma(-z.y, sn, z.x)), oy = fma(z.x, sn, fma(z.y, cm1, z.y));
        z.x = ox; z.y = oy;
    }
    return z;
}

// ---------------------------------------------------------------- pass A: one row per CTA
template <typename T, bool IMAG>
__global__ void __launch_bounds__(256) k_mix_row_fwd(const StepArgs<T, cx<T>> a, const MixPlan ply) {
    using C = cx<T>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int ny = a.ny;
    C *x = reinterpret_cast<C *>(smem_raw), *y = x + ny;
    const long row = blockIdx.x;
    const int b = (int)(row / a.nx), i = (int)(row % a.nx);
    const C *src = a.src + row * ny;
    C *dst = a.dst + row * ny;
    const bool pot = !(a.flags & F_NO_POT);
    T scale = T(1), A = T(0), Cc = T(0), Dc = T(0);
    if (pot) {
        const MemberState &ms = a.fin.st[b];
        scale = (T)ms.scale; A = (T)ms.A; Cc = (T)ms.C; Dc = (T)ms.D;
    }
    for (int n = threadIdx.x; n < ny; n += blockDim.x) {
        C z = __ldcg(src + n);
        if (pot) z = mx_potential<T, IMAG>(z, a, b, i, n, scale, A, Cc, Dc);
        x[n] = z;
    }
    mx_fft<-1, T>(x, y, ny, 1, ply, a.tw_y);
    for (int n = threadIdx.x; n < ny; n += blockDim.x) dst[n] = x[n];
}

// ---------------------------------------------------------------- pass B: W columns per CTA
// MODE 0: forward, kinetic factor, inverse.  MODE 1: forward only (observables).
template <typename T, bool IMAG, int MODE>
__global__ void __launch_bounds__(256) k_mix_col(const StepArgs<T, cx<T>> a, const MixPlan plx, int W) {
    using C = cx<T>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nx = a.nx, ny = a.ny;
    C *x = reinterpret_cast<C *>(smem_raw), *y = x + (size_t)nx * W;
    const int b = blockIdx.y, col0 = blockIdx.x * W;
    const C *src = a.src + (size_t)b * nx * ny + col0;
    C *dst = a.dst + (size_t)b * nx * ny + col0;
    if (MODE == 0 && blockIdx.x == 0 && threadIdx.x == 0 && a.fin.prepared) prepare_member(a.fin, b);
    for (int q = threadIdx.x; q < nx * W; q += blockDim.x) {
        const int n = q / W, c = q - n * W;
        x[q] = __ldcg(src + (size_t)n * ny + c);
    }
    mx_fft<-1, T>(x, y, nx, W, plx, a.tw_x);
    if constexpr (MODE == 0) {
        for (int q = threadIdx.x; q < nx * W; q += blockDim.x) {
            const int n = q / W, c = q - n * W;
            C z = x[q];
            if constexpr (IMAG) {
                const T fk = a.kin_xr[n] * a.kin_yr[col0 + c];
                z.x *= fk; z.y *= fk;
            } else {
                // (1 + a)(1 + b) / P with the "minus one" tables of gpe_api.cu: a' = a / P from the x table
                const C ap = a.kin_xc[n], bq = a.kin_yc[col0 + c];
                const T invp = a.inv_p, cb = T(1) + bq.x;
                const T gx = fma(ap.x, cb, fma(-ap.y, bq.y, bq.x * invp));
                const T gy = fma(ap.x, bq.y, fma(ap.y, cb, bq.y * invp));
                const T ox = fma(z.x, gx, fma(-z.y, gy, z.x * invp));
                const T oy = fma(z.x, gy, fma(z.y, gx, z.y * invp));
                z.x = ox; z.y = oy;
            }
            x[q] = z;
        }
        mx_fft<+1, T>(x, y, nx, W, plx, a.tw_x);
    }
    for (int q = threadIdx.x; q < nx * W; q += blockDim.x) {
        const int n = q / W, c = q - n * W;
        dst[(size_t)n * ny + c] = x[q];
    }
}

// ---------------------------------------------------------------- pass C: one row per CTA
template <typename T, bool IMAG>
__global__ void __launch_bounds__(256) k_mix_row_inv(const StepArgs<T, cx<T>> a, const MixPlan ply) {
    using C = cx<T>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[96];
    const int ny = a.ny;
    C *x = reinterpret_cast<C *>(smem_raw), *y = x + ny;
    const long row = blockIdx.x;
    const int b = (int)(row / a.nx), i = (int)(row % a.nx);
    const C *src = a.src + row * ny;
    C *dst = a.dst + row * ny;
    for (int n = threadIdx.x; n < ny; n += blockDim.x) x[n] = __ldcg(src + n);
    mx_fft<+1, T>(x, y, ny, 1, ply, a.tw_y);
    const MemberState &ms = a.fin.st[b];
    const T A = (T)ms.A, Cc = (T)ms.C, Dc = (T)ms.D;
    double sn = 0.0, st = 0.0;
    for (int n = threadIdx.x; n < ny; n += blockDim.x) {
        const C z = mx_potential<T, IMAG>(x[n], a, b, i, n, T(1), A, Cc, Dc);
        const double d = (double)z.x * (double)z.x + (double)z.y * (double)z.y;
        sn += d;
        if (a.flags & F_CAVITY) st += d * (double)a.cavy[n];
        dst[n] = z;
    }
    const double cxi = (a.flags & F_CAVITY) ? (double)a.cavx[i] : 0.0;
    block_reduce_and_finalize(a.fin, b, i, sn, st * cxi, (a.flags & F_CAV_FULL) ? sn * cxi * cxi : 0.0, red);
}

// ---------------------------------------------------------------- launchers
template <typename T> struct LaunchMix {
    using A = StepArgs<T, cx<T>>;
    using C = cx<T>;
    static int threads_for(int work) { return work >= 256 ? 256 : work >= 128 ? 128 : 64; }
    static int col_width(const A &a) { return (sizeof(T) == 4 && a.ny % 4 == 0) ? 4 : 2; }
    template <typename K> static cudaError_t optin(K kern, size_t smem) {
        if (smem <= 48 * 1024) return cudaSuccess;
        return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    }
    static cudaError_t row_fwd(const A &a, const MixPlan &ply, bool imag, cudaStream_t s) {
        const size_t smem = 2 * sizeof(C) * (size_t)a.ny;
        const unsigned grid = (unsigned)((long)a.batch * a.nx), bd = (unsigned)threads_for(a.ny / 4);
        if (imag) k_mix_row_fwd<T, true><<<grid, bd, smem, s>>>(a, ply);
        else k_mix_row_fwd<T, false><<<grid, bd, smem, s>>>(a, ply);
        return cudaGetLastError();
    }
    static cudaError_t row_inv(const A &a, const MixPlan &ply, bool imag, cudaStream_t s) {
        const size_t smem = 2 * sizeof(C) * (size_t)a.ny;
        const unsigned grid = (unsigned)((long)a.batch * a.nx), bd = (unsigned)threads_for(a.ny / 4);
        if (imag) k_mix_row_inv<T, true><<<grid, bd, smem, s>>>(a, ply);
        else k_mix_row_inv<T, false><<<grid, bd, smem, s>>>(a, ply);
        return cudaGetLastError();
    }
    static cudaError_t col(const A &a, const MixPlan &plx, bool imag, int mode, cudaStream_t s) {
        const int W = col_width(a);
        const size_t smem = 2 * sizeof(C) * (size_t)a.nx * W;
        const dim3 grid((unsigned)(a.ny / W), (unsigned)a.batch);
        const unsigned bd = (unsigned)threads_for(a.nx * W / 4);
        cudaError_t e;
        if (mode == 1) {
            if ((e = optin(k_mix_col<T, false, 1>, smem)) != cudaSuccess) return e;
            k_mix_col<T, false, 1><<<grid, bd, smem, s>>>(a, plx, W);
        } else if (imag) {
            if ((e = optin(k_mix_col<T, true, 0>, smem)) != cudaSuccess) return e;
            k_mix_col<T, true, 0><<<grid, bd, smem, s>>>(a, plx, W);
        } else {
            if ((e = optin(k_mix_col<T, false, 0>, smem)) != cudaSuccess) return e;
            k_mix_col<T, false, 0><<<grid, bd, smem, s>>>(a, plx, W);
        }
        return cudaGetLastError();
    }
};

}  // namespace gpe
