// gpe_fft.cuh -- register butterflies and the in-place shared-memory 1-D FFT used by every
// pass of the split-step (forward/inverse FFT of PAPER.md:73-76, Eq. 4).
//
// Formulation: N = 16 * R2 * R3 decimation-in-frequency Cooley-Tukey, done
// in place in shared memory; every thread owns 16 elements in registers at every stage.
//   stage 1: thread p holds x[p + (N/16) a], a = 0..15 -> 16-point DFT -> times w_N^{k1 p}
//   stage 2: inside block k1 (N/16 slots): radix R2 with twiddle w_{N/16}^{k2 q}
//   stage 3: radix R3 (absent when N <= 256)
// The output index k = k1 + 16 k2 + 16 R2 k3 ends up in slot k1*(N/16) + k2*R3 + k3, i.e. digit
// reversed.  The inverse is the exact mirror (conjugate twiddles, stages in reverse order), so
// a forward transform followed by a point-wise multiply and the mirrored inverse needs no
// reordering at all: that is what the column pass does (kinetic factor in the middle).
// Lanes of a warp always run over the oldest digit k1 (16 values) and the slot index carries
// one padding element per k1 block, which keeps all shared-memory accesses conflict free.
#pragma once
#include <cuda_runtime.h>

namespace gpe {

template <typename T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };
template <typename T> using cx = typename Vec2<T>::type;

template <typename T> __device__ __forceinline__ cx<T> mk(T x, T y) { cx<T> r; r.x = x; r.y = y; return r; }
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
    C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
// a * conj(b)
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) {
    C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r;
}

// z * exp(SIGN * 2 pi i m / 16), m = 0..7; m is a compile-time constant after unrolling.
// In fp32 the three constants cos(pi/8), sin(pi/8), sqrt(1/2) all round DOWN, so the rounded
// twiddles have modulus^2 = 1 - 3.4e-8 / 1 - 5.7e-8: a systematic (not random) loss that made
// the norm drift by -2e-7 per step in real time.  The float path therefore carries sqrt(1/2) as
// hi + lo and restores the modulus of the (cos, sin)(pi/8) pair with one extra FMA.
template <int SIGN, typename T> __device__ __forceinline__ cx<T> rot16(cx<T> z, int m) {
    constexpr T c1 = T(0.92387953251128675613), s1 = T(0.38268343236508977173),
                h = T(0.70710678118654752440);
    constexpr bool F32 = sizeof(T) == 4;
    constexpr T h_lo = F32 ? T(1.2101617152815436e-08) : T(0);   // sqrt(1/2) - float(sqrt(1/2))
    constexpr T eps_g = F32 ? T(2.8534284e-08) : T(0);            // 1/|(c1,s1)_fp32| - 1
    constexpr T sg = T(SIGN);
    cx<T> r;
    switch (m) {
    case 0: return z;
    case 4: return mk<T>(-sg * z.y, sg * z.x);
    case 2: r = mk<T>(z.x - sg * z.y, sg * z.x + z.y); break;
    case 6: r = mk<T>(-(z.x + sg * z.y), sg * z.x - z.y); break;
    case 1: r = mk<T>(z.x * c1 - z.y * (sg * s1), z.x * (sg * s1) + z.y * c1); break;
    case 3: r = mk<T>(z.x * s1 - z.y * (sg * c1), z.x * (sg * c1) + z.y * s1); break;
    case 5: r = mk<T>(-z.x * s1 - z.y * (sg * c1), z.x * (sg * c1) - z.y * s1); break;
    default: r = mk<T>(-z.x * c1 - z.y * (sg * s1), z.x * (sg * s1) - z.y * c1); break;
    }
    if (m == 2 || m == 6) {
        if constexpr (F32) return mk<T>(fma(r.x, h_lo, r.x * h), fma(r.y, h_lo, r.y * h));
        else return mk<T>(r.x * h, r.y * h);
    }
    if constexpr (F32) { r.x = fma(r.x, eps_g, r.x); r.y = fma(r.y, eps_g, r.y); }
    return r;
}

// In-register DFT of size R (2, 4, 8, 16): v[k] <- sum_a v[a] exp(SIGN 2 pi i a k / R),
// natural order in and out, radix-2 decimation in time with constant twiddles.
template <int R, int SIGN, typename T> __device__ __forceinline__ void dft(cx<T> *v) {
    if constexpr (R == 2) {
        cx<T> a = v[0];
        v[0] = cadd(a, v[1]);
        v[1] = csub(a, v[1]);
    } else {
        cx<T> e[R / 2], o[R / 2];
#pragma unroll
        for (int k = 0; k < R / 2; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
        dft<R / 2, SIGN, T>(e);
        dft<R / 2, SIGN, T>(o);
#pragma unroll
        for (int k = 0; k < R / 2; ++k) {
            cx<T> t = rot16<SIGN, T>(o[k], k * (16 / R));
            v[k] = cadd(e[k], t);
            v[k + R / 2] = csub(e[k], t);
        }
    }
}

template <int N> struct Fact;
template <> struct Fact<64> { static constexpr int R2 = 4, R3 = 1; };
template <> struct Fact<128> { static constexpr int R2 = 8, R3 = 1; };
template <> struct Fact<256> { static constexpr int R2 = 16, R3 = 1; };
template <> struct Fact<512> { static constexpr int R2 = 8, R3 = 4; };
template <> struct Fact<1024> { static constexpr int R2 = 8, R3 = 8; };
template <> struct Fact<2048> { static constexpr int R2 = 16, R3 = 8; };

// One 1-D FFT of length N worked on by N/16 threads (index j), S = element stride of the
// shared-memory tile (1 for a row, W for a tile of W columns).  tw[m] = exp(-2 pi i m / N).
template <int N, int S, typename T> struct Fft1D {
    using C = cx<T>;
    static constexpr int TPF = N / 16;
    static constexpr int M1 = N / 16;
    static constexpr int R2 = Fact<N>::R2, R3 = Fact<N>::R3;
    static constexpr int NST = R3 > 1 ? 3 : 2;
    static constexpr int SLOTS = N + 16;           // one padding slot per k1 block
    static constexpr int RL = NST == 3 ? R3 : R2;  // radix of the last stage
    static constexpr int GL = 16 / RL;             // butterflies per thread in the last stage

    __device__ __forceinline__ static int phys(int s) { return (s + s / M1) * S; }

    // natural output index of register (i*RL + r) of thread j after the forward transform
    __device__ __forceinline__ static int nat(int j, int i, int r) {
        int t = j + i * TPF;
        int k1 = t & 15, u = t >> 4;
        return NST == 3 ? k1 + 16 * u + 16 * R2 * r : k1 + 16 * r;
    }

    template <int R, int Mp> __device__ __forceinline__ static int base_slot(int t, int &q) {
        constexpr int M = Mp / R;
        int k1 = t & 15, u = t >> 4;
        int blk = u / M;
        q = u % M;
        return k1 * M1 + blk * Mp + q;
    }

    template <int R, int Mp, bool LAST>
    __device__ __forceinline__ static void stage_fwd(C *v, C *sm, int j, const C *__restrict__ tw) {
        constexpr int G = 16 / R, M = Mp / R;
#pragma unroll
        for (int i = 0; i < G; ++i) {
            int q, b = base_slot<R, Mp>(j + i * TPF, q);
#pragma unroll
            for (int a = 0; a < R; ++a) v[i * R + a] = sm[phys(b + M * a)];
        }
#pragma unroll
        for (int i = 0; i < G; ++i) dft<R, -1, T>(v + i * R);
        if constexpr (!LAST) {
#pragma unroll
            for (int i = 0; i < G; ++i) {
                int q, b = base_slot<R, Mp>(j + i * TPF, q);
#pragma unroll
                for (int k = 1; k < R; ++k) v[i * R + k] = cmul(v[i * R + k], tw[(N / Mp) * k * q]);
#pragma unroll
                for (int k = 0; k < R; ++k) sm[phys(b + M * k)] = v[i * R + k];
            }
        }
    }

    template <int R, int Mp, bool LAST>
    __device__ __forceinline__ static void stage_inv(C *v, C *sm, int j, const C *__restrict__ tw) {
        constexpr int G = 16 / R, M = Mp / R;
        if constexpr (!LAST) {
#pragma unroll
            for (int i = 0; i < G; ++i) {
                int q, b = base_slot<R, Mp>(j + i * TPF, q);
#pragma unroll
                for (int k = 0; k < R; ++k) v[i * R + k] = sm[phys(b + M * k)];
#pragma unroll
                for (int k = 1; k < R; ++k) v[i * R + k] = cmulc(v[i * R + k], tw[(N / Mp) * k * q]);
            }
        }
#pragma unroll
        for (int i = 0; i < G; ++i) dft<R, +1, T>(v + i * R);
#pragma unroll
        for (int i = 0; i < G; ++i) {
            int q, b = base_slot<R, Mp>(j + i * TPF, q);
#pragma unroll
            for (int a = 0; a < R; ++a) sm[phys(b + M * a)] = v[i * R + a];
        }
    }

    // in: v[a] = x[j + (N/16) a].  out: v[i*RL + r] = X[nat(j,i,r)] (unnormalised, e^{-i}).
    // All threads of the CTA must call this together (it contains __syncthreads()).
    __device__ __forceinline__ static void fwd(C *v, C *sm, int j, const C *__restrict__ tw) {
        dft<16, -1, T>(v);
#pragma unroll
        for (int k = 1; k < 16; ++k) v[k] = cmul(v[k], tw[k * j]);
#pragma unroll
        for (int k = 0; k < 16; ++k) sm[phys(j + M1 * k)] = v[k];
        __syncthreads();
        stage_fwd<R2, M1, NST == 2>(v, sm, j, tw);
        if constexpr (NST == 3) {
            __syncthreads();
            stage_fwd<R3, M1 / R2, true>(v, sm, j, tw);
        }
    }

    // exact mirror of fwd (unnormalised, e^{+i}): in: v[i*RL + r] = X[nat(j,i,r)],
    // out: v[a] = sum_k X[k] e^{+2 pi i k n / N} at n = j + (N/16) a.
    __device__ __forceinline__ static void inv(C *v, C *sm, int j, const C *__restrict__ tw) {
        if constexpr (NST == 3) {
            stage_inv<R3, M1 / R2, true>(v, sm, j, tw);
            __syncthreads();
            stage_inv<R2, M1, false>(v, sm, j, tw);
        } else {
            stage_inv<R2, M1, true>(v, sm, j, tw);
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = sm[phys(j + M1 * k)];
#pragma unroll
        for (int k = 1; k < 16; ++k) v[k] = cmulc(v[k], tw[k * j]);
        dft<16, +1, T>(v);
    }
};

}  // namespace gpe
