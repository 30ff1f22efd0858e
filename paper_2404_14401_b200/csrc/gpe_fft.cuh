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
// complex64 sums use the packed fp32x2 adder of sm_100 (FADD2 / FFMA2: one issue slot for both
// components; same rounding as two scalar adds).  GPE_PACKED_ADD=0 falls back to scalar adds.
#ifndef GPE_PACKED_ADD
#define GPE_PACKED_ADD 0
#endif
__device__ __forceinline__ float2 cadd(float2 a, float2 b) {
#if GPE_PACKED_ADD
    return __fadd2_rn(a, b);
#else
    a.x += b.x; a.y += b.y; return a;
#endif
}
__device__ __forceinline__ float2 csub(float2 a, float2 b) {
#if GPE_PACKED_ADD
    return __ffma2_rn(b, make_float2(-1.0f, -1.0f), a);
#else
    a.x -= b.x; a.y -= b.y; return a;
#endif
}
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { a.x += b.x; a.y += b.y; return a; }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
    C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
// a * conj(b)
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) {
    C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r;
}

// z * exp(SIGN * 2 pi i m / 16), m = 0..7; m is a compile-time constant after unrolling.
//
// In fp32 the constants cos(pi/8), sin(pi/8), sqrt(1/2) all round DOWN, so the rounded twiddles
// have modulus^2 = 1 - 5.7e-8 / 1 - 3.4e-8.  That loss is systematic, not random: every radix-16
// butterfly scaled the data by 1 - 1.4e-8 and the norm drifted by -2e-7 per step in real time
// (cuFFT and pocketfft show the same bias).  The float path therefore uses a unit-modulus pair:
// S = fl32(sin(pi/8)) exactly and C = sqrt(1 - S^2) = C_hi + C_lo, and sqrt(1/2) = H_hi + H_lo.
// The low parts must enter BEFORE the single final rounding -- fma(u, C_hi, u*C_lo), never
// fma(u, C_lo, u*C_hi), whose 0.2-ulp correction would be rounded away.
template <typename T> struct K16;
template <> struct K16<float> {
    static constexpr float C_hi = 0.9238795638084412f, C_lo = -2.8719358092582937e-08f,
                           S = 0.3826834261417389f, H_hi = 0.7071067690849304f,
                           H_lo = 1.210161710447897e-08f;
};
template <> struct K16<double> {
    static constexpr double C_hi = 0.92387953251128675613, C_lo = 0.0, S = 0.38268343236508977173,
                            H_hi = 0.70710678118654752440, H_lo = 0.0;
};
// u*C + t with a single rounding of the large terms (t = the S-term plus nothing else)
template <typename T> __device__ __forceinline__ T mulC_add(T u, T t) {
    if constexpr (sizeof(T) == 4) return fma(u, K16<T>::C_hi, fma(u, K16<T>::C_lo, t));
    else return fma(u, K16<T>::C_hi, t);
}
template <typename T> __device__ __forceinline__ T mulH(T u) {
    if constexpr (sizeof(T) == 4) return fma(u, K16<T>::H_hi, u * K16<T>::H_lo);
    else return u * K16<T>::H_hi;
}
template <int SIGN, typename T> __device__ __forceinline__ cx<T> rot16(cx<T> z, int m) {
    constexpr T S = K16<T>::S;
    constexpr T sg = T(SIGN);
    switch (m) {
    case 0: return z;
    case 4: return mk<T>(-sg * z.y, sg * z.x);
    case 2: return mk<T>(mulH<T>(z.x - sg * z.y), mulH<T>(sg * z.x + z.y));
    case 6: return mk<T>(mulH<T>(-(z.x + sg * z.y)), mulH<T>(sg * z.x - z.y));
    // (C + i sg S), (S + i sg C), (-S + i sg C), (-C + i sg S)
    case 1: return mk<T>(mulC_add<T>(z.x, -(sg * S) * z.y), mulC_add<T>(z.y, (sg * S) * z.x));
    case 3: return mk<T>(mulC_add<T>(-sg * z.y, S * z.x), mulC_add<T>(sg * z.x, S * z.y));
    case 5: return mk<T>(mulC_add<T>(-sg * z.y, -S * z.x), mulC_add<T>(sg * z.x, -S * z.y));
    default: return mk<T>(mulC_add<T>(-z.x, -(sg * S) * z.y), mulC_add<T>(-z.y, (sg * S) * z.x));
    }
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
    // tw1[k * M1 + j] = exp(-2 pi i k j / N): the first-stage twiddles transposed so that the
    // lanes of a warp (consecutive j) read consecutive addresses (tw[k * j] is a stride-k gather
    // that costs up to 30 L1 wavefronts per load).
    __device__ __forceinline__ static void fwd(C *v, C *sm, int j, const C *__restrict__ tw,
                                               const C *__restrict__ tw1) {
        dft<16, -1, T>(v);
#pragma unroll
        for (int k = 1; k < 16; ++k) v[k] = cmul(v[k], tw1[k * M1 + j]);
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
    __device__ __forceinline__ static void inv(C *v, C *sm, int j, const C *__restrict__ tw,
                                               const C *__restrict__ tw1) {
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
        for (int k = 1; k < 16; ++k) v[k] = cmulc(v[k], tw1[k * M1 + j]);
        dft<16, +1, T>(v);
    }
};

}  // namespace gpe
