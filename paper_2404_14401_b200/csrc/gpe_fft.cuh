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
//
// Element types.  The transform is written once over an element type E:
//   float2 / double2 : one complex number per element (scalar arithmetic);
//   cpair            : TWO complex64 numbers of two independent transforms in lock step, stored
//                      as (re0, re1), (im0, im1).  Every add, multiply and fma is then one packed
//                      fp32x2 instruction of sm_100 (FADD2 / FMUL2 / FFMA2 -- the twiddle enters
//                      as a broadcast scalar operand), so a butterfly costs half the issue slots
//                      per point, and a shared-memory exchange is one 128-bit access per pair.
#pragma once
#include <cuda_runtime.h>

namespace gpe {

template <typename T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };
template <typename T> using cx = typename Vec2<T>::type;

struct __align__(16) cpair { float2 re, im; };

template <typename E> struct El;
// T scalar type, R real vector (one value per lane), SE shared-memory element, PLANES of SE per element
template <> struct El<float2> { using T = float; using R = float; using SE = float2; static constexpr int PLANES = 1; };
template <> struct El<double2> { using T = double; using R = double; using SE = double2; static constexpr int PLANES = 1; };
template <> struct El<cpair> { using T = float; using R = float2; using SE = float2; static constexpr int PLANES = 2; };

template <typename T> __device__ __forceinline__ cx<T> mk(T x, T y) { cx<T> r; r.x = x; r.y = y; return r; }

// ---- "real vector" arithmetic: R = float | double | float2 (two lanes), s = scalar (broadcast)
__device__ __forceinline__ float radd(float a, float b) { return a + b; }
__device__ __forceinline__ float rsub(float a, float b) { return a - b; }
__device__ __forceinline__ float rneg(float a) { return -a; }
__device__ __forceinline__ float rmuls(float a, float s) { return a * s; }
__device__ __forceinline__ float rfmas(float a, float s, float c) { return fmaf(a, s, c); }
__device__ __forceinline__ double radd(double a, double b) { return a + b; }
__device__ __forceinline__ double rsub(double a, double b) { return a - b; }
__device__ __forceinline__ double rneg(double a) { return -a; }
__device__ __forceinline__ double rmuls(double a, double s) { return a * s; }
__device__ __forceinline__ double rfmas(double a, double s, double c) { return fma(a, s, c); }
__device__ __forceinline__ float2 rneg(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 radd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 rsub(float2 a, float2 b) { return __fadd2_rn(a, rneg(b)); }
__device__ __forceinline__ float2 rmuls(float2 a, float s) { return __fmul2_rn(a, make_float2(s, s)); }
__device__ __forceinline__ float2 rfmas(float2 a, float s, float2 c) { return __ffma2_rn(a, make_float2(s, s), c); }
__device__ __forceinline__ float2 rmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 rfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
template <int SG, typename R> __device__ __forceinline__ R rsg(R a) { if constexpr (SG > 0) return a; else return rneg(a); }

// ---- element access
__device__ __forceinline__ float ere(float2 z) { return z.x; }
__device__ __forceinline__ float eim(float2 z) { return z.y; }
__device__ __forceinline__ double ere(double2 z) { return z.x; }
__device__ __forceinline__ double eim(double2 z) { return z.y; }
__device__ __forceinline__ float2 ere(cpair z) { return z.re; }
__device__ __forceinline__ float2 eim(cpair z) { return z.im; }
template <typename E> __device__ __forceinline__ E emk(typename El<E>::R x, typename El<E>::R y);
template <> __device__ __forceinline__ float2 emk<float2>(float x, float y) { return make_float2(x, y); }
template <> __device__ __forceinline__ double2 emk<double2>(double x, double y) { return make_double2(x, y); }
template <> __device__ __forceinline__ cpair emk<cpair>(float2 x, float2 y) { cpair r; r.re = x; r.im = y; return r; }

// shared-memory exchange.  A cpair goes to two 64-bit planes (all real parts, then all imaginary
// parts, PLANE elements apart): the packed arithmetic keeps (re0, re1) and (im0, im1) in two
// unrelated register pairs, and a single 128-bit access would cost two MOVs per element to line
// them up in one aligned quad.
template <int PLANE> __device__ __forceinline__ void sst(float2 *sm, int i, float2 v) { sm[i] = v; }
template <int PLANE> __device__ __forceinline__ void sst(double2 *sm, int i, double2 v) { sm[i] = v; }
template <int PLANE> __device__ __forceinline__ void sst(float2 *sm, int i, cpair v) { sm[i] = v.re; sm[i + PLANE] = v.im; }
template <int PLANE, typename E> __device__ __forceinline__ E sld(const typename El<E>::SE *sm, int i) {
    if constexpr (El<E>::PLANES == 2) { E r; r.re = sm[i]; r.im = sm[i + PLANE]; return r; }
    else return sm[i];
}

template <typename E> __device__ __forceinline__ E cadd(E a, E b) { return emk<E>(radd(ere(a), ere(b)), radd(eim(a), eim(b))); }
template <typename E> __device__ __forceinline__ E csub(E a, E b) { return emk<E>(rsub(ere(a), ere(b)), rsub(eim(a), eim(b))); }
// a * w and a * conj(w); w = one twiddle (cos, sin) shared by all lanes of the element
template <typename E> __device__ __forceinline__ E cmul(E a, cx<typename El<E>::T> w) {
    return emk<E>(rfmas(ere(a), w.x, rmuls(eim(a), -w.y)), rfmas(ere(a), w.y, rmuls(eim(a), w.x)));
}
template <typename E> __device__ __forceinline__ E cmulc(E a, cx<typename El<E>::T> w) {
    return emk<E>(rfmas(ere(a), w.x, rmuls(eim(a), w.y)), rfmas(eim(a), w.x, rmuls(ere(a), -w.y)));
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
template <typename T, typename R> __device__ __forceinline__ R mulC_add(R u, R t) {
    if constexpr (sizeof(T) == 4) return rfmas(u, K16<T>::C_hi, rfmas(u, K16<T>::C_lo, t));
    else return rfmas(u, K16<T>::C_hi, t);
}
template <typename T, typename R> __device__ __forceinline__ R mulH(R u) {
    if constexpr (sizeof(T) == 4) return rfmas(u, K16<T>::H_hi, rmuls(u, K16<T>::H_lo));
    else return rmuls(u, K16<T>::H_hi);
}
template <int SIGN, typename E> __device__ __forceinline__ E rot16(E z, int m) {
    using T = typename El<E>::T;
    using R = typename El<E>::R;
    constexpr T S = K16<T>::S;
    constexpr T sS = T(SIGN) * S;
    const R x = ere(z), y = eim(z);
    switch (m) {
    case 0: return z;
    case 4: return emk<E>(rsg<-SIGN>(y), rsg<SIGN>(x));
    case 2: return emk<E>(mulH<T>(radd(x, rsg<-SIGN>(y))), mulH<T>(radd(rsg<SIGN>(x), y)));
    case 6: return emk<E>(mulH<T>(rneg(radd(x, rsg<SIGN>(y)))), mulH<T>(rsub(rsg<SIGN>(x), y)));
    // (C + i sg S), (S + i sg C), (-S + i sg C), (-C + i sg S)
    case 1: return emk<E>(mulC_add<T>(x, rmuls(y, -sS)), mulC_add<T>(y, rmuls(x, sS)));
    case 3: return emk<E>(mulC_add<T>(rsg<-SIGN>(y), rmuls(x, S)), mulC_add<T>(rsg<SIGN>(x), rmuls(y, S)));
    case 5: return emk<E>(mulC_add<T>(rsg<-SIGN>(y), rmuls(x, -S)), mulC_add<T>(rsg<SIGN>(x), rmuls(y, -S)));
    default: return emk<E>(mulC_add<T>(rneg(x), rmuls(y, -sS)), mulC_add<T>(rneg(y), rmuls(x, sS)));
    }
}

// In-register DFT of size R (2, 4, 8, 16): v[k] <- sum_a v[a] exp(SIGN 2 pi i a k / R),
// natural order in and out, radix-2 decimation in time with constant twiddles.
template <int R, int SIGN, typename E> __device__ __forceinline__ void dft(E *v) {
    if constexpr (R == 2) {
        E a = v[0];
        v[0] = cadd(a, v[1]);
        v[1] = csub(a, v[1]);
    } else {
        E e[R / 2], o[R / 2];
#pragma unroll
        for (int k = 0; k < R / 2; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
        dft<R / 2, SIGN, E>(e);
        dft<R / 2, SIGN, E>(o);
#pragma unroll
        for (int k = 0; k < R / 2; ++k) {
            E t = rot16<SIGN, E>(o[k], k * (16 / R));
            v[k] = cadd(e[k], t);
            v[k + R / 2] = csub(e[k], t);
        }
    }
}

// table fetch (plain cached load; the read-only path, __ldg, measured no faster on B200)
template <typename C> __device__ __forceinline__ C ldtw(const C *__restrict__ t, int i) { return t[i]; }

// N = P * R2 * R3: the radices of the second and third stage for P points per thread
template <int N, int P = 16> struct Fact;
template <> struct Fact<64, 16> { static constexpr int R2 = 4, R3 = 1; };
template <> struct Fact<128, 16> { static constexpr int R2 = 8, R3 = 1; };
template <> struct Fact<256, 16> { static constexpr int R2 = 16, R3 = 1; };
template <> struct Fact<512, 16> { static constexpr int R2 = 8, R3 = 4; };
template <> struct Fact<1024, 16> { static constexpr int R2 = 8, R3 = 8; };
template <> struct Fact<2048, 16> { static constexpr int R2 = 16, R3 = 8; };
// eight points per thread: twice the threads, half the dependent chain (the cluster kernel of gpe_chip.cuh)
template <> struct Fact<64, 8> { static constexpr int R2 = 8, R3 = 1; };
template <> struct Fact<128, 8> { static constexpr int R2 = 4, R3 = 4; };
template <> struct Fact<256, 8> { static constexpr int R2 = 8, R3 = 4; };

// One 1-D FFT of length N worked on by N/P threads (index j), every thread owning P points (16, or 8) at every
// stage; S = element stride of the shared-memory tile (1 for a row, W for a tile of W columns).
// tw[m] = exp(-2 pi i m / N).  E = element type (see the top of this file); twiddles are always one cx<T> per element.
template <int N, int S, typename E, int P = 16> struct Fft1D {
    using T = typename El<E>::T;
    using C = cx<T>;
    using SE = typename El<E>::SE;
    static constexpr int LOGP = P == 16 ? 4 : 3;
    static_assert(P == 16 || P == 8, "16 or 8 points per thread");
    static constexpr int TPF = N / P;
    static constexpr int M1 = N / P;
    static constexpr int R2 = Fact<N, P>::R2, R3 = Fact<N, P>::R3;
    static constexpr int NST = R3 > 1 ? 3 : 2;
    static constexpr int SLOTS = N + P;            // one padding slot per k1 block
    static constexpr int PLANE = SLOTS * S;        // distance between the planes of a cpair tile
    static constexpr int TILE = SLOTS * S * El<E>::PLANES;  // SE elements of one tile (S transforms)
    static constexpr int RL = NST == 3 ? R3 : R2;  // radix of the last stage
    static constexpr int GL = P / RL;              // butterflies per thread in the last stage

    __device__ __forceinline__ static int phys(int s) { return (s + s / M1) * S; }

    // natural output index of register (i*RL + r) of thread j after the forward transform
    __device__ __forceinline__ static int nat(int j, int i, int r) {
        int t = j + i * TPF;
        int k1 = t & (P - 1), u = t >> LOGP;
        return NST == 3 ? k1 + P * u + P * R2 * r : k1 + P * r;
    }

    template <int R, int Mp> __device__ __forceinline__ static int base_slot(int t, int &q) {
        constexpr int M = Mp / R;
        int k1 = t & (P - 1), u = t >> LOGP;
        int blk = u / M;
        q = u % M;
        return k1 * M1 + blk * Mp + q;
    }

    template <int R, int Mp, bool LAST>
    __device__ __forceinline__ static void stage_fwd(E *v, SE *sm, int j, const C *__restrict__ tw) {
        constexpr int G = P / R, M = Mp / R;
#pragma unroll
        for (int i = 0; i < G; ++i) {
            int q, b = base_slot<R, Mp>(j + i * TPF, q);
#pragma unroll
            for (int a = 0; a < R; ++a) v[i * R + a] = sld<PLANE, E>(sm, phys(b + M * a));
        }
#pragma unroll
        for (int i = 0; i < G; ++i) dft<R, -1, E>(v + i * R);
        if constexpr (!LAST) {
#pragma unroll
            for (int i = 0; i < G; ++i) {
                int q, b = base_slot<R, Mp>(j + i * TPF, q);
#pragma unroll
                for (int k = 1; k < R; ++k) v[i * R + k] = cmul(v[i * R + k], ldtw(tw, (N / Mp) * k * q));
#pragma unroll
                for (int k = 0; k < R; ++k) sst<PLANE>(sm, phys(b + M * k), v[i * R + k]);
            }
        }
    }

    template <int R, int Mp, bool LAST>
    __device__ __forceinline__ static void stage_inv(E *v, SE *sm, int j, const C *__restrict__ tw) {
        constexpr int G = P / R, M = Mp / R;
        if constexpr (!LAST) {
#pragma unroll
            for (int i = 0; i < G; ++i) {
                int q, b = base_slot<R, Mp>(j + i * TPF, q);
#pragma unroll
                for (int k = 0; k < R; ++k) v[i * R + k] = sld<PLANE, E>(sm, phys(b + M * k));
#pragma unroll
                for (int k = 1; k < R; ++k) v[i * R + k] = cmulc(v[i * R + k], ldtw(tw, (N / Mp) * k * q));
            }
        }
#pragma unroll
        for (int i = 0; i < G; ++i) dft<R, +1, E>(v + i * R);
#pragma unroll
        for (int i = 0; i < G; ++i) {
            int q, b = base_slot<R, Mp>(j + i * TPF, q);
#pragma unroll
            for (int a = 0; a < R; ++a) sst<PLANE>(sm, phys(b + M * a), v[i * R + a]);
        }
    }

    // ---- pair-mapped outer stage (row passes of gpe_pair.cuh).  Two transforms whose tiles are sm0
    // and sm1 are worked on by 2*TPF threads (slot u in [0, 2 TPF)); in the LAST forward stage (and
    // the mirrored FIRST inverse stage) thread u takes butterflies t = u + 2 TPF i, i < GL/2, of
    // BOTH transforms instead of GL butterflies of its own, so that it holds the same output
    // indices of the two transforms: register (2 i + w) * RL + r = X_w[nat_t(t, r)].  Needs GL >= 2.
    static constexpr int RLM = NST == 3 ? M1 / R2 : M1;   // Mp of the last stage
    __device__ __forceinline__ static int nat_t(int t, int r) {
        int k1 = t & (P - 1), u = t >> LOGP;
        return NST == 3 ? k1 + P * u + P * R2 * r : k1 + P * r;
    }
    __device__ __forceinline__ static void last_fwd_pair(E *v, const SE *sm0, const SE *sm1, int u) {
        constexpr int M = RLM / RL;
#pragma unroll
        for (int i = 0; i < GL / 2; ++i) {
            int q, b = base_slot<RL, RLM>(u + 2 * TPF * i, q);
#pragma unroll
            for (int a = 0; a < RL; ++a) {
                v[(2 * i) * RL + a] = sld<PLANE, E>(sm0, phys(b + M * a));
                v[(2 * i + 1) * RL + a] = sld<PLANE, E>(sm1, phys(b + M * a));
            }
        }
#pragma unroll
        for (int i = 0; i < GL; ++i) dft<RL, -1, E>(v + i * RL);
    }
    __device__ __forceinline__ static void first_inv_pair(E *v, SE *sm0, SE *sm1, int u) {
        constexpr int M = RLM / RL;
#pragma unroll
        for (int i = 0; i < GL; ++i) dft<RL, +1, E>(v + i * RL);
#pragma unroll
        for (int i = 0; i < GL / 2; ++i) {
            int q, b = base_slot<RL, RLM>(u + 2 * TPF * i, q);
#pragma unroll
            for (int a = 0; a < RL; ++a) {
                sst<PLANE>(sm0, phys(b + M * a), v[(2 * i) * RL + a]);
                sst<PLANE>(sm1, phys(b + M * a), v[(2 * i + 1) * RL + a]);
            }
        }
    }
    // forward transform whose last stage is pair-mapped; SYNC covers the threads of the own
    // transform, SYNC2 (before the pair-mapped stage) those of both transforms
    template <typename Sync, typename Sync2>
    __device__ __forceinline__ static void fwd_pairlast(E *v, SE *sm, const SE *sm0, const SE *sm1, int j, int u,
                                                        const C *__restrict__ tw, const C *__restrict__ tw1, Sync SYNC, Sync2 SYNC2) {
        dft<P, -1, E>(v);
#pragma unroll
        for (int k = 1; k < P; ++k) v[k] = cmul(v[k], ldtw(tw1, k * M1 + j));
#pragma unroll
        for (int k = 0; k < P; ++k) sst<PLANE>(sm, phys(j + M1 * k), v[k]);
        if constexpr (NST == 3) {
            SYNC();
            stage_fwd<R2, M1, false>(v, sm, j, tw);
        }
        SYNC2();
        last_fwd_pair(v, sm0, sm1, u);
    }
    // mirror: in: v[(2 i + w) * RL + r] = X_w[nat_t(u + 2 TPF i, r)]; out: v[a] of the own transform
    template <typename Sync, typename Sync2>
    __device__ __forceinline__ static void inv_pairfirst(E *v, SE *sm, SE *sm0, SE *sm1, int j, int u,
                                                         const C *__restrict__ tw, const C *__restrict__ tw1, Sync SYNC, Sync2 SYNC2) {
        first_inv_pair(v, sm0, sm1, u);
        SYNC2();
        if constexpr (NST == 3) {
            stage_inv<R2, M1, false>(v, sm, j, tw);
            SYNC();
        }
#pragma unroll
        for (int k = 0; k < P; ++k) v[k] = sld<PLANE, E>(sm, phys(j + M1 * k));
#pragma unroll
        for (int k = 1; k < P; ++k) v[k] = cmulc(v[k], ldtw(tw1, k * M1 + j));
        dft<P, +1, E>(v);
    }

    // in: v[a] = x[j + (N/16) a].  out: v[i*RL + r] = X[nat(j,i,r)] (unnormalised, e^{-i}).
    // All threads that share `sm` must call this together: SYNC() is the barrier between them
    // (__syncthreads, or a named barrier over the threads of one transform).
    // tw1[k * M1 + j] = exp(-2 pi i k j / N): the first-stage twiddles transposed so that the
    // lanes of a warp (consecutive j) read consecutive addresses (tw[k * j] is a stride-k gather
    // that costs up to 30 L1 wavefronts per load).
    template <typename Sync>
    __device__ __forceinline__ static void fwd(E *v, SE *sm, int j, const C *__restrict__ tw,
                                               const C *__restrict__ tw1, Sync SYNC) {
        dft<P, -1, E>(v);
#pragma unroll
        for (int k = 1; k < P; ++k) v[k] = cmul(v[k], ldtw(tw1, k * M1 + j));
#pragma unroll
        for (int k = 0; k < P; ++k) sst<PLANE>(sm, phys(j + M1 * k), v[k]);
        SYNC();
        stage_fwd<R2, M1, NST == 2>(v, sm, j, tw);
        if constexpr (NST == 3) {
            SYNC();
            stage_fwd<R3, M1 / R2, true>(v, sm, j, tw);
        }
    }
    __device__ __forceinline__ static void fwd(E *v, SE *sm, int j, const C *__restrict__ tw,
                                               const C *__restrict__ tw1) {
        fwd(v, sm, j, tw, tw1, [] { __syncthreads(); });
    }

    // exact mirror of fwd (unnormalised, e^{+i}): in: v[i*RL + r] = X[nat(j,i,r)],
    // out: v[a] = sum_k X[k] e^{+2 pi i k n / N} at n = j + (N/16) a.
    template <typename Sync>
    __device__ __forceinline__ static void inv(E *v, SE *sm, int j, const C *__restrict__ tw,
                                               const C *__restrict__ tw1, Sync SYNC) {
        if constexpr (NST == 3) {
            stage_inv<R3, M1 / R2, true>(v, sm, j, tw);
            SYNC();
            stage_inv<R2, M1, false>(v, sm, j, tw);
        } else {
            stage_inv<R2, M1, true>(v, sm, j, tw);
        }
        SYNC();
#pragma unroll
        for (int k = 0; k < P; ++k) v[k] = sld<PLANE, E>(sm, phys(j + M1 * k));
#pragma unroll
        for (int k = 1; k < P; ++k) v[k] = cmulc(v[k], ldtw(tw1, k * M1 + j));
        dft<P, +1, E>(v);
    }
    __device__ __forceinline__ static void inv(E *v, SE *sm, int j, const C *__restrict__ tw,
                                               const C *__restrict__ tw1) {
        inv(v, sm, j, tw, tw1, [] { __syncthreads(); });
    }
};

}  // namespace gpe
