// gpe_kernels.cuh -- the three fused passes of one split-step:
//   pass A (rows):    load psi [x lazy scale] -> potential half-step a1 -> FFT along y -> store
//   pass B (columns): load -> FFT along x -> kinetic factor a3 -> inverse FFT along x -> store
//   pass C (rows):    load -> inverse FFT along y -> potential half-step a5 -> partial sums of
//                     |psi|^2 and cos cos |psi|^2 (a6) -> store; the last block reduces the
//                     partials in a fixed order and writes the scalars of the next step
//                     (a0: A_{n+1}, C_{n+1}; a7: scale; a8: record) -- no host round trip.
// PAPER.md:62-76 (Eqs. 2-4), :116 (renormalisation), :183-186 (Eq. 14).
#pragma once
#include <cstdlib>
#include <utility>
#include "gpe_fft.cuh"
#include "gpe_types.h"

#ifndef GPE_ROW_MINB
#define GPE_ROW_MINB 3
#endif
namespace gpe {

// ---------------------------------------------------------------- programmatic dependent launch
// Small grids launch every pass with cudaLaunchAttributeProgrammaticStreamSerialization: its CTAs
// may be scheduled while the previous pass drains (launch latency and prologue off the critical
// path) and block in pdl_wait() until that pass has completed and its writes are visible.  Without
// the attribute both instructions are no-ops.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl, Args &&...args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

// ---------------------------------------------------------------- launch geometry
// Threads per CTA of the one-number-per-element passes (complex128, and complex64 at 64 points): 64 (or one row) for
// rows of 256 points and more, 128 for columns of 256 and 512 points, 256 otherwise.  Measured on B200 in complex128 (us per
// step, 256 -> 128 threads): 512^2 27.6 -> 22.0, 1024^2 42.5 -> 41.7 (rows; narrower column tiles lose there: 19.1 ->
// 20.4 us for pass B), 2048^2 135.5 -> 133.0 -- more, smaller CTAs overlap their load / transform / store phases.
#ifndef GPE_ROWG_THREADS
#define GPE_ROWG_THREADS 64    // 64 against 128: 1024^2 complex128 41.7 -> 40.2 us per step, 512^2 22.0 -> 21.7, 2048^2 unchanged
#endif
#ifndef GPE_COLG_THREADS
#define GPE_COLG_THREADS 128
#endif
template <int N> struct RowGeom {
    static constexpr int TPF = N / 16;
    static constexpr int TARGET = N >= 256 ? GPE_ROWG_THREADS : 256;
    static constexpr int RPC = (TARGET / TPF) < 1 ? 1 : (TARGET / TPF);  // rows per CTA
    static constexpr int THREADS = RPC * TPF;
};
template <typename T, int N> struct ColGeom {
    static constexpr int TPF = N / 16;
    static constexpr int WMIN = sizeof(T) == 4 ? 4 : 2;            // >= 32-byte row segments
    static constexpr int W0 = ((N >= 256 && N <= 512) ? GPE_COLG_THREADS : 256) / TPF;
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

// The part of row a0 that does not depend on the sums: A_n and the cavity constants of step n,
// alpha_n = N eta_n Theta_n / (Delta + i kappa) = (kre + i kim) Theta_n, C_n = 2 eta_n Re alpha_n = kc Theta_n
// (Eqs. 13-14).
// Probe (Eq. 17, real time): alpha_n += pre + i pim = Omega exp(i (Delta_p n dt + phi)) / (Delta + i kappa),
// C_n += pc = 2 eta_n pre.
// bunch = int cos^2(k_c x)|psi|^2 (full cavity model: Delta -> Delta - N U0 bunch, Eq. 15).
__device__ inline void step_coefficients(const FinalizeParams &f, int b, long long n, double bunch, double &A, double &kre, double &kim,
                                         double &kc, double &pre, double &pim, double &pc) {
    A = schedule_at(f, b, (double)n + f.sched_mid);
    kre = kim = kc = pre = pim = pc = 0.0;
    if (f.cavity_on) {
        const double eta = f.eta_mode == 0 ? f.eta_or_u[b] : sqrt(fabs(A) * f.eta_or_u[b]);
        const double D = f.delta[b] - (f.cav_u0 ? f.n_atoms[b] * f.cav_u0[b] * bunch : 0.0);
        const double K = f.kappa[b], den = D * D + K * K, ne = f.n_atoms[b] * eta;
        kre = ne * D / den;                       // 1 / (D + iK) = (D - iK) / (D^2 + K^2)
        kim = -ne * K / den;
        kc = 2.0 * eta * kre;
        if (f.probe_omega && f.probe_dt != 0.0 && f.probe_omega[b] != 0.0) {
            double sn, cs;
            sincos(f.probe_delta[b] * ((double)n * f.probe_dt) + f.probe_phi[b], &sn, &cs);
            const double Om = f.probe_omega[b];
            pre = Om * (cs * D + sn * K) / den;   // (cs + i sn)(D - iK) / (D^2 + K^2)
            pim = Om * (sn * D - cs * K) / den;
            pc = 2.0 * eta * pre;
        }
    }
}
// Called by one thread of pass B per member while step n runs: coefficients of step n + 1.
// `local`: the member's state when it does not live at f.st[b] (the cluster kernel keeps a copy per CTA)
__device__ inline void prepare_member(const FinalizeParams &f, int b, MemberState *local = nullptr) {
    MemberState &s = local ? *local : f.st[b];
    step_coefficients(f, b, s.step + 1, 0.0, s.nA, s.nKre, s.nKim, s.nKc, s.nPre, s.nPim, s.nPc);
}

// Called by one thread of the last block of member b with the raw sums over the stored psi.
__device__ inline void finalize_member(const FinalizeParams &f, int b, double sum_n, double sum_t, double sum_b,
                                       MemberState *local = nullptr) {
    MemberState &s = local ? *local : f.st[b];
    double norm = sum_n * f.dxdy, theta = sum_t * f.dxdy, bunch = sum_b * f.dxdy;
    if (!(norm == norm) || norm > 1e300 || norm < 0.0 || (f.normalise && !(norm > 0.0))) *f.nonfinite = 1;
    long long n1;
    if (f.advance) n1 = s.step + 1; else n1 = f.step0;
    double scale = 1.0;
    if (f.normalise) {
        scale = 1.0 / sqrt(norm);
        theta = theta / norm;
        bunch = bunch / norm;
        norm = 1.0;
    }
    double A, re_a = 0.0, im_a = 0.0, C = 0.0;
    if (f.advance && f.prepared) {
        A = s.nA; re_a = s.nKre * theta + s.nPre; im_a = s.nKim * theta + s.nPim; C = s.nKc * theta + s.nPc;
    } else {
        double kre, kim, kc, pre, pim, pc;
        step_coefficients(f, b, n1, bunch, A, kre, kim, kc, pre, pim, pc);
        re_a = kre * theta + pre; im_a = kim * theta + pim; C = kc * theta + pc;
    }
    const double Dc = f.cav_u0 ? f.cav_u0[b] * (re_a * re_a + im_a * im_a) : 0.0;   // Eq. 12
    // T/2 V T/2 (gpe.h `ordering`): the stored psi is the one that enters the potential factor, so both
    // halves of the merged multiply of the next pass A take the coefficients computed right here
    if (f.tvt) { s.A_pend = A; s.C_pend = C; s.D_pend = Dc; s.pend = 1; }
    else if (f.advance && f.merged) { s.A_pend = s.A; s.C_pend = s.C; s.D_pend = s.D; s.pend = 1; } else s.pend = 0;
    s.D = Dc;
    s.scale = scale; s.A = A; s.C = C; s.norm = norm; s.theta = theta;
    s.re_alpha = re_a; s.im_alpha = im_a; s.step = n1;
    if (!f.advance && b == 0) {
        f.call->record_every = f.record_every; f.call->rec_first = f.rec_first; f.call->records = f.records;
    }
    const CallParams cp = f.advance ? *f.call : CallParams{0, 0, nullptr};
    if (f.advance && cp.records && cp.record_every > 0 && (n1 % cp.record_every) == 0) {
        long long idx = n1 / cp.record_every - cp.rec_first - 1;
        double *r = cp.records + ((size_t)idx * f.batch + b) * 6;
        r[0] = (double)n1; r[1] = norm; r[2] = theta; r[3] = re_a; r[4] = im_a; r[5] = A;
    }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Last CTA of member b: thread t adds partials t, t + blockDim.x, ... in that order.  The loads go out
// four at a time (ld.global.cg: L2, where the other CTAs' partials are after their fence) -- one
// dependent L2 round trip per partial, as a volatile loop does, left a 3 us serial tail after pass C
// at 2048^2 (1024 partials, 8 per thread) and 10 us in complex128 (32 per lane of one warp).
__device__ __forceinline__ void sum_partials(const FinalizeParams &f, int b, double &s0, double &s1, double &s2) {
    __threadfence();
    const double2 *pp = f.partials + (size_t)b * f.cpm;
    const int nt = blockDim.x;
    s0 = 0.0; s1 = 0.0; s2 = 0.0;
    for (int q0 = threadIdx.x; q0 < f.cpm; q0 += 4 * nt) {
        double2 t[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { const int q = q0 + k * nt; t[k] = q < f.cpm ? __ldcg(pp + q) : make_double2(0.0, 0.0); }
#pragma unroll
        for (int k = 0; k < 4; ++k) { s0 += t[k].x; s1 += t[k].y; }
    }
    if (f.cav_u0) {
        const double *pb = f.partials_b + (size_t)b * f.cpm;
        for (int q0 = threadIdx.x; q0 < f.cpm; q0 += 4 * nt) {
            double u[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) { const int q = q0 + k * nt; u[k] = q < f.cpm ? __ldcg(pb + q) : 0.0; }
#pragma unroll
            for (int k = 0; k < 4; ++k) s2 += u[k];
        }
    }
}

// Block-level sum of (sn, st), one partial per CTA, last CTA of the member finalises.
// `red` is shared scratch of at least 2*32 doubles.  All threads of the CTA must call this.
__device__ inline void block_reduce_and_finalize(const FinalizeParams &f, int b, int cta_in_member,
                                                 double sn, double st, double sb, double *red) {
    sn = warp_sum(sn);
    st = warp_sum(st);
    if (f.cav_u0) sb = warp_sum(sb);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) { red[w] = sn; red[32 + w] = st; red[64 + w] = sb; }
    __syncthreads();
    __shared__ int is_last;
    if (threadIdx.x == 0) {
        double a = 0.0, c = 0.0, e = 0.0;
        for (int i = 0; i < nw; ++i) { a += red[i]; c += red[32 + i]; e += red[64 + i]; }
        f.partials[(size_t)b * f.cpm + cta_in_member] = make_double2(a, c);
        if (f.cav_u0) f.partials_b[(size_t)b * f.cpm + cta_in_member] = e;
        __threadfence();
        unsigned int old = atomicAdd(&f.counters[b], 1u);
        is_last = (old == (unsigned int)(f.cpm - 1));
    }
    __syncthreads();
    if (is_last) {   // uniform over the CTA: all its threads sum the partials of the member
        double a, c, e;
        sum_partials(f, b, a, c, e);
        a = warp_sum(a); c = warp_sum(c); e = warp_sum(e);
        __syncthreads();
        if (lane == 0) { red[w] = a; red[32 + w] = c; red[64 + w] = e; }
        __syncthreads();
        double t0 = 0.0, t1 = 0.0, t2 = 0.0;
        if (threadIdx.x == 0)
            for (int i = 0; i < nw; ++i) { t0 += red[i]; t1 += red[32 + i]; t2 += red[64 + i]; }
        if (f.knorm) {   // the norm from pass B's k-space partial sums (merged kinetic halves, see k_col)
            double k = 0.0;
            const double *pk = f.partials_k + (size_t)b * f.cpmk;
            for (int q = threadIdx.x; q < f.cpmk; q += blockDim.x) k += __ldcg(pk + q);
            k = warp_sum(k);
            __syncthreads();
            if (lane == 0) red[w] = k;
            __syncthreads();
            if (threadIdx.x == 0) {
                double tk = 0.0;
                for (int i = 0; i < nw; ++i) tk += red[i];
                t0 = tk * f.kscale;
            }
        }
        if (threadIdx.x == 0) {
            finalize_member(f, b, t0, t1, t2);
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

template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

// General-argument (cos w - 1, sin w) for the rare large phase: kept out of line so that the
// library range reduction is not inlined sixteen times into every pass.
static __device__ __noinline__ void sincosm1_general(float w, float *s, float *cm1) {
    float sh, ch;
    sincosf(0.5f * w, &sh, &ch);
    *s = 2.0f * sh * ch;
    *cm1 = -2.0f * sh * sh;
}
// |w| <= 0.5: odd/even Taylor polynomials, error < 1 ulp of the result
__device__ __forceinline__ void sincosm1_small(float w, float *s, float *cm1) {
    const float w2 = w * w;
    float ps = fmaf(w2, 2.7557319e-6f, -1.9841270e-4f);
    ps = fmaf(w2, ps, 8.3333333e-3f);
    ps = fmaf(w2, ps, -1.6666667e-1f);
    *s = fmaf(w * w2, ps, w);
    float pc = fmaf(w2, 2.4801587e-5f, -1.3888889e-3f);
    pc = fmaf(w2, pc, 4.1666667e-2f);
    pc = fmaf(w2, pc, -0.5f);
    *cm1 = w2 * pc;
}

// |w| <= 0.5, double: sin w and cos w - 1 by their Taylor series in w^2 (Horner, fused multiply-adds)
__device__ __forceinline__ void sincosm1_small(double w, double *s, double *cm1) {
    const double w2 = w * w;
    double ps = fma(w2, -1.0 / 1307674368000.0, 1.0 / 6227020800.0);
    ps = fma(w2, ps, -1.0 / 39916800.0);
    ps = fma(w2, ps, 1.0 / 362880.0);
    ps = fma(w2, ps, -1.0 / 5040.0);
    ps = fma(w2, ps, 1.0 / 120.0);
    ps = fma(w2, ps, -1.0 / 6.0);
    *s = fma(w * w2, ps, w);
    double pc = fma(w2, 1.0 / 20922789888000.0, -1.0 / 87178291200.0);
    pc = fma(w2, pc, 1.0 / 479001600.0);
    pc = fma(w2, pc, -1.0 / 3628800.0);
    pc = fma(w2, pc, 1.0 / 40320.0);
    pc = fma(w2, pc, -1.0 / 720.0);
    pc = fma(w2, pc, 1.0 / 24.0);
    pc = fma(w2, pc, -0.5);
    *cm1 = w2 * pc;
}

// Potential half-step on the 16 points of one thread (rows a1 / a5), y_k = j + M1 k:
//   psi <- psi * exp(-s (V + g|psi|^2) dt/2),  V = vrow + vy[y] + A cos^2(k_l y) + crow cos(k_c y) [+ V2d]
// (vrow = vx[i] + A cos^2(k_l x_i), crow = C_n cos(k_c x_i)).  All table loads of the 16 points
// are issued back to back (one 4-vector per point), the angles are formed, and only then is the
// phase applied -- with ONE warp-uniform decision between the small-angle polynomial and the
// general path, so the common case has no per-point branch at all.
// REDUCE: also returns sum |psi_new|^2 and sum cos(k_c y) |psi_new|^2 over the 16 points.
template <typename T, bool IMAG, bool REDUCE, int M1, int P = 16>
__device__ __forceinline__ void potential_step16(cx<T> (&v)[P], const StepArgs<T, cx<T>> &a, int b, int i, int j,
                                                 T scale, T fac, T A, T Cc, T vadd, T &sn, T &st) {
    using V4 = typename Vec4<T>::type;
    const int flags = a.flags;
    T vrow = vadd;   // per-row constant supplied by the caller (cavity lattice D cos^2(k_c x_i))
    // fac = 1, or 2 when the multiply also carries the pending second half-step of the previous
    // step (real time; A, Cc are then the sums of the two steps' coefficients)
    if (flags & F_HAS_SEP) vrow += fac * a.vx[i];
    if (flags & F_LAT_X) vrow += A * a.latx[i];
    const T crow = (flags & F_CAVITY) ? Cc * a.cavx[i] : T(0);
    const T Ay = (flags & F_LAT_Y) ? A : T(0);
    const T g = (flags & F_HAS_G) ? fac * a.g[b] : T(0);
    const T hdt = a.half_dt;
    const V4 *__restrict__ yt = reinterpret_cast<const V4 *>(a.ytab);
    T w[P];
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const V4 t = yt[j + M1 * k];
        if constexpr (IMAG) { v[k].x *= scale; v[k].y *= scale; }  // the lazy scale is 1 in real time
        const T d = v[k].x * v[k].x + v[k].y * v[k].y;
        const T V = fma(crow, t.z, fma(Ay, t.y, fma(fac, t.x, vrow)));
        w[k] = fma(g, d, V) * hdt;
    }
    if (flags & F_HAS_V2D) {
        const T *__restrict__ v2 = a.v2d + ((flags & F_V2D_BATCHED) ? (size_t)b * a.nx * a.ny : 0) + (size_t)i * a.ny;
#pragma unroll
        for (int k = 0; k < P; ++k) w[k] = fma(v2[j + M1 * k], fac * hdt, w[k]);
    }
    if constexpr (IMAG) {
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const T e = exp_t(-w[k]);
            v[k].x *= e; v[k].y *= e;
        }
    } else if constexpr (sizeof(T) == 4) {
        // psi <- psi + psi * (cos w - 1 - i sin w), three warp-uniform tiers by the largest |w|:
        //   |w| <= 2^-5: sin w = w - w^3/6, cos w - 1 = -w^2/2 + w^4/24 (truncation < 2^-27 relative)
        //   |w| <= 0.5 : degree-9 / degree-8 polynomials;   else: library range reduction
        float wmax = 0.f;
#pragma unroll
        for (int k = 0; k < P; ++k) wmax = fmaxf(wmax, fabsf(w[k]));
        if (__all_sync(0xffffffffu, wmax <= 0.03125f)) {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                const float w2 = w[k] * w[k];
                const float sn_ = -fmaf(w[k] * w2, -1.6666667e-1f, w[k]);   // sin(-w)
                const float cm1 = w2 * fmaf(w2, 4.1666667e-2f, -0.5f);
                const float nx_ = fmaf(v[k].x, cm1, fmaf(-v[k].y, sn_, v[k].x));
                const float ny_ = fmaf(v[k].x, sn_, fmaf(v[k].y, cm1, v[k].y));
                v[k].x = nx_; v[k].y = ny_;
            }
        } else if (__all_sync(0xffffffffu, wmax <= 0.5f)) {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                float sn_, cm1;
                sincosm1_small(-w[k], &sn_, &cm1);
                const float nx_ = fmaf(v[k].x, cm1, fmaf(-v[k].y, sn_, v[k].x));
                const float ny_ = fmaf(v[k].x, sn_, fmaf(v[k].y, cm1, v[k].y));
                v[k].x = nx_; v[k].y = ny_;
            }
        } else {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                float sn_, cm1;
                sincosm1_general(-w[k], &sn_, &cm1);
                const float nx_ = fmaf(v[k].x, cm1, fmaf(-v[k].y, sn_, v[k].x));
                const float ny_ = fmaf(v[k].x, sn_, fmaf(v[k].y, cm1, v[k].y));
                v[k].x = nx_; v[k].y = ny_;
            }
        }
    } else {
        // complex128: Taylor polynomials in w^2 up to w^15 / w^16 while every |w| of the warp is <= 0.5
        // (next terms 4e-20 / 6e-22 relative), the library's range reduction otherwise
        T wmax = T(0);
#pragma unroll
        for (int k = 0; k < P; ++k) wmax = fmax(wmax, fabs(w[k]));
        const bool small = __all_sync(0xffffffffu, wmax <= T(0.5));
#pragma unroll
        for (int k = 0; k < P; ++k) {
            T sn_, cm1;
            if (small) sincosm1_small(-w[k], &sn_, &cm1);
            else sincosm1_t(-w[k], &sn_, &cm1);
            const T tx = fma(v[k].x, cm1, -(v[k].y * sn_)), ty = fma(v[k].x, sn_, v[k].y * cm1);
            v[k].x += tx; v[k].y += ty;
        }
    }
    if constexpr (REDUCE) {
        sn = T(0); st = T(0);
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const T d = v[k].x * v[k].x + v[k].y * v[k].y;
            sn += d;
            if (flags & F_CAVITY) st = fma(d, a.ytab[4 * (j + M1 * k) + 2], st);
        }
    }
}

// ---------------------------------------------------------------- pass A
// complex128 rows: two 256-thread CTAs per SM (128 registers) from 512 points up -- measured on B200:
// 2048^2 real time 185 -> 157 us per step, 1024^2 53 -> 45; below 512 one CTA with all registers wins.
template <typename T, int NY, bool IMAG>
__global__ void __launch_bounds__(RowGeom<NY>::THREADS, (sizeof(T) == 4 ? GPE_ROW_MINB : (NY >= 512 ? 2 : 1)) * (256 / RowGeom<NY>::THREADS > 0 ? 256 / RowGeom<NY>::THREADS : 1)) k_row_fwd(const StepArgs<T, cx<T>> a) {
    using C = cx<T>;
    using F = Fft1D<NY, 1, cx<T>>;
    using G = RowGeom<NY>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    C *sm = smem + r * F::SLOTS;
    pdl_launch_dependents();
    pdl_wait();
    {   // one group of RPC rows per CTA
        const long grp = blockIdx.x;
        const long row = grp * G::RPC + r;
        const int b = (int)(row / a.nx), i = (int)(row % a.nx);
        C *dst = a.dst + row * NY;
        C v[16];
        const C *src = a.src + row * NY;
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = __ldcg(src + j + F::M1 * k);
        if (!(a.flags & F_NO_POT)) {
            const MemberState &ms = a.fin.st[b];
            T sn, st;
            const bool pend = !IMAG && ms.pend;
            const T cx2 = (a.flags & F_CAV_FULL) ? a.cavx[i] * a.cavx[i] : T(0);
            potential_step16<T, IMAG, false, F::M1>(v, a, b, i, j, (T)ms.scale, pend ? T(2) : T(1), (T)(pend ? ms.A + ms.A_pend : ms.A),
                                                    (T)(pend ? ms.C + ms.C_pend : ms.C), (T)(pend ? ms.D + ms.D_pend : ms.D) * cx2, sn, st);
        }
        F::fwd(v, sm, j, a.tw_y, a.tw1_y);
        {
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) dst[F::nat(j, ii, rr)] = v[ii * F::RL + rr];
        }
    }
}

// ---------------------------------------------------------------- pass B
// MODE 0: forward, kinetic factor, inverse (the step).  MODE 1: forward only, natural order
// (observables).
template <typename T, int NX, bool IMAG, int MODE>
__global__ void __launch_bounds__(ColGeom<T, NX>::THREADS, (256 / ColGeom<T, NX>::THREADS > 0 ? 256 / ColGeom<T, NX>::THREADS : 1)) k_col(const StepArgs<T, cx<T>> a) {
    using C = cx<T>;
    using G = ColGeom<T, NX>;
    using F = Fft1D<NX, G::W, cx<T>>;
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
    pdl_launch_dependents();
    pdl_wait();
    if (MODE != 1 && blockIdx.x == 0 && threadIdx.x == 0 && a.fin.prepared) prepare_member(a.fin, b);
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = __ldcg(src + (size_t)(j + F::M1 * k) * ny);
    F::fwd(v, sm, j, a.tw_x, a.tw1_x);
    if constexpr (MODE == 1) {
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) dst[(size_t)F::nat(j, ii, rr) * ny] = v[ii * F::RL + rr];
        return;
    } else {
        if constexpr (IMAG) {
            const T ey = a.kin_yr[col];
            T acc = T(0);
            const T bigp = T(1) / a.inv_p;   // nx ny: a power of two, exact
#pragma unroll
            for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
                for (int rr = 0; rr < F::RL; ++rr) {
                    T f = a.kin_xr[F::nat(j, ii, rr)] * ey;
                    v[ii * F::RL + rr].x *= f;
                    v[ii * F::RL + rr].y *= f;
                    if constexpr (MODE == 2) {   // merged kinetic halves: see k_col_p (gpe_pair.cuh)
                        acc = fma(v[ii * F::RL + rr].x, v[ii * F::RL + rr].x, fma(v[ii * F::RL + rr].y, v[ii * F::RL + rr].y, acc));
                        const T f2 = f * bigp;
                        v[ii * F::RL + rr].x *= f2;
                        v[ii * F::RL + rr].y *= f2;
                    }
                }
            if constexpr (MODE == 2) {
                __shared__ double redk[32];
                const double sk = warp_sum((double)acc);
                if ((threadIdx.x & 31) == 0) redk[threadIdx.x >> 5] = sk;
                __syncthreads();
                if (threadIdx.x == 0) {
                    double t = 0.0;
                    for (int q = 0; q < G::THREADS / 32; ++q) t += redk[q];
                    a.fin.partials_k[(size_t)b * a.fin.cpmk + blockIdx.x] = t;
                }
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
        F::inv(v, sm, j, a.tw_x, a.tw1_x);
#pragma unroll
        for (int k = 0; k < 16; ++k) dst[(size_t)(j + F::M1 * k) * ny] = v[k];
    }
}

// ---------------------------------------------------------------- pass C
template <typename T, int NY, bool IMAG, bool MERGED>
__global__ void __launch_bounds__(RowGeom<NY>::THREADS, (sizeof(T) == 4 ? GPE_ROW_MINB : (NY >= 512 ? 2 : 1)) * (256 / RowGeom<NY>::THREADS > 0 ? 256 / RowGeom<NY>::THREADS : 1)) k_row_inv(const StepArgs<T, cx<T>> a) {
    using C = cx<T>;
    using F = Fft1D<NY, 1, cx<T>>;
    using G = RowGeom<NY>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    __shared__ double red[96];
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    C *sm = smem + r * F::SLOTS;
    const int gpm = a.nx / G::RPC;  // groups per member: all rows of a group belong to one member
    pdl_launch_dependents();
    pdl_wait();
    {   // one group of RPC rows per CTA
        const long grp = blockIdx.x;
        const long row = grp * G::RPC + r;
        const int b = (int)(row / a.nx), i = (int)(row % a.nx);
        C *dst = a.dst + row * NY;
        C v[16];
        const C *src = a.src + row * NY;
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) v[ii * F::RL + rr] = __ldcg(src + F::nat(j, ii, rr));
        F::inv(v, sm, j, a.tw_y, a.tw1_y);
        const MemberState &ms = a.fin.st[b];
        T sn, st;
        if constexpr (MERGED) {   // real time: the multiply is left to the next pass A, sums of |psi|^2 only
            sn = T(0); st = T(0);
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const T d = v[k].x * v[k].x + v[k].y * v[k].y;
                sn += d;
                if (a.flags & F_CAVITY) st = fma(d, a.ytab[4 * (j + F::M1 * k) + 2], st);
            }
        } else potential_step16<T, IMAG, true, F::M1>(v, a, b, i, j, T(1), T(1), (T)ms.A, (T)ms.C,
                                                      (a.flags & F_CAV_FULL) ? (T)ms.D * a.cavx[i] * a.cavx[i] : T(0), sn, st);
#pragma unroll
        for (int k = 0; k < 16; ++k) dst[j + F::M1 * k] = v[k];
        double dn = (double)sn, dt_ = (a.flags & F_CAVITY) ? (double)st * (double)a.cavx[i] : 0.0;
        const double db_ = (a.flags & F_CAV_FULL) ? dn * ((double)a.cavx[i] * (double)a.cavx[i]) : 0.0;
        block_reduce_and_finalize(a.fin, b, (int)(grp % gpm), dn, dt_, db_, red);
    }
}

// ---------------------------------------------------------------- pass C of step n fused with pass A of step n+1
// The 2-pass form (see k_row_ca_p in gpe_pair.cuh for when it applies and why the imaginary-time scale may lag
// one step): load -> IFFT_y -> sum |psi|^2 -> both potential half-steps in one multiply -> FFT_y -> store.
// The member's coefficients are read before the sums are published (the last CTA advances the state).
template <typename T, int NY, bool IMAG>
__global__ void __launch_bounds__(RowGeom<NY>::THREADS, (sizeof(T) == 4 ? GPE_ROW_MINB : (NY >= 512 ? 2 : 1)) * (256 / RowGeom<NY>::THREADS > 0 ? 256 / RowGeom<NY>::THREADS : 1)) k_row_ca(const StepArgs<T, cx<T>> a) {
    using C = cx<T>;
    using F = Fft1D<NY, 1, cx<T>>;
    using G = RowGeom<NY>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    __shared__ double red[96];
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    C *sm = smem + r * F::SLOTS;
    const int gpm = a.nx / G::RPC;
    pdl_launch_dependents();
    pdl_wait();
    const long grp = blockIdx.x;
    const long row = grp * G::RPC + r;
    const int b = (int)(row / a.nx), i = (int)(row % a.nx);
    const MemberState &ms = a.fin.st[b];
    const T Asum = (T)(ms.A + ms.nA), scale = (T)ms.scale;
    C *dst = a.dst + row * NY;
    const C *src = a.src + row * NY;
    C v[16];
#pragma unroll
    for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
        for (int rr = 0; rr < F::RL; ++rr) v[ii * F::RL + rr] = __ldcg(src + F::nat(j, ii, rr));
    F::inv(v, sm, j, a.tw_y, a.tw1_y);
    T sn = T(0), st = T(0);
#pragma unroll
    for (int k = 0; k < 16; ++k) sn += v[k].x * v[k].x + v[k].y * v[k].y;
    block_reduce_and_finalize(a.fin, b, (int)(grp % gpm), (double)sn, 0.0, 0.0, red);
    potential_step16<T, IMAG, false, F::M1>(v, a, b, i, j, scale, T(2), Asum, T(0), T(0), sn, st);
    F::fwd(v, sm, j, a.tw_y, a.tw1_y);
#pragma unroll
    for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
        for (int rr = 0; rr < F::RL; ++rr) dst[F::nat(j, ii, rr)] = v[ii * F::RL + rr];
}

// ---------------------------------------------------------------- launchers (one per T, N)
template <typename T, int N> struct Launch {
    using C = cx<T>;
    using A = StepArgs<T, C>;
    static size_t row_smem() {
        return sizeof(C) * RowGeom<N>::RPC * Fft1D<N, 1, cx<T>>::SLOTS;
    }
    // Measured on B200: overlapping the next pass's launch with the tail of
    // the current one pays for launch-bound grids (<= 256^2 points) and costs 1-4 us per step above.
    static bool use_pdl(const A &a) { return (long)a.batch * a.nx * a.ny <= 65536L; }
    static unsigned row_grid(const A &a) { return (unsigned)((long)a.batch * a.nx / RowGeom<N>::RPC); }
    static size_t col_smem() { return sizeof(C) * ColGeom<T, N>::W * Fft1D<N, 1, cx<T>>::SLOTS; }

    // opt in to > 48 KB of dynamic shared memory once per (device, kernel) -- the attribute is per
    // device -- and not on every launch: the call costs microseconds of host time on a latency
    // critical path.  When the table is full the attribute is simply set again (slow but correct).
    template <typename K> static cudaError_t prep(K kern, size_t smem) {
        struct Slot { K k; int dev; };
        static thread_local Slot done_for[48] = {};
        if (smem <= 48 * 1024) return cudaSuccess;
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        for (const Slot &sl : done_for) if (sl.k == kern && sl.dev == dev) return cudaSuccess;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            for (Slot &sl : done_for) if (sl.k == nullptr) { sl.k = kern; sl.dev = dev; break; }
        return e;
    }
    // ny == N
    static cudaError_t row_fwd(const A &a, bool imag, cudaStream_t s) {
        dim3 grid(row_grid(a)), block(RowGeom<N>::THREADS);
        cudaError_t e;
        if (imag) {
            if ((e = prep(k_row_fwd<T, N, true>, row_smem())) != cudaSuccess) return e;
            { cudaError_t le = launch_pdl(k_row_fwd<T, N, true>, grid, block, row_smem(), s, use_pdl(a), a); if (le != cudaSuccess) return le; }
        } else {
            if ((e = prep(k_row_fwd<T, N, false>, row_smem())) != cudaSuccess) return e;
            { cudaError_t le = launch_pdl(k_row_fwd<T, N, false>, grid, block, row_smem(), s, use_pdl(a), a); if (le != cudaSuccess) return le; }
        }
        return cudaGetLastError();
    }
    static cudaError_t row_inv(const A &a, bool imag, cudaStream_t s) {
        dim3 grid(row_grid(a)), block(RowGeom<N>::THREADS);
        auto go = [&](auto kern) -> cudaError_t {
            cudaError_t e = prep(kern, row_smem());
            if (e != cudaSuccess) return e;
            e = launch_pdl(kern, grid, block, row_smem(), s, use_pdl(a), a);
            return e != cudaSuccess ? e : cudaGetLastError();
        };
        if (imag) return go(k_row_inv<T, N, true, false>);
        return a.fin.merged ? go(k_row_inv<T, N, false, true>) : go(k_row_inv<T, N, false, false>);
    }
    static cudaError_t row_ca(const A &a, bool imag, cudaStream_t s) {
        dim3 grid(row_grid(a)), block(RowGeom<N>::THREADS);
        auto go = [&](auto kern) -> cudaError_t {
            cudaError_t e = prep(kern, row_smem());
            if (e != cudaSuccess) return e;
            e = launch_pdl(kern, grid, block, row_smem(), s, use_pdl(a), a);
            return e != cudaSuccess ? e : cudaGetLastError();
        };
        return imag ? go(k_row_ca<T, N, true>) : go(k_row_ca<T, N, false>);
    }
    // nx == N
    static cudaError_t col(const A &a, bool imag, int mode, cudaStream_t s) {
        dim3 grid((unsigned)(a.ny / ColGeom<T, N>::W), (unsigned)a.batch), block(ColGeom<T, N>::THREADS);
        cudaError_t e;
        if (mode == 0 && imag && a.fin.knorm) {
            if ((e = prep(k_col<T, N, true, 2>, col_smem())) != cudaSuccess) return e;
            { cudaError_t le = launch_pdl(k_col<T, N, true, 2>, grid, block, col_smem(), s, use_pdl(a), a); if (le != cudaSuccess) return le; }
        } else if (mode == 1) {
            if ((e = prep(k_col<T, N, false, 1>, col_smem())) != cudaSuccess) return e;
            { cudaError_t le = launch_pdl(k_col<T, N, false, 1>, grid, block, col_smem(), s, use_pdl(a), a); if (le != cudaSuccess) return le; }
        } else if (imag) {
            if ((e = prep(k_col<T, N, true, 0>, col_smem())) != cudaSuccess) return e;
            { cudaError_t le = launch_pdl(k_col<T, N, true, 0>, grid, block, col_smem(), s, use_pdl(a), a); if (le != cudaSuccess) return le; }
        } else {
            if ((e = prep(k_col<T, N, false, 0>, col_smem())) != cudaSuccess) return e;
            { cudaError_t le = launch_pdl(k_col<T, N, false, 0>, grid, block, col_smem(), s, use_pdl(a), a); if (le != cudaSuccess) return le; }
        }
        return cudaGetLastError();
    }
    static int rows_per_cta() { return RowGeom<N>::RPC; }
    static int cols_per_cta() { return ColGeom<T, N>::W; }
};

}  // namespace gpe
