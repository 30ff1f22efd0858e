// gpe_chip.cuh -- small grids (64^2 .. 256^2): ALL steps of a gpe_evolve call in ONE kernel launch.
//
// At these sizes a pass is a few hundred nanoseconds of work and a step was three dependent launches of
// about 5 us each (profiles/r01_final.md: 256^2 15.2 us per step, 0.03 of its byte roofline).  Here one
// thread-block cluster per batch member (8 CTAs at 64^2, 16 from 128^2 on) stays resident for the whole call:
//   * CTA `rank` owns N / NC rows in the row phases and N / NC columns in the column phase;
//   * the kernel boundaries between the passes become hardware cluster barriers
//     (barrier.cluster.arrive.release / wait.acquire, about 0.2 us), the data crosses between the row and the
//     column ownership through the caller's psi buffer in L2 (in place, ld.global.cg / st.global: measured
//     DSMEM bandwidth, about 20 B/clk per SM, would make an all-to-all of the grid through distributed shared
//     memory slower than through L2);
//   * the rows stay in REGISTERS from the inverse transform along y of step n to the forward transform along
//     y of step n+1: the global scalars in between (norm, Theta, B -> A_{n+1}, C_{n+1}, D_{n+1}, 1/||psi||) are
//     summed per CTA, handed to every CTA of the cluster through distributed shared memory (one 24-byte
//     remote store per CTA pair), and every CTA then runs the same finalize_member on its own copy of the
//     member's state -- one cluster barrier, no round trip through CTA 0;
//   * CTA 0 alone writes records and, at the end, the member's state back to global memory.
// Same arithmetic as the one-number-per-element passes of gpe_kernels.cuh (potential_step16, Fft1D,
// finalize_member are shared): PAPER.md:62-76 Eqs. 2-4, :116, :183-188 Eqs. 14-15.
// The prologue reduction (k_reduce) and the epilogue (pending half-step / final rescale) stay separate launches.
#pragma once
#include <cooperative_groups.h>
#include "gpe_kernels.cuh"

#ifndef GPE_CHIP_NC16_MIN
#define GPE_CHIP_NC16_MIN 128   // from this size on 16 CTAs per cluster
#endif
// Points per thread (Fft1D's P).  Eight points per thread give twice the warps and half the dependent chain of
// sixteen.  Measured on B200, us per step (sweep / pulse / cavity workloads, complex64), P = 8 against P = 16:
// 64^2 4.7 / 4.7 / 5.6 against 7.3 / 7.1 / 8.0 (complex128 5.9 against 8.9); 128^2 6.6 / 6.6 / 7.6 against 7.8 / 7.5 / 8.4;
// 256^2 12.0 / 11.2 / 12.2 against 10.3 / 9.7 / 10.7 (one more exchange per transform).  The fp32 norm drift of a
// real-time step (a fixed bias of the few distinct rounded twiddles a small transform uses) is -6.2e-8 against
// -5.6e-8 at 64^2 but -1.0e-7 against -2.6e-8 at 128^2: eight points per thread at 64^2 only.
#ifndef GPE_CHIP_P8_MAX_N
#define GPE_CHIP_P8_MAX_N 64
#endif
namespace gpe {
namespace cg = cooperative_groups;

template <typename T, int N> struct ChipGeom {
    static constexpr int NC = N >= GPE_CHIP_NC16_MIN ? 16 : 8;   // CTAs per cluster (16 needs the non-portable opt-in)
    static constexpr int P = N <= GPE_CHIP_P8_MAX_N ? 8 : 16;          // points per thread
    static constexpr int RB = N / NC;                                  // rows (and columns) per CTA
    static constexpr int TPF = N / P;                                  // threads per transform
    static constexpr int THREADS = RB * TPF;                           // 64^2: 32, 128^2: 64, 256^2: 256
    using FR = Fft1D<N, 1, cx<T>, P>;                                  // a row in its own SLOTS-element tile
    using FC = Fft1D<N, RB, cx<T>, P>;                                 // RB columns interleaved in one tile
    static constexpr size_t SMEM = sizeof(cx<T>) * (size_t)RB * FR::SLOTS;
    static_assert(N >= 64 && N <= 256 && RB >= 1 && THREADS >= 32 && THREADS <= 512 && THREADS % 32 == 0, "small grids only");
};

// sum over the CTA of three doubles (fixed order), result valid in thread 0
template <int THREADS> __device__ __forceinline__ void cta_sum3(double &a, double &b, double &c, double *red) {
    a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
    constexpr int NW = THREADS / 32;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) { red[w] = a; red[16 + w] = b; red[32 + w] = c; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = 0.0; b = 0.0; c = 0.0;
#pragma unroll
        for (int q = 0; q < NW; ++q) { a += red[q]; b += red[16 + q]; c += red[32 + q]; }
    }
}

template <typename T, int N, bool IMAG>
__global__ void __launch_bounds__(ChipGeom<T, N>::THREADS, 1) k_chip(const StepArgs<T, cx<T>> a, long n_steps) {
    using G = ChipGeom<T, N>;
    using FR = typename G::FR;
    using FC = typename G::FC;
    using C = cx<T>;
    constexpr int NC = G::NC, RB = G::RB, TPF = G::TPF, M1 = FR::M1, P = G::P;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    __shared__ MemberState lms;          // this CTA's copy of the member's state (identical in all CTAs)
    __shared__ CallParams lcall;
    __shared__ double part[16][3];       // partial sums of every CTA of the cluster, written remotely
    __shared__ double red[48];
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int b = blockIdx.x / NC;
    const int tid = threadIdx.x;
    // row ownership
    const int r = tid / TPF, j = tid % TPF;
    const int i = rank * RB + r;                       // row of this thread
    C *smr = smem + r * FR::SLOTS;
    // column ownership
    const int cc = tid % RB, jc = tid / RB;
    const int col = rank * RB + cc;
    C *smc = smem + cc;
    C *psi = a.dst + (size_t)b * N * N;
    C *prow = psi + (size_t)i * N;
    C *pcol = psi + col;

    // first-stage twiddles transposed for P points per thread: [P][N/P] (the plan keeps both layouts)
    const C *tw1x = P == 16 ? a.tw1_x : a.tw1e_x, *tw1y = P == 16 ? a.tw1_y : a.tw1e_y;
    FinalizeParams f = a.fin;
    f.call = &lcall;                                   // the member's state is passed as `&lms` where it is needed
    if (tid == 0) {
        lms = a.fin.st[b];
        lcall = *a.fin.call;
        if (rank != 0) lcall.records = nullptr;        // CTA 0 alone writes records
    }
    __syncthreads();

    C v[P];
#pragma unroll
    for (int k = 0; k < P; ++k) v[k] = __ldcg(prow + j + M1 * k);

    for (long step = 0; step < n_steps; ++step) {
        // ---- pass A: potential half-step (merged with the pending one in real time) and FFT along y
        {
            const bool pend = !IMAG && lms.pend;
            const T cx2 = (a.flags & F_CAV_FULL) ? a.cavx[i] * a.cavx[i] : T(0);
            T sn, st;
            potential_step16<T, IMAG, false, M1>(v, a, b, i, j, (T)lms.scale, pend ? T(2) : T(1), (T)(pend ? lms.A + lms.A_pend : lms.A),
                                                 (T)(pend ? lms.C + lms.C_pend : lms.C), (T)(pend ? lms.D + lms.D_pend : lms.D) * cx2, sn, st);
        }
        FR::fwd(v, smr, j, a.tw_y, tw1y);
#pragma unroll
        for (int ii = 0; ii < FR::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < FR::RL; ++rr) prow[FR::nat(j, ii, rr)] = v[ii * FR::RL + rr];
        cluster.sync();
        // ---- pass B: FFT along x, kinetic factor, inverse FFT along x on this CTA's columns
        if (tid == 0 && f.prepared) prepare_member(f, b, &lms);
#pragma unroll
        for (int k = 0; k < P; ++k) v[k] = __ldcg(pcol + (size_t)(jc + FC::M1 * k) * N);
        FC::fwd(v, smc, jc, a.tw_x, tw1x);
        if constexpr (IMAG) {
            const T ey = a.kin_yr[col];
#pragma unroll
            for (int ii = 0; ii < FC::GL; ++ii)
#pragma unroll
                for (int rr = 0; rr < FC::RL; ++rr) {
                    const T fk = a.kin_xr[FC::nat(jc, ii, rr)] * ey;
                    v[ii * FC::RL + rr].x *= fk;
                    v[ii * FC::RL + rr].y *= fk;
                }
        } else {
            // (1+a)(1+b)/P as v/P + v*g, g = a' + b' + a'b: see k_col (gpe_kernels.cuh)
            const C bq = a.kin_yc[col];
            const T invp = a.inv_p, cb = T(1) + bq.x;
            const C bp = mk<T>(bq.x * invp, bq.y * invp);
#pragma unroll
            for (int ii = 0; ii < FC::GL; ++ii)
#pragma unroll
                for (int rr = 0; rr < FC::RL; ++rr) {
                    const C ap = a.kin_xc[FC::nat(jc, ii, rr)];
                    const T gx = fma(ap.x, cb, fma(-ap.y, bq.y, bp.x));
                    const T gy = fma(ap.x, bq.y, fma(ap.y, cb, bp.y));
                    C &z = v[ii * FC::RL + rr];
                    const T ox = fma(z.x, gx, fma(-z.y, gy, z.x * invp));
                    const T oy = fma(z.x, gy, fma(z.y, gx, z.y * invp));
                    z.x = ox; z.y = oy;
                }
        }
        FC::inv(v, smc, jc, a.tw_x, tw1x);
#pragma unroll
        for (int k = 0; k < P; ++k) pcol[(size_t)(jc + FC::M1 * k) * N] = v[k];
        cluster.sync();
        // ---- pass C: inverse FFT along y, second half-step (left pending in real time), sums
#pragma unroll
        for (int ii = 0; ii < FR::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < FR::RL; ++rr) v[ii * FR::RL + rr] = __ldcg(prow + FR::nat(j, ii, rr));
        FR::inv(v, smr, j, a.tw_y, tw1y);
        T sn = T(0), st = T(0);
        if (!IMAG && f.merged) {
#pragma unroll
            for (int k = 0; k < P; ++k) {
                const T d = v[k].x * v[k].x + v[k].y * v[k].y;
                sn += d;
                if (a.flags & F_CAVITY) st = fma(d, a.ytab[4 * (j + M1 * k) + 2], st);
            }
        } else {
            potential_step16<T, IMAG, true, M1>(v, a, b, i, j, T(1), T(1), (T)lms.A, (T)lms.C,
                                                (a.flags & F_CAV_FULL) ? (T)lms.D * a.cavx[i] * a.cavx[i] : T(0), sn, st);
        }
        double dn = (double)sn, dth = (a.flags & F_CAVITY) ? (double)st * (double)a.cavx[i] : 0.0;
        double dbn = (a.flags & F_CAV_FULL) ? dn * ((double)a.cavx[i] * (double)a.cavx[i]) : 0.0;
        cta_sum3<G::THREADS>(dn, dth, dbn, red);
        if (tid == 0) {
#pragma unroll 1
            for (int q = 0; q < NC; ++q) {
                double *dst = cluster.map_shared_rank(&part[0][0], q) + 3 * rank;
                dst[0] = dn; dst[1] = dth; dst[2] = dbn;
            }
        }
        cluster.sync();
        if (tid == 0) {
            double t0 = 0.0, t1 = 0.0, t2 = 0.0;
            for (int q = 0; q < NC; ++q) { t0 += part[q][0]; t1 += part[q][1]; t2 += part[q][2]; }
            finalize_member(f, b, t0, t1, t2, &lms);
        }
        __syncthreads();
    }
#pragma unroll
    for (int k = 0; k < P; ++k) prow[j + M1 * k] = v[k];
    if (rank == 0 && tid == 0) a.fin.st[b] = lms;
}

// ---------------------------------------------------------------- launcher
template <typename T, int N> struct LaunchChip {
    using A = StepArgs<T, cx<T>>;
    using G = ChipGeom<T, N>;
    template <typename K> static cudaError_t setup(K kern) {
        cudaError_t e = cudaSuccess;
        if (G::SMEM > 48 * 1024) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM);
        if (e == cudaSuccess && G::NC > 8) e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        return e;
    }
    template <typename K> static cudaError_t go(K kern, const A &a, long n_steps, cudaStream_t s) {
        cudaError_t e = setup(kern);
        if (e != cudaSuccess) return e;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(a.batch * G::NC)); cfg.blockDim = dim3(G::THREADS);
        cfg.dynamicSmemBytes = G::SMEM; cfg.stream = s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = G::NC; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, kern, a, n_steps);
        return e != cudaSuccess ? e : cudaGetLastError();
    }
    // can a cluster of this shape be resident on the current device at all?
    static bool available() {
        auto kern = k_chip<T, N, false>;
        if (setup(kern) != cudaSuccess) { cudaGetLastError(); return false; }
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(G::NC); cfg.blockDim = dim3(G::THREADS); cfg.dynamicSmemBytes = G::SMEM;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = G::NC; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) { cudaGetLastError(); return false; }
        return n >= 1;
    }
    static cudaError_t run(const A &a, bool imag, long n_steps, cudaStream_t s) {
        return imag ? go(k_chip<T, N, true>, a, n_steps, s) : go(k_chip<T, N, false>, a, n_steps, s);
    }
};

}  // namespace gpe
