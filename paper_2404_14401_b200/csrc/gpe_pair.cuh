// gpe_pair.cuh -- the complex64 hot path: the three passes of gpe_kernels.cuh with every
// thread working on TWO complex numbers in lock step (element type cpair of gpe_fft.cuh), so that
// all butterfly and twiddle arithmetic is packed fp32x2 (FADD2 / FMUL2 / FFMA2 of sm_100), the
// shared-memory exchange moves whole lane pairs (two 64-bit planes) and every access to the
// intermediate array is 128 or 256 bits wide.
//
//   pass B (columns): the two lanes are two ADJACENT COLUMNS (two independent transforms).
//   pass A (rows):    the two lanes are the even and the odd half of ONE row transform: a
//                     decimation-in-frequency radix-2 layer, written with scalar instructions
//                     right after the potential half-step (which is scalar anyway and so converts
//                     the interleaved (re, im) input to the split lane layout for free), followed
//                     by two independent NY/2-point transforms.  Lane 0 ends with psi^[2k'],
//                     lane 1 with psi^[2k'+1]: exactly the column pair pass B wants.
//   pass C (rows):    the mirror of pass A.
// Intermediate layout (between A and C, inside the caller's psi buffer, same bytes per row pair):
//   [batch][nx/2][ny/2][2] of cpair; element (i, k') = (Re psi^[i][2k'], Re psi^[i][2k'+1], Im .., Im ..)
//   sits at ((i/2) * ny/2 + k') * 2 + i%2: rows 2m and 2m+1 are interleaved so that the column pass,
//   whose tile is only two column pairs wide, still moves 64 contiguous bytes per row pair
//   (measured on B200: 32-byte segments cost pass B 4 us of 35 at 2048^2).
// Same mathematics as gpe_kernels.cuh (PAPER.md:62-76 Eqs. 2-4, :116, :183-186 Eq. 14).
#pragma once
#include "gpe_kernels.cuh"

// exp of the imaginary-time potential factor: ex2.approx (relative error <= 2^-21 plus 1.2e-7 |w| from
// the argument scaling; |w| = |V + g|psi|^2| dtau / 2 is O(1e-2) on the paper's workloads) against the
// 1e-5 per step of the parity bar; measured on B200: config 5 197 -> 190 us per step, 2048^2 66.3 -> 63.6
#ifndef GPE_EXPF
#define GPE_EXPF __expf
#endif
#ifndef GPE_ROWP_THREADS
#define GPE_ROWP_THREADS 64    // measured: 64 / 128 beat 128 / 256 below 2048 (more, smaller CTAs fill the 148 SMs)
#endif
#ifndef GPE_ROWP_MINB
#define GPE_ROWP_MINB 4         // 128-thread row CTAs per SM the row passes are compiled for (3 and 5 measured slower)
#endif
#ifndef GPE_COLP_RESIDENT
#define GPE_COLP_RESIDENT 512   // threads per SM the column pass is compiled for (128 registers each)
#endif
#ifndef GPE_COLP_THREADS
#define GPE_COLP_THREADS 128   // threads per column CTA where the transform allows (2048: 256 = two column pairs)
#endif

namespace gpe {

template <int N> struct RowGeomP {
    static constexpr int H = N / 2;
    static constexpr int TPF = H / 16;                               // threads per row
    static constexpr int RPC = (GPE_ROWP_THREADS / TPF) < 2 ? 2 : (GPE_ROWP_THREADS / TPF);    // rows per CTA (>= one row pair)
    static constexpr int THREADS = RPC * TPF;                        // 128 at 2048, 64 below
    static constexpr bool NAMED = RPC > 1 && TPF % 32 == 0;          // rows own whole warps
    // outer stage pair-mapped (Fft1D::last_fwd_pair): a thread holds the same output indices of rows
    // 2m and 2m+1, i.e. 32 contiguous bytes of the row-pair-interleaved intermediate array
    static constexpr bool PAIRMAP = RPC >= 2 && (16 / (Fact<H>::R3 > 1 ? Fact<H>::R3 : Fact<H>::R2)) >= 2;
    static constexpr bool PAIRNAMED = RPC > 2 && (2 * TPF) % 32 == 0;  // a row pair owns whole warps
};
template <int N> struct ColGeomP {
    static constexpr int TPF = N / 16;                               // threads per column pair
    static constexpr int CPW0 = GPE_COLP_THREADS / TPF;
    // column pairs per CTA; 2048: ONE (128 threads, 1024 CTAs: 6.92 per SM, at most 7 -- two pairs per
    // CTA gave 512 CTAs, 3 on 80 SMs and 4 on 68, and the pass waited for the 68: 27.4 against 21 us)
    static constexpr int CPW = CPW0 < 2 ? (N >= GPE_IL4_MIN_N ? 1 : 2) : CPW0;
    static constexpr int THREADS = CPW * TPF;
};

__device__ __forceinline__ void bar_named(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ cpair ldcg_pair(const cpair *p) {
    const float4 t = __ldcg(reinterpret_cast<const float4 *>(p));
    cpair r; r.re = make_float2(t.x, t.y); r.im = make_float2(t.z, t.w); return r;
}
__device__ __forceinline__ void st_pair(cpair *p, cpair v) {
    *reinterpret_cast<float4 *>(p) = make_float4(v.re.x, v.re.y, v.im.x, v.im.y);
}

// 256-bit accesses (sm_100): the two cpairs of one column pair of rows 2m and 2m+1, 32 contiguous bytes
__device__ __forceinline__ void st_pair2(cpair *p, cpair v0, cpair v1) {
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(v0.re.x), "f"(v0.re.y), "f"(v0.im.x),
                 "f"(v0.im.y), "f"(v1.re.x), "f"(v1.re.y), "f"(v1.im.x), "f"(v1.im.y) : "memory");
}
__device__ __forceinline__ void ldcg_pair2(const cpair *p, cpair &v0, cpair &v1) {
    asm volatile("ld.global.cg.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];" : "=f"(v0.re.x), "=f"(v0.re.y), "=f"(v0.im.x),
                 "=f"(v0.im.y), "=f"(v1.re.x), "=f"(v1.re.y), "=f"(v1.im.x), "=f"(v1.im.y) : "l"(p) : "memory");
}

// position of element (row i, column pair kp) of the intermediate array, hy = ny/2 (rows counted
// through the whole batch: nx is even, so a row pair never straddles two members)
// il = log2 of the number of interleaved rows: 1, or 2 when nx and ny >= GPE_IL4_MIN_N (il_of)
__device__ __forceinline__ size_t ipos(long i, int kp, size_t hy, int il) { return (((size_t)(i >> il) * hy + kp) << il) + (i & ((1 << il) - 1)); }
// N = the kernel's own compile-time axis length, other = the other one: both must reach GPE_IL4_MIN_N
// single grids only: the out-of-place passes double the footprint, and two 2048^2 grids no longer fit in L2
template <int N> __device__ __forceinline__ int il_of(int other, int batch) { return (N >= GPE_IL4_MIN_N && other >= GPE_IL4_MIN_N && batch == 1) ? 2 : 1; }

// Potential half-step (rows a1 / a5) on the 32 points of one thread: p0[k] at y = j + M1 k,
// p1[k] at y + H, same row i.  ytab2[n] = {vy[n], vy[n+H], cos^2(k_l y_n), cos^2(k_l y_{n+H})},
// {cos(k_c y_n), cos(k_c y_{n+H}), 0, 0}.  The angle and its polynomial are packed over the two
// points; |psi|^2 and the final rotation are scalar (they read / write the interleaved layout).
// REDUCE: sn += |psi_new|^2, st += cos(k_c y) |psi_new|^2 (one lane per point).
template <bool IMAG, bool REDUCE, int M1, int H>
__device__ __forceinline__ void potential_pair16(float2 (&p0)[16], float2 (&p1)[16], const StepArgs<float, float2> &a,
                                                 int b, int i, int j, float scale, float fac, float A, float Cc,
                                                 float vadd, float2 &sn, float2 &st) {
    const int flags = a.flags;
    float vrow = vadd;   // per-row constant from the caller: cavity lattice D cos^2(k_c x_i) (Eq. 12)
    // fac = 1, or 2 when this multiply also carries the pending second half-step of the previous
    // step (then A, Cc are the sums of the two steps' coefficients): static terms and g count twice
    if (flags & F_HAS_SEP) vrow += fac * a.vx[i];
    if (flags & F_LAT_X) vrow += A * a.latx[i];
    const float crow = (flags & F_CAVITY) ? Cc * a.cavx[i] : 0.f;
    const float Ay = (flags & F_LAT_Y) ? A : 0.f;
    const float g = (flags & F_HAS_G) ? fac * a.g[b] : 0.f;
    const float hdt = a.half_dt;
    const float4 *__restrict__ yt = reinterpret_cast<const float4 *>(a.ytab2);
    // in chunks of CH points per half row: bounds the live angles (registers); the tier vote is per chunk
    constexpr int CH = 8;
#pragma unroll
    for (int k0 = 0; k0 < 16; k0 += CH) {
        float2 w[16];   // only the CH entries of the current chunk are live
    #pragma unroll
        for (int k = k0; k < k0 + CH; ++k) {
            const int n = j + M1 * k;
            const float4 t0 = ldtw(yt, 2 * n);
            const float2 cav = ldtw(reinterpret_cast<const float2 *>(yt), 4 * n + 2);
            if constexpr (IMAG) { p0[k].x *= scale; p0[k].y *= scale; p1[k].x *= scale; p1[k].y *= scale; }
            const float2 d = make_float2(fmaf(p0[k].x, p0[k].x, p0[k].y * p0[k].y), fmaf(p1[k].x, p1[k].x, p1[k].y * p1[k].y));
            const float2 V = rfmas(cav, crow, rfmas(make_float2(t0.z, t0.w), Ay, rfmas(make_float2(t0.x, t0.y), fac, make_float2(vrow, vrow))));
            w[k] = rmuls(rfmas(d, g, V), hdt);
        }
        if (flags & F_HAS_V2D) {
            const float *__restrict__ v2 = a.v2d + ((flags & F_V2D_BATCHED) ? (size_t)b * a.nx * a.ny : 0) + (size_t)i * a.ny;
    #pragma unroll
            for (int k = k0; k < k0 + CH; ++k) w[k] = rfmas(make_float2(v2[j + M1 * k], v2[j + M1 * k + H]), fac * hdt, w[k]);
        }
        if constexpr (IMAG) {
    #pragma unroll
            for (int k = k0; k < k0 + CH; ++k) {
                const float e0 = GPE_EXPF(-w[k].x), e1 = GPE_EXPF(-w[k].y);
                p0[k].x *= e0; p0[k].y *= e0; p1[k].x *= e1; p1[k].y *= e1;
            }
        } else {
            // psi <- psi + psi * (cos w - 1 - i sin w); warp-uniform tiers by the largest |w| (see
            // potential_step16 in gpe_kernels.cuh for the polynomials and why the "minus one" form).
            float wmax = 0.f;
    #pragma unroll
            for (int k = k0; k < k0 + CH; ++k) wmax = fmaxf(wmax, fmaxf(fabsf(w[k].x), fabsf(w[k].y)));
            auto rotate = [&](int k, float2 sn_, float2 cm1) {
                const float ax = fmaf(p0[k].x, cm1.x, fmaf(-p0[k].y, sn_.x, p0[k].x));
                const float ay = fmaf(p0[k].x, sn_.x, fmaf(p0[k].y, cm1.x, p0[k].y));
                const float bx = fmaf(p1[k].x, cm1.y, fmaf(-p1[k].y, sn_.y, p1[k].x));
                const float by = fmaf(p1[k].x, sn_.y, fmaf(p1[k].y, cm1.y, p1[k].y));
                p0[k] = make_float2(ax, ay); p1[k] = make_float2(bx, by);
            };
            if (__all_sync(0xffffffffu, wmax <= 0.03125f)) {
    #pragma unroll
                for (int k = k0; k < k0 + CH; ++k) {
                    const float2 w2 = rmul(w[k], w[k]);
                    const float2 sn_ = rneg(rfmas(rmul(w[k], w2), -1.6666667e-1f, w[k]));   // sin(-w)
                    const float2 cm1 = rmul(w2, rfmas(w2, 4.1666667e-2f, make_float2(-0.5f, -0.5f)));
                    rotate(k, sn_, cm1);
                }
            } else if (__all_sync(0xffffffffu, wmax <= 0.5f)) {
    #pragma unroll
                for (int k = k0; k < k0 + CH; ++k) {
                    float2 sn_, cm1;
                    sincosm1_small(-w[k].x, &sn_.x, &cm1.x);
                    sincosm1_small(-w[k].y, &sn_.y, &cm1.y);
                    rotate(k, sn_, cm1);
                }
            } else {
    #pragma unroll
                for (int k = k0; k < k0 + CH; ++k) {
                    float2 sn_, cm1;
                    sincosm1_general(-w[k].x, &sn_.x, &cm1.x);
                    sincosm1_general(-w[k].y, &sn_.y, &cm1.y);
                    rotate(k, sn_, cm1);
                }
            }
        }
    }
    if constexpr (REDUCE) {
        sn = make_float2(0.f, 0.f); st = make_float2(0.f, 0.f);
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const float2 d = make_float2(fmaf(p0[k].x, p0[k].x, p0[k].y * p0[k].y), fmaf(p1[k].x, p1[k].x, p1[k].y * p1[k].y));
            sn = radd(sn, d);
            if (flags & F_CAVITY) st = rfma(d, *reinterpret_cast<const float2 *>(yt + 2 * (j + M1 * k) + 1), st);
        }
    }
}

// sums only (merged real-time half-steps: pass C leaves the multiply to the next pass A; a phase
// factor does not change |psi|^2, so norm and Theta of the stored array are those of psi_{n+1})
template <int M1>
__device__ __forceinline__ void reduce_pair16(const float2 (&p0)[16], const float2 (&p1)[16], const StepArgs<float, float2> &a,
                                              int j, float2 &sn, float2 &st) {
    const float4 *__restrict__ yt = reinterpret_cast<const float4 *>(a.ytab2);
    sn = make_float2(0.f, 0.f); st = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const float2 d = make_float2(fmaf(p0[k].x, p0[k].x, p0[k].y * p0[k].y), fmaf(p1[k].x, p1[k].x, p1[k].y * p1[k].y));
        sn = radd(sn, d);
        if (a.flags & F_CAVITY) st = rfma(d, *reinterpret_cast<const float2 *>(yt + 2 * (j + M1 * k) + 1), st);
    }
}

// ---------------------------------------------------------------- pass A (rows, forward)
template <int NY, bool IMAG, bool LATE>
__global__ void __launch_bounds__(RowGeomP<NY>::THREADS, (GPE_ROWP_MINB * 128) / RowGeomP<NY>::THREADS) k_row_fwd_p(const StepArgs<float, float2> a) {
    using G = RowGeomP<NY>;
    using F = Fft1D<G::H, 1, cpair>;
    constexpr int H = G::H, M1 = F::M1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    float2 *sm = reinterpret_cast<float2 *>(smem_raw) + r * F::TILE;
    const long row = (long)blockIdx.x * G::RPC + r;
    const int b = (int)(row / a.nx), i = (int)(row % a.nx), il = il_of<NY>(a.nx, a.batch);
    const float2 *src = a.src + row * NY;
    if constexpr (!LATE) pdl_launch_dependents();
    pdl_wait();
    float2 p0[16], p1[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        p0[k] = __ldcg(src + j + M1 * k); p1[k] = __ldcg(src + H + j + M1 * k);
    }
    {
        const MemberState &ms = a.fin.st[b];
        float2 sn, st;
        const bool pend = !IMAG && ms.pend;
        const float cx2 = (a.flags & F_CAV_FULL) ? a.cavx[i] * a.cavx[i] : 0.f;
        potential_pair16<IMAG, false, M1, H>(p0, p1, a, b, i, j, (float)ms.scale, pend ? 2.f : 1.f,
                                             (float)(pend ? ms.A + ms.A_pend : ms.A), (float)(pend ? ms.C + ms.C_pend : ms.C),
                                             (float)(pend ? ms.D + ms.D_pend : ms.D) * cx2, sn, st);
    }
    // radix-2 decimation in frequency across the two halves of the row: lane 0 <- x[n] + x[n+H],
    // lane 1 <- (x[n] - x[n+H]) w_NY^n; scalar instructions, they write the split lane layout
    cpair v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const float2 w = ldtw(a.tw_y, j + M1 * k);
        const float dx = p0[k].x - p1[k].x, dy = p0[k].y - p1[k].y;
        v[k].re = make_float2(p0[k].x + p1[k].x, fmaf(dx, w.x, -(dy * w.y)));
        v[k].im = make_float2(p0[k].y + p1[k].y, fmaf(dx, w.y, dy * w.x));
    }
    cpair *dst = reinterpret_cast<cpair *>(a.dst);
    if constexpr (G::PAIRMAP) {
        const int rp = r >> 1, u = j + (r & 1) * G::TPF;
        float2 *sm0 = reinterpret_cast<float2 *>(smem_raw) + (2 * rp) * F::TILE, *sm1 = sm0 + F::TILE;
        // every barrier spans the row pair: its first one also orders the pair's loads before its stores
        auto sync_row = [r] { if constexpr (G::NAMED) bar_named(1 + r, G::TPF); else __syncthreads(); };
        auto sync_pair = [rp] { if constexpr (G::PAIRNAMED) bar_named(9 + rp, 2 * G::TPF); else __syncthreads(); };
        F::fwd_pairlast(v, sm, sm0, sm1, j, u, a.tw_hy, a.tw1_hy, sync_row, sync_pair);
        const long rowp = (long)blockIdx.x * G::RPC + 2 * rp;
#pragma unroll
        for (int ii = 0; ii < F::GL / 2; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                const size_t pos = ipos(rowp, F::nat_t(u + 2 * G::TPF * ii, rr), H, il);
                st_pair2(dst + pos, v[(2 * ii) * F::RL + rr], v[(2 * ii + 1) * F::RL + rr]);
            }
    } else {
        // the rows of a pair are interleaved in the output: no store before every row's loads are done
        if (G::RPC > 1) __syncthreads();
        if constexpr (G::NAMED) F::fwd(v, sm, j, a.tw_hy, a.tw1_hy, [r] { bar_named(1 + r, G::TPF); });
        else F::fwd(v, sm, j, a.tw_hy, a.tw1_hy, [] { __syncthreads(); });
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) st_pair(dst + ipos(row, F::nat(j, ii, rr), H, il), v[ii * F::RL + rr]);
    }
    // after the CTA's last store, and only when asked for: even without the launch attribute the
    // instruction is not free after a burst of stores (measured: config 5 +6 us, 16 x 1024^2 +13 us per step)
    if constexpr (LATE) pdl_launch_dependents();
}

// ---------------------------------------------------------------- pass B (columns)
// KNORM (imaginary time, T/2 V T/2 with merged kinetic halves): the tables hold HALF a kinetic step h; the factor is
// applied twice and the k-space sum of |psi^ h / P|^2 taken in between (Parseval: the norm of the wavefunction at the
// step boundary, FinalizeParams::partials_k)
template <int NX, bool IMAG, bool LATE, bool KNORM = false>
__global__ void __launch_bounds__(ColGeomP<NX>::THREADS, GPE_COLP_RESIDENT / ColGeomP<NX>::THREADS) k_col_p(const StepArgs<float, float2> a) {
    using G = ColGeomP<NX>;
    using F = Fft1D<NX, G::CPW, cpair>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int c = threadIdx.x % G::CPW, j = threadIdx.x / G::CPW;
    const int cp = blockIdx.x * G::CPW + c;      // column pair: columns 2 cp, 2 cp + 1
    const int b = blockIdx.y;
    const size_t hy = a.ny / 2;
    // rows j + M1 k, k = 0..15 (M1 even): ipos(j + M1 k, cp) = ipos(j, cp) + k * M1 * hy
    const size_t base = (size_t)b * NX * hy + ipos(j, cp, hy, il_of<NX>(a.ny, a.batch)), kstr = (size_t)F::M1 * hy;
    const cpair *src = reinterpret_cast<const cpair *>(a.src) + base;
    cpair *dst = reinterpret_cast<cpair *>(a.dst) + base;
    float2 *sm = reinterpret_cast<float2 *>(smem_raw) + c;
    cpair v[16];
    if constexpr (!LATE) pdl_launch_dependents();
    pdl_wait();
    if (blockIdx.x == 0 && threadIdx.x == 0 && a.fin.prepared) prepare_member(a.fin, b);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        v[k] = ldcg_pair(src + k * kstr);
    }
    F::fwd(v, sm, j, a.tw_x, a.tw1_x);
    if constexpr (IMAG) {
        const float2 ey = *reinterpret_cast<const float2 *>(a.kin_yr + 2 * cp);
        float2 acc = make_float2(0.f, 0.f);
        const float bigp = 1.0f / a.inv_p;   // nx ny: a power of two, exact
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                const float2 f = rmuls(ey, a.kin_xr[F::nat(j, ii, rr)]);
                cpair &z = v[ii * F::RL + rr];
                z.re = rmul(z.re, f); z.im = rmul(z.im, f);
                if constexpr (KNORM) {
                    acc = rfma(z.re, z.re, rfma(z.im, z.im, acc));
                    const float2 f2 = rmuls(f, bigp);
                    z.re = rmul(z.re, f2); z.im = rmul(z.im, f2);
                }
            }
        if constexpr (KNORM) {
            __shared__ double redk[32];
            const double s = warp_sum((double)acc.x + (double)acc.y);
            if ((threadIdx.x & 31) == 0) redk[threadIdx.x >> 5] = s;
            __syncthreads();
            if (threadIdx.x == 0) {
                double t = 0.0;
                for (int q = 0; q < G::THREADS / 32; ++q) t += redk[q];
                a.fin.partials_k[(size_t)b * a.fin.cpmk + blockIdx.x] = t;
            }
        }
    } else {
        // kinetic factor (1+a)(1+b)/P applied as v/P + v*g, g = a' + b' + a'b (k_col of
        // gpe_kernels.cuh); b differs between the two columns (lanes), a is common to both
        // (kin_y2: the per-column constants in split lane layout, so no register shuffling is needed)
        const float4 k0 = ldtw(reinterpret_cast<const float4 *>(a.kin_y2), 2 * cp), k1 = ldtw(reinterpret_cast<const float4 *>(a.kin_y2), 2 * cp + 1);
        const float2 cb = make_float2(k0.x, k0.y), bqy = make_float2(k0.z, k0.w), bpx = make_float2(k1.x, k1.y), bpy = make_float2(k1.z, k1.w);
        const float invp = a.inv_p;
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                const float2 ap = ldtw(a.kin_xc, F::nat(j, ii, rr));
                const float2 gx = rfmas(cb, ap.x, rfmas(bqy, -ap.y, bpx));
                const float2 gy = rfmas(bqy, ap.x, rfmas(cb, ap.y, bpy));
                cpair &z = v[ii * F::RL + rr];
                const float2 ox = rfma(z.re, gx, rfma(rneg(z.im), gy, rmuls(z.re, invp)));
                const float2 oy = rfma(z.re, gy, rfma(z.im, gx, rmuls(z.im, invp)));
                z.re = ox; z.im = oy;
            }
    }
    F::inv(v, sm, j, a.tw_x, a.tw1_x);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        st_pair(dst + k * kstr, v[k]);
    }
    if constexpr (LATE) pdl_launch_dependents();
}

// ---------------------------------------------------------------- pass C (rows, inverse)
template <int NY, bool IMAG, bool MERGED, bool LATE>
__global__ void __launch_bounds__(RowGeomP<NY>::THREADS, (GPE_ROWP_MINB * 128) / RowGeomP<NY>::THREADS) k_row_inv_p(const StepArgs<float, float2> a) {
    using G = RowGeomP<NY>;
    using F = Fft1D<G::H, 1, cpair>;
    constexpr int H = G::H, M1 = F::M1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[128];
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    float2 *sm = reinterpret_cast<float2 *>(smem_raw) + r * F::TILE;
    const long row = (long)blockIdx.x * G::RPC + r;
    const int b = (int)(row / a.nx), i = (int)(row % a.nx), il = il_of<NY>(a.nx, a.batch);
    const int gpm = a.nx / G::RPC;
    const cpair *src = reinterpret_cast<const cpair *>(a.src);
    if constexpr (!LATE) pdl_launch_dependents();
    pdl_wait();
    cpair v[16];
    if constexpr (G::PAIRMAP) {
        // mirror of pass A: 32 contiguous bytes (rows 2m, 2m+1, same column pair) per thread and index
        const int rp = r >> 1, u = j + (r & 1) * G::TPF;
        float2 *sm0 = reinterpret_cast<float2 *>(smem_raw) + (2 * rp) * F::TILE, *sm1 = sm0 + F::TILE;
        const long rowp = (long)blockIdx.x * G::RPC + 2 * rp;
#pragma unroll
        for (int ii = 0; ii < F::GL / 2; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                const size_t pos = ipos(rowp, F::nat_t(u + 2 * G::TPF * ii, rr), H, il);
                ldcg_pair2(src + pos, v[(2 * ii) * F::RL + rr], v[(2 * ii + 1) * F::RL + rr]);
            }
        auto sync_row = [r] { if constexpr (G::NAMED) bar_named(1 + r, G::TPF); else __syncthreads(); };
        auto sync_pair = [rp] { if constexpr (G::PAIRNAMED) bar_named(9 + rp, 2 * G::TPF); else __syncthreads(); };
        F::inv_pairfirst(v, sm, sm0, sm1, j, u, a.tw_hy, a.tw1_hy, sync_row, sync_pair);
    } else {
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                v[ii * F::RL + rr] = ldcg_pair(src + ipos(row, F::nat(j, ii, rr), H, il));
            }
        if constexpr (G::NAMED) F::inv(v, sm, j, a.tw_hy, a.tw1_hy, [r] { bar_named(1 + r, G::TPF); });
        else F::inv(v, sm, j, a.tw_hy, a.tw1_hy, [] { __syncthreads(); });
    }
    // mirror of pass A's radix-2 layer: x[n] = e[n] + conj(w^n) o[n], x[n+H] = e[n] - conj(w^n) o[n]
    float2 p0[16], p1[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const float2 w = ldtw(a.tw_y, j + M1 * k);
        const float tx = fmaf(v[k].re.y, w.x, v[k].im.y * w.y), ty = fmaf(v[k].im.y, w.x, -(v[k].re.y * w.y));
        p0[k] = make_float2(v[k].re.x + tx, v[k].im.x + ty);
        p1[k] = make_float2(v[k].re.x - tx, v[k].im.x - ty);
    }
    const MemberState &ms = a.fin.st[b];
    float2 sn = make_float2(0.f, 0.f), st = sn;
    if constexpr (MERGED) reduce_pair16<M1>(p0, p1, a, j, sn, st);
    else potential_pair16<IMAG, true, M1, H>(p0, p1, a, b, i, j, 1.f, 1.f, (float)ms.A, (float)ms.C,
                                             (a.flags & F_CAV_FULL) ? (float)ms.D * a.cavx[i] * a.cavx[i] : 0.f, sn, st);
    float2 *dst = a.dst + row * NY;
    // Reduction first, wavefunction stores second: the partial sums of this CTA are published
    // (store, fence, counter increment) while thread 0 has no stores in flight, so the fence does
    // not wait for 16 KB of psi to be acknowledged by L2, and the counter's round trip overlaps
    // the stores.  Fixed summation order everywhere (bitwise reproducible, batch == single).
    const FinalizeParams &f = a.fin;
    const int cim = (int)(blockIdx.x % gpm);
    const double rown = (double)sn.x + (double)sn.y;
    double dn = warp_sum(rown);
    double dt_ = (a.flags & F_CAVITY) ? warp_sum(((double)st.x + (double)st.y) * (double)a.cavx[i]) : 0.0;
    const bool full = a.flags & F_CAV_FULL;   // third sum: cos^2(k_c x_i) times the row's |psi|^2 (Eq. 15)
    double db_ = full ? warp_sum(rown * ((double)a.cavx[i] * (double)a.cavx[i])) : 0.0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    constexpr int NW = G::THREADS / 32;
    __shared__ int is_last;
    if (lane == 0) { red[wid] = dn; red[32 + wid] = dt_; red[64 + wid] = db_; }
    __syncthreads();
    unsigned int old = 0;
    if (threadIdx.x == 0) {
        double s0 = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll
        for (int q = 0; q < NW; ++q) { s0 += red[q]; s1 += red[32 + q]; s2 += red[64 + q]; }
        f.partials[(size_t)b * f.cpm + cim] = make_double2(s0, s1);
        if (full) f.partials_b[(size_t)b * f.cpm + cim] = s2;
        __threadfence();
        old = atomicAdd(&f.counters[b], 1u);
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) { dst[j + M1 * k] = p0[k]; dst[H + j + M1 * k] = p1[k]; }
    if constexpr (LATE) pdl_launch_dependents();
    if (threadIdx.x == 0) is_last = (old == (unsigned int)(f.cpm - 1));
    __syncthreads();
    if (is_last) {   // the last CTA of the member: all its threads sum the partials
        __threadfence();
        const volatile double2 *pp = f.partials + (size_t)b * f.cpm;
        double s0 = 0.0, s1 = 0.0, s2 = 0.0;
        for (int q = threadIdx.x; q < f.cpm; q += G::THREADS) { s0 += pp[q].x; s1 += pp[q].y; }
        if (full) {
            const volatile double *pb = f.partials_b + (size_t)b * f.cpm;
            for (int q = threadIdx.x; q < f.cpm; q += G::THREADS) s2 += pb[q];
            s2 = warp_sum(s2);
        }
        s0 = warp_sum(s0); s1 = warp_sum(s1);
        double s3 = 0.0;
        if (f.knorm) {   // the norm from pass B's k-space partial sums (merged kinetic halves, see k_col_p)
            const double *pk = f.partials_k + (size_t)b * f.cpmk;
            for (int q = threadIdx.x; q < f.cpmk; q += G::THREADS) s3 += __ldcg(pk + q);
            s3 = warp_sum(s3);
        }
        __syncthreads();
        if (lane == 0) { red[wid] = s0; red[32 + wid] = s1; red[64 + wid] = s2; red[96 + wid] = s3; }
        __syncthreads();
        if (threadIdx.x == 0) {
            double t0 = 0.0, t1 = 0.0, t2 = 0.0, t3 = 0.0;
#pragma unroll
            for (int q = 0; q < NW; ++q) { t0 += red[q]; t1 += red[32 + q]; t2 += red[64 + q]; t3 += red[96 + q]; }
            finalize_member(f, b, f.knorm ? t3 * f.kscale : t0, t1, t2);
            f.counters[b] = 0u;
        }
    }
}

// ---------------------------------------------------------------- pass C of step n fused with pass A of step n+1
// The 2-pass form of SURVEY.md 8(a): when the potential factor between two kinetic steps needs no global
// scalar of the array it acts on, the rows never leave the SM between the inverse transform along y of
// step n and the forward transform along y of step n+1:
//   load (intermediate layout) -> IFFT_y -> partial sums of |psi|^2 -> psi *= exp(-s (V_n + V_{n+1} + 2 g|psi|^2) dt/2)
//   -> FFT_y -> store (intermediate layout, in place).
//   real time, no cavity term (a phase leaves |psi|^2 alone, and without Eq. 14 nothing else
//     couples the points): both half-steps in one multiply, exactly the merged multiply of pass A;
//   imaginary time with g = 0 and no cavity term (the paper's own benchmark workload): the
//     step is linear, so the renormalisation of PAPER.md:116 commutes with it.  The 1/||psi|| applied here is the
//     one of the PREVIOUS step (it only keeps the magnitudes near one); the last step of every gpe_evolve is the
//     plain pass C, whose norm and final rescale are exact.
// A_n is the member's current coefficient, A_{n+1} the one prepare_member left in nA during pass B; both are
// read BEFORE this CTA publishes its partial sums, because the last CTA to publish advances the member's state.
template <int NY, bool IMAG, bool LATE>
__global__ void __launch_bounds__(RowGeomP<NY>::THREADS, (GPE_ROWP_MINB * 128) / RowGeomP<NY>::THREADS) k_row_ca_p(const StepArgs<float, float2> a) {
    using G = RowGeomP<NY>;
    using F = Fft1D<G::H, 1, cpair>;
    constexpr int H = G::H, M1 = F::M1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[96];
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    float2 *sm = reinterpret_cast<float2 *>(smem_raw) + r * F::TILE;
    const long row = (long)blockIdx.x * G::RPC + r;
    const int b = (int)(row / a.nx), i = (int)(row % a.nx), il = il_of<NY>(a.nx, a.batch);
    const int gpm = a.nx / G::RPC;
    const cpair *src = reinterpret_cast<const cpair *>(a.src);
    cpair *dst = reinterpret_cast<cpair *>(a.dst);
    if constexpr (!LATE) pdl_launch_dependents();
    pdl_wait();
    const MemberState &ms = a.fin.st[b];
    const float Asum = (float)(ms.A + ms.nA), scale = (float)ms.scale;
    cpair v[16];
    const int rp = r >> 1, u = j + (r & 1) * G::TPF;
    float2 *sm0 = reinterpret_cast<float2 *>(smem_raw) + (2 * rp) * F::TILE, *sm1 = sm0 + F::TILE;
    const long rowp = (long)blockIdx.x * G::RPC + 2 * rp;
    auto sync_row = [r] { if constexpr (G::NAMED) bar_named(1 + r, G::TPF); else __syncthreads(); };
    auto sync_pair = [rp] { if constexpr (G::PAIRNAMED) bar_named(9 + rp, 2 * G::TPF); else __syncthreads(); };
    if constexpr (G::PAIRMAP) {
#pragma unroll
        for (int ii = 0; ii < F::GL / 2; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                const size_t pos = ipos(rowp, F::nat_t(u + 2 * G::TPF * ii, rr), H, il);
                ldcg_pair2(src + pos, v[(2 * ii) * F::RL + rr], v[(2 * ii + 1) * F::RL + rr]);
            }
        F::inv_pairfirst(v, sm, sm0, sm1, j, u, a.tw_hy, a.tw1_hy, sync_row, sync_pair);
    } else {
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) v[ii * F::RL + rr] = ldcg_pair(src + ipos(row, F::nat(j, ii, rr), H, il));
        if constexpr (G::NAMED) F::inv(v, sm, j, a.tw_hy, a.tw1_hy, [r] { bar_named(1 + r, G::TPF); });
        else F::inv(v, sm, j, a.tw_hy, a.tw1_hy, [] { __syncthreads(); });
    }
    float2 p0[16], p1[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const float2 w = ldtw(a.tw_y, j + M1 * k);
        const float tx = fmaf(v[k].re.y, w.x, v[k].im.y * w.y), ty = fmaf(v[k].im.y, w.x, -(v[k].re.y * w.y));
        p0[k] = make_float2(v[k].re.x + tx, v[k].im.x + ty);
        p1[k] = make_float2(v[k].re.x - tx, v[k].im.x - ty);
    }
    // partial sums of the array as it stands (norm of psi_{n+1} in real time; records), published at once
    float2 sn, st;
    reduce_pair16<M1>(p0, p1, a, j, sn, st);
    const FinalizeParams &f = a.fin;
    const int cim = (int)(blockIdx.x % gpm);
    double dn = warp_sum((double)sn.x + (double)sn.y);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    constexpr int NW = G::THREADS / 32;
    __shared__ int is_last;
    if (lane == 0) red[wid] = dn;
    __syncthreads();
    unsigned int old = 0;
    if (threadIdx.x == 0) {
        double s0 = 0.0;
#pragma unroll
        for (int q = 0; q < NW; ++q) s0 += red[q];
        f.partials[(size_t)b * f.cpm + cim] = make_double2(s0, 0.0);
        __threadfence();
        old = atomicAdd(&f.counters[b], 1u);
    }
    // both potential half-steps in one multiply, then pass A's radix-2 layer and forward transform
    {
        float2 dn_, dt_;
        potential_pair16<IMAG, false, M1, H>(p0, p1, a, b, i, j, scale, 2.f, Asum, 0.f, 0.f, dn_, dt_);
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const float2 w = ldtw(a.tw_y, j + M1 * k);
        const float dx = p0[k].x - p1[k].x, dy = p0[k].y - p1[k].y;
        v[k].re = make_float2(p0[k].x + p1[k].x, fmaf(dx, w.x, -(dy * w.y)));
        v[k].im = make_float2(p0[k].y + p1[k].y, fmaf(dx, w.y, dy * w.x));
    }
    if constexpr (G::PAIRMAP) {
        F::fwd_pairlast(v, sm, sm0, sm1, j, u, a.tw_hy, a.tw1_hy, sync_row, sync_pair);
#pragma unroll
        for (int ii = 0; ii < F::GL / 2; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                const size_t pos = ipos(rowp, F::nat_t(u + 2 * G::TPF * ii, rr), H, il);
                st_pair2(dst + pos, v[(2 * ii) * F::RL + rr], v[(2 * ii + 1) * F::RL + rr]);
            }
    } else {
        // in place: every row of the CTA was loaded before the first barrier of the inverse transform
        if constexpr (G::NAMED) F::fwd(v, sm, j, a.tw_hy, a.tw1_hy, [r] { bar_named(1 + r, G::TPF); });
        else F::fwd(v, sm, j, a.tw_hy, a.tw1_hy, [] { __syncthreads(); });
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) st_pair(dst + ipos(row, F::nat(j, ii, rr), H, il), v[ii * F::RL + rr]);
    }
    if constexpr (LATE) pdl_launch_dependents();
    if (threadIdx.x == 0) is_last = (old == (unsigned int)(f.cpm - 1));
    __syncthreads();
    if (is_last) {
        __threadfence();
        const volatile double2 *pp = f.partials + (size_t)b * f.cpm;
        double s0 = 0.0;
        for (int q = threadIdx.x; q < f.cpm; q += G::THREADS) s0 += pp[q].x;
        s0 = warp_sum(s0);
        __syncthreads();
        if (lane == 0) red[wid] = s0;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t0 = 0.0;
#pragma unroll
            for (int q = 0; q < NW; ++q) t0 += red[q];
            finalize_member(f, b, t0, 0.0, 0.0);
            f.counters[b] = 0u;
        }
    }
}

// ---------------------------------------------------------------- launchers
template <int N> struct LaunchP {
    using A = StepArgs<float, float2>;
    static size_t row_smem() { return sizeof(float2) * RowGeomP<N>::RPC * Fft1D<N / 2, 1, cpair>::TILE; }
    static size_t col_smem() { return sizeof(float2) * Fft1D<N, ColGeomP<N>::CPW, cpair>::TILE; }
    // launch-bound grids (<= 256^2 points): release the dependent launch at the top (measured on B200)
    static bool use_pdl(const A &a) { return (long)a.batch * a.nx * a.ny <= 65536L; }
    // Where a pass releases its dependent launch (programmatic dependent launch, gpe_kernels.cuh):
    // at the top for launch-bound grids (<= 256^2 points), after its last store -- a compile-time
    // variant, LATE -- for single grids of a wave or two (measured on B200, us per step: 512^2 17.4 -> 16.3,
    // 1024^2 23.0 -> 22.1, 2048^2 57.2 -> 56.4; released at the top these sizes lose 4-5 us), and not at
    // all for batches of many waves.  The instruction after the stores is not free even when predicated
    // off at run time (config 5: +6 us per step), hence the template parameter.
    static bool late(const A &a) {
        const long pts = (long)a.batch * a.nx * a.ny;
        return pts > 65536L && pts < (1L << 23);
    }
    template <typename K> static cudaError_t go(K kern, dim3 grid, dim3 block, size_t smem, cudaStream_t s, const A &a) {
        cudaError_t e = Launch<float, N>::prep(kern, smem);
        if (e != cudaSuccess) return e;
        e = launch_pdl(kern, grid, block, smem, s, use_pdl(a) || late(a), a);
        return e != cudaSuccess ? e : cudaGetLastError();
    }
    static cudaError_t row_fwd(const A &a, bool imag, cudaStream_t s) {   // ny == N
        dim3 grid((unsigned)((long)a.batch * a.nx / RowGeomP<N>::RPC)), block(RowGeomP<N>::THREADS);
        if (late(a)) return imag ? go(k_row_fwd_p<N, true, true>, grid, block, row_smem(), s, a) : go(k_row_fwd_p<N, false, true>, grid, block, row_smem(), s, a);
        return imag ? go(k_row_fwd_p<N, true, false>, grid, block, row_smem(), s, a) : go(k_row_fwd_p<N, false, false>, grid, block, row_smem(), s, a);
    }
    static cudaError_t row_inv(const A &a, bool imag, cudaStream_t s) {   // ny == N
        dim3 grid((unsigned)((long)a.batch * a.nx / RowGeomP<N>::RPC)), block(RowGeomP<N>::THREADS);
        if (late(a)) {
            if (imag) return go(k_row_inv_p<N, true, false, true>, grid, block, row_smem(), s, a);
            return a.fin.merged ? go(k_row_inv_p<N, false, true, true>, grid, block, row_smem(), s, a) : go(k_row_inv_p<N, false, false, true>, grid, block, row_smem(), s, a);
        }
        if (imag) return go(k_row_inv_p<N, true, false, false>, grid, block, row_smem(), s, a);
        return a.fin.merged ? go(k_row_inv_p<N, false, true, false>, grid, block, row_smem(), s, a) : go(k_row_inv_p<N, false, false, false>, grid, block, row_smem(), s, a);
    }
    static cudaError_t row_ca(const A &a, bool imag, cudaStream_t s) {   // ny == N
        dim3 grid((unsigned)((long)a.batch * a.nx / RowGeomP<N>::RPC)), block(RowGeomP<N>::THREADS);
        if (late(a)) return imag ? go(k_row_ca_p<N, true, true>, grid, block, row_smem(), s, a) : go(k_row_ca_p<N, false, true>, grid, block, row_smem(), s, a);
        return imag ? go(k_row_ca_p<N, true, false>, grid, block, row_smem(), s, a) : go(k_row_ca_p<N, false, false>, grid, block, row_smem(), s, a);
    }
    static cudaError_t col(const A &a, bool imag, cudaStream_t s) {       // nx == N
        dim3 grid((unsigned)(a.ny / 2 / ColGeomP<N>::CPW), (unsigned)a.batch), block(ColGeomP<N>::THREADS);
        if (imag && a.fin.knorm) return late(a) ? go(k_col_p<N, true, true, true>, grid, block, col_smem(), s, a) : go(k_col_p<N, true, false, true>, grid, block, col_smem(), s, a);
        if (late(a)) return imag ? go(k_col_p<N, true, true>, grid, block, col_smem(), s, a) : go(k_col_p<N, false, true>, grid, block, col_smem(), s, a);
        return imag ? go(k_col_p<N, true, false>, grid, block, col_smem(), s, a) : go(k_col_p<N, false, false>, grid, block, col_smem(), s, a);
    }
};

}  // namespace gpe
