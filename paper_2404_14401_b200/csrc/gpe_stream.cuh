// gpe_stream.cuh -- persistent, bulk-copy-fed forms of the three paired complex64 passes of
// gpe_pair.cuh (same mathematics, same intermediate layout, same per-thread arithmetic).
//
// Why.  ncu on the one-tile-per-CTA passes at 2048^2 (profiles/r01_final.md): no unit above 60 %,
// 16 warps per SM of which those of one CTA in four sit in their global-load phase, a second,
// three-quarters-full wave of CTAs in every pass.  Here ONE CTA per SM stays resident for the whole
// pass: four groups of 128 threads (the shape of the old CTAs, so the transform code is shared) each
// loop over tiles, and the NEXT tiles are already on their way into shared memory while the current
// ones are transformed:
//   * the tile of a group arrives by cp.async.bulk / cp.async.bulk.tensor (TMA) into one of two
//     32 KB staging buffers, completion on an mbarrier -- no registers and no LSU issue slots are
//     tied up by loads in flight, and all 16 warps of the SM are always in their arithmetic phase;
//   * a group copies its 16 elements per thread out of the staging buffer (conflict-free LDS), and
//     as soon as its 128 threads have done so (one named barrier, which is also the write-after-read
//     barrier of the group's exchange buffer) its thread 0 issues the copy of the tile two places
//     further down the CTA's list into the same buffer.  The group that frees a buffer refills it,
//     so there is no "empty" barrier and no producer warp;
//   * results go straight from registers to global memory as before (fire and forget).
// Tiles: CTA c takes tiles c, c + gridDim.x, ...; in the CTA's list tile number s belongs to group
// s % 4, sits in staging buffer s % 2 and completes on mbarrier s % 4 (the n-th use of an mbarrier has
// parity n & 1; its next use is armed only after the tile two places back has been consumed, which is
// after its own previous use completed).
// Shared memory per CTA: 2 x 32 KB staging + 4 exchange tiles of about 33 KB = 194 KB.
#pragma once
#include <cuda.h>
#include <cstdint>
#include "gpe_pair.cuh"

namespace gpe {

constexpr int kPsGroups = 4;          // groups of kPsGT threads per CTA
constexpr int kPsGT = 128;            // threads per group
constexpr int kPsThreads = kPsGroups * kPsGT;
constexpr int kPsStage = 32768;       // bytes of one tile = 128 threads x 16 elements x 16 B
constexpr int kPsNStage = 2;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// contiguous global -> shared bulk copy (bytes a multiple of 16, both addresses 16-byte aligned)
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_g2s_2d(void *dst, const CUtensorMap *map, int c0, int c1, uint64_t *bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(smem_u32(dst)),
                 "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_g2s_3d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, uint64_t *bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(smem_u32(dst)),
                 "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ cpair lds_pair(const unsigned char *p) {
    const float4 t = *reinterpret_cast<const float4 *>(p);
    cpair r; r.re = make_float2(t.x, t.y); r.im = make_float2(t.z, t.w); return r;
}

// ---------------------------------------------------------------- pass B (columns)
template <int NX> struct ColGeomS {
    static constexpr int TPF = NX / 16;                 // threads per column pair
    static constexpr int CPW = kPsGT / TPF < 1 ? 1 : kPsGT / TPF;   // column pairs per group tile
    static_assert(TPF * CPW == kPsGT, "a group is 128 threads");
    using F = Fft1D<NX, CPW, cpair>;
    static constexpr size_t EXCH = sizeof(float2) * F::TILE;
    static constexpr size_t SMEM = kPsNStage * kPsStage + kPsGroups * EXCH + 64;
    __host__ __device__ static constexpr int box_lines(int il) { return (NX >> il) < 256 ? (NX >> il) : 256; }
};

template <int NX, bool IMAG>
__global__ void __launch_bounds__(kPsThreads, 1) k_col_s(const __grid_constant__ CUtensorMap tmap, const StepArgs<float, float2> a) {
    using G = ColGeomS<NX>;
    using F = typename G::F;
    extern __shared__ __align__(1024) unsigned char smem_s[];
    unsigned char *smem_raw = smem_s;
    unsigned char *stage = smem_raw;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + kPsNStage * kPsStage + kPsGroups * G::EXCH);
    const int g = threadIdx.x / kPsGT, t = threadIdx.x % kPsGT;
    const int c = t % G::CPW, j = t / G::CPW;
    float2 *sm = reinterpret_cast<float2 *>(smem_raw + kPsNStage * kPsStage + g * G::EXCH) + c;
    const int il = il_of<NX>(a.ny, a.batch), ilm = (1 << il) - 1;
    const int hy = a.ny / 2, tpm = hy / G::CPW;           // tiles per member
    const int ntiles = a.batch * tpm;
    const int nseq = ((int)blockIdx.x < ntiles) ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    const int lines = NX >> il, bl = G::box_lines(il), nbox = lines / bl;
    auto issue = [&](int s) {   // one thread: arm the mbarrier of list entry s and start its copies
        const int tile = blockIdx.x + s * gridDim.x, b = tile / tpm, cp0 = (tile % tpm) * G::CPW;
        uint64_t *bar = full + (s % kPsGroups);
        unsigned char *dstb = stage + (s % kPsNStage) * kPsStage;
        mbar_expect_tx(bar, kPsStage);
        for (int q = 0; q < nbox; ++q)
            tma_g2s_2d(dstb + q * (kPsStage / nbox), &tmap, cp0 << (il + 2), b * lines + q * bl, bar);
    };
    if (threadIdx.x == 0) {
        for (int i = 0; i < kPsGroups; ++i) mbar_init(full + i, 1);
        fence_mbar_init();
    }
    __syncthreads();
    pdl_wait();
    if (threadIdx.x == 0)
        for (int s = 0; s < kPsNStage && s < nseq; ++s) issue(s);
    const float invp = a.inv_p;
    for (int s = g; s < nseq; s += kPsGroups) {
        const int tile = blockIdx.x + s * gridDim.x, b = tile / tpm, cp = (tile % tpm) * G::CPW + c;
        if (t == 0 && (tile % tpm) == 0 && a.fin.prepared) prepare_member(a.fin, b);
        const size_t hys = (size_t)hy;
        const size_t base = (size_t)b * NX * hys + ipos(j, cp, hys, il), kstr = (size_t)F::M1 * hys;
        cpair *dst = reinterpret_cast<cpair *>(a.dst) + base;
        cpair v[16];
        mbar_wait(full + g, (s / kPsGroups) & 1);
        {
            const unsigned char *st = stage + (s % kPsNStage) * kPsStage;
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const int i = j + F::M1 * k;
                v[k] = lds_pair(st + 16 * ((((i >> il) * G::CPW + c) << il) + (i & ilm)));
            }
        }
        // every thread of the group has its elements: the staging buffer is free for the tile two places
        // on, and the group's exchange tile is free of the previous tile's last reads
        bar_named(1 + g, kPsGT);
        if (t == 0 && s + kPsNStage < nseq) { fence_proxy_async(); issue(s + kPsNStage); }
        auto sync = [g] { bar_named(1 + g, kPsGT); };
        F::fwd(v, sm, j, a.tw_x, a.tw1_x, sync);
        if constexpr (IMAG) {
            const float2 ey = *reinterpret_cast<const float2 *>(a.kin_yr + 2 * cp);
#pragma unroll
            for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
                for (int rr = 0; rr < F::RL; ++rr) {
                    const float2 f = rmuls(ey, a.kin_xr[F::nat(j, ii, rr)]);
                    cpair &z = v[ii * F::RL + rr];
                    z.re = rmul(z.re, f); z.im = rmul(z.im, f);
                }
        } else {
            // kinetic factor (1+a)(1+b)/P as v/P + v*g, g = a' + b' + a'b: see k_col_p (gpe_pair.cuh)
            const float4 k0 = ldtw(reinterpret_cast<const float4 *>(a.kin_y2), 2 * cp), k1 = ldtw(reinterpret_cast<const float4 *>(a.kin_y2), 2 * cp + 1);
            const float2 cb = make_float2(k0.x, k0.y), bqy = make_float2(k0.z, k0.w), bpx = make_float2(k1.x, k1.y), bpy = make_float2(k1.z, k1.w);
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
        F::inv(v, sm, j, a.tw_x, a.tw1_x, sync);
#pragma unroll
        for (int k = 0; k < 16; ++k) st_pair(dst + k * kstr, v[k]);
    }
    pdl_launch_dependents();
}

// ---------------------------------------------------------------- passes A and C (rows)
// A group tile is RPG = 128 / (NY/32) whole rows (2 at 2048, 4 at 1024, ...): 32 KB.  Pass A copies them
// as one contiguous block of psi; pass C takes the same rows of the intermediate array -- contiguous too
// when two rows are interleaved (il = 1), a 3-D tensor box per 256 column pairs when four are (il = 2,
// 2048^2 only: the tile is one half of a four-row group).  Either way the staging buffer holds
// [row pair][column pair][row in pair][16 B].
template <int N> struct RowGeomS {
    static constexpr int H = N / 2;
    static constexpr int TPF = H / 16;                   // threads per row
    static constexpr int RPG = kPsGT / TPF;              // rows per group tile (even)
    static_assert(TPF * RPG == kPsGT && RPG >= 2, "a group is 128 threads and at least one row pair");
    using F = Fft1D<H, 1, cpair>;
    static constexpr bool PAIRMAP = F::GL >= 2;          // see RowGeomP (gpe_pair.cuh)
    static constexpr size_t EXCH = sizeof(float2) * RPG * F::TILE;
    static constexpr size_t BARS = kPsNStage * kPsStage + kPsGroups * EXCH;   // offset of the mbarriers
    static constexpr size_t SMEM = BARS + 64 + kPsGroups * (12 * sizeof(double) + 16);
};

// barriers: id 1 + g = the 128 threads of group g; 5 + 2 g + q = row q (2048) or row pair q (1024) of the
// group, 64 threads; anything of 32 threads or fewer lives inside one warp
template <int TPF> __device__ __forceinline__ void sync_row_s(int g, int r) {
    if constexpr (TPF == 64) bar_named(5 + 2 * g + r, 64);
    else if constexpr (TPF <= 32) __syncwarp();
    else bar_named(1 + g, kPsGT);
}
template <int TPF> __device__ __forceinline__ void sync_pair_s(int g, int rp) {
    if constexpr (2 * TPF == 64) bar_named(5 + 2 * g + rp, 64);
    else if constexpr (2 * TPF <= 32) __syncwarp();
    else bar_named(1 + g, kPsGT);
}

template <int NY, bool IMAG>
__global__ void __launch_bounds__(kPsThreads, 1) k_row_fwd_s(const StepArgs<float, float2> a) {
    using G = RowGeomS<NY>;
    using F = typename G::F;
    constexpr int H = G::H, M1 = F::M1, TPF = G::TPF, RPG = G::RPG;
    extern __shared__ __align__(1024) unsigned char smem_s[];
    unsigned char *stage = smem_s;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_s + G::BARS);
    const int g = threadIdx.x / kPsGT, t = threadIdx.x % kPsGT;
    const int r = t / TPF, j = t % TPF;
    float2 *exch = reinterpret_cast<float2 *>(smem_s + kPsNStage * kPsStage + g * G::EXCH);
    float2 *sm = exch + r * F::TILE;
    const int il = il_of<NY>(a.nx, a.batch);
    const int ntiles = (int)((long)a.batch * a.nx / RPG);
    const int nseq = ((int)blockIdx.x < ntiles) ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    auto issue = [&](int s) {
        const long tile = blockIdx.x + (long)s * gridDim.x;
        uint64_t *bar = full + (s % kPsGroups);
        mbar_expect_tx(bar, kPsStage);
        bulk_g2s(stage + (s % kPsNStage) * kPsStage, a.src + tile * RPG * NY, kPsStage, bar);
    };
    if (threadIdx.x == 0) {
        for (int i = 0; i < kPsGroups; ++i) mbar_init(full + i, 1);
        fence_mbar_init();
    }
    __syncthreads();
    pdl_wait();
    if (threadIdx.x == 0)
        for (int s = 0; s < kPsNStage && s < nseq; ++s) issue(s);
    cpair *dst = reinterpret_cast<cpair *>(a.dst);
    for (int s = g; s < nseq; s += kPsGroups) {
        const long tile = blockIdx.x + (long)s * gridDim.x;
        const long row = tile * RPG + r;
        const int b = (int)(row / a.nx), i = (int)(row % a.nx);
        float2 p0[16], p1[16];
        mbar_wait(full + g, (s / kPsGroups) & 1);
        {
            const float2 *st = reinterpret_cast<const float2 *>(stage + (s % kPsNStage) * kPsStage) + r * NY + j;
#pragma unroll
            for (int k = 0; k < 16; ++k) { p0[k] = st[M1 * k]; p1[k] = st[H + M1 * k]; }
        }
        bar_named(1 + g, kPsGT);   // staging buffer and exchange tile of the group are free (see k_col_s)
        if (t == 0 && s + kPsNStage < nseq) { fence_proxy_async(); issue(s + kPsNStage); }
        {
            const MemberState &ms = a.fin.st[b];
            float2 sn, st_;
            const bool pend = !IMAG && ms.pend;
            const float cx2 = (a.flags & F_CAV_FULL) ? a.cavx[i] * a.cavx[i] : 0.f;
            potential_pair16<IMAG, false, M1, H>(p0, p1, a, b, i, j, (float)ms.scale, pend ? 2.f : 1.f,
                                                 (float)(pend ? ms.A + ms.A_pend : ms.A), (float)(pend ? ms.C + ms.C_pend : ms.C),
                                                 (float)(pend ? ms.D + ms.D_pend : ms.D) * cx2, sn, st_);
        }
        // radix-2 decimation in frequency across the two halves of the row (k_row_fwd_p, gpe_pair.cuh)
        cpair v[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const float2 w = ldtw(a.tw_y, j + M1 * k);
            const float dx = p0[k].x - p1[k].x, dy = p0[k].y - p1[k].y;
            v[k].re = make_float2(p0[k].x + p1[k].x, fmaf(dx, w.x, -(dy * w.y)));
            v[k].im = make_float2(p0[k].y + p1[k].y, fmaf(dx, w.y, dy * w.x));
        }
        auto sync_row = [g, r] { sync_row_s<TPF>(g, r); };
        if constexpr (G::PAIRMAP) {
            const int rp = r >> 1, u = j + (r & 1) * TPF;
            float2 *sm0 = exch + (2 * rp) * F::TILE, *sm1 = sm0 + F::TILE;
            auto sync_pair = [g, rp] { sync_pair_s<TPF>(g, rp); };
            F::fwd_pairlast(v, sm, sm0, sm1, j, u, a.tw_hy, a.tw1_hy, sync_row, sync_pair);
            const long rowp = tile * RPG + 2 * rp;
#pragma unroll
            for (int ii = 0; ii < F::GL / 2; ++ii)
#pragma unroll
                for (int rr = 0; rr < F::RL; ++rr) {
                    const size_t pos = ipos(rowp, F::nat_t(u + 2 * TPF * ii, rr), H, il);
                    st_pair2(dst + pos, v[(2 * ii) * F::RL + rr], v[(2 * ii + 1) * F::RL + rr]);
                }
        } else {
            F::fwd(v, sm, j, a.tw_hy, a.tw1_hy, sync_row);
#pragma unroll
            for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
                for (int rr = 0; rr < F::RL; ++rr) st_pair(dst + ipos(row, F::nat(j, ii, rr), H, il), v[ii * F::RL + rr]);
        }
    }
    pdl_launch_dependents();
}

template <int NY, bool IMAG, bool MERGED>
__global__ void __launch_bounds__(kPsThreads, 1) k_row_inv_s(const __grid_constant__ CUtensorMap tmap, const StepArgs<float, float2> a) {
    using G = RowGeomS<NY>;
    using F = typename G::F;
    constexpr int H = G::H, M1 = F::M1, TPF = G::TPF, RPG = G::RPG;
    extern __shared__ __align__(1024) unsigned char smem_s[];
    unsigned char *stage = smem_s;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_s + G::BARS);
    const int g = threadIdx.x / kPsGT, t = threadIdx.x % kPsGT;
    const int r = t / TPF, j = t % TPF;
    double *red = reinterpret_cast<double *>(smem_s + G::BARS + 64) + g * 12;          // [3][4 warps] of the group
    int *is_last = reinterpret_cast<int *>(smem_s + G::BARS + 64 + kPsGroups * 12 * sizeof(double)) + g * 4;
    float2 *exch = reinterpret_cast<float2 *>(smem_s + kPsNStage * kPsStage + g * G::EXCH);
    float2 *sm = exch + r * F::TILE;
    const int il = il_of<NY>(a.nx, a.batch);
    const int gpm = a.nx / RPG;                          // tiles per member (= f.cpm)
    const int ntiles = a.batch * gpm;
    const int nseq = ((int)blockIdx.x < ntiles) ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    auto issue = [&](int s) {
        const long tile = blockIdx.x + (long)s * gridDim.x;
        uint64_t *bar = full + (s % kPsGroups);
        unsigned char *dstb = stage + (s % kPsNStage) * kPsStage;
        mbar_expect_tx(bar, kPsStage);
        if (il == 1) {
            bulk_g2s(dstb, reinterpret_cast<const cpair *>(a.src) + tile * RPG * H, kPsStage, bar);
        } else {   // RPG == 2: rows 2 tile, 2 tile + 1 = half (tile & 1) of row group tile / 2
            for (int q = 0; q < H / 256; ++q)
                tma_g2s_3d(dstb + q * 8192, &tmap, 0, (int)(tile & 1), (int)(tile >> 1) * H + q * 256, bar);
        }
    };
    if (threadIdx.x == 0) {
        for (int i = 0; i < kPsGroups; ++i) mbar_init(full + i, 1);
        fence_mbar_init();
    }
    __syncthreads();
    pdl_wait();
    if (threadIdx.x == 0)
        for (int s = 0; s < kPsNStage && s < nseq; ++s) issue(s);
    const FinalizeParams &f = a.fin;
    const int lane = t & 31, wid = t >> 5;
    for (int s = g; s < nseq; s += kPsGroups) {
        const long tile = blockIdx.x + (long)s * gridDim.x;
        const long row = tile * RPG + r;
        const int b = (int)(row / a.nx), i = (int)(row % a.nx);
        cpair v[16];
        mbar_wait(full + g, (s / kPsGroups) & 1);
        const unsigned char *st = stage + (s % kPsNStage) * kPsStage;
        auto sync_row = [g, r] { sync_row_s<TPF>(g, r); };
        if constexpr (G::PAIRMAP) {
            // 32 bytes per column pair = rows 2m, 2m+1.  A quarter warp reads eight consecutive column
            // pairs with one 128-bit access each: lanes 4-7 take the OTHER row first, so that the eight
            // 16-byte pieces fall into eight different bank groups (conflict free); the two transforms are
            // symmetric, so only the destination tiles of the first exchange swap with it.
            const int rp = r >> 1, u = j + (r & 1) * TPF, sw = (lane >> 2) & 1;
            float2 *sm0 = exch + (2 * rp) * F::TILE, *sm1 = sm0 + F::TILE;
            const unsigned char *sp = st + (size_t)rp * H * 32 + sw * 16;
#pragma unroll
            for (int ii = 0; ii < F::GL / 2; ++ii)
#pragma unroll
                for (int rr = 0; rr < F::RL; ++rr) {
                    const int kp = F::nat_t(u + 2 * TPF * ii, rr);
                    v[(2 * ii) * F::RL + rr] = lds_pair(sp + kp * 32);
                    v[(2 * ii + 1) * F::RL + rr] = lds_pair(sp + kp * 32 + 16 - 32 * sw);
                }
            bar_named(1 + g, kPsGT);
            if (t == 0 && s + kPsNStage < nseq) { fence_proxy_async(); issue(s + kPsNStage); }
            auto sync_pair = [g, rp] { sync_pair_s<TPF>(g, rp); };
            F::inv_pairfirst(v, sm, sw ? sm1 : sm0, sw ? sm0 : sm1, j, u, a.tw_hy, a.tw1_hy, sync_row, sync_pair);
        } else {
            const unsigned char *sp = st + (size_t)(r >> 1) * H * 32 + (r & 1) * 16;
#pragma unroll
            for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
                for (int rr = 0; rr < F::RL; ++rr) v[ii * F::RL + rr] = lds_pair(sp + F::nat(j, ii, rr) * 32);
            bar_named(1 + g, kPsGT);
            if (t == 0 && s + kPsNStage < nseq) { fence_proxy_async(); issue(s + kPsNStage); }
            F::inv(v, sm, j, a.tw_hy, a.tw1_hy, sync_row);
        }
        // mirror of pass A's radix-2 layer (k_row_inv_p, gpe_pair.cuh)
        float2 p0[16], p1[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const float2 w = ldtw(a.tw_y, j + M1 * k);
            const float tx = fmaf(v[k].re.y, w.x, v[k].im.y * w.y), ty = fmaf(v[k].im.y, w.x, -(v[k].re.y * w.y));
            p0[k] = make_float2(v[k].re.x + tx, v[k].im.x + ty);
            p1[k] = make_float2(v[k].re.x - tx, v[k].im.x - ty);
        }
        const MemberState &ms = a.fin.st[b];
        float2 sn = make_float2(0.f, 0.f), stt = sn;
        if constexpr (MERGED) reduce_pair16<M1>(p0, p1, a, j, sn, stt);
        else potential_pair16<IMAG, true, M1, H>(p0, p1, a, b, i, j, 1.f, 1.f, (float)ms.A, (float)ms.C,
                                                 (a.flags & F_CAV_FULL) ? (float)ms.D * a.cavx[i] * a.cavx[i] : 0.f, sn, stt);
        float2 *drow = a.dst + row * NY;
        // partial sums of the tile first, wavefunction stores second (k_row_inv_p); fixed summation order
        const int cim = (int)(tile % gpm);
        const double rown = (double)sn.x + (double)sn.y;
        double dn = warp_sum(rown);
        double dt_ = (a.flags & F_CAVITY) ? warp_sum(((double)stt.x + (double)stt.y) * (double)a.cavx[i]) : 0.0;
        const bool fullm = a.flags & F_CAV_FULL;
        double db_ = fullm ? warp_sum(rown * ((double)a.cavx[i] * (double)a.cavx[i])) : 0.0;
        if (lane == 0) { red[wid] = dn; red[4 + wid] = dt_; red[8 + wid] = db_; }
        bar_named(1 + g, kPsGT);
        unsigned int old = 0;
        if (t == 0) {
            double s0 = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll
            for (int q = 0; q < 4; ++q) { s0 += red[q]; s1 += red[4 + q]; s2 += red[8 + q]; }
            f.partials[(size_t)b * f.cpm + cim] = make_double2(s0, s1);
            if (fullm) f.partials_b[(size_t)b * f.cpm + cim] = s2;
            __threadfence();
            old = atomicAdd(&f.counters[b], 1u);
        }
#pragma unroll
        for (int k = 0; k < 16; ++k) { drow[j + M1 * k] = p0[k]; drow[H + j + M1 * k] = p1[k]; }
        if (t == 0) *is_last = (old == (unsigned int)(f.cpm - 1));
        bar_named(1 + g, kPsGT);
        if (*is_last) {   // the last tile of the member: the group's threads sum the partials
            double s0, s1, s2;
            sum_partials_n(f, b, t, kPsGT, s0, s1, s2);
            s0 = warp_sum(s0); s1 = warp_sum(s1); s2 = warp_sum(s2);
            bar_named(1 + g, kPsGT);
            if (lane == 0) { red[wid] = s0; red[4 + wid] = s1; red[8 + wid] = s2; }
            bar_named(1 + g, kPsGT);
            if (t == 0) {
                double t0 = 0.0, t1 = 0.0, t2 = 0.0;
#pragma unroll
                for (int q = 0; q < 4; ++q) { t0 += red[q]; t1 += red[4 + q]; t2 += red[8 + q]; }
                finalize_member(f, b, t0, t1, t2);
                f.counters[b] = 0u;
            }
        }
        bar_named(1 + g, kPsGT);   // red / is_last are reused by the group's next tile
    }
    pdl_launch_dependents();
}

// ---------------------------------------------------------------- launchers
template <int N> struct LaunchS {
    using A = StepArgs<float, float2>;
    template <typename K> static cudaError_t go(K kern, int grid, size_t smem, cudaStream_t s, const CUtensorMap &map, const A &a) {
        cudaError_t e = Launch<float, N>::prep(kern, smem);
        if (e != cudaSuccess) return e;
        e = launch_pdl(kern, dim3((unsigned)grid), dim3(kPsThreads), smem, s, true, map, a);
        return e != cudaSuccess ? e : cudaGetLastError();
    }
    static cudaError_t row_fwd(const A &a, bool imag, int nsm, cudaStream_t s) {   // ny == N
        const int ntiles = (int)((long)a.batch * a.nx / RowGeomS<N>::RPG);
        const int grid = ntiles < nsm ? ntiles : nsm;
        auto go2 = [&](auto kern) -> cudaError_t {
            cudaError_t e = Launch<float, N>::prep(kern, RowGeomS<N>::SMEM);
            if (e != cudaSuccess) return e;
            e = launch_pdl(kern, dim3((unsigned)grid), dim3(kPsThreads), RowGeomS<N>::SMEM, s, true, a);
            return e != cudaSuccess ? e : cudaGetLastError();
        };
        return imag ? go2(k_row_fwd_s<N, true>) : go2(k_row_fwd_s<N, false>);
    }
    static cudaError_t row_inv(const A &a, const CUtensorMap &map, bool imag, int nsm, cudaStream_t s) {   // ny == N
        const int ntiles = (int)((long)a.batch * a.nx / RowGeomS<N>::RPG);
        const int grid = ntiles < nsm ? ntiles : nsm;
        if (imag) return go(k_row_inv_s<N, true, false>, grid, RowGeomS<N>::SMEM, s, map, a);
        return a.fin.merged ? go(k_row_inv_s<N, false, true>, grid, RowGeomS<N>::SMEM, s, map, a)
                            : go(k_row_inv_s<N, false, false>, grid, RowGeomS<N>::SMEM, s, map, a);
    }
    static int col_cpw() { return ColGeomS<N>::CPW; }
    static cudaError_t col(const A &a, const CUtensorMap &map, bool imag, int nsm, cudaStream_t s) {   // nx == N
        const int ntiles = a.batch * (a.ny / 2 / ColGeomS<N>::CPW);
        const int grid = ntiles < nsm ? ntiles : nsm;
        return imag ? go(k_col_s<N, true>, grid, ColGeomS<N>::SMEM, s, map, a) : go(k_col_s<N, false>, grid, ColGeomS<N>::SMEM, s, map, a);
    }
};

}  // namespace gpe
