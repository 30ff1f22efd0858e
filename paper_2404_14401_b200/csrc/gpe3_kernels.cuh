// gpe3_kernels.cuh -- the split-step of PAPER.md:60-76 (Eqs. 2-4) on a THREE-dimensional grid (the first item of the
// paper's outlook, second half).  psi is [nz][nx][ny], y fastest.
//
// The kinetic factor exp(-sigma |k|^2 dt/2) is a product over the axes, and the transforms of different axes commute,
// so  IFFT3 . K . FFT3  =  (F_z^-1 K_z F_z) (F_x^-1 K_x F_x) (F_y^-1 K_y F_y)  exactly: a step is THREE passes over
// the array, each one loading a line (or a tile of lines) into registers, transforming it, multiplying by the
// factor of that axis, transforming back and storing in place -- natural layout throughout, no transposed copy:
//   pass Y (rows, contiguous):      load [x lazy scale] -> first potential half-step ->
//                                   FFT_y -> K_y -> IFFT_y -> store
//   pass X (lines of stride ny):    tiles of W neighbouring y per CTA: FFT_x -> K_x -> IFFT_x
//   pass Z (lines of stride nx ny): tiles of W neighbouring (x, y) per CTA: FFT_z -> K_z -> IFFT_z
//                                   [imaginary time: -> second potential half-step -> one partial sum of |psi|^2 per
//                                   CTA; the one-CTA kernel k3_finalize adds them in a fixed order, sets the lazy scale
//                                   1/sqrt(norm) and writes the record: no host round trip]
// Real time: the second half-step of step n and the first of step n+1 see the same |psi|^2 and are applied as ONE
// factor by pass Y of step n+1 (fac = 2); the first step of a call takes fac = 1 and a point-wise kernel closes the
// call (k3_point).  Three passes are the floor for three axes held one at a time in registers / shared memory:
// 6 P s bytes of psi traffic per step (P points, s bytes per complex number) plus the potential array.
#pragma once
#include "gpe_kernels.cuh"

// resident CTAs per SM asked of the compiler for complex64 (measured on B200, 256^3 real time: column passes 1 -> 2
// CTAs and row pass 2 -> 3: 304 -> 249 us per step; 3 CTAs of the column pass spill and lose: 263 us)
#ifndef GPE3_COL_MINB
#define GPE3_COL_MINB 2
#endif
#ifndef GPE3_ROW_MINB
#define GPE3_ROW_MINB 3
#endif
// complex128 lines of 512 points and more in 128-thread column CTAs of four columns (64-byte row segments), two per SM,
// instead of eight columns in 256 threads (measured: 512 x 512 x 256 2458 -> 2287 us per step, 256 x 256 x 512 1007 -> 931)
#ifndef GPE3_COL_D512_NARROW
#define GPE3_COL_D512_NARROW 1
#endif
#ifndef GPE3_PDL_MAX
#define GPE3_PDL_MAX (128L * 128L * 128L)
#endif

namespace gpe {

// launch geometry of the 3-D passes (64^3 with 256-thread CTAs had 64 CTAs per pass on 148 SMs).
// Threads per CTA by line length.  Rows: 64 at 64 points, 128 at 128, 64 again from 256 points up (measured on
// B200, 256^3 complex64 real time, with 256 -> 128 threads in both kinds of pass: 245 -> 208 us per step, complex128 574 -> 419: more, smaller CTAs
// overlap their load / transform / store phases better).  Columns of 256 points come in two widths: NARROW (128
// threads, 8 columns) and WIDE (256 threads, 16 columns); narrow wins while the plane nx ny is small (256^3: 208
// against 236 us) and loses when the lines are 2 MB apart (512 x 512 x 256: 1060 against 1013 us), see col_wide().
#ifndef GPE3_ROW_T
#define GPE3_ROW_T 64     // rows of 256 points and more: 64 threads (4 rows of 256 points); against 128: 256^3 complex64
#endif                    // 209.4 -> 206.1 us per step, 512 x 512 x 256 1013 -> 1000, complex128 imaginary time 488 -> 473

template <int N> struct RowTarget3 { static constexpr int THREADS = N <= 64 ? 64 : (N <= 128 ? 128 : GPE3_ROW_T); };
template <int N, bool WIDE> struct ColTarget3 { static constexpr int THREADS = N <= 64 ? 64 : (N <= 128 ? 128 : (N <= 256 ? (WIDE ? 256 : 128) : 256)); };
template <int N> struct RowGeom3 {
    static constexpr int TPF = N / 16;
    static constexpr int RPC = (RowTarget3<N>::THREADS / TPF) < 1 ? 1 : (RowTarget3<N>::THREADS / TPF);   // rows per CTA
    static constexpr int THREADS = RPC * TPF;
};
template <typename T, int N, bool WIDE = false> struct ColGeom3 {
    static constexpr int TPF = N / 16;
    static constexpr int WMIN = sizeof(T) == 4 ? 4 : 2;            // >= 32-byte row segments
    // complex128 lines of 512 points and more: 128 threads (4 columns = 64-byte row segments)
    static constexpr int W0 = ((sizeof(T) == 8 && N >= 512 && GPE3_COL_D512_NARROW) ? 128 : ColTarget3<N, WIDE>::THREADS) / TPF;
    static constexpr int W = W0 < WMIN ? WMIN : W0;                // columns per CTA
    static constexpr int THREADS = W * TPF;
};

struct State3 {
    double scale;      // lazy renormalisation: the stored psi times `scale` is the wavefunction
    double norm;       // sum |psi|^2 dV after the last reduced step (1 in imaginary time)
    double norm_pre;   // the same sum before the renormalisation of that step
    long long step;    // step counter
};

template <typename T> struct Args3 {
    cx<T> *psi;
    int nx, ny, nz;
    long line_stride, slab_stride;   // column passes: distance between the points of a line, between slabs
    const T *v3d;                    // [nz][nx][ny] or nullptr
    const T *vx, *vy, *vz;           // separable part (always present, zeros when not given)
    T g, half_dt, fac;               // fac: 1, or 2 when the factor carries the previous step's second half too
    int pot;                         // pass Y: factor on load; final pass Z (imaginary time): factor before the sums
    const T *kin;                    // step: the factor of this axis (imag: real [N], real time: complex (w - 1)/N);
                                     // measure: k^2 of this axis
    T inv_n;                         // 1/N of this axis
    const cx<T> *tw, *tw1;           // twiddles of this axis (gpe_fft.cuh)
    State3 *st;
    double *partials;                // one per CTA
    unsigned int *counter;
    int *nonfinite;
    double dV;
    int sums;                        // final pass: reduce |psi|^2 and finalise
    int final_axis;                  // column pass: 1 when the lines run along z
    long long step_index;            // index of the step being taken
    double *record;                  // {step, norm, norm_pre} of this step, or nullptr
    double *measure_out;             // measure mode: where the last CTA writes the total
    int rev;                         // 1: CTAs take their tiles in descending order (see evolve3 in gpe3_api.cu)
};

// tile index of this CTA: blocks are dispatched in ascending order, rev walks the array the other way
__device__ __forceinline__ unsigned tile_x(int rev) { return rev ? gridDim.x - 1u - blockIdx.x : blockIdx.x; }
__device__ __forceinline__ unsigned tile_y(int rev) { return rev ? gridDim.y - 1u - blockIdx.y : blockIdx.y; }
__device__ __forceinline__ void sincosm1_any(float w, float *s, float *cm1) { sincosm1_general(w, s, cm1); }
__device__ __forceinline__ void sincosm1_any(double w, double *s, double *cm1) { sincosm1_t(w, s, cm1); }

// ---------------------------------------------------------------- potential factor on the 16 points of a thread
// psi <- psi * exp(-sigma fac (V + g|psi|^2) dt/2) with V[k] supplied by the caller; see potential_step16 of
// gpe_kernels.cuh for the "minus one" form of the real-time phase and its warp-uniform tiers.
template <typename T, bool IMAG>
__device__ __forceinline__ void potential16(cx<T> (&v)[16], const T (&V)[16], T g, T hdt) {
    T w[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) w[k] = fma(g, v[k].x * v[k].x + v[k].y * v[k].y, V[k]) * hdt;
    if constexpr (IMAG) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const T e = exp_t(-w[k]);
            v[k].x *= e; v[k].y *= e;
        }
    } else {
        T wmax = T(0);
#pragma unroll
        for (int k = 0; k < 16; ++k) wmax = fmax(wmax, fabs(w[k]));
        const bool small = __all_sync(0xffffffffu, wmax <= T(0.5));
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            T sn_, cm1;
            if (small) sincosm1_small(-w[k], &sn_, &cm1);
            else sincosm1_any(-w[k], &sn_, &cm1);
            const T ox = fma(v[k].x, cm1, fma(-v[k].y, sn_, v[k].x));
            const T oy = fma(v[k].x, sn_, fma(v[k].y, cm1, v[k].y));
            v[k].x = ox; v[k].y = oy;
        }
    }
}

// kinetic factor of one axis on the registers of a thread after the forward transform (digit-reversed order)
template <typename T, typename F, bool IMAG>
__device__ __forceinline__ void kinetic16(cx<T> (&v)[16], const Args3<T> &a, int j) {
#pragma unroll
    for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
        for (int rr = 0; rr < F::RL; ++rr) {
            cx<T> &z = v[ii * F::RL + rr];
            const int q = F::nat(j, ii, rr);
            if constexpr (IMAG) {
                const T f = a.kin[q];
                z.x *= f; z.y *= f;
            } else {
                const cx<T> t = reinterpret_cast<const cx<T> *>(a.kin)[q];
                const T ox = fma(z.x, t.x, fma(-z.y, t.y, z.x * a.inv_n));
                const T oy = fma(z.x, t.y, fma(z.y, t.x, z.y * a.inv_n));
                z.x = ox; z.y = oy;
            }
        }
}

// sum over the CTA of `acc`, one partial per CTA, the last CTA adds the partials in a fixed order.
// Returns true in thread 0 of the last CTA with the total in `total`.
__device__ __forceinline__ bool reduce_ctas(double acc, double *partials, unsigned int *counter, unsigned int cta,
                                            unsigned int nctas, double &total) {
    __shared__ double red[32];
    __shared__ int is_last;
    acc = warp_sum(acc);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) red[w] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int q = 0; q < nw; ++q) t += red[q];
        partials[cta] = t;
        __threadfence();
        is_last = (atomicAdd(counter, 1u) == nctas - 1u);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    double t = 0.0;
    for (unsigned int q = threadIdx.x; q < nctas; q += blockDim.x) t += __ldcg(partials + q);
    t = warp_sum(t);
    __syncthreads();
    if (lane == 0) red[w] = t;
    __syncthreads();
    if (threadIdx.x != 0) return false;
    total = 0.0;
    for (int q = 0; q < nw; ++q) total += red[q];
    *counter = 0u;
    return true;
}

// end of a step, one thread: norm, lazy scale, record (include/gpe.h, gpe3_evolve)
template <bool IMAG>
__device__ __forceinline__ void finalize3(State3 *st, double total, double dV, long long step_index, double *record,
                                          int *nonfinite) {
    const double pre = total * dV;
    if (!(pre > 0.0) || !isfinite(pre)) *nonfinite = 1;
    if (IMAG) { st->scale = 1.0 / sqrt(pre); st->norm = 1.0; }
    else st->norm = pre;
    st->norm_pre = pre;
    st->step = step_index >= 0 ? step_index + 1 : st->step + 1;
    if (record) { record[0] = (double)(step_index + 1); record[1] = IMAG ? 1.0 : pre; record[2] = pre; }
}

// ---------------------------------------------------------------- pass Y: rows
// MODE 0: the step.  MODE 1: measure: sum kin[q] |psi^_y|^2 over the grid (kin = k_y^2) -> *measure_out.
template <typename T, int NY, bool IMAG, int MODE>
__global__ void __launch_bounds__(RowGeom3<NY>::THREADS, (sizeof(T) == 4 ? GPE3_ROW_MINB : 1) * (256 / RowGeom3<NY>::THREADS)) k3_row(const Args3<T> a) {
    using C = cx<T>;
    using F = Fft1D<NY, 1, cx<T>>;
    using G = RowGeom3<NY>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    const int r = threadIdx.x / G::TPF, j = threadIdx.x % G::TPF;
    C *sm = smem + r * F::SLOTS;
    const long row = (long)tile_x(a.rev) * G::RPC + r;
    const int l = (int)(row / a.nx), i = (int)(row % a.nx);
    C *p = a.psi + row * NY;
    C v[16];
    pdl_launch_dependents();   // small grids are launched with programmatic stream serialisation (Launch3::go)
    pdl_wait();
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = __ldcg(p + j + F::M1 * k);
    if constexpr (MODE == 0) {
        if constexpr (IMAG) {
            const T s = (T)a.st->scale;
#pragma unroll
            for (int k = 0; k < 16; ++k) { v[k].x *= s; v[k].y *= s; }
        }
        if (a.pot) {
            const T vrow = a.vz[l] + a.vx[i];
            T V[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) V[k] = vrow + a.vy[j + F::M1 * k];
            if (a.v3d) {
                const T *__restrict__ v3 = a.v3d + row * NY;
#pragma unroll
                for (int k = 0; k < 16; ++k) V[k] += v3[j + F::M1 * k];
            }
            potential16<T, IMAG>(v, V, a.g, a.half_dt * a.fac);
        }
    }
    F::fwd(v, sm, j, a.tw, a.tw1);
    if constexpr (MODE == 0) {
        kinetic16<T, F, IMAG>(v, a, j);
        F::inv(v, sm, j, a.tw, a.tw1);
#pragma unroll
        for (int k = 0; k < 16; ++k) p[j + F::M1 * k] = v[k];
    } else {
        double acc = 0.0;
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                const C z = v[ii * F::RL + rr];
                acc += (double)a.kin[F::nat(j, ii, rr)] * ((double)z.x * (double)z.x + (double)z.y * (double)z.y);
            }
        double total;
        if (reduce_ctas(acc, a.partials, a.counter, blockIdx.x, gridDim.x, total)) *a.measure_out = total;
    }
}

#ifndef GPE3_COL_D128
#define GPE3_COL_D128 3   // resident 128-thread CTAs per SM asked of the compiler for the complex128 column passes (168 registers, no
                          // spills; against 2: 256^3 414 -> 401 us per step real time, 471 -> 441 imaginary time)
#endif
template <typename T, int N, bool WIDE> constexpr int col_minb3() {
    constexpr int th = ColGeom3<T, N, WIDE>::THREADS;
    return sizeof(T) == 4 ? GPE3_COL_MINB * (256 / th) : (th == 128 ? (N <= 256 ? GPE3_COL_D128 : 2) : 256 / th);
}
// ---------------------------------------------------------------- passes X and Z: lines of stride line_stride
// grid = (columns of a slab / W, slabs).  FINAL: the last pass of the step (lines along z).
template <typename T, int N, bool IMAG, int MODE, bool WIDE>
__global__ void __launch_bounds__(ColGeom3<T, N, WIDE>::THREADS, col_minb3<T, N, WIDE>()) k3_col(const Args3<T> a) {
    using C = cx<T>;
    using G = ColGeom3<T, N, WIDE>;
    using F = Fft1D<N, G::W, cx<T>>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *smem = reinterpret_cast<C *>(smem_raw);
    const int c = threadIdx.x % G::W, j = threadIdx.x / G::W;
    const long col = (long)tile_x(a.rev) * G::W + c;
    C *p = a.psi + (long)tile_y(a.rev) * a.slab_stride + col;
    C *sm = smem + c;
    const long ls = a.line_stride;
    C v[16];
    pdl_launch_dependents();
    pdl_wait();
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = __ldcg(p + (long)(j + F::M1 * k) * ls);
    F::fwd(v, sm, j, a.tw, a.tw1);
    if constexpr (MODE == 1) {
        double acc = 0.0;
#pragma unroll
        for (int ii = 0; ii < F::GL; ++ii)
#pragma unroll
            for (int rr = 0; rr < F::RL; ++rr) {
                const C z = v[ii * F::RL + rr];
                acc += (double)a.kin[F::nat(j, ii, rr)] * ((double)z.x * (double)z.x + (double)z.y * (double)z.y);
            }
        double total;
        if (reduce_ctas(acc, a.partials, a.counter, blockIdx.y * gridDim.x + blockIdx.x, gridDim.x * gridDim.y, total))
            *a.measure_out = total;
        return;
    } else {
        kinetic16<T, F, IMAG>(v, a, j);
        F::inv(v, sm, j, a.tw, a.tw1);
        if (a.final_axis && a.pot) {   // imaginary time: the second half-step; l = j + M1 k
            const int i = (int)(col / a.ny), y = (int)(col % a.ny);
            const T vcol = a.vx[i] + a.vy[y];
            T V[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) V[k] = vcol + a.vz[j + F::M1 * k];
            if (a.v3d) {
                const T *__restrict__ v3 = a.v3d + col;
#pragma unroll
                for (int k = 0; k < 16; ++k) V[k] += v3[(long)(j + F::M1 * k) * ls];
            }
            potential16<T, IMAG>(v, V, a.g, a.half_dt);
        }
#pragma unroll
        for (int k = 0; k < 16; ++k) p[(long)(j + F::M1 * k) * ls] = v[k];
        if (a.final_axis && a.sums) {
            // One partial per CTA, added up by k3_finalize after the pass.  A fence + counter + broadcast at the end of
            // every CTA (the last-CTA pattern of reduce_ctas) held each CTA slot ~3 us longer: 124 instead of 82 us for
            // this pass at 256^3 complex64; publishing the partial before the stores, as pass C of the 2-D path does,
            // recovered only part of it (step 261 against 247 us).
            // The 16 terms of a thread in T (one conversion per thread), the rest in double.
            __shared__ double red[32];
            T part = T(0);
#pragma unroll
            for (int k = 0; k < 16; ++k) part = fma(v[k].x, v[k].x, fma(v[k].y, v[k].y, part));
            const double acc = warp_sum((double)part);
            if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
            __syncthreads();
            if (threadIdx.x == 0) {
                double t = 0.0;
                for (int q = 0; q < G::THREADS / 32; ++q) t += red[q];
                a.partials[blockIdx.y * gridDim.x + blockIdx.x] = t;
            }
        }
    }
}

// one CTA: the partial sums of the last pass in a fixed order, then the end of the step (finalize3)
template <bool IMAG>
__global__ void __launch_bounds__(256) k3_finalize(State3 *st, const double *partials, unsigned int n, double dV,
                                                   long long step_index, double *record, int *nonfinite) {
    __shared__ double red[8];
    pdl_launch_dependents();
    pdl_wait();
    double t = 0.0;
    for (unsigned int q0 = threadIdx.x; q0 < n; q0 += 4 * 256) {   // four loads in flight per thread, fixed order of the adds
        double u[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { const unsigned int q = q0 + 256u * k; u[k] = q < n ? __ldcg(partials + q) : 0.0; }
#pragma unroll
        for (int k = 0; k < 4; ++k) t += u[k];
    }
    t = warp_sum(t);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double total = 0.0;
        for (int q = 0; q < 8; ++q) total += red[q];
        finalize3<IMAG>(st, total, dV, step_index, record, nonfinite);
    }
}

// ---------------------------------------------------------------- point-wise kernels
// MODE 0: psi <- psi * exp(-i (V + g|psi|^2) dt/2) (the closing half-step of a real-time call)
// MODE 1: psi <- psi * scale (end of an imaginary-time call; the scale is reset by the next kernel on the stream)
// Four independent points per thread and iteration, so that four loads are in flight per thread.
template <typename T, int MODE>
__global__ void __launch_bounds__(256) k3_point(const Args3<T> a) {
    const long slab = (long)a.nx * a.ny, npts = slab * a.nz, stride = (long)gridDim.x * blockDim.x;
    const T s = MODE == 1 ? (T)a.st->scale : T(1);
    for (long q0 = (long)blockIdx.x * blockDim.x + threadIdx.x; q0 < npts; q0 += 4 * stride) {
        cx<T> z[4];
        T V[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const long q = q0 + k * stride;
            z[k] = q < npts ? a.psi[q] : mk<T>(T(0), T(0));
            if constexpr (MODE == 0) V[k] = (q < npts && a.v3d) ? a.v3d[q] : T(0);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const long q = q0 + k * stride;
            if (q >= npts) break;
            if constexpr (MODE == 1) { z[k].x *= s; z[k].y *= s; }
            else {
                const int l = (int)(q / slab), rem = (int)(q % slab), i = rem / a.ny, y = rem % a.ny;
                const T Vt = V[k] + a.vz[l] + a.vx[i] + a.vy[y];
                const T w = fma(a.g, z[k].x * z[k].x + z[k].y * z[k].y, Vt) * a.half_dt;
                T sn, cm1;
                sincosm1_t(-w, &sn, &cm1);
                const T ox = fma(z[k].x, cm1, fma(-z[k].y, sn, z[k].x)), oy = fma(z[k].x, sn, fma(z[k].y, cm1, z[k].y));
                z[k].x = ox; z[k].y = oy;
            }
            a.psi[q] = z[k];
        }
    }
}

// observables that need no transform: out6 = sums of {|psi|^2, V|psi|^2, (g/2)|psi|^4, x^2|psi|^2, y^2|psi|^2, z^2|psi|^2}
// (coordinates x_i = -Lx/2 + i Lx/nx); one partial sextet per CTA, added by the host in CTA order.
template <typename T>
__global__ void __launch_bounds__(256) k3_observe(const Args3<T> a, double Lx, double Ly, double Lz, double *part6) {
    __shared__ double red[6][8];
    const long slab = (long)a.nx * a.ny, npts = slab * a.nz;
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (long q = (long)blockIdx.x * blockDim.x + threadIdx.x; q < npts; q += (long)gridDim.x * blockDim.x) {
        const cx<T> z = a.psi[q];
        const int l = (int)(q / slab), rem = (int)(q % slab), i = rem / a.ny, y = rem % a.ny;
        double V = (double)a.vz[l] + (double)a.vx[i] + (double)a.vy[y];
        if (a.v3d) V += (double)a.v3d[q];
        const double d = (double)z.x * (double)z.x + (double)z.y * (double)z.y;
        const double X = -0.5 * Lx + (double)i * Lx / (double)a.nx, Y = -0.5 * Ly + (double)y * Ly / (double)a.ny,
                     Z = -0.5 * Lz + (double)l * Lz / (double)a.nz;
        s[0] += d; s[1] += V * d; s[2] += 0.5 * (double)a.g * d * d; s[3] += X * X * d; s[4] += Y * Y * d; s[5] += Z * Z * d;
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int m = 0; m < 6; ++m) {
        const double t = warp_sum(s[m]);
        if (lane == 0) red[m][w] = t;
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double t = 0.0;
        for (int q = 0; q < 8; ++q) t += red[threadIdx.x][q];
        part6[(size_t)blockIdx.x * 6 + threadIdx.x] = t;
    }
}

// kinetic tables of one axis, written on the stream (fp64 arithmetic, rounded once): see k_make_kinetic (gpe_api.cu)
//   imag: kin[q] = exp(-k^2 dt/2)/n; real time: kin[q] = (exp(-i k^2 dt/2) - 1)/n (complex); k2[q] = k^2
template <typename T>
__global__ void k3_make_tables(T *kin, T *k2, int n, double L, double dt, int imag) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    const double k = 2.0 * 3.14159265358979323846 * (double)(q < n / 2 ? q : q - n) / L, w = k * k * dt * 0.5, inv = 1.0 / (double)n;
    if (k2) k2[q] = (T)(k * k);
    if (!kin) return;
    if (imag) kin[q] = (T)(exp(-w) * inv);
    else {
        const double sh = sin(0.5 * w);
        kin[2 * q] = (T)(-2.0 * sh * sh * inv);
        kin[2 * q + 1] = (T)(-sin(w) * inv);
    }
}

// ---------------------------------------------------------------- launchers of one (dtype, N)
template <typename T> struct Ops3 {
    cudaError_t (*row)(const Args3<T> &, bool imag, int mode, cudaStream_t);                 // ny == N
    // line length == N; cols columns per slab, slabs of them; returns the number of CTAs (= partial sums) in *nctas
    cudaError_t (*col)(const Args3<T> &, bool imag, int mode, long cols, unsigned slabs, unsigned *nctas, cudaStream_t);
};

template <typename T, int N> struct Launch3 {
    using C = cx<T>;
    static size_t row_smem() { return sizeof(C) * RowGeom3<N>::RPC * Fft1D<N, 1, C>::SLOTS; }
    template <bool WIDE> static size_t col_smem() { return sizeof(C) * ColGeom3<T, N, WIDE>::W * Fft1D<N, 1, C>::SLOTS; }
    template <typename K> static cudaError_t go(K kern, dim3 grid, unsigned threads, size_t smem, cudaStream_t s, const Args3<T> &a) {
        cudaError_t e = Launch<T, N>::prep(kern, smem);
        if (e != cudaSuccess) return e;
        // grids up to GPE3_PDL_MAX points: the CTAs of a pass may be scheduled while the previous one drains
        // (launch latency and prologue off the critical path); they block in pdl_wait() until it has completed
        const bool pdl = (long)a.nx * a.ny * a.nz <= GPE3_PDL_MAX;
        return launch_pdl(kern, grid, dim3(threads), smem, s, pdl, a);
    }
    static cudaError_t row(const Args3<T> &a, bool imag, int mode, cudaStream_t s) {
        const dim3 grid((unsigned)((long)a.nz * a.nx / RowGeom3<N>::RPC));
        const unsigned th = RowGeom3<N>::THREADS;
        if (mode == 1) return go(k3_row<T, N, false, 1>, grid, th, row_smem(), s, a);
        return imag ? go(k3_row<T, N, true, 0>, grid, th, row_smem(), s, a) : go(k3_row<T, N, false, 0>, grid, th, row_smem(), s, a);
    }
    // the wide tile where the lines of a 256-point column pass are at least 2 MB apart (see ColTarget3)
    static bool col_wide(const Args3<T> &a) { return N == 256 && (size_t)a.line_stride * sizeof(C) >= (size_t)(2u << 20); }
    template <bool WIDE> static cudaError_t col_w(const Args3<T> &a, bool imag, int mode, long cols, unsigned slabs, unsigned *nctas, cudaStream_t s) {
        using G = ColGeom3<T, N, WIDE>;
        const dim3 grid((unsigned)(cols / G::W), slabs);
        if (nctas) *nctas = grid.x * grid.y;
        if (mode == 1) return go(k3_col<T, N, false, 1, WIDE>, grid, G::THREADS, col_smem<WIDE>(), s, a);
        return imag ? go(k3_col<T, N, true, 0, WIDE>, grid, G::THREADS, col_smem<WIDE>(), s, a)
                    : go(k3_col<T, N, false, 0, WIDE>, grid, G::THREADS, col_smem<WIDE>(), s, a);
    }
    static cudaError_t col(const Args3<T> &a, bool imag, int mode, long cols, unsigned slabs, unsigned *nctas, cudaStream_t s) {
        if constexpr (N == 256) { if (col_wide(a)) return col_w<true>(a, imag, mode, cols, slabs, nctas, s); }
        return col_w<false>(a, imag, mode, cols, slabs, nctas, s);
    }
};

#define GPE3_DECL_OPS(N)                  \
    extern const Ops3<float> ops3_f_##N;  \
    extern const Ops3<double> ops3_d_##N;
GPE3_DECL_OPS(64)
GPE3_DECL_OPS(128)
GPE3_DECL_OPS(256)
GPE3_DECL_OPS(512)
GPE3_DECL_OPS(1024)
#undef GPE3_DECL_OPS

template <typename T> inline const Ops3<T> *get_ops3(int n);
template <> inline const Ops3<float> *get_ops3<float>(int n) {
    switch (n) { case 64: return &ops3_f_64; case 128: return &ops3_f_128; case 256: return &ops3_f_256; case 512: return &ops3_f_512; case 1024: return &ops3_f_1024; }
    return nullptr;
}
template <> inline const Ops3<double> *get_ops3<double>(int n) {
    switch (n) { case 64: return &ops3_d_64; case 128: return &ops3_d_128; case 256: return &ops3_d_256; case 512: return &ops3_d_512; case 1024: return &ops3_d_1024; }
    return nullptr;
}

}  // namespace gpe
