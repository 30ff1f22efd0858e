// gpe_types.h -- plain structs shared by the host side (gpe_api.cu) and the kernels.
#pragma once
#include <cuda_runtime.h>

// Paired complex64 passes (gpe_pair.cuh): from this nx on, FOUR rows (not two) are interleaved in the
// intermediate array, so that a column CTA with one column pair still moves 64 contiguous bytes.  A row
// CTA owns two rows, so the passes can then no longer work in place: pass A writes the plan's scratch
// buffer, pass B works inside it, pass C writes psi (gpe_api.cu, evolve_impl).
#ifndef GPE_IL4_MIN_N
#define GPE_IL4_MIN_N 2048
#endif
namespace gpe {

// Per-member device scalars: written by the last block of the
// reducing pass, read by the next pass.  Never read by the host inside gpe_evolve.
struct MemberState {
    double scale;      // lazy renormalisation: the stored psi times `scale` is the wavefunction
    double A;          // schedule amplitude A_n of the upcoming step
    double C;          // cavity coefficient C_n = 2 eta_n Re(alpha_n) of the upcoming step
    double norm;       // sum |psi|^2 dx dy of the current wavefunction
    double theta;      // cavity overlap Theta (Eq. 14)
    double re_alpha, im_alpha;
    long long step;    // step counter n
    // real-time merged half-steps (gpe_pair.cuh): when pend == 1 the stored psi still lacks the
    // second potential half-step of the step just taken, whose coefficients are A_pend, C_pend
    double A_pend, C_pend;
    int pend;
    // coefficients of step `step + 1` that do not depend on the sums, prepared by one thread of
    // pass B while the step runs (prepare_member), so the last block of pass C has little left to do:
    // A_{n+1}; Re alpha = nKre Theta, Im alpha = nKim Theta, C = nKc Theta
    double nA, nKre, nKim, nKc;
    double nPre, nPim, nPc;   // probe: alpha += nPre + i nPim, C += nPc (zero without a probe)
    // full cavity model (Eq. 12): coefficient D_n = U0 |alpha_n|^2 of cos^2(k_c x) of the
    // upcoming step, and the one of the pending half-step
    double D, D_pend;
};

// Per-gpe_evolve-call parameters kept in device memory (written by the prologue kernel), so that
// the kernel arguments of a step do not change from call to call and its CUDA graph is reusable.
struct CallParams {
    long long record_every, rec_first;  // rec_first = floor(step0 / record_every)
    double *records;                    // [n_rec][batch][6] or nullptr
};

// Everything the finalising block needs (schedule, cavity parameters, records).
struct FinalizeParams {
    MemberState *st;          // [batch]
    double2 *partials;        // [batch][cpm] (sum |psi|^2, sum cos cos |psi|^2)
    double *partials_b;       // [batch][cpm] sum cos^2(k_c x) |psi|^2 (full cavity model only)
    unsigned int *counters;   // [batch]
    int *nonfinite;           // sticky flag
    int cpm;                  // CTAs per member in the reducing pass
    int sched_len;
    const double *sched_step; // [sched_len]
    const double *sched_amp;  // [sched_len] or [batch][sched_len]
    int sched_batched;
    double sched_mid;         // 0, or 0.5: sample the schedule at the middle of the step
    int cavity_on, eta_mode;
    const double *eta_or_u, *n_atoms, *delta, *kappa;  // [batch]
    const double *probe_omega, *probe_delta, *probe_phi;  // [batch] or nullptr (Eq. 17)
    const double *cav_u0;     // [batch] U0 of Eqs. 12 and 15, or nullptr (three-term model)
    double probe_dt;          // dt of the running real-time evolution; 0 = no probe (imaginary time)
    double dxdy;
    long long record_every, rec_first;  // prologue only (advance == 0): copied into *call
    double *records;          // prologue only
    CallParams *call;         // device; read by the step kernels
    int batch;
    int normalise;            // 1: imaginary-time step (scale <- 1/sqrt(norm), Theta /= norm)
    int advance;              // 1: a step was taken (step += 1); 0: prologue reduction
    int prepared;             // 1: pass B has run prepare_member for the step being finalised
    int merged;               // 1: pass C left the second half-step pending (real time, paired passes)
    int tvt;                  // 1: T/2 V T/2 ordering in real time: the pending factor takes the coefficients of THIS psi
    long long step0;          // used when advance == 0: sets the step counter
    // T/2 V T/2 in imaginary time with merged kinetic halves (gpe_api.cu): pass B leaves per-CTA partial sums of
    // |psi^ h / P|^2 (h = half a kinetic step) in partials_k; the last block of pass C takes the norm from them,
    // norm = kscale * sum * dxdy (kscale = nx ny), instead of from its own real-space sum
    int knorm, cpmk;
    double kscale;
    double *partials_k;       // [batch][cpmk]
};

enum : int {
    F_HAS_V2D = 1,    // general 2-D static potential array
    F_V2D_BATCHED = 2,
    F_HAS_SEP = 4,    // separable static part vx[i] + vy[j]
    F_LAT_X = 8,      // A cos^2(k_l x)
    F_LAT_Y = 16,     // A cos^2(k_l y)
    F_CAVITY = 32,
    F_HAS_G = 64,
    F_NO_POT = 128,   // plain FFT pass (observables)
    F_CAV_FULL = 256  // cavity lattice D_n cos^2(k_c x) and dispersive shift (needs the third sum)
};

// Arguments of the three passes of one step.  T = float / double.
template <typename T, typename C> struct StepArgs {
    const C *src;  // [batch][nx][ny]
    C *dst;        // same buffer as src inside gpe_evolve
    int nx, ny, batch, flags;
    const T *v2d;                  // [nx][ny] or [batch][nx][ny]
    const T *vx, *vy;              // separable static part
    const T *latx, *laty;          // cos^2(k_l x_i), cos^2(k_l y_j)
    const T *cavx, *cavy;          // cos(k_c x_i), cos(k_c y_j)
    const T *ytab;                 // [ny][4] = {vy[j], cos^2(k_l y_j), cos(k_c y_j), 0}: one 4-vector load per point
    const T *g;                    // [batch]
    T half_dt;                     // dt/2
    const C *tw_x, *tw_y;          // exp(-2 pi i m / nx), exp(-2 pi i m / ny)
    const C *tw1_x, *tw1_y;        // first-stage twiddles transposed: [16][n/16], exp(-2 pi i k j / n)
    const C *tw1e_x, *tw1e_y;      // the same for eight points per thread: [8][n/8] (cluster kernel, n <= 256)
    const C *tw_hy, *tw1_hy;       // the same two tables for length ny/2 (paired row passes, gpe_pair.cuh)
    const T *ytab2;                // [ny/2][8] = {vy[n], vy[n+ny/2], lat[n], lat[n+ny/2], cav[n], cav[n+ny/2], 0, 0}
    const C *kin_xc, *kin_yc;      // real time: (exp(-i kx^2 dt/2) - 1)/(nx ny), exp(-i ky^2 dt/2) - 1
    const T *kin_y2;               // real time, paired column pass: per column pair {1+bx0, 1+bx1, by0, by1, bx0/P, bx1/P, by0/P, by1/P}, b = exp(-i ky^2 dt/2) - 1
    T inv_p;                       // 1/(nx ny)
    const T *kin_xr, *kin_yr;      // imaginary time: exp(-kx^2 dt/2)/(nx ny), exp(-ky^2 dt/2)
    FinalizeParams fin;
};

}  // namespace gpe
