/*
 * gpe.h -- C ABI of libgpe: symmetric split-step Fourier propagation of the 2-D
 * Gross-Pitaevskii equation on one NVIDIA B200 (sm_100a).
 *
 * What the library computes is the method of arXiv 2404.14401 (TorchGPE), cited below as
 * PAPER.md:<line> (the copy under /root/reference), in the readings listed in DESIGN.md:
 *
 *   i d(psi)/dt = [ -1/2 nabla^2 + V_ext(r,t,psi) + g |psi|^2 ] psi          (Eq. 1)
 *
 * hbar = m = 1 (oscillator units).  One step of size dt is the Strang
 * splitting V/2 . T . V/2 (Eqs. 2-4; order of factors: DESIGN.md reading Q1):
 *   psi <- psi * exp(-s (V_n + g|psi|^2) dt/2)        s = i (real time), s = 1 (imaginary time)
 *   psi <- IFFT2[ exp(-s (kx^2+ky^2) dt/2) * FFT2[psi] ]
 *   psi <- psi * exp(-s (V_n + g|psi|^2) dt/2)        |psi|^2 recomputed
 *   imaginary time: psi <- psi / sqrt(sum |psi|^2 dx dy) after every step
 * with V_n(x,y) = V_static(x,y) + A_n cos^2(k_l r_axis) + C_n cos(k_c x) cos(k_c y)
 * (PAPER.md:154 Eq. 9, :175-179 Eqs. 11, 13), A_n a piecewise-linear schedule sampled at the
 * start of step n, and the self-consistent cavity coefficient recomputed once per step from
 * the current density (Eq. 14):
 *   Theta_n = sum cos(k_c x) cos(k_c y) |psi_n|^2 dx dy
 *   alpha_n = N_at eta_n Theta_n / (Delta + i kappa),  C_n = 2 eta_n Re(alpha_n),
 *   eta_n = eta (eta_mode 0) or sqrt(|A_n| u) (eta_mode 1; eta = sqrt(V0 U0) in Eq. 13).
 * Optional (gpe_potential_desc.cav_u0, off in BASELINE.json's configs, reading Q6): the full
 * cavity model adds the cavity lattice U_0 |alpha_n|^2 cos^2(k_c x) (Eq. 12) and the dispersive shift
 * Delta -> Delta - N_at U_0 sum cos^2(k_c x)|psi_n|^2 dx dy (Eq. 15; the printed equation has no N_at:
 * with psi normalised to 1 the atom number is explicit, reading Q5).
 *
 * Grid: x_i = -Lx/2 + i Lx/nx, i = 0..nx-1 (periodic), likewise y_j; psi is stored
 * [batch][nx][ny], y fastest, interleaved (re, im); integrals are sums times dx dy.
 * FFT convention: forward unnormalised with exp(-i(kx x + ky y)), inverse with 1/(nx ny).
 *
 * All pointers named *_dev / marked DEVICE are CUDA device pointers on the current device;
 * all others are host pointers.  Nothing here takes or returns a torch / C++ type.
 * Every call returns a gpe_status and never throws; gpe_last_error() gives the text of the
 * last failure on that plan.  The library has no CPU fallback: without a CUDA device every
 * compute call returns GPE_ECUDA.
 */
#ifndef GPE_H
#define GPE_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define GPE_API __attribute__((visibility("default")))
#else
#define GPE_API
#endif

typedef struct gpe_plan gpe_plan; /* opaque; owns tables, workspace and the device scalar block */

typedef enum { GPE_C64 = 0, GPE_C128 = 1 } gpe_dtype;     /* complex64 / complex128 */
typedef enum { GPE_REAL_TIME = 0, GPE_IMAG_TIME = 1 } gpe_mode;
typedef enum {
    GPE_OK = 0,
    GPE_EINVAL = 1,       /* bad argument (NULL, non-finite, misaligned, wrong size) */
    GPE_EUNSUPPORTED = 2, /* nx or ny outside the supported sizes (see gpe_plan_create) */
    GPE_ENOMEM = 3,       /* host or device allocation failed */
    GPE_ECUDA = 4,        /* a CUDA runtime call failed (text in gpe_last_error) */
    GPE_ESTATE = 5,       /* call order: gpe_evolve / gpe_observables before gpe_set_potential */
    GPE_ENONFINITE = 6    /* the device saw a non-finite norm during an earlier gpe_evolve */
} gpe_status;

#define GPE_NREC 6 /* doubles per record: {step, norm, theta, re_alpha, im_alpha, A} */

/* Bumped whenever a struct layout or a signature below changes; the Python binding refuses to run
 * against a library whose gpe_abi_version() or gpe_sizeof_potential_desc() differ from its own. */
#define GPE_ABI_VERSION 4

/*
 * gpe_plan_create -- the discretised problem of Eq. 1: an nx x ny periodic grid
 * over the box [-Lx/2, Lx/2) x [-Ly/2, Ly/2), `batch` independent wavefunctions (parameter
 * sweeps, north_star (4)).  nx, ny in [64, 2048], even, with no prime factor above 5, else
 * GPE_EUNSUPPORTED.  Powers of two run the fast kernels (the paper benchmarks powers of two and notes
 * only that other sizes are slower); any other allowed size runs mixed-radix passes
 * (radices 8, 5, 4, 3, 2), about an order of magnitude slower per point, without ordering = 1 and
 * without gpe_profile_passes.  Lx, Ly > 0 and finite, batch >= 1, else GPE_EINVAL.
 * Allocates the twiddle / wavenumber tables and the per-member device scalars on the current
 * device.  *out is set only on GPE_OK and is released with gpe_plan_destroy.
 */
GPE_API gpe_status gpe_plan_create(gpe_plan **out, int nx, int ny, double Lx, double Ly, gpe_dtype dtype,
                           int batch);

/* All work of the plan is enqueued on this cudaStream_t (default: the legacy stream 0). */
GPE_API gpe_status gpe_plan_set_stream(gpe_plan *p, void *cuda_stream);

/* Frees everything the plan owns (synchronises its stream first).  NULL is a no-op. */
GPE_API gpe_status gpe_plan_destroy(gpe_plan *p);

/*
 * gpe_potential_desc -- V_ext of Eq. 1 in the fixed form used by the paper's examples
 * (PAPER.md:154 Eq. 9; :170-186 Eqs. 10, 11, 13, 14) plus the contact coupling g.
 * "real" below is float for GPE_C64 and double for GPE_C128.
 */
typedef struct {
    const void *v_static;     /* DEVICE real [nx][ny] (or [batch][nx][ny]); NULL = none          */
    int v_static_batched;     /* 0: one array shared by all members; 1: one per member           */
    const double *vx, *vy;    /* HOST, optional separable static part vx[i] + vy[j]; NULL = none
                                 (added to v_static if both are given)                           */
    const double *g;          /* HOST [batch] contact coupling, norm-1 convention; NULL = 0      */
    int lattice_axis;         /* -1 none; 0: A cos^2(k_l x); 1: A cos^2(k_l y)   (Eqs. 9, 11)    */
    double lattice_k;
    int sched_len;            /* knots of the piecewise-linear amplitude A(step); 0 = A == 0     */
    const double *sched_step; /* HOST [sched_len], non-decreasing, in units of steps. A_n is
                                 interpolated on the segment starting at the LAST knot with
                                 step <= n; constant before the first and after the last knot   */
    const double *sched_amp;  /* HOST [sched_len], or [batch][sched_len] if sched_batched        */
    int sched_batched;
    int cavity_on;            /* adds C_n cos(k_c x) cos(k_c y)                  (Eqs. 13, 14)   */
    double cavity_k;
    int eta_mode;             /* 0: eta given; 1: eta_n = sqrt(|A_n| u)                          */
    const double *eta_or_u;   /* HOST [batch] (required if cavity_on)                            */
    const double *n_atoms;    /* HOST [batch] N_at of Eq. 14; NULL = 1                           */
    const double *delta;      /* HOST [batch] cavity detuning Delta (required if cavity_on)      */
    const double *kappa;      /* HOST [batch] cavity decay kappa  (required if cavity_on)        */
    /* On-axis cavity probe (Eq. 17), real time only (ignored in imaginary time):
     * alpha'_n = alpha_n + Omega_c exp(i (Delta_p t_n + phi)) / (Delta + i kappa), t_n = n dt, n the
     * plan's step counter; alpha' replaces alpha in C_n = 2 eta_n Re(alpha'_n) (Eq. 18) and in the
     * records.  gpe_observables reports the self-consistent alpha_n without the probe.  All three
     * NULL = no probe; otherwise probe_omega is required, the other two default to 0.  Needs cavity_on. */
    const double *probe_omega; /* HOST [batch] Omega_c                                            */
    const double *probe_delta; /* HOST [batch] Delta_p                                            */
    const double *probe_phi;   /* HOST [batch] phi                                                */
    /* Full cavity model (Eqs. 12 and 15): with U_0 = cav_u0[b] the potential gains the
     * cavity lattice U_0 |alpha_n|^2 cos^2(k_c x) and Delta is replaced, in alpha_n and in the probe,
     * by Delta - N_at U_0 B_n, B_n = sum cos^2(k_c x)|psi_n|^2 dx dy (a third fused reduction).
     * NULL = the three-term model.  Needs cavity_on. */
    const double *cav_u0;      /* HOST [batch]                                                    */
    /* 1: the schedule amplitude of step n is sampled at the middle of the step, A(n + 1/2), instead
     * of its start A(n) (reading Q4); records and observables report the same sample. */
    int sched_midpoint;
    /* Order of the factors of one step (reading Q1).  0 (default): V/2 T V/2 as north_star
     * spells out.  1: T/2 V T/2, the form the paper prints (Eqs. 3-4): half a kinetic
     * step, then A_n, Theta_n, alpha_n and |psi|^2 taken from the psi that ENTERS the potential factor,
     * one full factor exp(-sigma (V_n + g|psi|^2) dt), half a kinetic step, and in imaginary time the
     * renormalisation.  Both time modes run three fused passes per step (adjacent kinetic halves merge --
     * in imaginary time around the renormalisation, whose norm is then taken in k space; one extra
     * kinetic-only unit per call and per record boundary).  With ordering = 1 gpe_evolve fills a second
     * set of kinetic tables (dt/2) on the device the first time a (dt, mode) pair is seen.  Powers of two only. */
    int ordering;
} gpe_potential_desc;

/*
 * gpe_set_potential -- copies everything it needs (the caller may free all arrays on return;
 * the device array v_static is copied device-to-device on the plan's stream).  May be called
 * again at any time between gpe_evolve calls.  GPE_EINVAL on inconsistent fields: all of them are
 * checked before the plan is touched, so the previous potential stays in force.  A CUDA failure while
 * the new one is being uploaded leaves the plan without a potential (GPE_ESTATE until the next
 * successful call).  Synchronises the plan's stream.
 */
GPE_API gpe_status gpe_set_potential(gpe_plan *p, const gpe_potential_desc *d);

/*
 * gpe_evolve -- n_steps split-step steps (see the top of this file) in place on
 * psi: DEVICE [batch][nx][ny] complex of the plan's dtype, 16-byte aligned, caller-owned.
 * dt: time step; must be finite and non-zero, and > 0 for GPE_IMAG_TIME.
 * The plan keeps a step counter n (time origin of the schedule, A_n = A(n)); it starts at 0,
 * advances by n_steps per call and is read / set with gpe_get_step / gpe_set_step.
 * record_every > 0: after every step whose new counter value is a multiple of record_every,
 * GPE_NREC doubles per member are written to
 * records: DEVICE [n_rec][batch][GPE_NREC] = {step, norm, Theta, Re alpha, Im alpha, A}, evaluated on
 * the wavefunction after that step (after the renormalisation in imaginary time), with
 * n_rec = floor((n0+n_steps)/record_every) - floor(n0/record_every).  record_every = 0: none.
 * The call only ENQUEUES work on the plan's stream: no host synchronisation (the kinetic tables of a
 * new (dt, mode) pair are written by a kernel on the same stream, nothing is allocated), no host
 * round trip of the per-step scalars (norm, Theta, alpha live in device memory; north_star (3)).
 * The plan's device must be current (GPE_EINVAL otherwise; this holds for every call on a plan).
 * How the steps are run is chosen per call and does not change what is computed: three
 * fused passes per step; two where no global scalar sits between pass C and the next pass A (real time without the
 * cavity term; imaginary time with g = 0 and no cavity term); every step inside ONE thread-block-cluster kernel for
 * square grids up to 256^2; mixed-radix passes for sizes that are not powers of two.
 * GPE_ESTATE before gpe_set_potential; GPE_EINVAL on bad arguments; GPE_ECUDA on launch errors;
 * GPE_EUNSUPPORTED for ordering = 1 on a size that is not a power of two.
 */
GPE_API gpe_status gpe_evolve(gpe_plan *p, void *psi_dev, double dt, long n_steps, gpe_mode mode,
                      long record_every, double *records_dev);

/*
 * gpe_observables -- norm, energies and cavity quantities of psi:
 *   norm  = sum |psi|^2 dx dy
 *   e_kin = 1/2 sum (kx^2+ky^2)|psi^|^2 / sum |psi^|^2 * norm
 *   e_pot = sum (V_static + A_n cos^2) |psi|^2 dx dy          (n = the plan's step counter)
 *   e_int = g/2 sum |psi|^4 dx dy
 *   e_cav = N_at eta_n^2 Theta^2 Delta / (Delta^2 + kappa^2)  [Delta -> Delta~ with cav_u0]  (its functional derivative is
 *           the interference potential of Eq. 13)
 *   theta, re_alpha, im_alpha as in Eq. 14.
 * out_host: HOST [batch].  density_dev (DEVICE real [batch][nx][ny], or NULL): |psi|^2.
 * kdensity_dev (DEVICE real [batch][nx][ny], or NULL): |psi^|^2 / sum |psi^|^2 in FFT order
 * ("directly from the wave-function amplitude in reciprocal space").
 * Synchronises the plan's stream (it returns host values).  psi is not modified.
 * Returns GPE_ENONFINITE if an earlier gpe_evolve on this plan produced a non-finite norm: reported
 * ONCE (the flag is then cleared); out_host and the density buffers are filled all the same.
 */
typedef struct {
    double norm, e_kin, e_pot, e_int, e_cav, theta, re_alpha, im_alpha;
} gpe_obs;
GPE_API gpe_status gpe_observables(gpe_plan *p, const void *psi_dev, gpe_obs *out_host, void *density_dev,
                           void *kdensity_dev);

/*
 * gpe_populations -- momentum-order populations after a lattice pulse:
 *   out_host[b][m + m_max] = sum over |k_axis - 2 m k_l| < k_l (all k on the other axis)
 *                            of |psi^|^2 / sum |psi^|^2,   m = -m_max .. m_max
 * axis: 0 (x) or 1 (y).  out_host: HOST [batch][2 m_max + 1].  Synchronises the stream.
 */
GPE_API gpe_status gpe_populations(gpe_plan *p, const void *psi_dev, int axis, double k_l, int m_max,
                           double *out_host);

/*
 * gpe_fft2_forward -- the library's own forward 2-D FFT on its own: for every
 * member dst[p][q] = sum_{ij} src[i][j] exp(-2 pi i (p i / nx + q j / ny)), unnormalised, natural
 * (fftfreq) order.  src, dst: DEVICE [batch][nx][ny] complex of the plan's dtype; dst may equal
 * src.  Enqueued on the plan's stream, no synchronisation.  Used by the observables and exposed
 * so the transform can be tested alone.
 */
GPE_API gpe_status gpe_fft2_forward(gpe_plan *p, const void *src_dev, void *dst_dev);

/*
 * gpe_profile_passes -- measurement aid for the roofline report: runs n_steps
 * steps exactly as gpe_evolve does (psi evolves, the step counter advances, no records), with
 * CUDA events on the plan's stream around ONE of the three fused passes per step (round-robin),
 * and returns the mean device time per launch in milliseconds:
 * ms_out_host[0] = pass A (potential half-step + FFT along y), [1] = pass B (FFT along x, kinetic
 * factor, inverse FFT along x), [2] = pass C (inverse FFT along y, potential half-step, fused
 * norm / overlap reduction and scalar update).  3 <= n_steps <= 30000.  Synchronises the stream.
 */
GPE_API gpe_status gpe_profile_passes(gpe_plan *p, void *psi_dev, double dt, long n_steps, gpe_mode mode,
                              double *ms_out_host);

/*
 * gpe_measure_roofs -- the denominators of the roofline report, measured on the current device
 * ("L2 peak is not in MEASURED_PEAKS.json -- the builder measures it"; plain-ALU rates
 * "to be replaced by a measured FMA-loop probe").  Not part of the method.  out_host[5] =
 *   [0] GB/s of an in-place read + write (128-bit accesses, persistent CTAs) over a 32 MiB buffer --
 *       the size of the 2048^2 complex64 wavefunction, resident in L2 --, [1] the same over 64 MiB
 *       (2048^2 complex128), [2] the same over 1 GiB (HBM),
 *   [3] Tflop/s of independent fp32 fused multiply-add chains, [4] the same in fp64.
 * Runs on cuda_stream and synchronises it.  GPE_ENOMEM if the 1 GiB scratch buffer cannot be had.
 */
GPE_API gpe_status gpe_measure_roofs(void *cuda_stream, double *out_host);

/* Step counter n (schedule time origin); see gpe_evolve.  n >= 0: gpe_set_step returns GPE_EINVAL for a
 * negative value (shift the schedule knots instead). */
GPE_API gpe_status gpe_get_step(const gpe_plan *p, long *step);
GPE_API gpe_status gpe_set_step(gpe_plan *p, long step);

/* Text of the last error on this plan ("" if none).  p == NULL: text of the last
 * gpe_plan_create failure on this thread.  The pointer stays valid until the next call. */
GPE_API const char *gpe_last_error(const gpe_plan *p);

/*
 * gpe_norm_theta_noalloc -- the fused norm / cavity-overlap reduction of one step (PAPER.md:116 and PAPER.md:183,
 * Eq. 14) as an entry point that ALLOCATES NOTHING: no plan, no cudaMalloc / cudaFree inside.  For callers that
 * cannot allocate (CUDA graph capture, tight serving loops).  For every member b of
 * psi_dev: DEVICE [batch][nx][ny] complex (dtype; aligned to one complex number), grid as in gpe_plan_create,
 *   out_dev[b][0] = sum |psi|^2 dx dy,   out_dev[b][1] = sum cos(k x_i) cos(k y_j) |psi|^2 dx dy   (k = cavity_k)
 * out_dev: DEVICE [batch][2] doubles, 16-byte aligned, caller-owned.  Enqueued on cuda_stream, no synchronisation.
 * Scratch (per-CTA partial sums and counters) is a fixed 65 792-byte device array inside the library, held by every
 * GPU that loads it; hence the limits batch <= 64 and nx, ny <= 4096 (GPE_EUNSUPPORTED beyond, GPE_EINVAL on bad
 * arguments; text from gpe_noalloc_last_error).  Every call shares that array: calls that overlap on the GPU
 * (different streams or threads) race and must be serialised by the caller.
 */
GPE_API gpe_status gpe_norm_theta_noalloc(const void *psi_dev, int nx, int ny, double Lx, double Ly, gpe_dtype dtype,
                                          int batch, double cavity_k, double *out_dev, void *cuda_stream);
GPE_API const char *gpe_noalloc_last_error(void);

/*
 * ---- Three dimensions (second half; the first item of the paper's outlook) ----
 * The same split-step (Eqs. 2-4; imaginary time PAPER.md:112-116) for ONE wavefunction on an
 * nx x ny x nz periodic grid over [-Lx/2, Lx/2) x [-Ly/2, Ly/2) x [-Lz/2, Lz/2):
 *   psi <- exp(-s (V + g|psi|^2) dt/2)  IFFT3[ exp(-s |k|^2 dt/2) FFT3[ exp(-s (V + g|psi|^2) dt/2) psi ] ],
 * s = i (real time) or 1 (imaginary time, followed by psi <- psi / sqrt(sum |psi|^2 dx dy dz)); the second
 * potential factor takes |psi|^2 of the psi that enters it.  V = v_static + vx[i] + vy[j] + vz[l].
 * Layout: psi and v_static are [nz][nx][ny], y fastest, z slowest.  No cavity terms, schedule or batch here.
 * A step is three passes over the array, one per axis (csrc/gpe3_kernels.cuh); nothing is transposed.
 *
 * gpe3_plan_create: nx, ny, nz each one of 64, 128, 256, 512, 1024 (else GPE_EUNSUPPORTED); Lx, Ly, Lz > 0 and finite,
 * dtype as above (else GPE_EINVAL).  Allocates tables and a few KB of reduction scratch on the current device; the
 * caller owns psi.  *out is set only on GPE_OK; release with gpe3_plan_destroy (NULL is accepted).
 */
typedef struct gpe3_plan gpe3_plan;
GPE_API gpe_status gpe3_plan_create(gpe3_plan **out, int nx, int ny, int nz, double Lx, double Ly, double Lz,
                                    gpe_dtype dtype);
GPE_API gpe_status gpe3_plan_set_stream(gpe3_plan *p, void *cuda_stream);   /* all later work of the plan goes there */
GPE_API gpe_status gpe3_plan_destroy(gpe3_plan *p);

/*
 * gpe3_set_potential -- v_static_dev: DEVICE real array [nz][nx][ny] of the plan's real type (float for GPE_C64,
 * double for GPE_C128), or NULL; vx, vy, vz: HOST doubles [nx], [ny], [nz], each may be NULL (= 0); g: contact
 * coupling in the norm-1 convention.  Everything is copied (v_static device-to-device on the plan's stream); the
 * call synchronises the stream.  GPE_EINVAL on a non-finite g / vx / vy / vz or a misaligned v_static_dev.
 */
GPE_API gpe_status gpe3_set_potential(gpe3_plan *p, const void *v_static_dev, const double *vx, const double *vy,
                                      const double *vz, double g);

#define GPE3_NREC 3 /* doubles per record: {step, norm, norm_pre} */
/*
 * gpe3_evolve -- n_steps steps in place on psi_dev: DEVICE [nz][nx][ny] complex of the plan's dtype, 16-byte
 * aligned, caller-owned.  dt finite and non-zero, > 0 in imaginary time.  The plan keeps a step counter
 * (gpe3_get_step / gpe3_set_step) that only numbers the records.  records_dev: DEVICE doubles, NULL or
 * [n_rec][GPE3_NREC] with n_rec = floor((step + n_steps) / record_every) - floor(step / record_every): after every
 * step whose index is a multiple of record_every, {index, sum |psi|^2 dV, the same sum before that step's
 * renormalisation} (the two are equal in real time; in imaginary time the second gives the chemical potential
 * estimate -log(norm_pre) / (2 dt)).  The call only ENQUEUES work on the plan's stream and returns; errors of the
 * device side (a non-finite or zero norm) are reported by the next gpe3_synchronize.
 * GPE_ESTATE before gpe3_set_potential or on another device than the plan's; GPE_EINVAL on bad arguments.
 */
GPE_API gpe_status gpe3_evolve(gpe3_plan *p, void *psi_dev, double dt, long long n_steps, gpe_mode mode,
                               long long record_every, double *records_dev);

/*
 * gpe3_observables -- out_host[8] = {norm, e_kin, e_pot, e_int, <x^2>, <y^2>, <z^2>, 0} of psi_dev (not modified):
 * norm = sum |psi|^2 dV, e_kin = (1/2) sum |k|^2 |psi^|^2 / sum |psi^|^2 * norm, e_pot = sum V |psi|^2 dV,
 * e_int = (g/2) sum |psi|^4 dV, <x^2> = sum x_i^2 |psi|^2 dV (not divided by the norm).  Synchronises the stream.
 */
GPE_API gpe_status gpe3_observables(gpe3_plan *p, const void *psi_dev, double *out_host);

/* Waits for the plan's stream; GPE_ENONFINITE (once) if an earlier gpe3_evolve saw a non-finite or zero norm. */
GPE_API gpe_status gpe3_synchronize(gpe3_plan *p);
GPE_API gpe_status gpe3_get_step(const gpe3_plan *p, long long *step);
GPE_API gpe_status gpe3_set_step(gpe3_plan *p, long long step);   /* GPE_EINVAL for step < 0 */
/* Text of the last error of the plan, or of the last failed gpe3_plan_create of this thread when p is NULL. */
GPE_API const char *gpe3_last_error(const gpe3_plan *p);

/* Library build information: "libgpe <version> sm_100a". */
GPE_API const char *gpe_version(void);

/* GPE_ABI_VERSION and sizeof(gpe_potential_desc) of the built library (checked by the binding on load). */
GPE_API int gpe_abi_version(void);
GPE_API size_t gpe_sizeof_potential_desc(void);

#ifdef __cplusplus
}
#endif
#endif /* GPE_H */
