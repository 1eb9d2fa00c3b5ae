/*
 * sso.h -- C ABI of the B200-native Fourier split-operator library.
 *
 * One call of sso_step advances a complex wavefunction (Schroedinger, 1 component)
 * or a Dirac spinor (2 or 4 components) on a regular periodic lattice by `nsteps`
 * Fourier split-operator time steps
 *
 *     w(t+tau) = U_A1(1/2) F^-1{ U~_A2(1) F{ U_A1(1/2) w(t) } }
 *
 * i.e. PAPER.md:71 (eq. 7, Strang factorisation) in the Fourier form of
 * PAPER.md:76 (eq. 8), on the lattice of PAPER.md:80 (all line numbers refer to
 * the paper text, Bauke & Keitel, arXiv:1012.3911).  U_A1 is the position-space
 * phase exp(-i Vbar tau/2) of PAPER.md:98 (eq. 11) / 165 (eq. 22); U~_A2 is, in
 * momentum space, the phase exp(-i tau (k - q Abar)^2 / 2m) of PAPER.md:107
 * (eq. 13) for Schroedinger and the per-k 2x2 / 4x4 unitary
 * exp(-i tau (c alpha.(k - q Abar) + m c^2 beta)) of PAPER.md:203-232
 * (eq. 27-33) and 240-242 (eq. 35) for Dirac.  Units: atomic units, hbar = 1
 * (PAPER.md:323).
 *
 * Conventions:
 *   grid      r_j = (j - n/2) dx per axis, half open, periodic (G14, G18)
 *   momenta   k_j = 2 pi j/(n dx), j < n/2;  2 pi (j-n)/(n dx), j >= n/2 (Nyquist negative)
 *   DFT       forward = exp(-i k.r), unnormalised; inverse carries 1/N (eq. 12)
 *   layout    psi[ncomp][n0][n1][n2], C order, last axis contiguous, interleaved (re, im),
 *             float2 (SSO_C64) or double2 (SSO_C128)
 *   Dirac     ncomp = 4: Dirac representation, PAPER.md:127-129 (eq. 16);
 *             ncomp = 2: alpha_1 = sigma_x, alpha_2 = sigma_y, beta = sigma_z
 *             (eq. 17 and the {1,4} block of eq. 16, reading G7)
 *   fields    time integrals over a step are supplied by the caller as step AVERAGES
 *             (reading G12); both potential half steps of step n use the same average (G13)
 *
 * All device work is enqueued on the caller's CUDA stream (a cudaStream_t passed
 * as void*; NULL = the legacy default stream) and is asynchronous, except
 * sso_norm, sso_step_host and the table uploads of sso_set_*, which synchronise
 * that stream.  There is no CPU fallback: every entry point that needs the GPU
 * fails with SSO_ERR_CUDA when no device is usable.
 *
 * Error behaviour: every function returns an int status (0 = SSO_OK); nothing is
 * thrown across the ABI.  sso_last_error(plan) returns a plan-owned, NUL-terminated
 * description of the most recent failure on that plan (or, for plan == NULL, of the
 * most recent failed sso_plan_create or sso_norm_static on this thread).
 */
#ifndef SSO_H_
#define SSO_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SSO_OK 0
#define SSO_ERR_INVALID 1     /* bad argument (NULL, range, alignment, non-finite)          */
#define SSO_ERR_UNSUPPORTED 2 /* valid request this build does not implement                */
#define SSO_ERR_ALLOC 3       /* host or device allocation failed                           */
#define SSO_ERR_CUDA 4        /* CUDA runtime error, or no device                           */
#define SSO_ERR_STATE 5       /* call sequence error (e.g. field table too short for nsteps) */

#define SSO_C64 0  /* complex64:  float2  */
#define SSO_C128 1 /* complex128: double2 */

#define SSO_FIELD_NONE 0
#define SSO_FIELD_E 1 /* length gauge: adds r . Ebar_n to the potential energy (eq. 11) */
#define SSO_FIELD_A 2 /* velocity gauge, homogeneous A(t): pi = k - q Abar_n in the kinetic factor
                         (eq. 13; for Dirac reading G16)                              */

/* options for sso_set_option */
#define SSO_OPT_LINES_PER_TILE_CONTIG 1  /* lines per CTA in contiguous-axis passes (0 = auto)   */
#define SSO_OPT_LINES_PER_TILE_STRIDED 2 /* adjacent lines per CTA in strided-axis passes (0=auto) */
#define SSO_OPT_POTENTIAL_PHASE 3        /* 0 = complex phase table exp(-i V tau/2) (default),
                                            1 = real angle table + in-kernel sincos.  The plan keeps
                                            no copy of V: CHANGING this option discards the potential,
                                            and sso_step fails with SSO_ERR_STATE until
                                            sso_set_potential has been called again                */
#define SSO_OPT_GROUPS_PER_CTA 4         /* independent line groups per CTA (0 = auto)              */
#define SSO_OPT_RING_BUFFERS 5           /* tile buffers per CTA of the pass pipelines (0 = auto: as many as fit)  */
#define SSO_OPT_THREADS_PER_CTA 6        /* ring pipeline CTA size: 512 (128 regs/thread) or 384 (168); 0 = auto */
#define SSO_OPT_STRIDED_RING 7           /* strided-axis passes: 0 auto, 1 force the TMA ring, 2 direct kernel only */
#define SSO_OPT_DIRAC_TABLE 8            /* Dirac plans without a field, ndim >= 2: 0 = cos(E tau), sin(E tau)/E of every k point
                                            evaluated in the kinetic pass, 1 = read from a table (16 bytes per k point) */
#define SSO_OPT_TILE_ORDER 9              /* order in which the passes walk their tiles: 0 = auto; otherwise value - 1 is a mask of
                                            the passes that go from the highest address down (bit 0 contiguous-axis passes,
                                            1 middle-axis forward, 2 middle-axis inverse, 3 kinetic); results do not depend on it */
#define SSO_OPT_LINES_PER_TILE_MIDDLE 10 /* adjacent lines per tile in the middle-axis passes of a 3D lattice (0 = auto)  */
#define SSO_OPT_CLUSTER_1D 11            /* 1D Schroedinger steps on a thread-block cluster: 0 = auto, 1 = off (single CTA; lattices
                                            beyond SSO_MAX_AXIS then fail), 4 or 8 = CTAs per cluster (needs sizes[0]/value in [512, 4096]) */

#define SSO_MIN_AXIS 16   /* smallest supported axis length                       */
#define SSO_MAX_AXIS 8192 /* largest supported axis length: one CTA of 512 threads holds a line (16 points per thread) */
#define SSO_MAX_AXIS_1D 32768 /* 1D Schroedinger lattices (ncomp = 1, no SSO_FIELD_E, no position-space A): the line is
                                 spread over a thread-block cluster of 8 SMs                                         */

typedef struct sso_plan sso_plan; /* opaque; owned by the library */

/*
 * Create a plan for a lattice of `ndim` (1..3) axes with sizes[a] points (powers
 * of two in [SSO_MIN_AXIS, SSO_MAX_AXIS]; up to SSO_MAX_AXIS_1D for ndim = 1, ncomp = 1) and spacings dx[a] > 0, time step dt
 * (finite, may be negative: the Strang step is symmetric, so -dt undoes +dt),
 * ncomp = 1 (Schroedinger), 2 (Dirac, ndim 1 or 2) or 4 (Dirac, ndim 1..3); a 1D Dirac plan needs
 * ncomp * sizes[0] <= 8192 (SSO_ERR_UNSUPPORTED otherwise).
 * sizes and dx are host arrays, read during the call only.  Builds the radix
 * schedule, twiddle tables and k grids.  Defaults: V = 0, no
 * field, mass 1, c 137.036, charge -1 (electron), time index 0.
 * On failure *out is set to NULL.
 */
int sso_plan_create(sso_plan **out, int ndim, const int64_t *sizes, const double *dx, double dt,
                    int ncomp, int precision);

/* Particle constants m, c, q (eq. 9, 117 eq. 14).  mass > 0, c > 0, all finite. */
int sso_set_constants(sso_plan *plan, double mass, double c, double charge);

/*
 * Real potential ENERGY q phi(r) on the lattice, double[n0][n1][n2] in C order
 * (host pointer if on_device == 0, device pointer otherwise); NULL means V = 0.
 * The array is consumed during the call (the plan keeps its own phase table
 * exp(-i V tau/2), eq. 11 with delta = 1/2); the caller keeps
 * ownership.  Synchronises `stream`.
 */
int sso_set_potential(sso_plan *plan, const double *V, int on_device, void *stream);

/*
 * Homogeneous, time-dependent field.  step_avg is a HOST array
 * double[nvals][ndim]: row n holds the average over [n dt, (n+1) dt] of E(t)
 * (SSO_FIELD_E) or A(t) (SSO_FIELD_A).  Copied; kind SSO_FIELD_NONE ignores the
 * other arguments.  Stepping past row nvals-1 fails with SSO_ERR_STATE.
 */
int sso_set_field(sso_plan *plan, int kind, const double *step_avg, int64_t nvals);

/*
 * Position-dependent vector potential A(r) of a Dirac plan, applied in POSITION space as the paper does
 * (eq. 18a: c sum_i alpha_i (-q A_i(x,t)) belongs to A_1, next to q phi):  both potential half
 * steps of a step also multiply every spinor by
 *     exp(i sum_i a_i alpha_i) = cos a + i (sum_i a_i alpha_i / a) sin a,   a_i = (tau/2) q c A_i(r),  a = |a|
 * (eq. 23/24; with q = -1 this is eq. 26 as printed; eq. 34, in
 * one dimension).  A is the STEP AVERAGE of the field on the lattice (its time integral over a step divided by
 * tau, reading G12), double[ndim][n0][n1][n2] in C order, host or device pointer; copied, the caller keeps
 * ownership; a HOST array is checked for non-finite values (SSO_ERR_INVALID), a DEVICE array is not (a NaN there ends
 * up in psi: the caller's responsibility); it is used for every following step until replaced (a time-dependent A(r,t) is set step by step);
 * NULL switches the factor off.  Independent of SSO_FIELD_A, whose homogeneous A(t) enters the kinetic factor
 * (reading G16); the two splittings agree to O(tau^2).  ncomp = 1 gives SSO_ERR_UNSUPPORTED.  In this version the
 * factor runs as a kernel of its own where psi is in position space on every axis, i.e. before the first and after
 * the last pass of a step: while it is set, consecutive potential half steps are not merged (a 2D step costs an
 * opening, a kinetic and a closing pass) and the factor itself costs one kernel per step inside a call (the closing
 * half of one step and the opening half of the next are one rotation) plus a half rotation at each end of the call.
 * Synchronises `stream`.
 */
int sso_set_vector_potential(sso_plan *plan, const double *A, int on_device, void *stream);

/* Step counter n used to index step_avg (t_n = n dt, reading G21); sso_step advances it. */
int sso_set_time_index(sso_plan *plan, int64_t n);
int sso_get_time_index(const sso_plan *plan, int64_t *n);

/*
 * Advance psi in place by nsteps >= 0 steps.  psi is a DEVICE pointer to
 * ncomp * prod(sizes) complex numbers in the plan's precision, 16-byte aligned;
 * the caller owns it.  Asynchronous on `stream`; only kernels are enqueued (the
 * call can be captured into a CUDA graph), from the first call on: every device
 * table whose shape depends on the configuration is (re)allocated by the call that
 * sets the configuration (sso_plan_create, sso_set_option, sso_set_field,
 * sso_set_potential, sso_set_vector_potential), never by sso_step; if such an
 * allocation failed there, sso_step returns SSO_ERR_STATE instead of allocating.
 * Consecutive potential half steps inside one call are merged into one phase
 * (identical up to rounding).
 */
int sso_step(sso_plan *plan, void *psi, int64_t nsteps, void *stream);

/*
 * Same, for a HOST buffer: copies psi to a plan-owned device buffer, steps,
 * copies back and synchronises (the paper's protocol: one upload before the
 * first step, one download after the last).
 */
int sso_step_host(sso_plan *plan, void *psi_host, int64_t nsteps);

/*
 * *out_host = sum_c sum_r |psi_c(r)|^2 prod(dx), the lattice form of the norm integral of |psi|^2 that every
 * factor of the step preserves (the step is a product of unitary factors, eq. 7 and 76 eq. 8; the
 * paper plots this density).  psi is a DEVICE pointer laid out as for sso_step; the sum is
 * accumulated in double also for SSO_C64, in a fixed order (deterministic).  Synchronises `stream`.
 */
int sso_norm(sso_plan *plan, const void *psi, double *out_host, void *stream);

/*
 * The same norm for callers that cannot allocate device memory -- no plan, no cudaMalloc, no cudaFree, no call into
 * an allocating library, on any call.  Meant for: a process whose own arena (or the framework around it) already
 * owns all of HBM, where an allocation made by this library would simply fail; a time loop that must not stall,
 * since cudaMalloc and cudaFree wait for everything running on the device; a monitor that is handed a pointer to a
 * wavefunction some other component propagates and has no plan of its own (creating one allocates tables).
 *
 *   *out_dev = vol * sum_{i < count} |psi[i]|^2        (the quantity of sso_norm; eq. 7, 76 eq. 8, 331)
 *
 * psi      DEVICE pointer to `count` complex numbers (all components and lattice points of the state, any lattice
 *          shape), float2 for SSO_C64 or double2 for SSO_C128, aligned to one complex number; caller-owned, read only.
 * vol      prod(dx) of the lattice (there is no plan to take it from); finite.
 * out_dev  DEVICE pointer to one double, 8-byte aligned, caller-owned; written by the last kernel of the call.
 * stream   the two kernels are enqueued on it; the call does not wait for them and copies nothing to the host.
 *
 * The per-chunk partial sums (one per SSO_NORM_STATIC_CHUNK elements, accumulated in double in a fixed order, so the
 * result is deterministic and does not depend on the GPU model) go to an array built into the library image, of
 * SSO_NORM_STATIC_MAX_COUNT / SSO_NORM_STATIC_CHUNK doubles = 256 KiB; every GPU that loads libsso.so holds it until
 * the process exits.  Hence the limit: count > SSO_NORM_STATIC_MAX_COUNT returns SSO_ERR_INVALID (split the state
 * and add the pieces, or use sso_norm).  count = 0 gives *out_dev = 0.
 *
 * All calls on a device share that one array, and it keeps what the last call left in it.  A call overwrites every
 * slot it later reads, so nothing needs clearing between calls -- but two calls whose kernels can overlap on the
 * GPU (different streams without an ordering between them, or two host threads) race on it and may both return
 * garbage; order them with events or keep them on one stream.  Different devices have separate copies.
 *
 * The first call on each device (with that device current, as for every call) also looks up the array's address
 * on that device, which can make the CUDA runtime load the library's device code there.  Make that first call
 * during set-up, before starting any stream capture.  Later calls only launch the two kernels.
 *
 * Errors are reported through sso_last_error(NULL), like those of sso_plan_create.  The value agrees with sso_norm
 * to rounding (the order of the additions differs), not bit for bit.
 */
#define SSO_NORM_STATIC_CHUNK 8192                 /* complex numbers summed into one partial sum           */
#define SSO_NORM_STATIC_MAX_COUNT (1LL << 28)      /* largest count per call (4 GiB of complex128)          */
int sso_norm_static(const void *psi, int precision, int64_t count, double vol, double *out_dev, void *stream);

/*
 * Observables (section V.2).  psi, psi_a, psi_b are DEVICE pointers laid out as for sso_step, in
 * position space (i.e. between sso_step calls); results go to HOST memory; every sum is accumulated in double, also
 * for SSO_C64, in a fixed order (deterministic); integrals are sums over the lattice times prod(dx).  All of these
 * synchronise `stream` except sso_filter_accumulate.
 *
 * sso_overlap: out_host[0..1] = (re, im) of <a|b> = sum_c sum_r conj(a_c(r)) b_c(r) prod(dx) -- the autocorrelation
 *   function chi(t) of PAPER.md:359 eq. 40 for a = Psi(., 0), b = Psi(., t).
 * sso_expect_position: out_host[a] = sum r_a |psi|^2 prod(dx), a < ndim, on the grid r_j = (j - n/2) dx (reading G14).
 * sso_expect_momentum: out_host[a] = sum_k k_a |psi~(k)|^2 prod(dx) / N, the canonical momentum (hbar = 1), psi~ the
 *   unnormalised forward transform of PAPER.md:103 eq. 12 taken on a plan-owned copy (psi is not modified; the copy
 *   is allocated on first use and costs as much device memory as psi).  Axes of at most SSO_MAX_AXIS points: for a
 *   longer 1D lattice (SSO_MAX_AXIS_1D) the call returns SSO_ERR_UNSUPPORTED before it allocates or enqueues anything.
 */
int sso_overlap(sso_plan *plan, const void *psi_a, const void *psi_b, double *out_host, void *stream);
int sso_expect_position(sso_plan *plan, const void *psi, double *out_host, void *stream);
int sso_expect_momentum(sso_plan *plan, const void *psi, double *out_host, void *stream);

/*
 * Windowed spectrum of an autocorrelation function (eq. 41):
 *   out[e] = sum_{n < nt} chi(n dts) (1 - cos(2 pi n / nt)) exp(i n dts E[e]) dts,      T = nt dts,
 * the integral of eq. 41 as the sum over the samples (reading G30).  chi_host: nt complex128 samples (re, im
 * interleaved), E_host: nE energies, out_host: nE complex128 values; all HOST arrays, copied.  nt, nE > 0.
 */
int sso_spectrum(sso_plan *plan, const double *chi_host, int64_t nt, double dts, const double *E_host, int64_t nE,
                 double *out_host, void *stream);

/*
 * One term of the eigenfunction filter (eq. 42):  acc(r) += psi(r) (1 - cos(2 pi t/T)) exp(i E t) dts
 * for every component.  acc is a DEVICE array of ncomp * prod(sizes) complex128 numbers whatever the plan's
 * precision (the caller zeroes it before the first term and owns it); psi as for sso_step.  Asynchronous on `stream`.
 */
int sso_filter_accumulate(sso_plan *plan, void *acc, const void *psi, double t, double T, double E, double dts,
                          void *stream);

/*
 * Observables FUSED INTO THE LAST PASS of a call: advances psi by nsteps >= 1 steps exactly like
 * sso_step and returns, for the resulting psi(t),
 *   out_host[0]      sum |psi|^2 prod(dx)                                   (the norm)
 *   out_host[1..2]   Re, Im of <psi_ref | psi(t)>  (eq. 40; 0 when psi_ref is NULL)
 *   out_host[3..5]   <r_a>, a < ndim (the rest 0)
 * and, when filter_acc is not NULL, adds the term psi(t) (1 - cos(2 pi filter_t/filter_T)) exp(i filter_E filter_t)
 * filter_dts of the eigenfunction filter (eq. 42) to the complex128 DEVICE array filter_acc
 * (ncomp * prod(sizes) numbers, caller-owned).  On 2D/3D lattices all of it is accumulated by the closing pass of the
 * call while the result is still in registers: psi(t) makes no extra trip through HBM (psi_ref and filter_acc are
 * read, filter_acc written, once).  1D lattices (psi does not leave the SM during a call) and plans with a
 * position-space vector potential use the separate kernels above after the steps; the results are the same.  The sums
 * are accumulated in double; their last bits may differ from run to run (which tiles a warp meets is decided at run
 * time).  psi_ref is a DEVICE array laid out like psi.  Synchronises `stream`.
 */
int sso_step_observe(sso_plan *plan, void *psi, int64_t nsteps, const void *psi_ref, void *filter_acc, double filter_t,
                     double filter_T, double filter_E, double filter_dts, double *out_host, void *stream);

/* Tuning knobs (SSO_OPT_*); invalid values give SSO_ERR_INVALID. */
int sso_set_option(sso_plan *plan, int option, int64_t value);

/*
 * Number of kernel launches sso_step(nsteps) enqueues for this plan in its
 * current state (for launch accounting in benchmarks).
 */
int sso_launch_count(const sso_plan *plan, int64_t nsteps, int64_t *count);

/*
 * Measurement aid: advances psi by nsteps exactly like sso_step, but brackets every pass launch with CUDA
 * events (which keeps consecutive passes from overlapping) and returns, per pass kind, the number of launches
 * in count[SSO_PASS_KINDS] and their mean duration in microseconds in mean_us[SSO_PASS_KINDS] (host arrays).
 * The pass kinds are the passes of the fused step (eq. 8 factor by
 * factor).  Synchronises `stream`.  sso_pass_name returns a static description of a kind.
 */
#define SSO_PASS_OPENING 0        /* V/2 and the forward transform along the last axis            */
#define SSO_PASS_POTENTIAL 1      /* inverse transform, merged potential phase, forward transform  */
#define SSO_PASS_CLOSING 2        /* inverse transform along the last axis and V/2                 */
#define SSO_PASS_KINETIC 3        /* forward transform, kinetic factor, inverse transform (axis 0) */
#define SSO_PASS_MIDDLE_FORWARD 4 /* 3D: forward transform along the middle axis                   */
#define SSO_PASS_MIDDLE_INVERSE 5 /* 3D: inverse transform along the middle axis                   */
#define SSO_PASS_LINE_1D 6        /* 1D: every step of the call in one persistent launch           */
#define SSO_PASS_TABLES 7         /* small per-step table kernels (field phases, kinetic phases)   */
#define SSO_PASS_ROTATION 8       /* position-space vector-potential factor (sso_set_vector_potential) */
#define SSO_PASS_KINDS 9
int sso_profile_step(sso_plan *plan, void *psi, int64_t nsteps, void *stream, int64_t *count, double *mean_us);
const char *sso_pass_name(int kind);

/* Frees every table; NULL is a no-op returning SSO_OK. */
int sso_destroy(sso_plan *plan);

const char *sso_last_error(const sso_plan *plan);

/* Library version string, e.g. "sso 0.1 (sm_100a)". */
const char *sso_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SSO_H_ */
