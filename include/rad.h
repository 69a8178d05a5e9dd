/*
 * rad.h -- C ABI of the B200-native far-field radiation detector.
 *
 * The operation (BASELINE.json north_star; "the far-field radiation
 * plugin calculates radiation emissions using the Lienard-Wiechert potential approach";
 * line 74 "a weighted sum of all contributions from all particles"; lines 79-81 "at each
 * PIConGPU time step ... the sum of the contributions from all radiating particles ...
 * the complex amplitude and phase for each wavelength and direction"):
 *
 *   A(n, w_j) = sum over steps t, particles k of
 *                 w_k * [ n x ((n - beta_k) x betadot_k) ] / (1 - beta_k.n)^2
 *                     * exp( i w_j ( t0 + t*dt - n.r_k/c ) ) * dt
 *   S(n, w_j) = scale * |A(n, w_j)|^2              (d^2 I / dOmega dw)
 *
 * on a grid of n_dir observation directions n and n_omega angular frequencies w_j.
 *
 * Per-region (sub-volume) detectors (rad_config.n_regions > 1): the ML application of the
 * paper learns from pairs (particles of a sub-volume, radiation of that sub-volume) --
 * PAPER.md line 184 "which type of local particle dynamics ... gave rise to an observed
 * radiation spectrum observed in one direction", line 196 (the 3e4 particles of one sample),
 * line 285 "a selected example sub-volume".  The handle then holds one amplitude per region,
 *   A_r(n, w_j) = the same sum over the particles of region r only,
 * fed by rad_accumulate_step_regions(); sum_r A_r is the detector of all particles
 * (rad_spectrum_total).
 * Units are SI: r [m], beta = v/c [1], betadot [1/s], omega [rad/s], dt [s];
 * c = 299 792 458 m/s.  Readings of the paper where it is silent: DESIGN.md.
 *
 * Conventions
 *   - No C++/torch types cross this boundary: plain pointers, sizes and scalars.
 *     Every pointer argument says HOST or DEVICE.
 *   - Particle state is structure-of-arrays: 10 arrays (rx ry rz bx by bz bdx bdy bdz w)
 *     of n_particles elements of `state_dtype` (40 B per particle in fp32).
 *     The caller owns them; the library never copies (except the *_host entry), frees or
 *     writes them; they must stay valid until the work queued on `cuda_stream` completes.
 *   - Every call is asynchronous on `cuda_stream` (a cudaStream_t passed as void*, NULL =
 *     the legacy default stream) unless it returns data to HOST memory, in which case it
 *     synchronises that stream before returning.
 *   - A handle is not thread-safe; distinct handles are independent.  All work of a
 *     handle must be issued on streams the caller orders correctly (the library adds no
 *     cross-stream dependency between calls).
 *   - No exception crosses the ABI.  Every function returns a rad_status; details via
 *     rad_last_error().  Particle values are not scanned: NaN/Inf or 1 - beta.n = 0 in the
 *     state give NaN/Inf in every bin the particle contributes to, for fp32 and fp64 state
 *     alike (documented, caller's responsibility; tests/test_gpu_parity.py
 *     test_non_finite_particle_state_propagates).
 *   - An entry point makes the handle's device current while it runs and restores the calling
 *     thread's current device before it returns.
 *   - There is no CPU fallback: without a CUDA device rad_create fails with RAD_ERR_CUDA.
 */
#ifndef RAD_H_
#define RAD_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RAD_API __attribute__((visibility("default")))

typedef struct rad_handle rad_handle; /* opaque, library-owned */

typedef enum {
    RAD_OK = 0,
    RAD_ERR_INVALID_ARG = 1, /* NULL/negative/non-finite argument, zero direction, unsorted omega */
    RAD_ERR_ALLOC = 2,       /* host or device allocation failed */
    RAD_ERR_CUDA = 3,        /* a CUDA runtime call or kernel launch failed / no device */
    RAD_ERR_STATE = 4,       /* handle unusable (a previous CUDA error) */
    RAD_ERR_UNSUPPORTED = 5  /* valid request this build does not implement */
} rad_status;

typedef enum { RAD_F32 = 0, RAD_F64 = 1 } rad_dtype;

/* rad_config.flags */
#define RAD_FLAG_DETERMINISTIC 1u /* bit 0: no floating-point atomics; results are
                                     bit-reproducible run to run (slower, more memory) */
#define RAD_FLAG_FORCE_GENERAL 2u /* bit 1: never use the grid-specific variants (the uniform-grid
                                     recurrence kernel, the dyadic-grid squaring chains): always the
                                     general-grid kernel */
#define RAD_FLAG_OVERLAP_STEPS 4u /* bit 2: consecutive calls on one stream may overlap (below) */
#define RAD_FLAG_FAST_GRIDDED 8u  /* bit 3: approximate fast path (gridded in retarded time, below) */
#define RAD_FLAG_PRECISE 16u      /* bit 4: every sin/cos by the fp32 polynomial (abs. error 2-3e-7) instead of the
                                     special-function unit (4-5e-7), on the general-grid kernel whatever the grid:
                                     about 0.55 x the speed; for spectra with bins near 1e-6 of the peak fed by few
                                     thousand particles, where the cancellation between terms amplifies the
                                     per-term error.  Not with the Nyquist limiter, a
                                     Gaussian / CIC form factor or RAD_FLAG_FAST_GRIDDED (RAD_ERR_UNSUPPORTED) */

/* RAD_FLAG_OVERLAP_STEPS.  The accumulate and result kernels are then launched with
 * programmatic stream serialization: the blocks of a call may start while the last blocks of
 * the handle's previous kernel on the same stream are still running (they fill the SMs that
 * the tail of that grid leaves idle) and wait, just before they touch the accumulator, until
 * everything queued before them has completed.  Results are the same; what changes is the
 * contract for the INPUT arrays: a call may read its particle arrays before earlier work on
 * cuda_stream has finished, so with this flag the arrays passed to rad_accumulate_step*
 * must be complete when the call is made -- written before a stream / event synchronisation,
 * or by work on another stream that cuda_stream waits for through an event (as the *_host
 * entry points do internally), not by a kernel queued on cuda_stream directly before the call.
 * Worth 1 % on steps of several 1e9 updates and up to 25 % on steps that fill the GPU only
 * once (a few 1e8 updates).  Combines with RAD_FLAG_DETERMINISTIC (results stay bit-identical);
 * not exercised under CUDA stream capture (capture handles without this flag). */

typedef struct {
    uint32_t struct_size;  /* = sizeof(rad_config); ABI versioning                         */
    int32_t device;        /* CUDA device ordinal                                          */
    int32_t n_dir;         /* >= 1                                                         */
    int32_t n_omega;       /* >= 1                                                         */
    const double *dirs;    /* HOST [n_dir][3]; any non-zero length, normalised in fp64     */
    const double *omega;   /* HOST [n_omega] rad/s; finite, > 0, strictly increasing       */
    double dt;             /* s, > 0: the quadrature weight of every term                  */
    double t0;             /* s: time of step_index 0                                      */
    double scale;          /* S = scale*|A|^2; 0 -> SI e^2/(16 pi^3 eps0 c) J s            */
    int32_t state_dtype;   /* a rad_dtype value (RAD_F32 / RAD_F64) for the 10 particle arrays;
                              declared int32_t, not the enum, so the struct layout does not
                              depend on the compiler's enum size                            */
    uint32_t flags;        /* RAD_FLAG_*                                                   */
    int32_t n_regions;     /* 0 or 1: one detector; R > 1: R per-region detectors          */
    int32_t window_type;   /* RAD_WINDOW_*: spatial window on the macro weights (below)    */
    double window_origin[3]; /* m: lower corner o of the window box                        */
    double window_extent[3]; /* m: edge lengths L; L_c <= 0: axis c is not windowed        */
    double nyquist_factor; /* nu >= 0; 0: off.  Nyquist limiter (below)                      */
    int32_t form_factor_type;     /* RAD_FF_*: macro-particle form factor (below); 0: none   */
    int32_t reserved0;            /* must be 0                                               */
    double form_factor_size[3];   /* m: s_x, s_y, s_z of the macro-particle shape, >= 0      */
    /* RAD_FLAG_FAST_GRIDDED only (ignored otherwise): */
    double fast_box_min[3];       /* m: a box that contains every particle position of the   */
    double fast_box_max[3];       /*    accumulation window                                   */
    int64_t fast_step_min;        /* step indices of the window: fast_step_min <= step_index  */
    int64_t fast_step_max;        /*    <= fast_step_max in every accumulate call             */
    double fast_tolerance;        /* target relative accuracy of the gridding, 0 -> 1e-6      */
} rad_config;

/* RAD_FLAG_FAST_GRIDDED -- the approximate fast path (PAPER.md line
 * 142: the plugin's cost, "scaling with the number of particles, frequencies, and directions,
 * easily exceed[s] the computational limits of the underlying particle-in-cell simulation").
 * For one direction n the sum is a non-uniform Fourier sum over the retarded times
 * tau = t - n.r/c of all (particle, step) terms,
 *     A(n, w_j) = sum a(n) exp(i w_j tau),        a = the real transverse amplitude (A1, A2).
 * Instead of W sin/cos pairs per term, every term is SPREAD onto a uniform grid in tau that the
 * handle keeps per direction (spacing h = pi / (2 w_max), i.e. twofold oversampling of the highest
 * frequency; a compactly supported "exponential of semicircle" kernel of width 4..12 grid points,
 * chosen from fast_tolerance), at a cost independent of W: 4 vector atomics per (particle,
 * direction) at the default width.  rad_spectrum / rad_amplitude then evaluate
 *     A(n, w_j) = (1 / Phi(w_j)) sum_m g_m(n) exp(i w_j tau_m)
 * exactly (a direct sum over the grid points with the integer-phase sin/cos of the direct path,
 * no FFT) and divide by the kernel's Fourier transform Phi.  The result approximates the exact
 * sum to about fast_tolerance (relative to the typical |A| of a bin); the oracle and the parity
 * tolerances are those of the exact path.  Worth it when spectra are taken every many steps.
 * Restrictions: one region, no Nyquist limiter, no form factor, no RAD_FLAG_DETERMINISTIC
 * (RAD_ERR_UNSUPPORTED at rad_create); particles outside fast_box or steps outside the window
 * are not deposited and make the next rad_spectrum / rad_amplitude fail with RAD_ERR_STATE.
 * rad_export_accumulator / rad_import_accumulator / rad_add_amplitude are not available
 * (RAD_ERR_UNSUPPORTED); rad_reset clears the grid. */

/* Macro-particle form factor (the plugin "correctly quantif[ies] coherent and
 * incoherent radiation [39]"; ref [39], line 338, "a general form factor formalism for
 * macro-particles"; the formula is not printed in the paper -- reading FF1 of DESIGN.md).  A
 * macro-particle of weight w stands for w real particles distributed with a shape whose Fourier
 * transform at the emitted wave vector k = w_j n / c is F(n, w_j), 0 <= F <= 1; their fields add
 * coherently for the fraction F^2 and incoherently for the rest (intensity w^2 F^2 + w (1 - F^2)),
 * so with form_factor_type != RAD_FF_NONE the weight of a term in the amplitude sum is
 *     g_k(n, w_j) = sqrt( w_k + (w_k^2 - w_k) F^2(n, w_j) )         instead of w_k
 * (the spatial window, if any, still multiplies it; weights must be >= 0).
 *     RAD_FF_GAUSSIAN    F = exp( -1/2 sum_c (w_j n_c s_c / c)^2 )           s_c: standard deviations
 *     RAD_FF_CIC         F = prod_c sinc^2( w_j n_c s_c / (2c) )             s_c: cell sizes (cloud in cell)
 *     RAD_FF_INCOHERENT  F = 0: g = sqrt(w) (a per-particle weight: costs nothing per update)
 * w = 1 is the identity for every shape; zero sizes give F = 1, g = w (the detector as
 * BASELINE.json states it).  F^2 is tabulated per (direction, frequency) at rad_create in fp64;
 * the square root is taken per update (a third special-function operation per update). */
#define RAD_FF_NONE 0
#define RAD_FF_GAUSSIAN 1
#define RAD_FF_CIC 2
#define RAD_FF_INCOHERENT 3

/* Nyquist limiter (not in the paper; reading N1 of DESIGN.md): with nyquist_factor = nu > 0 the
 * term of particle k at a step is left out of bin (n, w_j) when
 *     w_j * dt * (1 - beta_k.n) >= pi * nu,
 * i.e. when the wave the particle emits towards n, whose phase advances by w (1 - beta.n) dt per
 * step, is sampled fewer than 2/nu times per period (nu = 1: the Nyquist limit itself).  The
 * comparison is made in fp64, exactly as written.  Detectors with nu > 0 use the general-grid
 * kernel for every shape. */

/* Spatial window (not in the paper, which cites the plugin [37] for such details; reading W1 of
 * DESIGN.md): with window_type != RAD_WINDOW_NONE the macro weight of every particle is
 * multiplied, at every step, by
 *     Wn(r) = product over the axes c with L_c > 0 of w1((r_c - o_c) / L_c),
 *     w1(u) = 0 for u outside [0, 1];  TRIANGLE: 1 - |2u - 1|;  HAMMING: 0.54 - 0.46 cos(2 pi u),
 * which tapers the contribution of particles near the faces of the box (particles entering
 * or leaving a finite simulation volume otherwise ring in the spectrum). */
#define RAD_WINDOW_NONE 0
#define RAD_WINDOW_TRIANGLE 1
#define RAD_WINDOW_HAMMING 2

/* Frequency grids.  Any strictly increasing grid is served by the general-grid kernel (one sin/cos
 * per update).  Two structures are detected at rad_create and served by faster variants with the same
 * results to rounding (same tolerances, tests/test_gpu_parity.py): a LINEAR grid w_j = w_0 + j dw
 * (rotation recurrence, BASELINE.json north_star) and a DYADIC log grid, w_(j+b) = 2 w_j for an integer
 * number b in {4, 8, 16, 32, 64} of bins per octave (z(2w) = z(w)^2).
 * rad_kernel_variant() names the variant in use; RAD_FLAG_FORCE_GENERAL switches both off.
 * Detector shapes: any n_dir >= 1, n_omega >= 1.  n_dir * n_omega <= 16 (up to 2 directions) runs the
 * particle-streaming kernel; detectors with few directions and a moderate number of frequencies let the lane
 * groups of a warp split the particles instead of idling ("+split" in the variant name). */

/* Create a detector for a grid of observation directions n and frequencies w_j (BASELINE.json
 * north_star "on a grid of observation directions n and frequencies w"; the
 * plugin records "for each wavelength and direction"): copies dirs/omega, builds the device
 * tables, zeroes A.  *out is set to NULL on failure. */
RAD_API rad_status rad_create(const rad_config *cfg, rad_handle **out);

/* A += contributions of n_particles particles at time t0 + step_index*dt: one PIC step of the
 * sum ("at each PIConGPU time step ... the sum of the contributions from all
 * radiating particles"; the summand is north_star's, stated at the top of this header).
 * All 10 arrays DEVICE, `state_dtype` elements, 16-byte aligned not required.
 * n_particles == 0 is a no-op.  Calls are additive: several calls with the same
 * step_index superpose (particle subsets), any order of steps gives the same A up to
 * rounding. */
RAD_API rad_status rad_accumulate_step(rad_handle *h, int64_t step_index, int64_t n_particles,
                                       const void *rx, const void *ry, const void *rz,
                                       const void *bx, const void *by, const void *bz,
                                       const void *bdx, const void *bdy, const void *bdz,
                                       const void *w, void *cuda_stream);

/* n_steps consecutive PIC steps in ONE launch: exactly the result (up to rounding order) of
 *   for s in 0 .. n_steps-1: rad_accumulate_step(h, first_step_index + s, n_particles,
 *                                                 rx + s*step_stride, ..., w + s*step_stride)
 * i.e. each of the 10 DEVICE arrays holds the state of step s at elements
 * [s*step_stride, s*step_stride + n_particles) (step_stride >= n_particles, in elements).
 * For trajectories that are resident (replay, or a simulation that buffers a few steps):
 * the grid covers (step, particle chunk) pairs, so launch latency, ramp and tail of the grid
 * are paid once per call instead of once per step -- this is what makes small steps (a few
 * 1e5 updates) run at the rate of large ones.  Per-region handles: rad_accumulate_steps_regions
 * (this call returns RAD_ERR_UNSUPPORTED there).  Few-bin (streaming-kernel) detectors and RAD_FLAG_DETERMINISTIC
 * handles run it as n_steps launches. */
RAD_API rad_status rad_accumulate_steps(rad_handle *h, int64_t first_step_index, int32_t n_steps,
                                        int64_t n_particles, int64_t step_stride,
                                        const void *rx, const void *ry, const void *rz,
                                        const void *bx, const void *by, const void *bz,
                                        const void *bdx, const void *bdy, const void *bdz,
                                        const void *w, void *cuda_stream);

/* The multi-step form of rad_accumulate_step_regions: n_steps consecutive steps, step s of every
 * array at elements [s*step_stride, ...), the same region_offsets (relative to the start of each
 * step's row) for all steps; step_stride >= region_offsets[n_regions]. */
RAD_API rad_status rad_accumulate_steps_regions(rad_handle *h, int64_t first_step_index, int32_t n_steps,
                                                int64_t step_stride, int32_t n_regions,
                                                const int64_t *region_offsets,
                                                const void *rx, const void *ry, const void *rz,
                                                const void *bx, const void *by, const void *bz,
                                                const void *bdx, const void *bdy, const void *bdz,
                                                const void *w, void *cuda_stream);

/* Same, state in HOST memory (pinned memory makes the copies asynchronous).  The
 * library stages the arrays through its own double-buffered device buffer: the
 * host->device copy of one call overlaps the kernels of the previous call.  The host
 * arrays may be reused as soon as the call returns only if they are pageable; pinned
 * arrays must stay untouched until `cuda_stream` has passed this call. */
RAD_API rad_status rad_accumulate_step_host(rad_handle *h, int64_t step_index, int64_t n_particles,
                                            const void *rx, const void *ry, const void *rz,
                                            const void *bx, const void *by, const void *bz,
                                            const void *bdx, const void *bdy, const void *bdz,
                                            const void *w, void *cuda_stream);

/* Per-region form (handles created with n_regions = R > 1; also valid with R = 1).
 * The particle arrays are sorted by region: region r owns the particles
 * [region_offsets[r], region_offsets[r+1]); region_offsets is HOST memory, n_regions + 1
 * non-decreasing entries, region_offsets[0] >= 0; it is copied before the call returns.
 * Particles before region_offsets[0] or from region_offsets[n_regions] on belong to no
 * region and are not read.  Empty regions are allowed.  A_r += contributions of region r's
 * particles at time t0 + step_index*dt, for every r, in ONE kernel launch.
 * n_regions must equal the handle's.  rad_accumulate_step() on a handle with R > 1 fails
 * with RAD_ERR_INVALID_ARG (it would not say which region the particles belong to). */
RAD_API rad_status rad_accumulate_step_regions(rad_handle *h, int64_t step_index, int32_t n_regions,
                                               const int64_t *region_offsets,
                                               const void *rx, const void *ry, const void *rz,
                                               const void *bx, const void *by, const void *bz,
                                               const void *bdx, const void *bdy, const void *bdz,
                                               const void *w, void *cuda_stream);

/* Same with the state in HOST memory (see rad_accumulate_step_host); the arrays are read
 * from element region_offsets[0] to region_offsets[n_regions] - 1. */
RAD_API rad_status rad_accumulate_step_regions_host(rad_handle *h, int64_t step_index, int32_t n_regions,
                                                    const int64_t *region_offsets,
                                                    const void *rx, const void *ry, const void *rz,
                                                    const void *bx, const void *by, const void *bz,
                                                    const void *bdx, const void *bdy, const void *bdz,
                                                    const void *w, void *cuda_stream);

/* In rad_spectrum, rad_amplitude and rad_add_amplitude a handle with R = n_regions > 1 adds a
 * leading region dimension: spectrum out[R][n_dir][n_omega], amplitude
 * out/amp[R][n_dir][n_omega][3][2]. */

/* Where a result goes (the `out_on_device` argument of rad_spectrum / rad_spectrum_total /
 * rad_amplitude). */
#define RAD_OUT_HOST 0       /* HOST memory; the call returns after the data has arrived          */
#define RAD_OUT_DEVICE 1     /* DEVICE memory; asynchronous on cuda_stream                          */
#define RAD_OUT_HOST_ASYNC 2 /* HOST memory (pinned, else the copy blocks); asynchronous: the data
                                is there once cuda_stream has passed this call (event / sync by
                                the caller) -- lets the next step's work be queued meanwhile      */

/* out[n_dir][n_omega] (row-major, fp64) = scale * sum_c |A_c|^2.  Non-destructive.
 * out_on_device: RAD_OUT_HOST, RAD_OUT_DEVICE or RAD_OUT_HOST_ASYNC. */
RAD_API rad_status rad_spectrum(rad_handle *h, double *out, int out_on_device, void *cuda_stream);

/* out[n_dir][n_omega] = scale * sum_c |sum_r A_r,c|^2: the detector of all particles of all
 * regions (amplitudes, not intensities, add up: PAPER.md line 80).  Equals rad_spectrum for
 * R = 1.  Same HOST/DEVICE convention as rad_spectrum. */
RAD_API rad_status rad_spectrum_total(rad_handle *h, double *out, int out_on_device, void *cuda_stream);

/* out[n_dir][n_omega][3][2] fp64: (re, im) of the x, y, z components of A
 * ("complex amplitude and phase for each wavelength and direction"). */
RAD_API rad_status rad_amplitude(rad_handle *h, double *out, int out_on_device, void *cuda_stream);

/* A := A + amp, amp DEVICE [n_dir][n_omega][3][2] fp64 in the rad_amplitude layout.
 * For the multi-GPU sum: ranks all-reduce rad_amplitude() buffers (amplitudes, not
 * intensities, must be summed -- PAPER.md line 80 "sum of the contributions from all
 * radiating particles in the simulation"), rad_reset(), then add the reduced buffer. */
RAD_API rad_status rad_add_amplitude(rad_handle *h, const double *amp_device, void *cuda_stream);

/* The accumulator itself, for the multi-GPU sum and for checkpoints.  A is perpendicular to n
 * (it is n x something), so the library keeps its two components on a fixed orthonormal pair
 * e1, e2 _|_ n chosen at rad_create from n alone (e1 = normalise(z^ x n), x^ x n if |n_z| > 0.9;
 * e2 = n x e1): handles created with the same dirs share the basis, whatever the device.
 *   out_device[(R)][n_dir][n_omega][4] fp64 = (Re A1, Im A1, Re A2, Im A2), A = A1 e1 + A2 e2.
 * PAPER.md line 80 ("the sum of the contributions from all radiating particles in the
 * simulation") with particles sharded over GPUs (line 138) means: every rank exports, ONE sum
 * all-reduce over these n_dir*n_omega*4 doubles (two thirds of the Cartesian rad_amplitude
 * buffer), then rad_spectrum_of() on the sum -- amplitudes, never intensities, are added.
 * A device-to-device copy on cuda_stream; asynchronous. */
RAD_API rad_status rad_export_accumulator(rad_handle *h, double *out_device, void *cuda_stream);

/* A := A + amp4, amp4_device in the rad_export_accumulator layout (restart from a checkpoint,
 * or fold another rank's amplitude into this handle).  Asynchronous on cuda_stream. */
RAD_API rad_status rad_import_accumulator(rad_handle *h, const double *amp4_device, void *cuda_stream);

/* out[(R)][n_dir][n_omega] = scale * (|A1|^2 + |A2|^2) of an amplitude buffer in the
 * rad_export_accumulator layout (DEVICE) instead of the handle's own accumulator, which is not
 * touched: the |A|^2 step after the all-reduce.  out_on_device as in rad_spectrum. */
RAD_API rad_status rad_spectrum_of(rad_handle *h, const double *amp4_device, double *out, int out_on_device,
                                   void *cuda_stream);

/* A := 0: start a new accumulation window.  PAPER.md line 74 "the observed intensity at each
 * wavelength and direction varies between time steps", line 80 "calculate the radiation spectrum
 * ... at each time step": a caller that wants per-step or per-window spectra resets between them. */
RAD_API rad_status rad_reset(rad_handle *h, void *cuda_stream);

/* Frees everything the handle owns after synchronising the device.  NULL-safe. */
RAD_API void rad_destroy(rad_handle *h);

/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
RAD_API int64_t rad_launch_count(const rad_handle *h);

/* Name of the accumulation kernel variant the last rad_accumulate_step used
 * ("general", "uniform", ...), static storage. */
RAD_API const char *rad_kernel_variant(const rad_handle *h);

RAD_API const char *rad_status_string(rad_status s);
/* Message of the last failing call on this handle (h == NULL: last rad_create failure). */
RAD_API const char *rad_last_error(const rad_handle *h);
RAD_API const char *rad_version(void);

/* The detector as ONE call that allocates nothing -- for callers that cannot call cudaMalloc (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it).  No handle:
 *   out_device[n_dir][n_omega] (DEVICE, fp64, overwritten) = scale * |A(n, w_j)|^2,
 *   A = the sum at the top of this header over the steps first_step_index ... + n_steps - 1 and
 *       n_particles particles per step (plain detector: one region, no window, limiter or form factor),
 * with every argument the caller's: dirs_device DEVICE [n_dir][3] fp64 (any non-zero length),
 * omega_device DEVICE [n_omega] fp64 rad/s (NOT validated: device memory is not read back), the 10
 * state arrays DEVICE in the rad_accumulate_steps layout (step s at elements [s*step_stride,
 * s*step_stride + n_particles), `state_dtype` elements), dt/t0/scale as in rad_config (scale 0 ->
 * SI).  n_steps == 0 or n_particles == 0 gives out = 0.  Runs on the calling thread's CURRENT
 * device, asynchronously on cuda_stream.
 * The fp64 amplitude accumulator the kernel folds into is a static __device__ array inside the
 * library, RAD_STATIC_MAX_BINS * 32 B = 2 MiB, which every GPU that loads the library holds until the
 * process exits: n_dir * n_omega > RAD_STATIC_MAX_BINS fails with RAD_ERR_UNSUPPORTED.  The call
 * uses no cudaMalloc / cudaFree or other allocating routine (it clears the part of the array it
 * uses, launches the accumulate kernel -- a variant of the general-grid kernel that needs no set-up
 * tables, same tolerances against the oracle, about 0.55 x the speed -- and the |A|^2 kernel); its first call on a device
 * looks up the array's address (cudaGetSymbolAddress), so make one call before capturing.
 * ALL calls on a device share the array: calls that overlap on the GPU (different streams without
 * an ordering, or several threads) race on it and give wrong results; calls on one stream are safe.
 * Other error codes: RAD_ERR_INVALID_ARG (NULL pointer, negative size, dt <= 0, bad dtype,
 * step_stride < n_particles), RAD_ERR_CUDA; message via rad_static_last_error() (per thread). */
#define RAD_STATIC_MAX_BINS 65536
RAD_API rad_status rad_spectrum_static(int32_t n_dir, const double *dirs_device, int32_t n_omega,
                                       const double *omega_device, double dt, double t0, double scale,
                                       int32_t state_dtype, int64_t first_step_index, int32_t n_steps,
                                       int64_t n_particles, int64_t step_stride,
                                       const void *rx, const void *ry, const void *rz,
                                       const void *bx, const void *by, const void *bz,
                                       const void *bdx, const void *bdy, const void *bdz,
                                       const void *w, double *out_device, void *cuda_stream);
RAD_API const char *rad_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* RAD_H_ */
