/*
 * rad_oracle.c -- fp64 CPU ORACLE for the far-field (Lienard-Wiechert) radiation detector.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing on the product path (paper_2501_03383_b200/) may
 * include, link, import or call this file; only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs use it.  It shares no code, header,
 * table or constant generator with the CUDA path.
 *
 * What it computes (BASELINE.json north_star; "weighted sum of all
 * contributions from all particles"; lines 79-81 "at each time step ... sum of the
 * contributions from all radiating particles ... complex amplitude and phase for each
 * wavelength and direction"; line 142 "Lienard-Wiechert potential approach [38]";
 * SURVEY.md section 8(c)):
 *
 *   for each call (step t, particles k), each direction n, each frequency w_j:
 *      d    = 1 - beta_k . n
 *      a    = w_k * dt * [ n x ((n - beta_k) x betadot_k) ] / d^2          (3-vector)
 *      tau  = (t0 + t*dt) - (n . r_k)/c
 *      A[n][j][c] += a_c * (cos(w_j tau) + i sin(w_j tau)),   c in {x,y,z}
 *   S[n][j] = scale * (|A_x|^2 + |A_y|^2 + |A_z|^2)
 *
 * Written exactly in that order with the two explicit cross products, plain double
 * arithmetic, libm sin/cos, plain summation in particle order; no blocking, no
 * reordering, no fast-math.  OpenMP only splits the independent (n, j) bins over
 * threads; every bin's sum is sequential in k, so results do not depend on the
 * thread count.
 *
 * Readings of the paper: Q1 phase sign +i w (t - n.r/c);
 * Q2 time of step t is t0 + t*dt; Q3 rectangle rule, every term times dt, no window;
 * Q4 spectrum = scale*|A|^2, default scale e^2/(16 pi^3 eps0 c); Q5 amplitude linear
 * in the macro weight; Q8 n normalised in fp64; Q9 far field (1/R dropped).
 *
 * Pins (tests/test_oracle_pins.py): zero for unaccelerated motion, Dirichlet kernel
 * (magnitude and complex phase), Doppler-shifted Dirichlet kernel, two-particle
 * interference, linearity/superposition, cyclotron (Schott) harmonics, SI constant,
 * mpmath/numpy brute force.  The spectra of the five BASELINE.json configs themselves
 * have no published values: "parity unpinned" except through those pins.
 *
 * Per-region detectors ("which type of local
 * particle dynamics ... gave rise to an observed radiation spectrum", line 196 the 3e4
 * particles of one sample, line 285 "a selected example sub-volume"):
 * oracle_accumulate_step_regions() is the same sum restricted to the particles of each
 * region, A_r = sum over k in region r; pins: sum_r A_r = A of all particles, an empty
 * region is exactly zero, regions are independent, masked numpy brute force.
 *
 * Spatial window (reading W1 of DESIGN.md; not in the paper, which
 * only cites the plugin [37]): the macro weight of a particle is multiplied by
 *   Wn(r) = prod over axes c with extent L_c > 0 of w1((r_c - o_c)/L_c),
 *   w1(u) = 0 outside [0,1];  TRIANGLE: 1 - |2u - 1|;  HAMMING: 0.54 - 0.46 cos(2 pi u)
 * evaluated at the particle's position of that step.  Pins: type NONE and all-zero extents
 * change nothing; closed-form window values times the Dirichlet kernel; outside -> exactly 0;
 * equals the unwindowed oracle fed w*Wn(r) computed independently in numpy.
 *
 * Nyquist limiter (NEXT-3, reading N1 of DESIGN.md; at dt = 1e-17 s the top of
 * the BASELINE.json frequency range is beyond the sampling limit): with nyquist_factor nu > 0
 * the term of particle k is dropped from bin (n, w_j) when
 *     w_j * dt * (1 - beta_k.n) >= pi * nu,
 * i.e. when the phase of the emitted wave, which advances by w (1 - beta.n) dt per step along
 * the trajectory, is sampled fewer than 2/nu times per period.  Pins: nu = 0 and nu = huge change
 * nothing; a static particle loses exactly the bins w_j dt >= pi nu; the cut-off of a moving
 * particle is Doppler shifted by direction; kept bins equal the closed forms.
 * (nu is the last argument of the _w entry points; 0 = off.)
 *
 * Macro-particle form factor (NEXT-3, reading FF1 of DESIGN.md; the plugin
 * "correctly quantif[ies] coherent and incoherent radiation [39]", ref [39] "a general form
 * factor formalism for macro-particles", formula not printed in the paper): a macro-particle of
 * weight w stands for w real particles distributed with a shape whose Fourier transform at the
 * emitted wave vector k = w_j n / c is F(n, w_j), 0 <= F <= 1.  Their fields add coherently for
 * the fraction F^2 and incoherently for the rest, intensity factor w^2 F^2 + w (1 - F^2), so the
 * weight of a term in the amplitude sum becomes
 *     g_k(n, w_j) = sqrt( w_k + (w_k^2 - w_k) F^2(n, w_j) )        instead of w_k
 * (the spatial window, if any, still multiplies it).  Shapes (ff_size = s_x, s_y, s_z in metres):
 *     1 GAUSSIAN    F = exp( -1/2 sum_c (w_j n_c s_c / c)^2 )             (s_c = standard deviations)
 *     2 CIC         F = prod_c sinc^2( w_j n_c s_c / (2 c) ), sinc x = sin x / x   (s_c = cell sizes)
 *     3 INCOHERENT  F = 0   (g = sqrt w)
 *     0 none        g = w   (the detector as BASELINE.json states it; F = 1 gives the same)
 * Pins (test_p14_*): w = 1 is the identity bit for bit; F = 1 (zero size) reproduces the plain
 * sum; F = 0 makes the intensity of one macro-particle proportional to w, not w^2; closed forms
 * g^2 x Dirichlet kernel for the Gaussian (anisotropic, direction dependent) and at the first
 * zero of the CIC shape; numpy brute force.  (ff_type, ff_size are the last arguments of the _ff
 * entry points.)
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C_LIGHT 299792458.0 /* m/s, exact (SI) */

/* e^2 / (16 pi^3 eps0 c) in J s, from CODATA-2018 e and eps0 (SURVEY.md Q4 / pin P9). */
double oracle_default_scale(void)
{
    const double e = 1.602176634e-19;     /* C, exact */
    const double eps0 = 8.8541878128e-12; /* F/m */
    const double pi = 3.14159265358979323846;
    return (e * e) / (16.0 * pi * pi * pi * eps0 * ORACLE_C_LIGHT);
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static void cross3(const double a[3], const double b[3], double out[3])
{
    out[0] = a[1] * b[2] - a[2] * b[1];
    out[1] = a[2] * b[0] - a[0] * b[2];
    out[2] = a[0] * b[1] - a[1] * b[0];
}

/* w1(u) of the spatial window, see the header. */
static double window_1d(int type, double u)
{
    if (u < 0.0 || u > 1.0) return 0.0;
    if (type == 1) return 1.0 - fabs(2.0 * u - 1.0);
    if (type == 2) return 0.54 - 0.46 * cos(2.0 * 3.14159265358979323846 * u);
    return 1.0;
}

/*
 * Accumulate one PIC step into A.
 *   dirs   [n_dir][3]   fp64, any non-zero length (normalised here, Q8)
 *   omega  [n_omega]    rad/s
 *   state  10 SoA arrays of length n_part; is_f32 != 0 -> float arrays promoted
 *          value-for-value to double, else double arrays
 *   bin_idx optional list of n_bins flat bin indices (dir*n_omega + j) to compute;
 *          NULL -> all bins.  Bins are independent sums, so a subset is exact.
 *   A      [n_dir][n_omega][3][2] (re, im) fp64, accumulated in place (only the
 *          selected bins are touched)
 *   win_type 0 none / 1 triangle / 2 Hamming; win = {o_x, o_y, o_z, L_x, L_y, L_z} (NULL or
 *          type 0: no window; L_c <= 0: axis c not windowed)
 *   nyquist nu of the Nyquist limiter (0: off)
 * Returns 0, or 1 on a bad argument.
 */
/* F(n, w) of the macro-particle shape, see the header (reading FF1). */
static double form_factor(int type, const double size[3], const double n[3], double om)
{
    if (type == 1) {
        double q = 0.0;
        for (int c = 0; c < 3; ++c) {
            const double x = om * n[c] * size[c] / ORACLE_C_LIGHT;
            q += x * x;
        }
        return exp(-0.5 * q);
    }
    if (type == 2) {
        double F = 1.0;
        for (int c = 0; c < 3; ++c) {
            const double x = om * n[c] * size[c] / (2.0 * ORACLE_C_LIGHT);
            const double sinc = (x == 0.0) ? 1.0 : sin(x) / x;
            F *= sinc * sinc;
        }
        return F;
    }
    if (type == 3) return 0.0;
    return 1.0;
}

/*   ff_type 0 none / 1 Gaussian / 2 CIC / 3 incoherent; ff_size = {s_x, s_y, s_z} (NULL with type 0) */
int oracle_accumulate_step_ff(int n_dir, const double *dirs, int n_omega, const double *omega,
                              double dt, double t0, long long step_index, long long n_part,
                              int is_f32, const void *rx, const void *ry, const void *rz,
                              const void *bx, const void *by, const void *bz, const void *bdx,
                              const void *bdy, const void *bdz, const void *w,
                              long long n_bins, const long long *bin_idx, double *A,
                              int win_type, const double *win, double nyquist,
                              int ff_type, const double *ff_size)
{
    if (ff_type != 0 && !ff_size) return 1;
    if (n_dir <= 0 || n_omega <= 0 || !dirs || !omega || !A || n_part < 0) return 1;
    const long long total = bin_idx ? n_bins : (long long)n_dir * n_omega;
    const double t_step = t0 + (double)step_index * dt;
    const double nyq_lim = 3.14159265358979323846 * nyquist; /* pi nu; 0 = limiter off */

#define LOAD(p, k) (is_f32 ? (double)((const float *)(p))[k] : ((const double *)(p))[k])

#pragma omp parallel for schedule(dynamic, 1)
    for (long long b = 0; b < total; ++b) {
        const long long flat = bin_idx ? bin_idx[b] : b;
        const int id = (int)(flat / n_omega);
        const int j = (int)(flat % n_omega);
        double n[3] = {dirs[3 * id + 0], dirs[3 * id + 1], dirs[3 * id + 2]};
        const double nn = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
        n[0] /= nn; n[1] /= nn; n[2] /= nn;
        const double om = omega[j];
        const double F = ff_type != 0 ? form_factor(ff_type, ff_size, n, om) : 1.0;
        double acc[6] = {0, 0, 0, 0, 0, 0};
        for (long long k = 0; k < n_part; ++k) {
            const double r[3] = {LOAD(rx, k), LOAD(ry, k), LOAD(rz, k)};
            const double be[3] = {LOAD(bx, k), LOAD(by, k), LOAD(bz, k)};
            const double bd[3] = {LOAD(bdx, k), LOAD(bdy, k), LOAD(bdz, k)};
            double wk = LOAD(w, k);
            if (ff_type != 0) wk = sqrt(wk + (wk * wk - wk) * F * F); /* g_k(n, w_j), reading FF1 */
            if (win_type != 0 && win)
                for (int c = 0; c < 3; ++c)
                    if (win[3 + c] > 0.0) wk *= window_1d(win_type, (r[c] - win[c]) / win[3 + c]);
            const double d = 1.0 - (be[0] * n[0] + be[1] * n[1] + be[2] * n[2]);
            const double nmb[3] = {n[0] - be[0], n[1] - be[1], n[2] - be[2]};
            double inner[3], outer[3];
            cross3(nmb, bd, inner);   /* (n - beta) x betadot        */
            cross3(n, inner, outer);  /* n x ((n - beta) x betadot)  */
            const double pre = wk * dt / (d * d);
            const double tau = t_step - (n[0] * r[0] + n[1] * r[1] + n[2] * r[2]) / ORACLE_C_LIGHT;
            if (nyq_lim > 0.0 && om * dt * d >= nyq_lim) continue; /* Nyquist limiter, reading N1 */
            const double ph = om * tau;
            const double cs = cos(ph), sn = sin(ph);
            for (int c = 0; c < 3; ++c) {
                const double a = pre * outer[c];
                acc[2 * c + 0] += a * cs;
                acc[2 * c + 1] += a * sn;
            }
        }
        double *dst = A + (size_t)flat * 6;
        for (int c = 0; c < 6; ++c) dst[c] += acc[c];
    }
#undef LOAD
    return 0;
}

/* No form factor. */
int oracle_accumulate_step_w(int n_dir, const double *dirs, int n_omega, const double *omega,
                             double dt, double t0, long long step_index, long long n_part,
                             int is_f32, const void *rx, const void *ry, const void *rz,
                             const void *bx, const void *by, const void *bz, const void *bdx,
                             const void *bdy, const void *bdz, const void *w,
                             long long n_bins, const long long *bin_idx, double *A,
                             int win_type, const double *win, double nyquist)
{
    return oracle_accumulate_step_ff(n_dir, dirs, n_omega, omega, dt, t0, step_index, n_part, is_f32, rx, ry,
                                     rz, bx, by, bz, bdx, bdy, bdz, w, n_bins, bin_idx, A, win_type, win,
                                     nyquist, 0, NULL);
}

/* The plain detector: no window. */
int oracle_accumulate_step(int n_dir, const double *dirs, int n_omega, const double *omega,
                           double dt, double t0, long long step_index, long long n_part,
                           int is_f32, const void *rx, const void *ry, const void *rz,
                           const void *bx, const void *by, const void *bz, const void *bdx,
                           const void *bdy, const void *bdz, const void *w,
                           long long n_bins, const long long *bin_idx, double *A)
{
    return oracle_accumulate_step_w(n_dir, dirs, n_omega, omega, dt, t0, step_index, n_part, is_f32, rx, ry,
                                    rz, bx, by, bz, bdx, bdy, bdz, w, n_bins, bin_idx, A, 0, NULL, 0.0);
}

/*
 * Per-region detectors: particles are sorted by region, region r owns the particles
 * [offsets[r], offsets[r+1]) (offsets non-decreasing, n_regions+1 entries), and
 *   A_r[n][j][c] += the sum above over the particles of region r only.
 * A is [n_regions][n_dir][n_omega][3][2]; bin_idx (optional) selects the same (n, j) bins in
 * every region.  Written as the definition: one plain oracle_accumulate_step per region
 * on that region's slice of the state arrays.
 */
int oracle_accumulate_step_regions_ff(int n_dir, const double *dirs, int n_omega, const double *omega,
                                      double dt, double t0, long long step_index, long long n_regions,
                                      const long long *offsets, int is_f32, const void *rx,
                                      const void *ry, const void *rz, const void *bx, const void *by,
                                      const void *bz, const void *bdx, const void *bdy,
                                      const void *bdz, const void *w, long long n_bins,
                                      const long long *bin_idx, double *A, int win_type, const double *win,
                                      double nyquist, int ff_type, const double *ff_size)
{
    if (n_regions <= 0 || !offsets || offsets[0] < 0) return 1;
    for (long long r = 0; r < n_regions; ++r)
        if (offsets[r + 1] < offsets[r]) return 1;
    const size_t es = is_f32 ? sizeof(float) : sizeof(double);
#define AT(p, k) ((const void *)((const char *)(p) + (size_t)(k) * es))
    for (long long r = 0; r < n_regions; ++r) {
        const long long k0 = offsets[r], n_r = offsets[r + 1] - offsets[r];
        double *A_r = A + (size_t)r * n_dir * n_omega * 6;
        const int rc = oracle_accumulate_step_ff(n_dir, dirs, n_omega, omega, dt, t0, step_index, n_r,
                                                 is_f32, AT(rx, k0), AT(ry, k0), AT(rz, k0), AT(bx, k0),
                                                 AT(by, k0), AT(bz, k0), AT(bdx, k0), AT(bdy, k0),
                                                 AT(bdz, k0), AT(w, k0), n_bins, bin_idx, A_r, win_type, win, nyquist,
                                                 ff_type, ff_size);
        if (rc != 0) return rc;
    }
#undef AT
    return 0;
}

int oracle_accumulate_step_regions_w(int n_dir, const double *dirs, int n_omega, const double *omega,
                                     double dt, double t0, long long step_index, long long n_regions,
                                     const long long *offsets, int is_f32, const void *rx,
                                     const void *ry, const void *rz, const void *bx, const void *by,
                                     const void *bz, const void *bdx, const void *bdy,
                                     const void *bdz, const void *w, long long n_bins,
                                     const long long *bin_idx, double *A, int win_type, const double *win,
                                     double nyquist)
{
    return oracle_accumulate_step_regions_ff(n_dir, dirs, n_omega, omega, dt, t0, step_index, n_regions, offsets,
                                             is_f32, rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w, n_bins, bin_idx, A,
                                             win_type, win, nyquist, 0, NULL);
}

int oracle_accumulate_step_regions(int n_dir, const double *dirs, int n_omega, const double *omega,
                                   double dt, double t0, long long step_index, long long n_regions,
                                   const long long *offsets, int is_f32, const void *rx,
                                   const void *ry, const void *rz, const void *bx, const void *by,
                                   const void *bz, const void *bdx, const void *bdy,
                                   const void *bdz, const void *w, long long n_bins,
                                   const long long *bin_idx, double *A)
{
    return oracle_accumulate_step_regions_w(n_dir, dirs, n_omega, omega, dt, t0, step_index, n_regions, offsets,
                                            is_f32, rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w, n_bins, bin_idx, A,
                                            0, NULL, 0.0);
}

/* Per-region detectors, detector of all particles: S_total[n][j] = scale * sum_c |sum_r A_r,c|^2
 * (amplitudes, not intensities, add up: PAPER.md line 80).  A is [n_regions][n_bins][3][2]. */
int oracle_spectrum_total(long long n_regions, long long n_bins, const double *A, double scale, double *S)
{
    if (!A || !S || n_bins < 0 || n_regions <= 0) return 1;
    const double sc = (scale == 0.0) ? oracle_default_scale() : scale;
    for (long long b = 0; b < n_bins; ++b) {
        double tot[6] = {0, 0, 0, 0, 0, 0};
        for (long long r = 0; r < n_regions; ++r)
            for (int c = 0; c < 6; ++c) tot[c] += A[((size_t)r * n_bins + b) * 6 + c];
        double s = 0.0;
        for (int c = 0; c < 6; ++c) s += tot[c] * tot[c];
        S[b] = sc * s;
    }
    return 0;
}

/* S[n][j] = scale * sum_c |A_c|^2 ; scale == 0 -> SI default (Q4). */
int oracle_spectrum(long long n_bins_total, const double *A, double scale, double *S)
{
    if (!A || !S || n_bins_total < 0) return 1;
    const double sc = (scale == 0.0) ? oracle_default_scale() : scale;
    for (long long b = 0; b < n_bins_total; ++b) {
        const double *a = A + (size_t)b * 6;
        double s = 0.0;
        for (int c = 0; c < 6; ++c) s += a[c] * a[c];
        S[b] = sc * s;
    }
    return 0;
}
