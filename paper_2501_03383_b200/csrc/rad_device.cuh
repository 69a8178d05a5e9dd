// rad_device.cuh -- device helpers shared by the accumulate kernels: particle load, per
// (particle, direction) staging (a1) and the integer-phase sincos (a2).  See rad_kernels.cu
// and DESIGN.md "Phase arithmetic" for the derivation.
#pragma once
#include "rad_internal.h"

namespace rad {
namespace dev {

constexpr double kMagic = 6755399441055744.0;  // 1.5 * 2^52: fp64 round-to-integer constant
constexpr float kTwoPi = 6.283185307179586f;
constexpr float kUnitToRad = 1.4629180792671596e-09f;  // 2 pi / 2^32

// Programmatic dependent launch (RAD_FLAG_OVERLAP_STEPS; no-ops in a normally launched grid):
// pdl_trigger() lets the next kernel of the stream start once every block of this grid has
// started; pdl_wait() blocks until all work queued before this grid has completed and is visible.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// state element -> fp64: exact for every fp32 value (zero, subnormals, Inf and NaN included, so
// non-finite particle state propagates into the result as include/rad.h documents).
// F2F.F64.F32 is not an XU-rate instruction (>= 61 results/clk/SM, bench.py alu_peaks), unlike the
// opposite direction; round 1's integer-pipe version mapped 0 to 2^-127 and Inf/NaN to finite
// values for no measurable gain.
__device__ __forceinline__ double to_f64(double x) { return x; }
__device__ __forceinline__ double to_f64(float x) { return (double)x; }

// fp64 -> fp32 as ONE F2F: with -ftz the plain cast also emits a DSETP + select per conversion
// to flush fp32 subnormals, which these values (|x| >= 1e-30 or exactly 0) never are.
__device__ __forceinline__ float to_f32(double x)
{
    float f;
    asm("cvt.rn.f32.f64 %0, %1;" : "=f"(f) : "d"(x));
    return f;
}

// two fp32 in one 64-bit register pair, for the packed fma.rn.f32x2 / mul.rn.f32x2 (SASS FFMA2 / FMUL2:
// 59.6 instructions = 119 FMA per clock per SM against 85.8 for plain FFMA, bench.py alu_peaks)
__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ void fma2(unsigned long long &acc, unsigned long long a, unsigned long long b)
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ unsigned long long fma2r(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ unsigned long long mul2(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

// fp64 -> fp32 by TRUNCATION on the integer pipe (exponent re-bias + funnel shift: LOP3, IADD3, SHF, LOP3) instead of
// F2F.F32.F64, which is an XU-rate instruction (14 per clock per SM) and competes with MUFU.SIN/COS.  Values outside
// the fp32 normal range (zero, |x| < 2^-126, |x| >= 2^128, Inf, NaN) take the real conversion, so non-finite state
// still propagates.  Used by the one-direction-per-warp tile only (stage_record<true>): there the XU pipe is THE
// limiter and the change is worth 0.5 % (config 2 129.47 -> 128.80 ms); on the narrower tiles and in the streaming
// kernel, whose issue slots are as busy as their XU pipe, the extra integer instructions cost more than they save.
__device__ __forceinline__ float to_f32_trunc(double x)
{
    const unsigned hi = (unsigned)__double2hiint(x), lo = (unsigned)__double2loint(x);
    const unsigned ha = hi & 0x7fffffffu;
    float r = __uint_as_float(__funnelshift_l(lo, ha - 0x38000000u, 3) | (hi & 0x80000000u));
    if (ha - 0x38100000u >= 0x0fe00000u) r = to_f32(x);
    return r;
}

template <typename ST>
__device__ __forceinline__ ST ld_state(const void *p, long long k)
{
    return __ldg(reinterpret_cast<const ST *>(p) + k);
}

// a1: stage one particle for one direction -> record {T, ql, a1, a2} + sf.
struct Particle {
    double rx, ry, rz, bx, by, bz;  // fp64 for the phase and the Doppler factor
    float bfx, bfy, bfz, bdx, bdy, bdz, wdt;
    float w, ww;  // form factor on: macro weight w and w^2 - w (wdt is then dt [x window] only)
};

// form-factor weight g = sqrt(w + (w^2 - w) F^2) of one update (rad.h, reading FF1): FFMA + MUFU.SQRT
__device__ __forceinline__ float ff_weight(float w, float ww, float F2)
{
    float g;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(g) : "f"(fmaf(ww, F2, w)));
    return g;
}

template <bool TRUNC = false>
__device__ __forceinline__ void stage_record(const Particle &p, const DirRec &dr, double ts32,
                                             float4 &rec, float &sf, uint32_t *T_out = nullptr,
                                             double *d_out = nullptr, float *inv_out = nullptr)
{
    // phase: s32 = (t - n.r/c) f_unit 2^32 in fp64, split into integer (mod 2^32) + residual
    const double s32 = ts32 - fma(dr.kx, p.rx, fma(dr.ky, p.ry, dr.kz * p.rz));
    const double m = s32 + kMagic;
    const uint32_t T = (uint32_t)__double2loint(m);
    const double res = s32 - (m - kMagic);
    // Doppler factor d = 1 - n.beta in fp64 (no cancellation error for beta -> 1)
    const double d64 = 1.0 - fma(dr.nx, p.bx, fma(dr.ny, p.by, dr.nz * p.bz));
    const float d = TRUNC ? to_f32_trunc(d64) : to_f32(d64);
    // amplitude: n x ((n-beta) x bd) = (n-beta)(n.bd) - bd (1-n.beta); it is _|_ n, so its
    // components on the transverse basis are a_i = -(e_i.beta)(n.bd) - (e_i.bd) d
    const float g = fmaf(dr.nfx, p.bdx, fmaf(dr.nfy, p.bdy, dr.nfz * p.bdz));
    const float e1b = fmaf(dr.e1x, p.bfx, fmaf(dr.e1y, p.bfy, dr.e1z * p.bfz));
    const float e2b = fmaf(dr.e2x, p.bfx, fmaf(dr.e2y, p.bfy, dr.e2z * p.bfz));
    const float e1d = fmaf(dr.e1x, p.bdx, fmaf(dr.e1y, p.bdy, dr.e1z * p.bdz));
    const float e2d = fmaf(dr.e2x, p.bdx, fmaf(dr.e2y, p.bdy, dr.e2z * p.bdz));
    const float inv = 1.0f / d;
    const float pre = -p.wdt * inv * inv;  // -w dt / d^2
    rec.x = __uint_as_float(T);
    rec.y = (TRUNC ? to_f32_trunc(res) : to_f32(res)) * kUnitToRad;
    rec.z = pre * fmaf(e1b, g, e1d * d);
    rec.w = pre * fmaf(e2b, g, e2d * d);
    sf = (TRUNC ? to_f32_trunc(s32) : to_f32(s32)) * kUnitToRad;
    if (T_out) *T_out = T;
    if (d_out) *d_out = d64;
    if (inv_out) *inv_out = inv;
}

// Nyquist limiter (rad.h, reading N1): number of bins j with w_j dt d < pi nu.  The predicate is
// the oracle's expression in fp64 (two correctly rounded multiplications, in its order), monotone
// in j over the sorted w_j.  On log-spaced and linear grids (detected at rad_create) the count is
// first GUESSED in closed form from the fp32 Doppler factor -- w_cut = pi nu / (dt d), j = log_q(w_cut / w_0)
// or (w_cut - w_0) / dw, good to ~1e-4 of a bin -- and then CHECKED with the exact predicate (two independent
// evaluations: bin guess - 1 must be kept, bin guess must not), so the keep/drop set stays the oracle's bit
// for bit; when the check fails (the cut-off within the guess's error of a bin: ~1 in 5000) and on other
// grids the count is bisected (10-12 dependent steps).
__device__ __forceinline__ bool nyquist_keeps(const AccumParams &P, int j, double d)
{
    return __dmul_rn(__dmul_rn(__ldg(P.omega64 + j), P.dt64), d) < P.nyq_lim;
}
__device__ __forceinline__ int nyquist_count(const AccumParams &P, double d, float inv_d)
{
    int lo = 0, hi = P.n_omega;
    if (d != d) return hi;  // NaN state: the comparison is false for every bin, nothing is dropped (NaN propagates)
    if (P.nyq_mode != 0) {
        const float g = P.nyq_mode == 1 ? P.nyq_a * __log2f(P.nyq_b * inv_d) : fmaf(P.nyq_a, inv_d, P.nyq_b);
        const int c = (int)fminf(fmaxf(ceilf(g), 0.0f), (float)hi);  // (NaN / Inf / d <= 0 land on an end of the range)
        const bool above = c < hi ? nyquist_keeps(P, c, d) : false;     // bin c must be dropped ...
        const bool below = c > 0 ? nyquist_keeps(P, c - 1, d) : true;   // ... and bin c - 1 kept (independent loads)
        if (!above && below) return c;
        // the cut-off lies within the guess's error of a bin (or d <= 0): bisect
    }
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (nyquist_keeps(P, mid, d)) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

// exp(i 2 pi f tau) for one frequency f = (F + phi) f_unit from a staged record (integer phase)
__device__ __forceinline__ void phase_sincos(uint32_t F, float Ff, float fl, uint32_t T, float ql,
                                             float sf, float &sn, float &cs)
{
    const uint32_t u = F * T;
    const float v = __uint_as_float(0x3f800000u | (u >> 9));  // 1 + frac, in turns
    const float q = fmaf(fl, sf, Ff * ql);
    __sincosf(fmaf(v, kTwoPi, q), &sn, &cs);
}

// exp(i 2 pi f tau) for the evaluation sweep of the fast gridded path.  There the terms sit on a
// regular grid and carry the coherent low-frequency content of the signal, so a SYSTEMATIC error of
// the sin/cos at the phases a bin visits periodically (w_max visits the quarter turns: h w_max =
// pi / 2) leaks that content into the bin.  Hence the argument stays in TURNS and exact:
// v = frac - 1/2 in [-1/2, 1/2) (exact), t = v + phi_j T' / 2^32 (the small fraction term), and
// sin.approx / cos.approx see x = t * C with C = 0x40c90fdc, the fp32 just above 2 pi for which
// C * 0.15915494f = 1 + 6.3e-8: their own first instruction, x * 0.15915494f rounded towards zero,
// then returns t itself (exactly for every t whose mantissa is below 1.88, one ulp high otherwise),
// i.e. MUFU.SIN/COS are fed the exact turn -- 0, 1/4, 1/2 give exact 0 and 1.  The centring shifts
// every phase by half a turn: the caller's per-bin factor (g_corr) carries the -1.
__device__ __forceinline__ void phase_sincos_grid(uint32_t F, float fl, uint32_t T, float sf_turns,
                                                  float &sn, float &cs)
{
    const uint32_t u = F * T;
    const float v = __uint_as_float(0x3f800000u | (u >> 9)) - 1.5f;
    const float t = fmaf(fl, sf_turns, v);
    __sincosf(t * __uint_as_float(0x40c90fdcu), &sn, &cs);
}

// The same exp(i 2 pi f tau) WITHOUT the XU pipe: the reduced phase goes through FMA-pipe
// polynomials.  t = frac + q/(2 pi) turns; r = t - rint(2t)/2 in [-1/4, 1/4]; sin(2 pi r) and
// cos(2 pi r) by near-minimax odd/even polynomials (fp32 abs. error 1.9e-7 / 2.9e-7, below
// MUFU.SIN/COS's ~4e-7); the half-turn parity flips both signs.  27 FMA/ALU-pipe instructions
// instead of 10 + 2 MUFU: used for a fraction of the bins to take load off the XU pipe, the
// bound of the general kernel (DESIGN.md section 5.1 "hybrid").
__device__ __forceinline__ void phase_sincos_poly(uint32_t F, float Ff, float fl, uint32_t T, float ql,
                                                  float sf, float &sn, float &cs)
{
    constexpr float kMagicF = 12582912.0f;  // 1.5 * 2^23
    const uint32_t u = F * T;
    const float v = __uint_as_float(0x3f800000u | (u >> 9));  // 1 + frac, in turns
    const float q = fmaf(fl, sf, Ff * ql);                    // radians
    const float t = fmaf(q, 0.15915494309189535f, v);         // turns, in [0.5, 2.5]
    const float kf = fmaf(t, 2.0f, kMagicF);                  // low mantissa bits = rint(2t)
    const float r = fmaf(kf - kMagicF, -0.5f, t);             // [-1/4, 1/4] turns
    const uint32_t sign = __float_as_uint(kf) << 31;          // odd half-turn: z -> -z
    const float r2 = r * r;
    float ps = fmaf(3.976161437e+01f, r2, -7.658139608e+01f);
    ps = fmaf(ps, r2, 8.160248510e+01f);
    ps = fmaf(ps, r2, -4.134168072e+01f);
    ps = fmaf(ps, r2, 6.283185280e+00f);
    float pc = fmaf(5.702861988e+01f, r2, -8.533239558e+01f);
    pc = fmaf(pc, r2, 6.493784751e+01f);
    pc = fmaf(pc, r2, -1.973920580e+01f);
    sn = __uint_as_float(__float_as_uint(ps * r) ^ sign);
    cs = __uint_as_float(__float_as_uint(fmaf(pc, r2, 1.0f)) ^ sign);
}

// Spatial window on the macro weight (rad.h, reading W1): product over the windowed axes of
// w1((r_c - o_c)/L_c).  Inside/outside is decided in fp64, the window value in fp32.
__device__ __forceinline__ float window_weight(const AccumParams &P, double rx, double ry, double rz)
{
    if (P.win_type == RAD_WINDOW_NONE) return 1.0f;
    const double r[3] = {rx, ry, rz};
    float W = 1.0f;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (P.win_il[c] > 0.0) {
            const double u = (r[c] - P.win_o[c]) * P.win_il[c];
            const float uf = to_f32(u);
            const float w1 = P.win_type == RAD_WINDOW_TRIANGLE ? 1.0f - fabsf(fmaf(2.0f, uf, -1.0f))
                                                               : fmaf(-0.46f, __cosf(kTwoPi * uf), 0.54f);
            W *= (u >= 0.0 && u <= 1.0) ? w1 : 0.0f;
        }
    }
    return W;
}

// ff: form factor on -- the macro weight stays out of the amplitude record (it enters per update
// through ff_weight); the record then carries dt [x window] only
template <typename ST, bool WIN = true>
__device__ __forceinline__ Particle load_particle(const AccumParams &P, long long k, bool valid, const bool ff = false)
{
    Particle p;
    if (valid) {
        const ST rx = ld_state<ST>(P.st[0], k), ry = ld_state<ST>(P.st[1], k),
                 rz = ld_state<ST>(P.st[2], k);
        const ST bx = ld_state<ST>(P.st[3], k), by = ld_state<ST>(P.st[4], k),
                 bz = ld_state<ST>(P.st[5], k);
        const ST dx = ld_state<ST>(P.st[6], k), dy = ld_state<ST>(P.st[7], k),
                 dz = ld_state<ST>(P.st[8], k);
        const ST w = ld_state<ST>(P.st[9], k);
        p.rx = to_f64(rx); p.ry = to_f64(ry); p.rz = to_f64(rz);
        p.bx = to_f64(bx); p.by = to_f64(by); p.bz = to_f64(bz);
        p.bfx = (float)bx; p.bfy = (float)by; p.bfz = (float)bz;
        p.bdx = (float)dx; p.bdy = (float)dy; p.bdz = (float)dz;
        p.w = (float)w;
        p.ww = fmaf(p.w, p.w, -p.w);
        p.wdt = ff ? P.dt : (P.w_sqrt ? __fsqrt_rn(p.w) : p.w) * P.dt;
        if (WIN) p.wdt *= window_weight(P, p.rx, p.ry, p.rz);
    } else {  // padding lane: zero amplitude, harmless phase
        p.rx = p.ry = p.rz = p.bx = p.by = p.bz = 0.0;
        p.bfx = p.bfy = p.bfz = p.bdx = p.bdy = p.bdz = p.wdt = p.w = p.ww = 0.0f;
    }
    return p;
}

}  // namespace dev
}  // namespace rad
