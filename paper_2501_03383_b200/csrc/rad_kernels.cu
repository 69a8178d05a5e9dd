// rad_kernels.cu -- accumulation kernels (SURVEY.md section 8(a) rows a1, a2, a2', a3) for sm_100a.
//
// Mapping ("bin owner"): a thread owns S frequency bins of one direction and keeps their
// transverse complex amplitudes (A1, A2) in fp32 registers; a warp owns DPW = 32/LW
// directions x (LW*S) frequencies; the 4 warps of a block own 4 such tiles and share one
// chunk of particles.  Per batch of 32 particles each lane stages ONE particle for the
// warp's directions (a1: coalesced SoA loads, fp64 phase set-up, fp32 amplitude) into the
// warp's private shared-memory records; then all lanes sweep the 32 records (a2), reading
// them as shared-memory broadcasts.  No block-level barrier anywhere.
//
// Work decomposition: a warp task = (warp tile, particle chunk); task id = 4*blockIdx.x + warp,
// warp tile = id mod n_wtiles, chunk = id / n_wtiles, so the 4 warps of a block share their
// chunk (L1 hits on the state) whenever n_wtiles is a multiple of 4 and no warp idles when it
// is not.  A chunk is [c*chunk, (c+1)*chunk) or, for per-region detectors, an entry of the
// chunk table (particles of ONE region; the fold goes to that region's accumulator).
//
// Phase: turns = f_j tau, tau = t - n.r/c.  With
// f_j = (F_j + phi_j) f_unit (F_j a 32-bit integer, |phi_j| <= 1/2) and
// s32 = tau f_unit 2^32 = I + res (I integer, |res| <= 1/2, both from fp64):
//   frac(turns) = frac( (F_j * (I mod 2^32) mod 2^32) / 2^32  +  F_j res / 2^32  +  phi_j s )
// The first term is ONE 32-bit integer multiply (wrap-around = exact reduction mod one turn
// for any |tau|); the other two are O(1/2 turn) and O(tau f_unit) and are added in fp32.
#include <math_constants.h>

#include <type_traits>

#include "rad_device.cuh"
#include "rad_internal.h"

namespace rad {

namespace {

using namespace dev;

// a3: fold one thread's fp32 partials into the fp64 accumulator (or the deterministic
// per-chunk workspace).
template <int S, int LW, bool GRID = false>
__device__ __forceinline__ void fold(const AccumParams &P, const float (&acc)[S][4], int dir,
                                     int jbase, int ci, int region)
{
    if (dir >= P.n_dir) return;
    if (GRID) {  // fast gridded path: the partial is divided by the spreading kernel's transform
        double *dst = P.acc + (size_t)dir * (size_t)P.w_pad * 4;
#pragma unroll
        for (int i = 0; i < S; ++i) {
            const int j = jbase + i * LW;
            if (j < P.n_omega) {
                // complex factor 1 / (Phi_j (1 - exp(i w_j h))): kernel transform and first differences
                const double2 c = __ldg(P.g_corr + j);
                const double p0 = acc[i][0], p1 = acc[i][1], p2 = acc[i][2], p3 = acc[i][3];
                atomicAdd(dst + (size_t)j * 4 + 0, c.x * p0 - c.y * p1);
                atomicAdd(dst + (size_t)j * 4 + 1, c.x * p1 + c.y * p0);
                atomicAdd(dst + (size_t)j * 4 + 2, c.x * p2 - c.y * p3);
                atomicAdd(dst + (size_t)j * 4 + 3, c.x * p3 + c.y * p2);
            }
        }
        return;
    }
    if (P.partial) {
        double *dst = P.partial + ((size_t)ci * P.n_dir + dir) * (size_t)P.w_pad * 4;
#pragma unroll
        for (int i = 0; i < S; ++i) {
            const int j = jbase + i * LW;
            double2 *q = reinterpret_cast<double2 *>(dst + (size_t)j * 4);
            q[0] = make_double2((double)acc[i][0], (double)acc[i][1]);
            q[1] = make_double2((double)acc[i][2], (double)acc[i][3]);
        }
    } else {
        double *dst = P.acc + ((size_t)region * P.n_dir + dir) * (size_t)P.w_pad * 4;
#pragma unroll
        for (int i = 0; i < S; ++i) {
            const int j = jbase + i * LW;
            if (j < P.n_omega) {
#pragma unroll
                for (int c = 0; c < 4; ++c) atomicAdd(dst + (size_t)j * 4 + c, (double)acc[i][c]);
            }
        }
    }
}

// warp task -> (warp tile, chunk index, particle range, region); false: no task for this warp
__device__ __forceinline__ bool decode_task(const AccumParams &P, int warp, int &wt, int &ci,
                                            long long &k0, long long &k1, int &region, double &ts32)
{
    const long long task = (long long)blockIdx.x * kWarpsPerBlock + warp;
    if (task >= (long long)P.n_wtiles * P.n_chunks) return false;
    ci = (int)(task / P.n_wtiles);
    wt = (int)(task - (long long)ci * P.n_wtiles);
    if (P.chunks) {
        const ChunkRec c = P.chunks[ci];
        k0 = c.k0; k1 = c.k0 + c.len; region = c.region;
        ts32 = fma((double)c.step, P.dts32, P.ts32);
    } else {
        ts32 = P.ts32;
        k0 = (long long)ci * P.chunk;
        k1 = min(P.n_particles, k0 + (long long)P.chunk);
        region = 0;
    }
    return true;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// a2 (UNI = false): general (non-uniform) frequency grid.  Per update: 1 IMAD + 1 LEA.HI + 3 FP32
// for the phase, FMUL + MUFU.SIN + MUFU.COS, 4 FFMA.
// a2' (UNI = true): uniform grid w_j = w_0 + j dw.  A thread's bins are LW dw apart, so they are
// the powers of rot = exp(i LW dw tau), staged once per (particle, direction).  The chain is
// anchored at the thread's middle bin by a direct integer-phase sincos; the next bin is one
// complex product with rot, and every other bin follows from the three-term recurrence
// z_(i+1) = 2 cos(theta) z_i - z_(i-1) (one packed FMA), S/2 steps forwards and S/2-1 backwards:
// 1 sincos + 1 complex product + (S-2) packed FMAs per S updates instead of S sincos.  Chain
// length <= S/2 keeps the recurrence drift (an error grows at most n-fold over n steps) below the
// MUFU error, which is the periodic re-anchoring BASELINE.json asks for.
// NYQ (general grid only): Nyquist limiter -- the staging lane also finds, per (particle,
// direction), how many bins lie below the cut-off (nyquist_count); the sweep accumulates bin j
// only if j < that count (one ISETP per update, the four FFMAs are predicated).
// FF: macro-particle form factor (rad.h, reading FF1) -- every update's (cos, sin) is scaled by
// g = sqrt(w + (w^2 - w) F^2): F^2 of the thread's S bins in registers, (w, w^2 - w) of the batch's
// particles in shared memory; one FFMA + MUFU.SQRT + 2 FMUL more per update.
// DY (general grid only): dyadic log grid, w_(j + DY*LW) = 2 w_j (an integer number of bins per octave that
// the tile shape divides: rad_api.cu).  Bins i and i + DY of a thread's strip are then one octave apart and
// z_(i+DY) = z_i^2 (4 FMA-pipe instructions instead of the phase arithmetic + MUFU.SIN/COS).  Chains are
// kDyadChain = 2 bins long: every second bin of a chain is anchored by a direct sincos, the other is its
// square.  A squaring doubles the phase error and the deviation of |z| from 1: measured maxrel against the
// oracle with one squaring per chain = the plain kernel's (2.5e-4 vs 2.9e-4 on a 6 x 300 detector), with two
// squarings 2.2e-3 (beyond the 1e-3 tolerance: the MUFU error x 4).
// GRID: evaluation of the fast gridded path (rad.h RAD_FLAG_FAST_GRIDDED) -- the "particles" are the
// points of the per-direction retarded-time grids: point m of direction n has phase s32 = g_s0[n] +
// m g_hs and amplitude g_master[n][m]; the sweep and the phase arithmetic are those of the general grid.
// Uniform-grid chain in packed form: sign s_n of y_n = s_n z_(MID+n) forwards (n >= 0: + + - - + + ...) and of
// y'_m = s'_m z_(MID-m) backwards (m >= 0: + - - + + - ...); with them s_(n+1) / s_(n-1) = -1, so the three-term
// recurrence has no subtraction.
__host__ __device__ constexpr int uni_sign(int n) { return (n & 3) >= 2 ? -1 : 1; }
__host__ __device__ constexpr int uni_sign_b(int m) { return ((m + 1) & 3) >= 2 ? -1 : 1; }
constexpr int kDyadChain = 2;  // dyadic grids: bins per squaring chain (1 anchor + kDyadChain - 1 squarings)

template <typename ST, int LW, int S, int MINB, bool UNI, bool NYQ, bool FF, bool GRID = false, int DY = 0, bool SPLIT = false,
          bool PREC = false>
__global__ void __launch_bounds__(kThreads, MINB) rad_accum(const AccumParams P)
{
    static_assert(!GRID || (!UNI && !NYQ && !FF), "grid evaluation runs the plain general-grid sweep");
    static_assert(DY == 0 || (!UNI && !NYQ && !FF && !GRID), "dyadic squaring runs on the plain general-grid sweep");
    static_assert(!SPLIT || (LW < 32 && !NYQ && !FF && !GRID && DY == 0), "particle split: plain general / uniform sweep, >= 2 lane groups");
    static_assert(!PREC || (!UNI && !NYQ && !FF && !GRID && DY == 0 && !SPLIT), "RAD_FLAG_PRECISE: the plain general-grid sweep, every bin by the polynomial");
    static_assert(!(UNI && NYQ), "the limiter runs on the general-grid kernel");
    constexpr int DPW = 32 / LW;
    // Shared-memory records are direction-major, rec[direction of the warp][particle of the batch], rows padded
    // by one record: the staging lanes store 16-byte records at consecutive addresses and the sweep's
    // DPW different broadcast reads (one per direction) fall into different banks.  (Particle-major
    // rec[particle][direction] made the stores of a warp 64 or 128 bytes apart: 4- / 8-way bank
    // conflicts, 1.26e8 conflict cycles per launch on config 3d, profiles/r2_ncu_rad_accum_general_cfg3d.md.)
    constexpr int PITCH = kBatch + (DPW > 1 ? 1 : 0);
    constexpr int NC = UNI ? 1 : S;  // per-thread frequency constants held in registers
    constexpr int MID = S / 2 - 1;   // anchor bin of the uniform-grid chain
    __shared__ float4 s_rec[kWarpsPerBlock][PITCH * DPW];
    __shared__ float s_sf[kWarpsPerBlock][PITCH * DPW];
    __shared__ float2 s_rot[UNI ? kWarpsPerBlock : 1][UNI ? PITCH * DPW : 1];
    __shared__ int s_jc[NYQ ? kWarpsPerBlock : 1][NYQ ? PITCH * DPW : 1];
    __shared__ float2 s_w[FF ? kWarpsPerBlock : 1][FF ? kBatch : 1];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int wt, ci, region;
    long long k0, k1;
    double ts32;
    pdl_trigger();
    if (!decode_task(P, warp, wt, ci, k0, k1, region, ts32)) return;  // whole warp leaves; no block barrier below
    const int dg = wt / P.n_ftiles, ft = wt - dg * P.n_ftiles;
    const int ld = lane / LW, lf = lane - ld * LW;
    const int jbase = ft * (LW * S) + lf;
    // Particle split (P.psplit = PS > 0; detectors with fewer directions than a warp holds, rad_api.cu
    // choose_tile): 2^PS lane groups share ONE direction and take every 2^PS-th record of a batch each, so no
    // lane idles on a padded direction; their partial sums meet in a shuffle reduction before the fold.
    const int PS = SPLIT ? P.psplit : 0;     // compile-time 0 in every other instantiation
    const int rl = ld >> PS;                    // row of this lane's direction in the staged records
    const int psub = ld & ((1 << PS) - 1);      // which records of a batch this lane group sweeps
    const int dir0 = (dg * DPW) >> PS;          // first direction of the warp
    const int n_rows = DPW >> PS;               // directions staged per warp

    uint32_t F[NC];
    float Ff[NC], fl[NC], acc[S][4];
#pragma unroll
    for (int i = 0; i < NC; ++i) {
        const int j = jbase + (UNI ? MID : i) * LW;
        F[i] = __ldg(P.F + j);
        Ff[i] = __ldg(P.Ff + j);
        fl[i] = __ldg(P.fl + j);
    }
#pragma unroll
    for (int i = 0; i < S; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.0f;
    // Packed (re, im) accumulators, two fma.rn.f32x2 per update instead of four FFMA (the scalar amplitude enters
    // as the broadcast operand form Rn.F32): measured where the issue slots matter more than the packed form's
    // longer stay in the FMA pipe -- uniform grid 3196 -> 3327 G/s, general grid with the form factor 1343 ->
    // 1416 G/s; NOT on the plain general kernel (config 2 -0.3 %, config 3d -6 %) nor the dyadic one (-1.4 %).
    constexpr bool PK = (UNI && !FF) || (!UNI && !NYQ && FF && !GRID);
    unsigned long long accA[PK ? S : 1], accB[PK ? S : 1];
#pragma unroll
    for (int i = 0; i < (PK ? S : 1); ++i) accA[i] = accB[i] = 0ull;
    float F2r[FF ? S : 1];
    if (FF) {
        const float *row = P.F2 + (size_t)min(dir0 + rl, P.n_dir - 1) * P.w_pad + jbase;
#pragma unroll
        for (int i = 0; i < S; ++i) F2r[FF ? i : 0] = __ldg(row + i * LW);
    }

    float4 *rec = s_rec[warp];
    float *sfs = s_sf[warp];
    float2 *rots = s_rot[UNI ? warp : 0];
    int *jcs = s_jc[NYQ ? warp : 0];
    float2 *ws = s_w[FF ? warp : 0];

    for (long long kb = k0; kb < k1; kb += kBatch) {
        if (GRID) {  // stage grid point m = kb + lane for the warp's directions
            // Phase unit of the evaluation = one grid step (frequency tables built with f_unit' =
            // 1 / (h 2^32), rad_api.cu): tau_m / h = g_s0[n] + m is an INTEGER, so the integer phase
            // F'_j * T mod 2^32 is the whole phase and no fp32 term depends on the position within a
            // period of f_max.  (With the direct path's unit the fractional part of tau f_max repeats
            // every 4 grid points; its fp32 rounding then modulates the coherent low-frequency content
            // of the grid with exactly the period of w_max and leaks 5e-7 of the PEAK into the top bin.)
            const long long m = kb + lane;
#pragma unroll(DPW > 2 ? 1 : DPW)
            for (int dd = 0; dd < DPW; ++dd) {
                const int dir = min(dg * DPW + dd, P.n_dir - 1);
                const double t_units = __ldg(P.g_s0 + dir) + (double)m;   // exact integer
                // Frequency tiles from bin g_jdiff on sum FIRST DIFFERENCES of the grid, g_m - g_(m-1) (fp64):
                // sum_m (g_m - g_(m-1)) z^m = (1 - z) sum_m g_m z^m, undone per bin at fold time (g_corr).
                // The grid is dominated by the coherent low-frequency part of the signal (all deposits of
                // one sign); the differences are not, so the systematic part of the fp32 sin/cos error (a
                // fixed function of the phase, sampled on a regular grid) has no coherent content left to
                // leak into the dark high-frequency bins (measured without: a white floor of 1e-7 of the
                // peak amplitude, 3e-4 ... 8e-4 on bins at 1e-6 of the peak).  Dividing by 1 - z amplifies
                // the rounding noise by 1 / (w h), so the low-frequency tiles (w h < 2.5e-3), where the
                // signal itself is the coherent peak, sum the grid as it is.
                double2 g = make_double2(0.0, 0.0);
                if (m < k1) {
                    const double2 *row = P.g_master + (size_t)dir * P.g_M;
                    g = __ldg(row + m);
                    if (m > 0 && ft * (LW * S) >= P.g_jdiff) {
                        const double2 gp = __ldg(row + m - 1);
                        g.x -= gp.x;
                        g.y -= gp.y;
                    }
                }
                rec[dd * PITCH + lane] = make_float4(__uint_as_float((uint32_t)__double2loint(t_units + kMagic)), 0.0f,
                                                   to_f32(g.x), to_f32(g.y));
                sfs[dd * PITCH + lane] = to_f32(t_units) * 2.3283064365386963e-10f;   // T' / 2^32 (turns per unit fraction)
            }
        } else {  // a1: stage
            const long long k = kb + lane;
            const Particle p = load_particle<ST, true>(P, k, k < k1, FF);
            if (FF) ws[lane] = make_float2(p.w, p.ww);
#pragma unroll(DPW > 2 ? 1 : DPW)  // 4 or 8 directions per warp: keep the staging code out of the register budget
            for (int dd = 0; dd < n_rows; ++dd) {
                const int dir = min(dir0 + dd, P.n_dir - 1);
                float4 r4;
                float sf;
                uint32_t T;
                double d64;
                float inv_d;
                stage_record<(DPW == 1 && !UNI && DY == 0 && !PREC)>(p, P.dirs[dir], ts32, r4, sf, &T, &d64, &inv_d);
                rec[dd * PITCH + lane] = r4;
                sfs[dd * PITCH + lane] = sf;
                // bins below the cut-off, relative to the first bin of the warp's frequency tile
                if (NYQ) jcs[dd * PITCH + lane] = nyquist_count(P, d64, inv_d) - ft * (LW * S);
                if (UNI) {
                    float sn, cs;
                    phase_sincos(P.rot_G, P.rot_Gf, P.rot_gl, T, r4.y, sf, sn, cs);
                    rots[dd * PITCH + lane] = make_float2(cs, sn);
                }
            }
        }
        __syncwarp();
        if (UNI) {
#pragma unroll 4
            for (int kk = psub; kk < kBatch; kk += 1 << PS) {  // a2': sweep with the rotation recurrence
                const float4 r4 = rec[rl * PITCH + kk];
                const float sf = sfs[rl * PITCH + kk];
                const float2 rot = rots[rl * PITCH + kk];
                float zi0, zr0;
                phase_sincos(F[0], Ff[0], fl[0], __float_as_uint(r4.x), r4.y, sf, zi0, zr0);
                const float2 wq = FF ? ws[kk] : make_float2(0.0f, 0.0f);
                const unsigned long long A1b = pack2(r4.z, r4.z), A2b = pack2(r4.w, r4.w);
                auto add = [&](const int i, const float zr_, const float zi_) {  // acc[i] += a (x) z [* g]
                    if constexpr (!FF) {
                        const unsigned long long Z = pack2(zr_, zi_);
                        fma2(accA[i], A1b, Z);
                        fma2(accB[i], A2b, Z);
                    } else {
                        const float g = ff_weight(wq.x, wq.y, F2r[FF ? i : 0]);
                        const float cr = zr_ * g, ci = zi_ * g;
                        acc[i][0] = fmaf(r4.z, cr, acc[i][0]);
                        acc[i][1] = fmaf(r4.z, ci, acc[i][1]);
                        acc[i][2] = fmaf(r4.w, cr, acc[i][2]);
                        acc[i][3] = fmaf(r4.w, ci, acc[i][3]);
                    }
                };
                add(MID, zr0, zi0);
                // One complex rotation gives z_(MID+1) = z_MID rot; every other bin of the strip follows from
                // the three-term recurrence of a rotation by a fixed angle, z_(i+-1) = 2 cos(theta) z_i - z_(i-+1)
                // (2 FFMA per bin instead of the 4 FMA-pipe instructions of a complex product).  A rounding error
                // delta grows like sin(n theta) / sin(theta) <= n over n <= S/2 steps from the anchor.
                const float c2 = rot.x + rot.x;
                const float fr = fmaf(zr0, rot.x, -zi0 * rot.y), fi = fmaf(zi0, rot.x, zr0 * rot.y);  // z_(MID+1)
                if constexpr (!FF) {
                    // Packed form, one fma.rn.f32x2 per bin and no negation: the chain carries y = s z with the
                    // signs s = + + - - + ... (uni_sign), for which y_(n+1) = (+-2c) y_n + y_(n-1); the bins with
                    // s = -1 accumulate -A and get their sign back after the sweep (below).
                    const unsigned long long Cp = pack2(c2, c2), Cn = pack2(-c2, -c2);
                    const unsigned long long Y0 = pack2(zr0, zi0);
                    auto addp = [&](const int i, const unsigned long long Y) {
                        fma2(accA[i], A1b, Y);
                        fma2(accB[i], A2b, Y);
                    };
                    unsigned long long P0 = Y0, Y = pack2(fr, fi);  // forwards: n = 1
                    addp(MID + 1, Y);
#pragma unroll
                    for (int i = MID + 2; i < S; ++i) {
                        const int n = i - MID;  // y_n from y_(n-1), y_(n-2): factor 2c s_n / s_(n-1)
                        const unsigned long long N = fma2r(uni_sign(n) == uni_sign(n - 1) ? Cp : Cn, Y, P0);
                        P0 = Y; Y = N;
                        addp(i, Y);
                    }
                    if (MID >= 1) {
                        P0 = Y0;
                        Y = fma2r(Cn, Y0, pack2(fr, fi));  // backwards: m = 1, y'_1 = -z_(MID-1) = -2c z_MID + z_(MID+1)
                        addp(MID - 1, Y);
#pragma unroll
                        for (int i = MID - 2; i >= 0; --i) {
                            const int m = MID - i;
                            const unsigned long long N = fma2r(uni_sign_b(m) == uni_sign_b(m - 1) ? Cp : Cn, Y, P0);
                            P0 = Y; Y = N;
                            addp(i, Y);
                        }
                    }
                } else {
                    float pr = zr0, pi = zi0, zr = fr, zi = fi;
                    const float br = fmaf(c2, zr0, -zr), bi = fmaf(c2, zi0, -zi);  // z_(MID-1)
                    add(MID + 1, zr, zi);
#pragma unroll
                    for (int i = MID + 2; i < S; ++i) {  // forwards
                        const float nr = fmaf(c2, zr, -pr), ni = fmaf(c2, zi, -pi);
                        pr = zr; pi = zi; zr = nr; zi = ni;
                        add(i, zr, zi);
                    }
                    if (MID >= 1) add(MID - 1, br, bi);
                    pr = zr0; pi = zi0; zr = br; zi = bi;
#pragma unroll
                    for (int i = MID - 2; i >= 0; --i) {  // backwards
                        const float nr = fmaf(c2, zr, -pr), ni = fmaf(c2, zi, -pi);
                        pr = zr; pi = zi; zr = nr; zi = ni;
                        add(i, zr, zi);
                    }
                }
            }
        } else {
            // a2: sweep.  Hybrid: of every two particles, kPolyEven / kPolyOdd of the S bins take
            // the FMA-pipe polynomial sincos instead of MUFU.SIN/COS (balances XU against issue).
            // One staged record against the S bins of the strip.  Limiter only: bins [0, KLO) are accumulated
            // unconditionally, the four FMAs of a bin in [KLO, KHI) are predicated on "bin below this record's
            // cut-off" (bins i*LW < m of the strip are kept), bins [KHI, S) are not computed at all.
            struct Rec { float4 r4; float sf; int m; float2 wq; };
            auto load_rec = [&](const int kk, const bool pred) {
                Rec r;
                r.r4 = rec[rl * PITCH + kk];
                r.sf = sfs[rl * PITCH + kk];
                r.m = pred ? jcs[rl * PITCH + kk] - lf : 0;
                r.wq = FF ? ws[kk] : make_float2(0.0f, 0.0f);
                return r;
            };
            auto sweep_bins = [&](const Rec &r, const int n_poly, auto klo_tag, auto khi_tag) {
                constexpr int KLO = decltype(klo_tag)::value, KHI = decltype(khi_tag)::value;
                const float4 r4 = r.r4;
                const float sf = r.sf;
                const uint32_t T = __float_as_uint(r4.x);
                float zs[S], zc[S];  // DY: the strip's (sin, cos), bin i + DY squares bin i
#pragma unroll
                for (int i = 0; i < (KHI < S ? KHI : S); ++i) {
                    float sn, cs;
                    if (DY > 0 && (i / (DY > 0 ? DY : 1)) % kDyadChain != 0) {
                        const float ps = zs[i >= DY ? i - DY : 0], pc = zc[i >= DY ? i - DY : 0];
                        cs = fmaf(pc, pc, -ps * ps);
                        sn = (pc + pc) * ps;
                    } else if (GRID)
                        phase_sincos_grid(F[i % NC], fl[i % NC], T, sf, sn, cs);
                    else if (i >= S - n_poly)
                        phase_sincos_poly(F[i % NC], Ff[i % NC], fl[i % NC], T, r4.y, sf, sn, cs);
                    else
                        phase_sincos(F[i % NC], Ff[i % NC], fl[i % NC], T, r4.y, sf, sn, cs);
                    zs[i] = sn;
                    zc[i] = cs;
                    if (FF) {
                        const float g = ff_weight(r.wq.x, r.wq.y, F2r[FF ? i : 0]);
                        sn *= g;
                        cs *= g;
                    }
                    if (i >= KLO) {
                        // limiter: one SETP + four predicated FFMAs written in PTX, so that the
                        // compiler keeps the bins' instruction streams interleaved (as C++ it
                        // sinks each bin's sincos into a branch of its own: 2.07 -> 3.08 ms)
                        asm("{\n\t.reg .pred p;\n\tsetp.lt.s32 p, %8, %9;\n\t"
                            "@p fma.rn.ftz.f32 %0, %4, %6, %0;\n\t@p fma.rn.ftz.f32 %1, %4, %7, %1;\n\t"
                            "@p fma.rn.ftz.f32 %2, %5, %6, %2;\n\t@p fma.rn.ftz.f32 %3, %5, %7, %3;\n\t}"
                            : "+f"(acc[i][0]), "+f"(acc[i][1]), "+f"(acc[i][2]), "+f"(acc[i][3])
                            : "f"(r4.z), "f"(r4.w), "f"(cs), "f"(sn), "r"(i * LW), "r"(r.m));
                    } else if constexpr (PK) {
                        const unsigned long long Z = pack2(cs, sn);
                        fma2(accA[i], pack2(r4.z, r4.z), Z);
                        fma2(accB[i], pack2(r4.w, r4.w), Z);
                    } else {
                        acc[i][0] = fmaf(r4.z, cs, acc[i][0]);
                        acc[i][1] = fmaf(r4.z, sn, acc[i][1]);
                        acc[i][2] = fmaf(r4.w, cs, acc[i][2]);
                        acc[i][3] = fmaf(r4.w, sn, acc[i][3]);
                    }
                }
            };
            using KS = std::integral_constant<int, S>;
            if constexpr (NYQ) {
                // The cut-offs of a batch's records lie close together (the Doppler factor moves them by a few
                // per cent): per BATCH the warp finds their range, [mn, mx) relative to the tile's first bin, and
                // runs the batch with the bins below every cut-off unconditional (klo = mn / LW bins of the strip:
                // the bins of a strip are LW apart, "bin i of every lane" is a block of LW frequencies), the
                // next two predicated and the rest not computed -- one of S + 1 straight-line sweeps, so nothing
                // inside a sweep branches.  A batch whose cut-offs span more than two blocks runs fully predicated.
                // (History, config 1 with nu = 1: every record predicated 2.26 ms; all / none / predicated paths
                // per pair of records 2.20 ms; skippable 2-bin groups inside the predicated strip 2.23 ms; 64-bin
                // tiles 2.42 ms.)
                int mn = jcs[lane], mx = mn;
                for (int dd = 1; dd < n_rows; ++dd) {
                    const int v = jcs[dd * PITCH + lane];
                    mn = min(mn, v);
                    mx = max(mx, v);
                }
                mn = __reduce_min_sync(0xffffffffu, mn);
                mx = __reduce_max_sync(0xffffffffu, mx);
                const int klo = min(S, max(mn, 0) / LW), khi = min(S, (max(mx, 0) + LW - 1) / LW);
                auto run = [&](auto klo_tag, auto khi_tag) {
                    constexpr bool pred = decltype(klo_tag)::value < decltype(khi_tag)::value;
#pragma unroll 1
                    for (int kk = 0; kk < kBatch; kk += 2) {
                        const Rec ra = load_rec(kk, pred), rb = load_rec(kk + 1, pred);
                        sweep_bins(ra, kPolyEven, klo_tag, khi_tag);
                        sweep_bins(rb, kPolyOdd, klo_tag, khi_tag);
                    }
                };
                using std::integral_constant;
                if (khi == 0) {
                    // every bin of the tile above every cut-off: nothing to add
                } else if (khi - klo > 2) {
                    run(integral_constant<int, 0>{}, KS{});
                } else {
                    static_assert(S == 8, "one sweep per number of unconditional bins");
                    switch (klo) {
                        case 0: run(integral_constant<int, 0>{}, integral_constant<int, 2>{}); break;
                        case 1: run(integral_constant<int, 1>{}, integral_constant<int, 3>{}); break;
                        case 2: run(integral_constant<int, 2>{}, integral_constant<int, 4>{}); break;
                        case 3: run(integral_constant<int, 3>{}, integral_constant<int, 5>{}); break;
                        case 4: run(integral_constant<int, 4>{}, integral_constant<int, 6>{}); break;
                        case 5: run(integral_constant<int, 5>{}, integral_constant<int, 7>{}); break;
                        case 6: run(integral_constant<int, 6>{}, KS{}); break;
                        case 7: run(integral_constant<int, 7>{}, KS{}); break;
                        default: run(KS{}, KS{}); break;
                    }
                }
            } else {
#pragma unroll 1
                for (int m2 = 0; m2 < (kBatch >> PS); m2 += 2) {
                    const int kk = (m2 << PS) + psub;
                    const Rec ra = load_rec(kk, false), rb = load_rec(kk + (1 << PS), false);
                    sweep_bins(ra, PREC ? S : DY > 0 ? 0 : kPolyEven, KS{}, KS{});   // dyadic: the XU pipe is not the bound
                    sweep_bins(rb, PREC ? S : DY > 0 ? 0 : kPolyOdd, KS{}, KS{});
                }
            }
        }
        __syncwarp();
    }
    if constexpr (PK) {
#pragma unroll
        for (int i = 0; i < S; ++i) {
            unpack2(accA[i], acc[i][0], acc[i][1]);
            unpack2(accB[i], acc[i][2], acc[i][3]);
            if (UNI && (i >= MID ? uni_sign(i - MID) : uni_sign_b(MID - i)) < 0) {  // bins whose chain carried -z
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[i][c] = -acc[i][c];
            }
        }
    }
    if (SPLIT) {  // particle split: sum the lane groups of a direction (fixed order), group 0 folds
        for (int o = LW; o < (LW << PS); o <<= 1) {
#pragma unroll
            for (int i = 0; i < S; ++i)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[i][c] += __shfl_xor_sync(0xffffffffu, acc[i][c], o);
        }
    }
    pdl_wait();  // the accumulator (and the deterministic workspace) belong to earlier work until here
    fold<S, LW, GRID>(P, acc, psub == 0 ? dir0 + rl : P.n_dir, jbase, ci, region);
}

// ------------------------------------------------------------------------------------------
// Launch logic.
template <typename ST, int LW, int S, int MINB, bool UNI, bool NYQ, bool FF>
static cudaError_t launch_one(const AccumParams &p, cudaStream_t s, bool overlap)
{
    const long long n_tasks = (long long)p.n_wtiles * p.n_chunks;
    const unsigned grid = (unsigned)((n_tasks + kWarpsPerBlock - 1) / kWarpsPerBlock);
    return launch_kernel(rad_accum<ST, LW, S, MINB, UNI, NYQ, FF>, dim3(grid), dim3(kThreads), 0, s, overlap, p);
}

template <typename ST, bool UNI, bool NYQ, bool FF>
static cudaError_t dispatch_lw(const Handle &h, const AccumParams &p, cudaStream_t s)
{
    // the form-factor variants need 8 more registers (F^2 of the strip): the narrow tile shapes and
    // the limiter variant would spill at the 128-register cap of 4 blocks per SM -> 3 blocks (168)
    constexpr int kMB = FF ? kMinBlocks - 1 : kMinBlocks;
    constexpr int kMBwide = (FF && NYQ) ? kMinBlocks - 1 : kMinBlocks;
    switch (h.lw) {
        case 32: return launch_one<ST, 32, kStrip, kMBwide, UNI, NYQ, FF>(p, s, h.overlap);
        case 16: return launch_one<ST, 16, kStrip, kMBwide, UNI, NYQ, FF>(p, s, h.overlap);
        case 8: return launch_one<ST, 8, kStrip, kMB, UNI, NYQ, FF>(p, s, h.overlap);
        default: return launch_one<ST, 4, kStrip, kMB, UNI, NYQ, FF>(p, s, h.overlap);
    }
}

template <typename ST, bool UNI, bool NYQ>
static cudaError_t dispatch(const Handle &h, const AccumParams &p, cudaStream_t s)
{
    return p.F2 ? dispatch_lw<ST, UNI, NYQ, true>(h, p, s) : dispatch_lw<ST, UNI, NYQ, false>(h, p, s);
}

// fast gridded path: A(n, w_j) = (1/Phi_j) sum_m g_m(n) exp(i w_j tau_m) over the grid points
cudaError_t launch_eval_grid(const Handle &h, const AccumParams &p, cudaStream_t s)
{
    const long long n_tasks = (long long)p.n_wtiles * p.n_chunks;
    const unsigned grid = (unsigned)((n_tasks + kWarpsPerBlock - 1) / kWarpsPerBlock);
    switch (h.lw) {
        case 32: return launch_kernel(rad_accum<float, 32, kStrip, kMinBlocks, false, false, false, true>, dim3(grid), dim3(kThreads), 0, s, h.overlap, p);
        case 16: return launch_kernel(rad_accum<float, 16, kStrip, kMinBlocks, false, false, false, true>, dim3(grid), dim3(kThreads), 0, s, h.overlap, p);
        case 8: return launch_kernel(rad_accum<float, 8, kStrip, kMinBlocks, false, false, false, true>, dim3(grid), dim3(kThreads), 0, s, h.overlap, p);
        default: return launch_kernel(rad_accum<float, 4, kStrip, kMinBlocks, false, false, false, true>, dim3(grid), dim3(kThreads), 0, s, h.overlap, p);
    }
}

template <typename ST, int DY>
static cudaError_t dispatch_dyadic(const Handle &h, const AccumParams &p, cudaStream_t s)
{
    const long long n_tasks = (long long)p.n_wtiles * p.n_chunks;
    const dim3 grid((unsigned)((n_tasks + kWarpsPerBlock - 1) / kWarpsPerBlock));
    switch (h.lw) {
        case 32: return launch_kernel(rad_accum<ST, 32, kStrip, kMinBlocks, false, false, false, false, DY>, grid, dim3(kThreads), 0, s, h.overlap, p);
        case 16: return launch_kernel(rad_accum<ST, 16, kStrip, kMinBlocks, false, false, false, false, DY>, grid, dim3(kThreads), 0, s, h.overlap, p);
        case 8: return launch_kernel(rad_accum<ST, 8, kStrip, kMinBlocks, false, false, false, false, DY>, grid, dim3(kThreads), 0, s, h.overlap, p);
        default: return launch_kernel(rad_accum<ST, 4, kStrip, kMinBlocks, false, false, false, false, DY>, grid, dim3(kThreads), 0, s, h.overlap, p);
    }
}

template <typename ST, bool UNI>
static cudaError_t dispatch_split(const Handle &h, const AccumParams &p, cudaStream_t s)
{
    const long long n_tasks = (long long)p.n_wtiles * p.n_chunks;
    const dim3 grid((unsigned)((n_tasks + kWarpsPerBlock - 1) / kWarpsPerBlock));
    switch (h.lw) {
        case 16: return launch_kernel(rad_accum<ST, 16, kStrip, kMinBlocks, UNI, false, false, false, 0, true>, grid, dim3(kThreads), 0, s, h.overlap, p);
        case 8: return launch_kernel(rad_accum<ST, 8, kStrip, kMinBlocks, UNI, false, false, false, 0, true>, grid, dim3(kThreads), 0, s, h.overlap, p);
        default: return launch_kernel(rad_accum<ST, 4, kStrip, kMinBlocks, UNI, false, false, false, 0, true>, grid, dim3(kThreads), 0, s, h.overlap, p);
    }
}

template <typename ST>
static cudaError_t dispatch_precise(const Handle &h, const AccumParams &p, cudaStream_t s)
{
    const long long n_tasks = (long long)p.n_wtiles * p.n_chunks;
    const dim3 grid((unsigned)((n_tasks + kWarpsPerBlock - 1) / kWarpsPerBlock));
    switch (h.lw) {
        case 32: return launch_kernel(rad_accum<ST, 32, kStrip, kMinBlocks, false, false, false, false, 0, false, true>, grid, dim3(kThreads), 0, s, h.overlap, p);
        case 16: return launch_kernel(rad_accum<ST, 16, kStrip, kMinBlocks, false, false, false, false, 0, false, true>, grid, dim3(kThreads), 0, s, h.overlap, p);
        case 8: return launch_kernel(rad_accum<ST, 8, kStrip, kMinBlocks, false, false, false, false, 0, false, true>, grid, dim3(kThreads), 0, s, h.overlap, p);
        default: return launch_kernel(rad_accum<ST, 4, kStrip, kMinBlocks, false, false, false, false, 0, false, true>, grid, dim3(kThreads), 0, s, h.overlap, p);
    }
}

cudaError_t launch_accumulate(const Handle &h, const AccumParams &p, bool state_f64,
                              cudaStream_t s, int *n_launches, const char **variant)
{
    *n_launches = 1;
    if (h.precise) {  // RAD_FLAG_PRECISE: every sincos by the fp32 polynomial (rad_create keeps the other variants off)
        *variant = "general+precise";
        return state_f64 ? dispatch_precise<double>(h, p, s) : dispatch_precise<float>(h, p, s);
    }
    if (p.psplit > 0) {  // few directions: lane groups split the particles (rad_create allows it on the plain sweeps only)
        *variant = h.uniform ? "uniform+split" : "general+split";
        if (h.uniform) return state_f64 ? dispatch_split<double, true>(h, p, s) : dispatch_split<float, true>(h, p, s);
        return state_f64 ? dispatch_split<double, false>(h, p, s) : dispatch_split<float, false>(h, p, s);
    }
    if (h.dyad_c > 0 && !h.uniform && p.nyq_lim == 0.0 && !p.F2) {
        *variant = "general+dyadic";
        if (h.dyad_c == 1) return state_f64 ? dispatch_dyadic<double, 1>(h, p, s) : dispatch_dyadic<float, 1>(h, p, s);
        return state_f64 ? dispatch_dyadic<double, 2>(h, p, s) : dispatch_dyadic<float, 2>(h, p, s);
    }
    if (h.uniform) {
        *variant = p.F2 ? "uniform+formfactor" : "uniform";
        return state_f64 ? dispatch<double, true, false>(h, p, s) : dispatch<float, true, false>(h, p, s);
    }
    if (p.nyq_lim > 0.0) {
        *variant = p.F2 ? "general+nyquist+formfactor" : "general+nyquist";
        return state_f64 ? dispatch<double, false, true>(h, p, s) : dispatch<float, false, true>(h, p, s);
    }
    *variant = p.F2 ? "general+formfactor" : "general";
    return state_f64 ? dispatch<double, false, false>(h, p, s) : dispatch<float, false, false>(h, p, s);
}

}  // namespace rad
