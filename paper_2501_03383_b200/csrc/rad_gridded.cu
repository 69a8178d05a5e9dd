// rad_gridded.cu -- the approximate fast path, RAD_FLAG_FAST_GRIDDED (include/rad.h; SURVEY.md
// section 8(f) NEXT-4; the direct sum's cost "scal[es] with the number of
// particles, frequencies, and directions").
//
// For one direction n the detector is a non-uniform Fourier sum over retarded times,
//     A(n, w_j) = sum_terms a exp(i w_j tau),    tau = t - n.r/c,   a = (A1, A2) real,
// a type-3 non-uniform transform.  Its first half is done here, per (particle, direction), at a
// cost that does not depend on the number of frequencies: the term is SPREAD onto a uniform grid
// in tau (spacing h = pi / (2 w_max): twofold oversampling) with the compactly supported
// "exponential of semicircle" kernel
//     phi(x) = exp(beta (sqrt(1 - x^2) - 1)),  |x| < 1,   x = (m - u) / (WD / 2),  u = (tau - tau_0(n)) / h,
// WD grid points wide (beta = 2.30 WD, the published choice for twofold oversampling: error about
// 10^-(WD-1)).  The second half -- sum over the grid points with exact phases, divided by the
// kernel's transform Phi(w_j) -- is the GRID variant of rad_accum (rad_kernels.cu), run by
// rad_spectrum / rad_amplitude.
//
// Mapping: thread <-> particle (coalesced SoA loads, state read once), loop over the directions of
// the launch; per (particle, direction): the fp64 phase and Doppler factor and the fp32 transverse
// amplitude of the direct path (stage_record), WD + 2 kernel values (FFMA, MUFU.SQRT, FFMA,
// MUFU.EX2 each), and WD / 2 16-byte vector reductions red.global.add.v4.f32 (SASS
// REDG.E.ADD.F32x4) of {a1 phi_m, a2 phi_m, a1 phi_m+1, a2 phi_m+1} into one of the two fp32 delta grids.
// A fold kernel adds the delta grid into the fp64 master grid after every call: the low-frequency
// (coherent) part of the signal makes all deposits of a grid point equal in sign, and the rounding
// of thousands of fp32 additions onto such a point shows up in the dark high-frequency bins
// (measured on config 2 with a fold every 32 calls: 2.8e-3 on the worst bin above 1e-6 of the peak).
#include "rad_device.cuh"
#include "rad_internal.h"

namespace rad {

namespace {

using namespace dev;

constexpr int kSpreadThreads = 256;

__device__ __forceinline__ void red_add_v4(float2 *addr, float a, float b, float c, float d)
{
    asm volatile("red.global.v4.f32.add [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d)
                 : "memory");
}

template <typename ST, int WD>
__global__ void __launch_bounds__(kSpreadThreads) rad_spread(const AccumParams P)
{
    static_assert(WD % 2 == 0 && WD >= 4 && WD <= 12, "kernel width");
    constexpr float kInvHalf = 2.0f / WD;
    pdl_trigger();
    const long long k = (long long)blockIdx.x * kSpreadThreads + threadIdx.x;
    const bool valid = k < P.n_particles;
    const Particle p = load_particle<ST, true>(P, valid ? k : 0, valid, false);
    pdl_wait();  // the delta grids belong to earlier work (a fold zeroes them) until here
    if (!valid) return;
    unsigned long long lost = 0;
    for (int dir = P.dir0; dir < P.dir1; ++dir) {
        const DirRec &dr = P.dirs[dir];  // the same record for all lanes: one broadcast load each
        // phase and amplitude exactly as the direct path stages them (rad_device.cuh stage_record)
        const double s32 = P.ts32 - fma(dr.kx, p.rx, fma(dr.ky, p.ry, dr.kz * p.rz));
        const double d64 = 1.0 - fma(dr.nx, p.bx, fma(dr.ny, p.by, dr.nz * p.bz));
        const float d = to_f32(d64);
        const float g = fmaf(dr.nfx, p.bdx, fmaf(dr.nfy, p.bdy, dr.nfz * p.bdz));
        const float e1b = fmaf(dr.e1x, p.bfx, fmaf(dr.e1y, p.bfy, dr.e1z * p.bfz));
        const float e2b = fmaf(dr.e2x, p.bfx, fmaf(dr.e2y, p.bfy, dr.e2z * p.bfz));
        const float e1d = fmaf(dr.e1x, p.bdx, fmaf(dr.e1y, p.bdy, dr.e1z * p.bdz));
        const float e2d = fmaf(dr.e2x, p.bdx, fmaf(dr.e2y, p.bdy, dr.e2z * p.bdz));
        const float inv = 1.0f / d;
        const float pre = -p.wdt * inv * inv;
        const float a1 = pre * fmaf(e1b, g, e1d * d), a2 = pre * fmaf(e2b, g, e2d * d);
        // grid coordinate u (fp64); the support |m - u| < WD/2 holds the WD points m_first ... m_first + WD - 1
        const double u = fma(s32, P.g_ihs, -__ldg(P.g_s0 + dir));  // tau / h - (index of grid point 0)
        const long long m_first = (long long)floor(u - 0.5 * WD) + 1;
        if (m_first < 1 || m_first + WD >= P.g_M) {  // outside the box / window given at rad_create
            ++lost;
            continue;
        }
        const float x0 = to_f32((double)m_first - u) * kInvHalf;  // x of point m_first, in (-1, -1 + 2/WD]
        float phi[WD];
#pragma unroll
        for (int i = 0; i < WD; ++i) {
            const float x = fmaf((float)i, kInvHalf, x0);
            const float t = fmaf(-x, x, 1.0f);
            // correctly rounded square root: beta multiplies its error (sqrt.approx's 2^-22 would put a
            // 5e-6 floor under the gridding error); the spreading is bound by the reductions, not by this
            const float sq = __fsqrt_rn(fmaxf(t, 0.0f));
            float e;
            asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(P.g_beta2 * (sq - 1.0f)));
            phi[i] = t > 0.0f ? e : 0.0f;
        }
        // WD / 2 16-byte reductions, never a half-empty one: a 16-byte chunk holds two consecutive grid points,
        // and there are TWO deposit grids per direction, one whose chunks start at even points and one whose
        // chunks start at odd points (stored one point to the left); the term goes to the grid whose chunk
        // boundaries coincide with its first point.  (The kernel is bound by the rate at which L2 takes these
        // reductions: a single even-aligned grid needs WD/2 + 1 chunks for every second term, measured 5.67 ms
        // per config-2 step with 4.5 chunks per term on average, 6.31 ms with 5.)
        const int odd = (int)(m_first & 1);
        float2 *row = P.g_delta + ((size_t)dir * 2 + odd) * P.g_M + (m_first - odd);
#pragma unroll
        for (int i = 0; i < WD; i += 2) red_add_v4(row + i, a1 * phi[i], a2 * phi[i], a1 * phi[i + 1], a2 * phi[i + 1]);
    }
    if (lost) atomicAdd(P.g_oob, lost);
}

// master += even-aligned deposits + odd-aligned deposits (stored one point to the left); both := 0
// (fp32 partial sums never grow beyond one call)
__global__ void rad_grid_fold_kernel(double2 *__restrict__ master, float2 *__restrict__ delta, int M, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const long long dir = i / M;
    const int m = (int)(i - dir * M);
    float2 *ev = delta + (size_t)dir * 2 * M, *od = ev + M;
    float2 dl = ev[m];
    const bool he = dl.x != 0.0f || dl.y != 0.0f;
    bool ho = false;
    if (m > 0) {
        const float2 q = od[m - 1];
        ho = q.x != 0.0f || q.y != 0.0f;
        dl.x += q.x;
        dl.y += q.y;
    }
    if (he || ho) {
        double2 mm = master[i];
        mm.x += (double)dl.x;
        mm.y += (double)dl.y;
        master[i] = mm;
        if (he) ev[m] = make_float2(0.0f, 0.0f);
        if (ho) od[m - 1] = make_float2(0.0f, 0.0f);
    }
}

template <typename ST>
cudaError_t dispatch_spread(const Handle &h, const AccumParams &p, cudaStream_t s)
{
    const unsigned grid = (unsigned)((p.n_particles + kSpreadThreads - 1) / kSpreadThreads);
    switch (h.g_w) {
        case 4: return launch_kernel(rad_spread<ST, 4>, dim3(grid), dim3(kSpreadThreads), 0, s, h.overlap, p);
        case 6: return launch_kernel(rad_spread<ST, 6>, dim3(grid), dim3(kSpreadThreads), 0, s, h.overlap, p);
        case 8: return launch_kernel(rad_spread<ST, 8>, dim3(grid), dim3(kSpreadThreads), 0, s, h.overlap, p);
        case 10: return launch_kernel(rad_spread<ST, 10>, dim3(grid), dim3(kSpreadThreads), 0, s, h.overlap, p);
        default: return launch_kernel(rad_spread<ST, 12>, dim3(grid), dim3(kSpreadThreads), 0, s, h.overlap, p);
    }
}

}  // namespace

cudaError_t launch_spread(const Handle &h, const AccumParams &p, bool state_f64, cudaStream_t s)
{
    return state_f64 ? dispatch_spread<double>(h, p, s) : dispatch_spread<float>(h, p, s);
}

cudaError_t launch_grid_fold(const Handle &h, cudaStream_t s)
{
    const long long n = (long long)h.D * h.g_M;
    rad_grid_fold_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(h.g_master_d, h.g_delta_d, h.g_M, n);
    return cudaGetLastError();
}

}  // namespace rad
