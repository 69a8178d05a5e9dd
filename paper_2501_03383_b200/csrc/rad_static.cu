// rad_static.cu -- rad_spectrum_static (include/rad.h): the detector as ONE call that allocates
// nothing.  For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
// loops, harnesses that forbid it): no handle, no tables, no workspace -- the caller passes the
// inputs and the output, and the fp64 amplitude accumulator, which the handle-based path keeps in
// cudaMalloc'ed memory (Handle::acc_d), lives in a file-scope __device__ array of fixed size.
//
// The kernel is a variant of the general-grid accumulate kernel (rad_kernels.cu) without anything
// that needs set-up tables: per (particle, direction) the retarded time tau = t - n.r/c, the Doppler
// factor and the transverse amplitude in fp64 (staged once per 512-particle chunk in shared memory),
// per update the phase f_j tau reduced to one turn in fp64 (two magic-number roundings), then the
// same fp32 MUFU sin/cos and fp32 partial sums, folded into the fp64 accumulator with red.f64 per
// chunk.  Self-contained: shares no code with the handle-based path.
#include <cuda_runtime.h>
#include <stdint.h>

#include <cmath>
#include <cstdio>
#include <mutex>

#include "rad.h"

namespace {

constexpr int kMaxBins = RAD_STATIC_MAX_BINS;  // n_dir * n_omega
constexpr int kThreads = 128;
constexpr int kChunk = 512;        // particles staged per block and work item
constexpr int kMaxGrid = 148 * 64;  // grid-stride loop beyond
constexpr int kMaxDevices = 64;
constexpr double kC = 299792458.0;                   // m/s
constexpr double kInvTwoPi = 0.15915494309189533577;  // turns per radian
constexpr double kMagic52 = 6755399441055744.0;       // 1.5 * 2^52: x + kMagic52 - kMagic52 = rint(x)
constexpr double kMagic20 = 1572864.0;                // 1.5 * 2^20: the low 32 mantissa bits of x + kMagic20 are x * 2^32
constexpr float kTwoPi = 6.283185307179586f;
constexpr float kUnitToRad = 1.4629180792671596e-09f;  // 2 pi / 2^32

// THE scratch: (Re A1, Im A1, Re A2, Im A2) per (direction, frequency), 2 MiB, held by every GPU that
// loads the library until the process exits.  In host code this name is a host-side stand-in, NOT a
// device address: the kernels get the address cudaGetSymbolAddress returns (scratch_for_current_device).
static __device__ __align__(256) double g_static_acc[(size_t)kMaxBins * 4];

struct StaticParams {
    const double *dirs;   // DEVICE [D][3]
    const double *omega;  // DEVICE [W]
    const void *st[10];   // DEVICE state arrays, [n_steps][stride]
    double *acc;          // device address of g_static_acc
    double dt, t0;
    long long first_step, n, stride, n_work;
    int D, W, chunks_per_step, nbp_log2;
};

template <typename ST>
__device__ __forceinline__ double ld(const void *p, long long k)
{
    return (double)__ldg(reinterpret_cast<const ST *>(p) + k);
}

template <typename ST>
__global__ void __launch_bounds__(kThreads) rad_accum_static(const StaticParams P)
{
    __shared__ double s_tau[kChunk];  // retarded time of the term, seconds
    __shared__ float2 s_a[kChunk];    // its real amplitude on the transverse basis (e1, e2)
    // thread layout: nbp = 2^nbp_log2 lanes along frequency (covering min(W, 128) bins), the remaining factor
    // G = 128 / nbp splits the particles of the chunk, so that detectors with few frequencies keep all lanes busy
    const int nbp = 1 << P.nbp_log2, G = kThreads >> P.nbp_log2;
    const int jb = threadIdx.x & (nbp - 1), g = threadIdx.x >> P.nbp_log2;
    for (long long work = blockIdx.x; work < P.n_work; work += gridDim.x) {
        // direction fastest: neighbouring blocks read the same particles (L2)
        const int dir = (int)(work % P.D);
        const long long cg = work / P.D;
        const long long step = cg / P.chunks_per_step;
        const long long c0 = (cg - step * P.chunks_per_step) * kChunk;
        const int cnt = (int)min((long long)kChunk, P.n - c0);
        // n normalised in fp64; e1 = normalise(z^ x n) (x^ x n if |n_z| > 0.9), e2 = n x e1 (rad.h)
        double nx = P.dirs[3 * dir], ny = P.dirs[3 * dir + 1], nz = P.dirs[3 * dir + 2];
        const double inn = 1.0 / sqrt(nx * nx + ny * ny + nz * nz);
        nx *= inn; ny *= inn; nz *= inn;
        double e1x, e1y, e1z;
        if (fabs(nz) > 0.9) { e1x = 0.0; e1y = -nz; e1z = ny; }
        else { e1x = -ny; e1y = nx; e1z = 0.0; }
        const double ie = 1.0 / sqrt(e1x * e1x + e1y * e1y + e1z * e1z);
        e1x *= ie; e1y *= ie; e1z *= ie;
        const double e2x = ny * e1z - nz * e1y, e2y = nz * e1x - nx * e1z, e2z = nx * e1y - ny * e1x;
        const double t = P.t0 + (double)(P.first_step + step) * P.dt;
        __syncthreads();  // the previous work item's records have been consumed
        for (int k = threadIdx.x; k < cnt; k += kThreads) {
            const long long i = step * P.stride + c0 + k;
            const double rx = ld<ST>(P.st[0], i), ry = ld<ST>(P.st[1], i), rz = ld<ST>(P.st[2], i);
            const double bx = ld<ST>(P.st[3], i), by = ld<ST>(P.st[4], i), bz = ld<ST>(P.st[5], i);
            const double ax = ld<ST>(P.st[6], i), ay = ld<ST>(P.st[7], i), az = ld<ST>(P.st[8], i);
            const double w = ld<ST>(P.st[9], i);
            // n x ((n - beta) x bd) = (n - beta)(n.bd) - bd (1 - n.beta) is _|_ n: on the transverse basis
            // a_i = -(e_i.beta)(n.bd) - (e_i.bd) d,  d = 1 - n.beta
            const double d = 1.0 - (nx * bx + ny * by + nz * bz);
            const double nb = nx * ax + ny * ay + nz * az;
            const double pre = -w * P.dt / (d * d);
            const double a1 = pre * ((e1x * bx + e1y * by + e1z * bz) * nb + (e1x * ax + e1y * ay + e1z * az) * d);
            const double a2 = pre * ((e2x * bx + e2y * by + e2z * bz) * nb + (e2x * ax + e2y * ay + e2z * az) * d);
            s_tau[k] = t - (nx * rx + ny * ry + nz * rz) / kC;
            s_a[k] = make_float2((float)a1, (float)a2);
        }
        __syncthreads();
        for (int j = jb; j < P.W; j += nbp) {
            const double f = __ldg(P.omega + j) * kInvTwoPi;  // turns per second
            float re1 = 0.0f, im1 = 0.0f, re2 = 0.0f, im2 = 0.0f;
            for (int k = g; k < cnt; k += G) {
                const double tau = s_tau[k];
                // f tau mod 1 in fp64: the integer part by the first magic rounding, the fraction exactly by the
                // fused multiply-add, then as a 32-bit fixed-point number u = frac * 2^32 (mod 2^32)
                const double r = fma(f, tau, kMagic52) - kMagic52;
                const double frac = fma(f, tau, -r);  // [-1/2, 1/2]
                const unsigned u = (unsigned)__double2loint(frac + kMagic20);
                // sin/cos argument 2 pi (1 + u / 2^32): the top 23 bits as the mantissa of v in [1, 2), the low 9 exact
                const float v = __uint_as_float(0x3f800000u | (u >> 9));
                const float lo = __uint_as_float(0x4b000000u | (u & 0x1ffu)) - 8388608.0f;
                float sn, cs;
                __sincosf(fmaf(v, kTwoPi, lo * kUnitToRad), &sn, &cs);
                const float2 a = s_a[k];
                re1 = fmaf(a.x, cs, re1); im1 = fmaf(a.x, sn, im1);
                re2 = fmaf(a.y, cs, re2); im2 = fmaf(a.y, sn, im2);
            }
            double *o = P.acc + ((size_t)dir * P.W + j) * 4;
            atomicAdd(o + 0, (double)re1); atomicAdd(o + 1, (double)im1);
            atomicAdd(o + 2, (double)re2); atomicAdd(o + 3, (double)im2);
        }
    }
}

// S = scale (|A1|^2 + |A2|^2)
__global__ void rad_spectrum_static_kernel(const double *__restrict__ acc, double *__restrict__ out, double scale, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double4 a = reinterpret_cast<const double4 *>(acc)[i];
    out[i] = scale * (a.x * a.x + a.y * a.y + a.z * a.z + a.w * a.w);
}

thread_local char g_error[256] = "";

rad_status fail(rad_status st, const char *msg, const char *detail = nullptr)
{
    snprintf(g_error, sizeof g_error, "%s%s%s", msg, detail ? ": " : "", detail ? detail : "");
    return st;
}

// Set-up, once per device, with that device current: the device address of g_static_acc.
std::mutex g_mutex;
double *g_acc_ptr[kMaxDevices] = {};

cudaError_t scratch_for_current_device(int device, double **out)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_acc_ptr[device]) {
        double *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_static_acc);
        if (e != cudaSuccess) return e;
        g_acc_ptr[device] = p;
    }
    *out = g_acc_ptr[device];
    return cudaSuccess;
}

double default_scale()  // SI e^2 / (16 pi^3 eps0 c), as rad_config.scale = 0
{
    const double pi = 3.14159265358979323846, e = 1.602176634e-19, eps0 = 8.8541878128e-12;
    return e * e / (16.0 * pi * pi * pi * eps0 * kC);
}

}  // namespace

extern "C" {

RAD_API rad_status rad_spectrum_static(int32_t n_dir, const double *dirs_device, int32_t n_omega,
                                       const double *omega_device, double dt, double t0, double scale,
                                       int32_t state_dtype, int64_t first_step_index, int32_t n_steps,
                                       int64_t n_particles, int64_t step_stride,
                                       const void *rx, const void *ry, const void *rz,
                                       const void *bx, const void *by, const void *bz,
                                       const void *bdx, const void *bdy, const void *bdz,
                                       const void *w, double *out_device, void *cuda_stream)
{
    if (n_dir < 1 || n_omega < 1 || !dirs_device || !omega_device || !out_device)
        return fail(RAD_ERR_INVALID_ARG, "n_dir, n_omega >= 1; dirs_device, omega_device, out_device non-NULL");
    if ((int64_t)n_dir * n_omega > kMaxBins) {
        char d[128];
        snprintf(d, sizeof d, "n_dir * n_omega = %lld exceeds RAD_STATIC_MAX_BINS = %d (the size of the static scratch)",
                 (long long)n_dir * n_omega, kMaxBins);
        return fail(RAD_ERR_UNSUPPORTED, "rad_spectrum_static", d);
    }
    if (!std::isfinite(dt) || dt <= 0.0 || !std::isfinite(t0) || !std::isfinite(scale) || scale < 0.0)
        return fail(RAD_ERR_INVALID_ARG, "dt must be finite and > 0; t0, scale finite; scale >= 0");
    if (state_dtype != RAD_F32 && state_dtype != RAD_F64)
        return fail(RAD_ERR_INVALID_ARG, "state_dtype must be RAD_F32 or RAD_F64");
    if (n_steps < 0 || n_particles < 0 || step_stride < n_particles)
        return fail(RAD_ERR_INVALID_ARG, "n_steps, n_particles >= 0; step_stride >= n_particles");
    const bool any = n_steps > 0 && n_particles > 0;
    if (any && (!rx || !ry || !rz || !bx || !by || !bz || !bdx || !bdy || !bdz || !w))
        return fail(RAD_ERR_INVALID_ARG, "NULL particle array");
    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) return fail(RAD_ERR_CUDA, "cudaGetDevice", cudaGetErrorString(e));
    if (device < 0 || device >= kMaxDevices) return fail(RAD_ERR_UNSUPPORTED, "device ordinal beyond 63");
    StaticParams P = {};
    e = scratch_for_current_device(device, &P.acc);
    if (e != cudaSuccess) return fail(RAD_ERR_CUDA, "cudaGetSymbolAddress(static scratch)", cudaGetErrorString(e));
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int bins = n_dir * n_omega;
    // the scratch keeps the previous call's amplitudes: clear what this call uses
    e = cudaMemsetAsync(P.acc, 0, (size_t)bins * 4 * sizeof(double), s);
    if (e != cudaSuccess) return fail(RAD_ERR_CUDA, "cudaMemsetAsync(static scratch)", cudaGetErrorString(e));
    if (any) {
        P.dirs = dirs_device; P.omega = omega_device;
        const void *st[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
        for (int i = 0; i < 10; ++i) P.st[i] = st[i];
        P.dt = dt; P.t0 = t0; P.first_step = first_step_index; P.n = n_particles; P.stride = step_stride;
        P.D = n_dir; P.W = n_omega;
        const int64_t cps = (n_particles + kChunk - 1) / kChunk;
        if (cps > INT32_MAX || cps * n_steps > ((int64_t)1 << 40) / n_dir)
            return fail(RAD_ERR_UNSUPPORTED, "rad_spectrum_static: more than 2^40 (chunk, direction) work items");
        P.chunks_per_step = (int)cps;
        P.n_work = cps * n_steps * n_dir;
        while ((1 << P.nbp_log2) < n_omega && (1 << P.nbp_log2) < kThreads) ++P.nbp_log2;
        const unsigned grid = (unsigned)(P.n_work < kMaxGrid ? P.n_work : kMaxGrid);
        if (state_dtype == RAD_F64) rad_accum_static<double><<<grid, kThreads, 0, s>>>(P);
        else rad_accum_static<float><<<grid, kThreads, 0, s>>>(P);
        e = cudaGetLastError();
        if (e != cudaSuccess) return fail(RAD_ERR_CUDA, "rad_accum_static launch", cudaGetErrorString(e));
    }
    rad_spectrum_static_kernel<<<(bins + 255) / 256, 256, 0, s>>>(P.acc, out_device, scale == 0.0 ? default_scale() : scale,
                                                                  bins);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(RAD_ERR_CUDA, "rad_spectrum_static_kernel launch", cudaGetErrorString(e));
    g_error[0] = 0;
    return RAD_OK;
}

RAD_API const char *rad_static_last_error(void) { return g_error; }

}  // extern "C"
