// rad_finalize.cu -- a4: |A|^2 and normalisation, amplitude export /
// import in Cartesian components, and the deterministic reduction of per-chunk partials.
// All fp64, one thread per (direction, frequency) bin; bandwidth-trivial (<= a few MB).
// Per-region handles: "row" = region * D + direction runs over R*D rows; the basis of a row is
// that of direction row mod D.
#include "rad_device.cuh"
#include "rad_internal.h"

namespace rad {

namespace {

// S[n][j] = scale * (|A1|^2 + |A2|^2); (e1, e2, n) is orthonormal and A . n = 0, so this
// equals scale * (|Ax|^2 + |Ay|^2 + |Az|^2).
__global__ void rad_spectrum_kernel(const double *__restrict__ acc, double *__restrict__ out,
                                    int D, int W, int w_pad, double scale)
{
    dev::pdl_trigger();
    dev::pdl_wait();  // A belongs to the accumulate kernels queued before
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= (long long)D * W) return;
    const int d = (int)(b / W), j = (int)(b - (long long)d * W);
    const double2 *a = reinterpret_cast<const double2 *>(acc + ((size_t)d * w_pad + j) * 4);
    const double2 a1 = a[0], a2 = a[1];
    out[b] = scale * (a1.x * a1.x + a1.y * a1.y + a2.x * a2.x + a2.y * a2.y);
}

// A_xyz = A1 e1 + A2 e2  ->  out[n][j][3][2]
__global__ void rad_amplitude_kernel(const double *__restrict__ acc, const DirRec *__restrict__ dirs,
                                     const double *__restrict__ basis, double *__restrict__ out,
                                     int rows, int D, int W, int w_pad)
{
    dev::pdl_trigger();
    dev::pdl_wait();  // A belongs to the accumulate kernels queued before
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= (long long)rows * W) return;
    const int d = (int)(b / W), j = (int)(b - (long long)d * W);
    const double2 *a = reinterpret_cast<const double2 *>(acc + ((size_t)d * w_pad + j) * 4);
    const double2 a1 = a[0], a2 = a[1];
    const double *e = basis + (size_t)(d % D) * 6;  // fp64 e1, e2
    double *o = out + (size_t)b * 6;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        o[2 * c + 0] = a1.x * e[c] + a2.x * e[3 + c];
        o[2 * c + 1] = a1.y * e[c] + a2.y * e[3 + c];
    }
}

// A1 += e1 . amp, A2 += e2 . amp
__global__ void rad_add_amplitude_kernel(double *__restrict__ acc, const double *__restrict__ basis,
                                         const double *__restrict__ amp, int rows, int D, int W, int w_pad)
{
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= (long long)rows * W) return;
    const int d = (int)(b / W), j = (int)(b - (long long)d * W);
    const double *e = basis + (size_t)(d % D) * 6;
    const double *in = amp + (size_t)b * 6;
    double r1 = 0, i1 = 0, r2 = 0, i2 = 0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        r1 += e[c] * in[2 * c];
        i1 += e[c] * in[2 * c + 1];
        r2 += e[3 + c] * in[2 * c];
        i2 += e[3 + c] * in[2 * c + 1];
    }
    double *a = acc + ((size_t)d * w_pad + j) * 4;
    a[0] += r1; a[1] += i1; a[2] += r2; a[3] += i2;
}

// deterministic mode: acc[region][e] += sum over the region's chunks (fixed order) of
// partial[chunk][e]; cstart[r] = first chunk of region r (NULL: one region, all chunks)
__global__ void rad_reduce_partials_kernel(double *__restrict__ acc, const double *__restrict__ partial,
                                           long long n_elem, int n_chunks, int R,
                                           const int *__restrict__ cstart)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_elem * R) return;
    const int r = (int)(t / n_elem);
    const long long e = t - (long long)r * n_elem;
    const int c0 = cstart ? cstart[r] : 0, c1 = cstart ? cstart[r + 1] : n_chunks;
    double s = 0.0;
    for (int c = c0; c < c1; ++c) s += partial[(size_t)c * n_elem + e];
    acc[t] += s;
}

// S_total[n][j] = scale * |sum_r A_r|^2 (amplitudes of the regions add up, then the modulus)
__global__ void rad_spectrum_total_kernel(const double *__restrict__ acc, double *__restrict__ out,
                                          int R, int D, int W, int w_pad, double scale)
{
    dev::pdl_trigger();
    dev::pdl_wait();  // A belongs to the accumulate kernels queued before
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= (long long)D * W) return;
    const int d = (int)(b / W), j = (int)(b - (long long)d * W);
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    for (int r = 0; r < R; ++r) {
        const double2 *a = reinterpret_cast<const double2 *>(acc + (((size_t)r * D + d) * w_pad + j) * 4);
        const double2 a1 = a[0], a2 = a[1];
        s0 += a1.x; s1 += a1.y; s2 += a2.x; s3 += a2.y;
    }
    out[b] = scale * (s0 * s0 + s1 * s1 + s2 * s2 + s3 * s3);
}

// A += amp4 (compact [rows][W][4] -> padded [rows][w_pad][4])
__global__ void rad_import_accumulator_kernel(double *__restrict__ acc, const double *__restrict__ amp4,
                                              int rows, int W, int w_pad)
{
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= (long long)rows * W) return;
    const int d = (int)(b / W), j = (int)(b - (long long)d * W);
    const double2 *in = reinterpret_cast<const double2 *>(amp4 + (size_t)b * 4);
    double2 *a = reinterpret_cast<double2 *>(acc + ((size_t)d * w_pad + j) * 4);
    const double2 i0 = in[0], i1 = in[1];
    double2 a0 = a[0], a1 = a[1];
    a0.x += i0.x; a0.y += i0.y; a1.x += i1.x; a1.y += i1.y;
    a[0] = a0; a[1] = a1;
}

inline unsigned blocks_for(long long n, int t) { return (unsigned)((n + t - 1) / t); }

}  // namespace

cudaError_t launch_spectrum(const Handle &h, double *out_dev, cudaStream_t s)
{
    const long long n = (long long)h.R * h.D * h.W;
    return launch_kernel(rad_spectrum_kernel, dim3(blocks_for(n, 256)), dim3(256), 0, s, h.overlap, h.acc_d, out_dev,
                         h.R * h.D, h.W, h.w_pad, h.scale);
}

cudaError_t launch_amplitude(const Handle &h, double *out_dev, cudaStream_t s)
{
    const long long n = (long long)h.R * h.D * h.W;
    return launch_kernel(rad_amplitude_kernel, dim3(blocks_for(n, 256)), dim3(256), 0, s, h.overlap, h.acc_d,
                         h.dirs_d, h.basis_d, out_dev, h.R * h.D, h.D, h.W, h.w_pad);
}

cudaError_t launch_add_amplitude(const Handle &h, const double *amp_dev, cudaStream_t s)
{
    const long long n = (long long)h.R * h.D * h.W;
    rad_add_amplitude_kernel<<<blocks_for(n, 256), 256, 0, s>>>(h.acc_d, h.basis_d, amp_dev, h.R * h.D,
                                                                h.D, h.W, h.w_pad);
    return cudaGetLastError();
}

cudaError_t launch_reduce_partials(const Handle &h, const double *partial, int n_chunks,
                                   const int *region_chunk_start, cudaStream_t s)
{
    const long long n = (long long)h.D * h.w_pad * 4;
    const int R = region_chunk_start ? h.R : 1;
    rad_reduce_partials_kernel<<<blocks_for(n * R, 256), 256, 0, s>>>(h.acc_d, partial, n, n_chunks, R,
                                                                     region_chunk_start);
    return cudaGetLastError();
}

// |A|^2 of a compact amplitude buffer (rad_export_accumulator layout: row pitch W, not w_pad)
cudaError_t launch_spectrum_of(const Handle &h, const double *amp4_dev, double *out_dev, cudaStream_t s)
{
    const long long n = (long long)h.R * h.D * h.W;
    return launch_kernel(rad_spectrum_kernel, dim3(blocks_for(n, 256)), dim3(256), 0, s, h.overlap, amp4_dev, out_dev,
                         h.R * h.D, h.W, h.W, h.scale);
}

cudaError_t launch_import_accumulator(const Handle &h, const double *amp4_dev, cudaStream_t s)
{
    const long long n = (long long)h.R * h.D * h.W;
    rad_import_accumulator_kernel<<<blocks_for(n, 256), 256, 0, s>>>(h.acc_d, amp4_dev, h.R * h.D, h.W, h.w_pad);
    return cudaGetLastError();
}

cudaError_t launch_spectrum_total(const Handle &h, double *out_dev, cudaStream_t s)
{
    const long long n = (long long)h.D * h.W;
    return launch_kernel(rad_spectrum_total_kernel, dim3(blocks_for(n, 256)), dim3(256), 0, s, h.overlap, h.acc_d,
                         out_dev, h.R, h.D, h.W, h.w_pad, h.scale);
}

}  // namespace rad
