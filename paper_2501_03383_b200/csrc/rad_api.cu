// rad_api.cu -- host runtime and the extern "C" boundary declared in include/rad.h.
// a0 (set-up at rad_create): normalise n, transverse basis, frequency
// tables (integer + fractional part in units of f_unit), tile-shape choice, zeroed A.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <new>

#include "rad_internal.h"

using namespace rad;

struct rad_handle {
    Handle h;
};

namespace {

thread_local std::string g_create_error;

const double kPi = 3.14159265358979323846;

double default_scale()
{
    const double e = 1.602176634e-19, eps0 = 8.8541878128e-12;
    return e * e / (16.0 * kPi * kPi * kPi * eps0 * kC);
}

rad_status fail(Handle *h, rad_status st, const std::string &msg)
{
    if (h) h->err = msg; else g_create_error = msg;
    return st;
}

rad_status cuda_fail(Handle *h, cudaError_t e, const char *what)
{
    if (h) h->broken = true;
    return fail(h, RAD_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define RAD_CUDA(h, call)                                         \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail((h), e_, #call);  \
    } while (0)

void free_all(Handle &h)
{
    cudaFree(h.dirs_d); cudaFree(h.basis_d); cudaFree(h.F_d); cudaFree(h.Ff_d); cudaFree(h.fl_d);
    cudaFree(h.acc_d); cudaFree(h.partial_d); cudaFree(h.stage_d[0]); cudaFree(h.stage_d[1]);
    cudaFree(h.out_d);
    for (int i = 0; i < 2; ++i) {
        if (h.copied[i]) cudaEventDestroy(h.copied[i]);
        if (h.consumed[i]) cudaEventDestroy(h.consumed[i]);
    }
    if (h.copy_stream) cudaStreamDestroy(h.copy_stream);
}

// Tile shape: lw lanes along frequency x 8 bins per lane, 32/lw directions per warp.
// Pick the shape wasting the fewest padded bins / padded directions; ties -> wider lw.
void choose_tile(Handle &h)
{
    double best = -1.0;
    for (int lw = 32; lw >= 4; lw >>= 1) {
        const int tile = lw * h.strip, dpw = 32 / lw;
        const int w_pad = (h.W + tile - 1) / tile * tile;
        const int d_pad = (h.D + dpw - 1) / dpw * dpw;
        const double eff = ((double)h.W / w_pad) * ((double)h.D / d_pad);
        if (eff > best + 1e-9) { best = eff; h.lw = lw; }
    }
    const int tile = h.lw * h.strip, dpw = 32 / h.lw;
    h.w_pad = (h.W + tile - 1) / tile * tile;
    h.n_ftiles = h.w_pad / tile;
    h.n_wtiles = ((h.D + dpw - 1) / dpw) * h.n_ftiles;
}

// Particles per block: enough blocks for >= ~8 waves of (SMs x resident blocks) so that the
// tail of the dynamically scheduled grid is small, fp32 partial sums span <= 4096 particles
// (rounding), and the fold (a3) stays ~1 % of the sweep.
int choose_chunk(const Handle &h, long long n)
{
    const long long gx = (h.n_wtiles + kWarpsPerBlock - 1) / kWarpsPerBlock;
    const long long want_blocks = 8LL * h.sm_count * kMinBlocks;
    long long n_chunks = (want_blocks + gx - 1) / gx;
    long long chunk = (n + n_chunks - 1) / n_chunks;
    chunk = (chunk + kBatch - 1) / kBatch * kBatch;
    if (chunk < 256) chunk = 256;
    if (chunk > 4096) chunk = 4096;
    // small inputs: prefer filling the SMs over amortising the fold
    while (chunk > kBatch && gx * ((n + chunk - 1) / chunk) < (long long)h.sm_count * kMinBlocks) chunk /= 2;
    chunk = (chunk + kBatch - 1) / kBatch * kBatch;
    return (int)chunk;
}

rad_status ensure_out(Handle &h, size_t bytes)
{
    if (h.out_bytes >= bytes) return RAD_OK;
    RAD_CUDA(&h, cudaDeviceSynchronize());
    cudaFree(h.out_d);
    h.out_d = nullptr; h.out_bytes = 0;
    if (cudaMalloc(&h.out_d, bytes) != cudaSuccess) {
        cudaGetLastError();
        return fail(&h, RAD_ERR_ALLOC, "cudaMalloc(result scratch) failed");
    }
    h.out_bytes = bytes;
    return RAD_OK;
}

rad_status check_handle(rad_handle *hh)
{
    if (!hh) return RAD_ERR_INVALID_ARG;
    if (hh->h.broken) return fail(&hh->h, RAD_ERR_STATE, "handle unusable after CUDA error: " + hh->h.err);
    RAD_CUDA(&hh->h, cudaSetDevice(hh->h.device));
    return RAD_OK;
}

rad_status accumulate_device(Handle &h, int64_t step, int64_t n, const void *const st[10], cudaStream_t s)
{
    AccumParams p{};
    for (int i = 0; i < 10; ++i) p.st[i] = st[i];
    p.n_particles = n;
    p.chunk = choose_chunk(h, n);
    if (const char *e = getenv("RAD_CHUNK")) {  // tuning/debug override (particles per block)
        const int c = atoi(e);
        if (c >= kBatch) p.chunk = c / kBatch * kBatch;
    }
    p.n_dir = h.D; p.n_omega = h.W; p.w_pad = h.w_pad;
    p.n_ftiles = h.n_ftiles; p.n_wtiles = h.n_wtiles;
    p.dirs = h.dirs_d; p.F = h.F_d; p.Ff = h.Ff_d; p.fl = h.fl_d;
    p.ts32 = (h.t0 + (double)step * h.dt) * h.f_unit * kTwo32;
    p.dt = (float)h.dt;
    p.acc = h.acc_d;
    p.partial = nullptr;
    p.rot_G = h.rot_G; p.rot_Gf = h.rot_Gf; p.rot_gl = h.rot_gl;
    int n_chunks = (int)((n + p.chunk - 1) / p.chunk);
    int stream_grid = 0;
    if (h.stream_nb) {  // few bins: persistent particle-streaming kernel, one partial slot per block
        const int tile = stream_tile_particles(h.state_f64);
        const long long n_tiles = (n + tile - 1) / tile;
        stream_grid = (int)std::min<long long>(n_tiles, (long long)stream_blocks_per_sm(h.stream_nb) * h.sm_count);
        for (int j = 0; j < 16; ++j) { p.sF[j] = h.sF[j]; p.sFf[j] = h.sFf[j]; p.sfl[j] = h.sfl[j]; }
        n_chunks = stream_grid;
    }
    if (h.deterministic) {
        const size_t need = (size_t)n_chunks * h.D * h.w_pad * 4 * sizeof(double);
        if (need > h.partial_bytes) {
            RAD_CUDA(&h, cudaDeviceSynchronize());
            cudaFree(h.partial_d);
            h.partial_d = nullptr; h.partial_bytes = 0;
            if (cudaMalloc(&h.partial_d, need) != cudaSuccess) {
                cudaGetLastError();
                return fail(&h, RAD_ERR_ALLOC, "cudaMalloc(deterministic workspace) failed");
            }
            h.partial_bytes = need;
        }
        p.partial = h.partial_d;
        if (h.stream_nb) RAD_CUDA(&h, cudaMemsetAsync(h.partial_d, 0, need, s));  // padded bins stay 0
    }
    if (h.stream_nb) {
        RAD_CUDA(&h, launch_accumulate_stream(h, p, h.state_f64, stream_grid, s));
        h.variant = "stream";
        h.launches += 1;
    } else {
        int nl = 0;
        RAD_CUDA(&h, launch_accumulate(h, p, h.state_f64, s, &nl, &h.variant));
        h.launches += nl;
    }
    if (h.deterministic) {
        RAD_CUDA(&h, launch_reduce_partials(h, h.partial_d, n_chunks, s));
        h.launches += 1;
    }
    return RAD_OK;
}

}  // namespace

extern "C" {

rad_status rad_create(const rad_config *cfg, rad_handle **out)
{
    if (out) *out = nullptr;
    if (!cfg || !out) return fail(nullptr, RAD_ERR_INVALID_ARG, "cfg/out is NULL");
    if (cfg->struct_size != sizeof(rad_config))
        return fail(nullptr, RAD_ERR_INVALID_ARG, "rad_config.struct_size mismatch (ABI version)");
    if (cfg->n_dir < 1 || cfg->n_omega < 1 || !cfg->dirs || !cfg->omega)
        return fail(nullptr, RAD_ERR_INVALID_ARG, "n_dir/n_omega must be >= 1 and dirs/omega non-NULL");
    if (!(cfg->dt > 0.0) || !std::isfinite(cfg->dt) || !std::isfinite(cfg->t0) ||
        !std::isfinite(cfg->scale) || cfg->scale < 0.0)
        return fail(nullptr, RAD_ERR_INVALID_ARG, "dt must be finite and > 0; t0, scale finite; scale >= 0");
    if (cfg->state_dtype != RAD_F32 && cfg->state_dtype != RAD_F64)
        return fail(nullptr, RAD_ERR_INVALID_ARG, "state_dtype must be RAD_F32 or RAD_F64");
    if (cfg->flags & ~(RAD_FLAG_DETERMINISTIC | RAD_FLAG_FORCE_GENERAL))
        return fail(nullptr, RAD_ERR_INVALID_ARG, "unknown flag bits");
    for (int j = 0; j < cfg->n_omega; ++j) {
        const double w = cfg->omega[j];
        if (!std::isfinite(w) || !(w > 0.0) || (j > 0 && !(w > cfg->omega[j - 1])))
            return fail(nullptr, RAD_ERR_INVALID_ARG, "omega must be finite, > 0 and strictly increasing");
    }
    rad_handle *hh = new (std::nothrow) rad_handle();
    if (!hh) return fail(nullptr, RAD_ERR_ALLOC, "out of host memory");
    Handle &h = hh->h;
    h.device = cfg->device; h.D = cfg->n_dir; h.W = cfg->n_omega;
    h.dt = cfg->dt; h.t0 = cfg->t0;
    h.scale = cfg->scale == 0.0 ? default_scale() : cfg->scale;
    h.state_f64 = cfg->state_dtype == RAD_F64;
    h.deterministic = (cfg->flags & RAD_FLAG_DETERMINISTIC) != 0;

    // directions: normalise in fp64 (Q8), build e1, e2 with e1 x e2 = n
    h.dirs_h.resize((size_t)h.D * 3);
    std::vector<DirRec> recs(h.D);
    std::vector<double> basis((size_t)h.D * 6);
    h.omega_h.assign(cfg->omega, cfg->omega + h.W);
    const double f_max = h.omega_h.back() / (2.0 * kPi);
    h.f_unit = f_max / 4294967040.0;  // F_j <= 2^32 - 256
    const double kscale = h.f_unit * kTwo32 / kC;
    for (int d = 0; d < h.D; ++d) {
        const double *v = cfg->dirs + 3 * d;
        const double nn = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        if (!std::isfinite(nn) || !(nn > 0.0)) {
            delete hh;
            return fail(nullptr, RAD_ERR_INVALID_ARG, "direction with zero or non-finite length");
        }
        const double n[3] = {v[0] / nn, v[1] / nn, v[2] / nn};
        double e1[3];
        if (std::fabs(n[2]) > 0.9) { e1[0] = 0.0; e1[1] = -n[2]; e1[2] = n[1]; }   // x^ x n
        else                       { e1[0] = -n[1]; e1[1] = n[0]; e1[2] = 0.0; }   // z^ x n
        const double l1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
        for (double &x : e1) x /= l1;
        const double e2[3] = {n[1] * e1[2] - n[2] * e1[1], n[2] * e1[0] - n[0] * e1[2],
                              n[0] * e1[1] - n[1] * e1[0]};                        // n x e1
        for (int c = 0; c < 3; ++c) {
            h.dirs_h[3 * d + c] = n[c];
            basis[6 * d + c] = e1[c];
            basis[6 * d + 3 + c] = e2[c];
        }
        DirRec &r = recs[d];
        r.kx = n[0] * kscale; r.ky = n[1] * kscale; r.kz = n[2] * kscale;
        r.nx = n[0]; r.ny = n[1]; r.nz = n[2];
        r.nfx = (float)n[0]; r.nfy = (float)n[1]; r.nfz = (float)n[2];
        r.e1x = (float)e1[0]; r.e1y = (float)e1[1]; r.e1z = (float)e1[2];
        r.e2x = (float)e2[0]; r.e2y = (float)e2[1]; r.e2z = (float)e2[2];
        r.pad[0] = r.pad[1] = r.pad[2] = 0.0f;
    }
    choose_tile(h);
    h.stream_nb = stream_shape(h.D, h.W, &h.stream_nd);
    // uniform grid?  w_j = w_0 + j dw to fp64 rounding -> rotation-recurrence kernel (a2')
    h.uniform = false;
    if (h.W >= 2 * h.strip && !(cfg->flags & RAD_FLAG_FORCE_GENERAL)) {
        const double dw = (h.omega_h.back() - h.omega_h.front()) / (h.W - 1);
        bool uni = true;
        for (int j = 0; j < h.W && uni; ++j)
            uni = std::fabs(h.omega_h[j] - (h.omega_h[0] + j * dw)) <= 4e-16 * h.omega_h.back() * (1 + j);
        if (uni) {
            const double step = dw / (2.0 * kPi) / h.f_unit * h.lw;  // rotator frequency, f_unit units
            const double G = std::nearbyint(step);
            h.uniform = true;
            h.rot_G = (uint32_t)G; h.rot_Gf = (float)G; h.rot_gl = (float)(step - G);
        }
    }
    std::vector<uint32_t> F(h.w_pad, 0u);
    std::vector<float> Ff(h.w_pad, 0.0f), fl(h.w_pad, 0.0f);
    for (int j = 0; j < h.W; ++j) {
        const double fu = h.omega_h[j] / (2.0 * kPi) / h.f_unit;
        const double Fi = std::nearbyint(fu);
        F[j] = (uint32_t)Fi;
        Ff[j] = (float)Fi;
        fl[j] = (float)(fu - Fi);
        if (j < 16) { h.sF[j] = F[j]; h.sFf[j] = Ff[j]; h.sfl[j] = fl[j]; }
    }

    cudaError_t e = cudaSetDevice(h.device);
    if (e != cudaSuccess) { delete hh; return cuda_fail(nullptr, e, "cudaSetDevice"); }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, h.device);
    if (e != cudaSuccess) { delete hh; return cuda_fail(nullptr, e, "cudaGetDeviceProperties"); }
    h.sm_count = prop.multiProcessorCount;
    const size_t acc_bytes = (size_t)h.D * h.w_pad * 4 * sizeof(double);
    bool ok = cudaMalloc(&h.dirs_d, sizeof(DirRec) * h.D) == cudaSuccess &&
              cudaMalloc(&h.basis_d, sizeof(double) * 6 * h.D) == cudaSuccess &&
              cudaMalloc(&h.F_d, sizeof(uint32_t) * h.w_pad) == cudaSuccess &&
              cudaMalloc(&h.Ff_d, sizeof(float) * h.w_pad) == cudaSuccess &&
              cudaMalloc(&h.fl_d, sizeof(float) * h.w_pad) == cudaSuccess &&
              cudaMalloc(&h.acc_d, acc_bytes) == cudaSuccess;
    if (!ok) {
        cudaGetLastError(); free_all(h); delete hh;
        return fail(nullptr, RAD_ERR_ALLOC, "cudaMalloc(tables/accumulator) failed");
    }
    ok = cudaMemcpy(h.dirs_d, recs.data(), sizeof(DirRec) * h.D, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(h.basis_d, basis.data(), sizeof(double) * 6 * h.D, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(h.F_d, F.data(), sizeof(uint32_t) * h.w_pad, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(h.Ff_d, Ff.data(), sizeof(float) * h.w_pad, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(h.fl_d, fl.data(), sizeof(float) * h.w_pad, cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemset(h.acc_d, 0, acc_bytes) == cudaSuccess &&
         cudaStreamCreateWithFlags(&h.copy_stream, cudaStreamNonBlocking) == cudaSuccess;
    for (int i = 0; ok && i < 2; ++i)
        ok = cudaEventCreateWithFlags(&h.copied[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&h.consumed[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {
        e = cudaGetLastError(); free_all(h); delete hh;
        return cuda_fail(nullptr, e, "table upload / stream set-up");
    }
    *out = hh;
    return RAD_OK;
}

rad_status rad_accumulate_step(rad_handle *hh, int64_t step_index, int64_t n_particles,
                               const void *rx, const void *ry, const void *rz, const void *bx,
                               const void *by, const void *bz, const void *bdx, const void *bdy,
                               const void *bdz, const void *w, void *cuda_stream)
{
    rad_status st = check_handle(hh);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    if (n_particles < 0) return fail(&h, RAD_ERR_INVALID_ARG, "n_particles < 0");
    if (n_particles == 0) return RAD_OK;
    const void *arr[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
    for (const void *p : arr)
        if (!p) return fail(&h, RAD_ERR_INVALID_ARG, "NULL state array");
    return accumulate_device(h, step_index, n_particles, arr, (cudaStream_t)cuda_stream);
}

rad_status rad_accumulate_step_host(rad_handle *hh, int64_t step_index, int64_t n_particles,
                                    const void *rx, const void *ry, const void *rz, const void *bx,
                                    const void *by, const void *bz, const void *bdx, const void *bdy,
                                    const void *bdz, const void *w, void *cuda_stream)
{
    rad_status st = check_handle(hh);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    if (n_particles < 0) return fail(&h, RAD_ERR_INVALID_ARG, "n_particles < 0");
    if (n_particles == 0) return RAD_OK;
    const void *arr[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
    for (const void *p : arr)
        if (!p) return fail(&h, RAD_ERR_INVALID_ARG, "NULL state array");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t esz = h.state_f64 ? 8 : 4;
    const size_t stride = ((size_t)n_particles * esz + 255) / 256 * 256;
    const int b = h.stage_next;
    h.stage_next ^= 1;
    if (h.stage_bytes[b] < stride * 10) {
        RAD_CUDA(&h, cudaDeviceSynchronize());
        cudaFree(h.stage_d[b]);
        h.stage_d[b] = nullptr; h.stage_bytes[b] = 0;
        if (cudaMalloc(&h.stage_d[b], stride * 10) != cudaSuccess) {
            cudaGetLastError();
            return fail(&h, RAD_ERR_ALLOC, "cudaMalloc(state staging) failed");
        }
        h.stage_bytes[b] = stride * 10;
        h.consumed_valid[b] = false;
    }
    // slot b may be overwritten only after the kernels that last read it are done
    if (h.consumed_valid[b]) RAD_CUDA(&h, cudaStreamWaitEvent(h.copy_stream, h.consumed[b], 0));
    const void *dev[10];
    for (int i = 0; i < 10; ++i) {
        char *dst = (char *)h.stage_d[b] + stride * i;
        RAD_CUDA(&h, cudaMemcpyAsync(dst, arr[i], (size_t)n_particles * esz, cudaMemcpyHostToDevice,
                                     h.copy_stream));
        dev[i] = dst;
    }
    RAD_CUDA(&h, cudaEventRecord(h.copied[b], h.copy_stream));
    RAD_CUDA(&h, cudaStreamWaitEvent(s, h.copied[b], 0));
    st = accumulate_device(h, step_index, n_particles, dev, s);
    if (st != RAD_OK) return st;
    RAD_CUDA(&h, cudaEventRecord(h.consumed[b], s));
    h.consumed_valid[b] = true;
    return RAD_OK;
}

static rad_status deliver(Handle &h, double *out, int out_on_device, size_t bytes, cudaStream_t s,
                          cudaError_t (*launch)(const Handle &, double *, cudaStream_t))
{
    if (!out) return fail(&h, RAD_ERR_INVALID_ARG, "out is NULL");
    if (out_on_device) {
        RAD_CUDA(&h, launch(h, out, s));
        h.launches += 1;
        return RAD_OK;
    }
    rad_status st = ensure_out(h, bytes);
    if (st != RAD_OK) return st;
    RAD_CUDA(&h, launch(h, h.out_d, s));
    h.launches += 1;
    RAD_CUDA(&h, cudaMemcpyAsync(out, h.out_d, bytes, cudaMemcpyDeviceToHost, s));
    RAD_CUDA(&h, cudaStreamSynchronize(s));
    return RAD_OK;
}

rad_status rad_spectrum(rad_handle *hh, double *out, int out_on_device, void *cuda_stream)
{
    rad_status st = check_handle(hh);
    if (st != RAD_OK) return st;
    return deliver(hh->h, out, out_on_device, (size_t)hh->h.D * hh->h.W * sizeof(double),
                   (cudaStream_t)cuda_stream, launch_spectrum);
}

rad_status rad_amplitude(rad_handle *hh, double *out, int out_on_device, void *cuda_stream)
{
    rad_status st = check_handle(hh);
    if (st != RAD_OK) return st;
    return deliver(hh->h, out, out_on_device, (size_t)hh->h.D * hh->h.W * 6 * sizeof(double),
                   (cudaStream_t)cuda_stream, launch_amplitude);
}

rad_status rad_add_amplitude(rad_handle *hh, const double *amp_device, void *cuda_stream)
{
    rad_status st = check_handle(hh);
    if (st != RAD_OK) return st;
    if (!amp_device) return fail(&hh->h, RAD_ERR_INVALID_ARG, "amp_device is NULL");
    RAD_CUDA(&hh->h, launch_add_amplitude(hh->h, amp_device, (cudaStream_t)cuda_stream));
    hh->h.launches += 1;
    return RAD_OK;
}

rad_status rad_reset(rad_handle *hh, void *cuda_stream)
{
    rad_status st = check_handle(hh);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    RAD_CUDA(&h, cudaMemsetAsync(h.acc_d, 0, (size_t)h.D * h.w_pad * 4 * sizeof(double),
                                 (cudaStream_t)cuda_stream));
    return RAD_OK;
}

void rad_destroy(rad_handle *hh)
{
    if (!hh) return;
    if (cudaSetDevice(hh->h.device) == cudaSuccess) {
        cudaDeviceSynchronize();
        free_all(hh->h);
    }
    cudaGetLastError();
    delete hh;
}

int64_t rad_launch_count(const rad_handle *hh) { return hh ? hh->h.launches : 0; }

const char *rad_kernel_variant(const rad_handle *hh) { return hh ? hh->h.variant : "none"; }

const char *rad_status_string(rad_status s)
{
    switch (s) {
        case RAD_OK: return "RAD_OK";
        case RAD_ERR_INVALID_ARG: return "RAD_ERR_INVALID_ARG";
        case RAD_ERR_ALLOC: return "RAD_ERR_ALLOC";
        case RAD_ERR_CUDA: return "RAD_ERR_CUDA";
        case RAD_ERR_STATE: return "RAD_ERR_STATE";
        case RAD_ERR_UNSUPPORTED: return "RAD_ERR_UNSUPPORTED";
    }
    return "RAD_ERR_UNKNOWN";
}

const char *rad_last_error(const rad_handle *hh) { return hh ? hh->h.err.c_str() : g_create_error.c_str(); }

const char *rad_version(void) { return "rad-b200 0.1 (sm_100a)"; }

}  // extern "C"
