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
    cudaFree(h.Fg_d); cudaFree(h.Ffg_d); cudaFree(h.flg_d);
    cudaFree(h.g_s0_d); cudaFree(h.g_corr_d); cudaFree(h.g_delta_d); cudaFree(h.g_master_d); cudaFree(h.g_oob_d);
    cudaFree(h.out_d); cudaFree(h.chunks_d); cudaFree(h.reg_cstart_d); cudaFree(h.omega_d); cudaFree(h.F2_d);

    if (h.chunks_h) cudaFreeHost(h.chunks_h);
    if (h.reg_cstart_h) cudaFreeHost(h.reg_cstart_h);
    if (h.reg_uploaded) cudaEventDestroy(h.reg_uploaded);
    for (int i = 0; i < 2; ++i) {
        if (h.copied[i]) cudaEventDestroy(h.copied[i]);
        if (h.consumed[i]) cudaEventDestroy(h.consumed[i]);
    }
    if (h.copy_stream) cudaStreamDestroy(h.copy_stream);
}

// Tile shape: lw lanes along frequency x 8 bins per lane, 32/lw directions per warp.  A detector with
// fewer directions than a warp holds (D <= dpw / 2) does not leave the other lane groups idle: 2^ps groups
// share one direction and split the particles of a batch between them ("particle split", rad_kernels.cu).
// -> fraction of the warp's lanes x bins that are real work; *ps = log2 of the groups per direction.
double tile_efficiency(const Handle &h, int lw, int *ps, bool allow_split)
{
    const int tile = lw * h.strip, dpw = 32 / lw;
    const int w_pad = (h.W + tile - 1) / tile * tile;
    *ps = 0;
    while (allow_split && h.D <= (dpw >> (*ps + 1))) ++*ps;   // D * 2^(ps+1) <= dpw, without shifting D
    const int d_pad = *ps > 0 ? dpw : (h.D + dpw - 1) / dpw * dpw;
    return ((double)h.W / w_pad) * ((double)(h.D << *ps) / d_pad);
}

void set_tile(Handle &h, int lw, int ps)
{
    const int tile = lw * h.strip, dpw = 32 / lw;
    h.lw = lw; h.psplit = ps;
    h.w_pad = (h.W + tile - 1) / tile * tile;
    h.n_ftiles = h.w_pad / tile;
    h.n_wtiles = (((h.D << ps) + dpw - 1) / dpw) * h.n_ftiles;
}

// Pick the shape wasting the fewest padded bins / padded directions; ties -> wider lw.
void choose_tile(Handle &h, bool allow_split)
{
    double best = -1.0;
    int best_lw = 32, best_ps = 0;
    for (int lw = 32; lw >= 4; lw >>= 1) {
        int ps;
        const double eff = tile_efficiency(h, lw, &ps, allow_split);
        if (eff > best + 1e-9) { best = eff; best_lw = lw; best_ps = ps; }
    }
    set_tile(h, best_lw, best_ps);
}

// Particles per block: enough blocks for >= ~8 waves of (SMs x resident blocks) so that the
// tail of the dynamically scheduled grid is small, fp32 partial sums span <= 4096 particles
// (rounding), and the fold (a3) stays ~1 % of the sweep.
int choose_chunk(const Handle &h, long long n)
{
    // a warp task = (warp tile, chunk); a block runs 4 tasks; cap blocks are resident at once
    const long long cap = (long long)h.sm_count * kMinBlocks;
    auto blocks_at = [&](long long chunk) {
        return (h.n_wtiles * ((n + chunk - 1) / chunk) + kWarpsPerBlock - 1) / kWarpsPerBlock;
    };
    if (blocks_at(256) >= 4 * cap) {  // large input: ~4 waves of full-length chunks; the tapered
                                      // chunk table (build_tapered_table) evens out the tail
        const long long want_tasks = 4 * cap * kWarpsPerBlock;
        const long long n_chunks = (want_tasks + h.n_wtiles - 1) / h.n_wtiles;
        long long chunk = (n + n_chunks - 1) / n_chunks;
        chunk = (chunk + kBatch - 1) / kBatch * kBatch;
        return (int)std::min<long long>(std::max<long long>(chunk, 256), 4096);
    }
    // small input (a few waves at most).  Cost model in particle-equivalents of one warp task:
    //   waves * (chunk + 32)   sweep of one chunk plus ~32 particles' worth of constants, stage latency, ramp;
    //   + n_chunks             the fold: every bin address receives one fp64 atomic per chunk, and atomics on
    //                          one address serialise in L2 (~110 cycles each, measured on config 0: with
    //                          1024 chunks of 32 particles 77 % of the kernel was the fold) -- about one
    //                          particle-equivalent per chunk, whatever the number of bins.
    long long best = 4096, best_cost = -1;
    for (long long chunk = kBatch; chunk <= 4096; chunk += kBatch) {
        const long long waves = (blocks_at(chunk) + cap - 1) / cap;
        const long long cost = waves * (chunk + 32) + (n + chunk - 1) / chunk;
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = chunk; }
        if (chunk >= n) break;
    }
    return (int)best;
}

// Pinned + device storage for `need` chunk records (and the R+1 region chunk starts); waits
// until the previous upload has left the pinned copy.
rad_status ensure_chunk_capacity(Handle &h, size_t need)
{
    if (h.reg_uploaded) RAD_CUDA(&h, cudaEventSynchronize(h.reg_uploaded));  // pinned copy is free again
    else RAD_CUDA(&h, cudaEventCreateWithFlags(&h.reg_uploaded, cudaEventDisableTiming));
    if (need > h.reg_cap || !h.reg_cstart_h) {
        RAD_CUDA(&h, cudaDeviceSynchronize());
        cudaFree(h.chunks_d); h.chunks_d = nullptr;
        if (h.chunks_h) cudaFreeHost(h.chunks_h);
        h.chunks_h = nullptr; h.reg_cap = 0;
        // whatever table was cached lived in these buffers: forget it, so that a failed
        // allocation below can never be followed by a cache hit on freed memory
        h.reg_chunk = 0; h.reg_offsets.clear(); h.tap_n = -1; h.tap_chunk = 0; h.reg_n_chunks = 0;
        const size_t cap = std::max<size_t>(need + need / 4, 64);
        bool ok = cudaMallocHost(&h.chunks_h, cap * sizeof(ChunkRec)) == cudaSuccess &&
                  cudaMalloc(&h.chunks_d, cap * sizeof(ChunkRec)) == cudaSuccess;
        if (ok && !h.reg_cstart_h)
            ok = cudaMallocHost(&h.reg_cstart_h, (h.R + 1) * sizeof(int)) == cudaSuccess &&
                 cudaMalloc(&h.reg_cstart_d, (h.R + 1) * sizeof(int)) == cudaSuccess;
        if (!ok) {
            cudaGetLastError();
            return fail(&h, RAD_ERR_ALLOC, "allocation of the chunk table failed");
        }
        h.reg_cap = cap;
    }
    return RAD_OK;
}

// Per-region calls: (re)build the chunk table for these offsets (shifted so that the first
// region starts at particle `base` of the device arrays) and upload it on stream s.  Chunks
// never straddle a region; a region of n_r particles is cut into ceil(n_r / chunk) chunks
// of equal length (rounded up to whole 32-particle batches).
rad_status build_chunk_table(Handle &h, const int64_t *off, long long base, int chunk, cudaStream_t s,
                             int n_steps = 1, long long stride = 0)
{
    bool same = h.reg_chunk == chunk && (int)h.reg_offsets.size() == h.R + 1 && h.reg_steps == n_steps &&
                h.reg_stride == stride;
    for (int r = 0; same && r <= h.R; ++r) same = h.reg_offsets[r] == off[r] - base;
    if (same) return RAD_OK;
    size_t need = 0;
    for (int r = 0; r < h.R; ++r) need += (size_t)((off[r + 1] - off[r] + chunk - 1) / chunk);
    need *= (size_t)n_steps;
    if (need > (size_t)INT32_MAX) return fail(&h, RAD_ERR_INVALID_ARG, "too many particle chunks");
    rad_status st_cap = ensure_chunk_capacity(h, need);
    if (st_cap != RAD_OK) return st_cap;
    int n = 0;
    for (int t = 0; t < n_steps; ++t)      // step-major (the region chunk starts serve single-step calls only)
        for (int r = 0; r < h.R; ++r) {
            if (t == 0) h.reg_cstart_h[r] = n;
            const long long n_r = off[r + 1] - off[r], k0 = off[r] - base + (long long)t * stride;
            if (n_r == 0) continue;
            const long long pieces = (n_r + chunk - 1) / chunk;
            long long len = (n_r + pieces - 1) / pieces;
            len = (len + kBatch - 1) / kBatch * kBatch;
            for (long long k = 0; k < n_r; k += len)
                h.chunks_h[n++] = ChunkRec{k0 + k, (int)std::min(len, n_r - k), r, t, 0};
        }
    h.reg_cstart_h[h.R] = n_steps == 1 ? n : 0;
    h.reg_n_chunks = n;
    h.reg_chunk = chunk;
    h.reg_steps = n_steps;
    h.reg_stride = stride;
    h.reg_offsets.resize(h.R + 1);
    for (int r = 0; r <= h.R; ++r) h.reg_offsets[r] = off[r] - base;
    if (n > 0)
        RAD_CUDA(&h, cudaMemcpyAsync(h.chunks_d, h.chunks_h, (size_t)n * sizeof(ChunkRec),
                                     cudaMemcpyHostToDevice, s));
    RAD_CUDA(&h, cudaMemcpyAsync(h.reg_cstart_d, h.reg_cstart_h, (h.R + 1) * sizeof(int),
                                 cudaMemcpyHostToDevice, s));
    RAD_CUDA(&h, cudaEventRecord(h.reg_uploaded, s));
    return RAD_OK;
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

// Makes the handle's device current for the duration of an entry point and restores the
// caller's device afterwards (a call must not change the calling thread's current device).
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t enter(int device)
    {
        cudaError_t e = cudaGetDevice(&prev);
        if (e != cudaSuccess) return e;
        if (prev == device) return cudaSuccess;
        e = cudaSetDevice(device);
        switched = e == cudaSuccess;
        return e;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

rad_status check_handle(rad_handle *hh, DeviceGuard &g)
{
    if (!hh) return RAD_ERR_INVALID_ARG;
    if (hh->h.broken) return fail(&hh->h, RAD_ERR_STATE, "handle unusable after CUDA error: " + hh->h.err);
    RAD_CUDA(&hh->h, g.enter(hh->h.device));
    return RAD_OK;
}

// Multi-step calls: chunk table over (step, particle chunk), all folding into region 0.  Cached per
// (n_steps, n, stride, chunk): a replay loop that calls with the same shape again uploads nothing and
// never waits for the previous upload (that wait serialised host and device: the table of call i+1 could
// only be written once the copy of call i, queued behind kernel i-1, had left the pinned buffer).
rad_status build_step_table(Handle &h, int n_steps, long long n, long long stride, int chunk, cudaStream_t s)
{
    if (h.reg_chunk == -2 && h.stp_steps == n_steps && h.stp_n == n && h.stp_stride == stride && h.stp_chunk == chunk)
        return RAD_OK;
    // (An entry spanning several steps of a small particle range -- so that an fp32 partial covers a full
    // chunk even when a step has fewer particles than that -- was measured: either form of the extra loop
    // level costs the single-step kernel 1.7 - 2.5 % (register pressure at the 128-register cap), for a case
    // that only arises below ~256 particles per step.  Not built.)
    const size_t per_step = (size_t)((n + chunk - 1) / chunk);
    const size_t need = per_step * (size_t)n_steps;
    if (need > (size_t)INT32_MAX) return fail(&h, RAD_ERR_INVALID_ARG, "too many particle chunks");
    rad_status st_cap = ensure_chunk_capacity(h, need);
    if (st_cap != RAD_OK) return st_cap;
    h.reg_chunk = 0; h.reg_offsets.clear(); h.tap_n = -1;  // the other cached tables (same buffers) are gone
    int m = 0;
    for (int t = 0; t < n_steps; ++t)
        for (long long k = 0; k < n; k += chunk)
            h.chunks_h[m++] = ChunkRec{(long long)t * stride + k, (int)std::min<long long>(chunk, n - k), 0, t, 0};
    h.reg_n_chunks = m;
    RAD_CUDA(&h, cudaMemcpyAsync(h.chunks_d, h.chunks_h, (size_t)m * sizeof(ChunkRec), cudaMemcpyHostToDevice, s));
    RAD_CUDA(&h, cudaEventRecord(h.reg_uploaded, s));
    h.reg_chunk = -2;  // marks "step table on the device"
    h.stp_steps = n_steps; h.stp_n = n; h.stp_stride = stride; h.stp_chunk = chunk;
    return RAD_OK;
}

// Plain single-step calls on large inputs: tapered chunk table ("guided" schedule).  The grid is
// ~8 waves of equal blocks; the last wave ends ragged while SMs idle.  Chunks keep the nominal
// length until ~2 waves of work are left, then each takes 1/taper of what remains (down to 128
// particles), so the blocks scheduled last are short and the tail of the grid is even.
// Cached per (n, chunk): no upload in the steady state.
rad_status build_tapered_table(Handle &h, long long n, int chunk, cudaStream_t s)
{
    if (h.tap_n == n && h.tap_chunk == chunk && h.reg_chunk == -1) return RAD_OK;
    const long long gx = (h.n_wtiles + kWarpsPerBlock - 1) / kWarpsPerBlock;   // blocks per chunk
    const double chunks_per_wave = (double)h.sm_count * kMinBlocks / (double)gx;
    // taper factor 1-4 x chunks-per-wave and a floor of 64-256 particles measured within 0.4 % of
    // each other; frozen at 1 x and 128
    const long long tmin = 4 * kBatch;
    const double taper = std::max(2.0, chunks_per_wave);
    std::vector<ChunkRec> recs;
    long long k = 0;
    while (k < n) {
        long long len = std::min<long long>(chunk, (long long)((double)(n - k) / taper));
        len = std::max<long long>(len, tmin) / kBatch * kBatch;
        len = std::min(len, n - k);
        recs.push_back(ChunkRec{k, (int)len, 0, 0, 0});
        k += len;
    }
    rad_status st_cap = ensure_chunk_capacity(h, recs.size());
    if (st_cap != RAD_OK) return st_cap;
    std::copy(recs.begin(), recs.end(), h.chunks_h);
    h.reg_n_chunks = (int)recs.size();
    h.reg_chunk = -1; h.reg_offsets.clear();     // marks "tapered table on the device"
    h.tap_n = n; h.tap_chunk = chunk;
    RAD_CUDA(&h, cudaMemcpyAsync(h.chunks_d, h.chunks_h, recs.size() * sizeof(ChunkRec), cudaMemcpyHostToDevice, s));
    RAD_CUDA(&h, cudaEventRecord(h.reg_uploaded, s));
    return RAD_OK;
}

// ---- fast gridded path (rad.h RAD_FLAG_FAST_GRIDDED; kernels in rad_gridded.cu) ----
constexpr int kGridFoldEvery = 1;  // accumulate calls between folds of the fp32 delta grid into the fp64 master
                                   // (rad_gridded.cu: more than one costs accuracy on dark bins; a fold is ~2 % of a call)

void grid_params(const Handle &h, AccumParams &p)
{
    p.g_delta = h.g_delta_d; p.g_master = h.g_master_d; p.g_s0 = h.g_s0_d; p.g_corr = h.g_corr_d;
    p.g_hs = h.g_hs; p.g_ihs = 1.0 / h.g_hs; p.g_M = h.g_M; p.g_jdiff = h.g_jdiff;
    p.g_beta2 = (float)(h.g_beta * 1.4426950408889634);
    p.g_oob = h.g_oob_d;
}

rad_status grid_fold(Handle &h, cudaStream_t s)
{
    if (h.g_pending == 0) return RAD_OK;
    RAD_CUDA(&h, launch_grid_fold(h, s));
    h.launches += 1;
    h.g_pending = 0;
    return RAD_OK;
}

// spread one step's particles onto the grids of all directions
rad_status accumulate_gridded(Handle &h, int64_t step, int64_t n, const void *const st[10], cudaStream_t s)
{
    if (step < h.g_step_min || step > h.g_step_max)
        return fail(&h, RAD_ERR_INVALID_ARG, "step_index outside [fast_step_min, fast_step_max] given at rad_create");
    AccumParams p{};
    for (int i = 0; i < 10; ++i) p.st[i] = st[i];
    p.n_particles = n;
    p.n_dir = h.D; p.n_omega = h.W; p.w_pad = h.w_pad;
    p.dirs = h.dirs_d;
    p.ts32 = (h.t0 + (double)step * h.dt) * h.f_unit * kTwo32;
    p.dt = (float)h.dt;
    p.win_type = h.win_type;
    for (int c = 0; c < 3; ++c) { p.win_o[c] = h.win_o[c]; p.win_il[c] = h.win_il[c]; }
    grid_params(h, p);
    // direction groups whose two deposit grids stay L2 resident (96 of the 126 MB); the 40 B/particle are re-read per
    // group (measured on config 2: 24 ... 112 MB per group within 5 %, smaller groups lose to the extra launches)
    const int per = (int)std::max<long long>(1, (96LL << 20) / ((long long)h.g_M * 2 * (long long)sizeof(float2)));
    for (int d0 = 0; d0 < h.D; d0 += per) {
        p.dir0 = d0; p.dir1 = std::min(h.D, d0 + per);
        RAD_CUDA(&h, launch_spread(h, p, h.state_f64, s));
        h.launches += 1;
    }
    h.variant = "gridded";
    h.g_acc_valid = false;
    if (++h.g_pending >= kGridFoldEvery) return grid_fold(h, s);
    return RAD_OK;
}

// A(n, w_j) := (1/Phi_j) sum_m g_m(n) exp(i w_j tau_m) into the accumulator (rad_spectrum / rad_amplitude)
rad_status evaluate_gridded(Handle &h, cudaStream_t s);

// st: DEVICE arrays.  region_off == NULL: particles [0, n) of the one detector; else n_regions+1
// HOST offsets into arrays whose element 0 is particle `region_base` of the caller's numbering
// and n = particles spanned by the regions.
// n_steps > 1: step t of every array starts step_stride elements after step t-1.
rad_status accumulate_device(Handle &h, int64_t step, int64_t n, const void *const st[10], cudaStream_t s,
                             const int64_t *region_off = nullptr, long long region_base = 0,
                             int n_steps = 1, long long step_stride = 0)
{
    if (h.fast) {  // approximate fast path: one spreading pass per step
        const size_t esz = h.state_f64 ? 8 : 4;
        for (int t = 0; t < n_steps; ++t) {
            const void *sub[10];
            for (int i = 0; i < 10; ++i) sub[i] = (const char *)st[i] + (size_t)t * step_stride * esz;
            rad_status st_ = accumulate_gridded(h, step + t, n, sub, s);
            if (st_ != RAD_OK) return st_;
        }
        return RAD_OK;
    }
    if (n_steps > 1 && (h.stream_nb || h.deterministic)) {
        // few-bin streaming kernel / deterministic workspace: one launch per step
        const size_t esz = h.state_f64 ? 8 : 4;
        for (int t = 0; t < n_steps; ++t) {
            const void *sub[10];
            for (int i = 0; i < 10; ++i) sub[i] = (const char *)st[i] + (size_t)t * step_stride * esz;
            rad_status st_ = accumulate_device(h, step + t, n, sub, s, region_off, region_base);
            if (st_ != RAD_OK) return st_;
        }
        return RAD_OK;
    }
    AccumParams p{};
    for (int i = 0; i < 10; ++i) p.st[i] = st[i];
    p.n_particles = n;
    // per-region calls: every region rounds its own chunk count up -> leave room for that
    p.chunk = choose_chunk(h, (region_off ? n + (long long)h.R * 64 : n) * n_steps);
    p.n_dir = h.D; p.n_omega = h.W; p.w_pad = h.w_pad;
    p.n_ftiles = h.n_ftiles; p.n_wtiles = h.n_wtiles; p.psplit = h.psplit;
    p.dirs = h.dirs_d; p.F = h.F_d; p.Ff = h.Ff_d; p.fl = h.fl_d; p.F2 = h.F2_d;
    p.w_sqrt = h.ff_type == RAD_FF_INCOHERENT;
    p.ts32 = (h.t0 + (double)step * h.dt) * h.f_unit * kTwo32;
    p.dts32 = h.dt * h.f_unit * kTwo32;
    p.nyq_lim = h.nyq_lim; p.dt64 = h.dt; p.omega64 = h.omega_d;
    p.nyq_mode = h.nyq_mode; p.nyq_a = h.nyq_a; p.nyq_b = h.nyq_b;
    p.win_type = h.win_type;
    for (int c = 0; c < 3; ++c) { p.win_o[c] = h.win_o[c]; p.win_il[c] = h.win_il[c]; }
    p.dt = (float)h.dt;
    p.acc = h.acc_d;
    p.partial = nullptr;
    p.rot_G = h.rot_G; p.rot_Gf = h.rot_Gf; p.rot_gl = h.rot_gl;
    int n_chunks = (int)((n + p.chunk - 1) / p.chunk);
    if (region_off) {
        rad_status st_ = build_chunk_table(h, region_off, region_base, p.chunk, s, n_steps, step_stride);
        if (st_ != RAD_OK) return st_;
        n_chunks = h.reg_n_chunks;
        p.chunks = h.chunks_d;
        if (n_chunks == 0) return RAD_OK;
    } else if (n_steps > 1) {
        rad_status st_ = build_step_table(h, n_steps, n, step_stride, p.chunk, s);
        if (st_ != RAD_OK) return st_;
        n_chunks = h.reg_n_chunks;
        p.chunks = h.chunks_d;
    } else if (!h.stream_nb && !h.deterministic &&
               (long long)n_chunks * h.n_wtiles >= 4LL * h.sm_count * kMinBlocks * kWarpsPerBlock) {
        rad_status st_ = build_tapered_table(h, n, p.chunk, s);
        if (st_ != RAD_OK) return st_;
        n_chunks = h.reg_n_chunks;
        p.chunks = h.chunks_d;
    }
    p.n_chunks = n_chunks;
    int stream_grid = 0;
    if (h.stream_nb) {  // few bins: persistent particle-streaming kernel, one partial slot per block
        const int tile = stream_tile_particles(h.stream_nb, h.state_f64);
        const long long n_tiles = (n + tile - 1) / tile;
        stream_grid = (int)std::min<long long>(n_tiles, (long long)stream_blocks_per_sm(h.stream_nb) * h.sm_count);
        for (int j = 0; j < 16; ++j) { p.sF[j] = h.sF[j]; p.sFf[j] = h.sFf[j]; p.sfl[j] = h.sfl[j]; }
        p.sdir[0] = h.sdir[0]; p.sdir[1] = h.sdir[1];
        if (h.F2_d) {  // bin b = d * WB + j of the streaming kernel
            const int wb = h.stream_nb / h.stream_nd;
            for (int d = 0; d < h.stream_nd && d < h.D; ++d)
                for (int j = 0; j < wb && j < h.W; ++j) p.sF2[d * wb + j] = h.F2_h[(size_t)d * h.w_pad + j];
        }
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
        RAD_CUDA(&h, launch_reduce_partials(h, h.partial_d, n_chunks, region_off ? h.reg_cstart_d : nullptr, s));
        h.launches += 1;
    }
    return RAD_OK;
}

rad_status evaluate_gridded(Handle &h, cudaStream_t s)
{
    if (h.g_acc_valid) return RAD_OK;
    rad_status st = grid_fold(h, s);
    if (st != RAD_OK) return st;
    RAD_CUDA(&h, cudaMemsetAsync(h.acc_d, 0, (size_t)h.D * h.w_pad * 4 * sizeof(double), s));
    AccumParams p{};
    p.n_particles = h.g_M;          // the "particles" of this sweep are the grid points
    // Short chunks: consecutive grid points are consecutive in retarded time, so below the highest
    // frequencies the fp32 partial sum of a chunk is COHERENT (large) and the bin's amplitude is what
    // survives the cancellation between chunks -- the rounding of the partial sums must stay below that.
    // (Measured on configs 2 and 3a with 4096-point chunks: a floor of 5e-7 of the peak amplitude,
    // 8e-4 relative on bins at 1e-6 of the peak, whatever the kernel width; the error scales with the chunk.)
    p.chunk = 8 * kBatch;
    p.n_chunks = (h.g_M + p.chunk - 1) / p.chunk;
    p.n_dir = h.D; p.n_omega = h.W; p.w_pad = h.w_pad;
    p.n_ftiles = h.n_ftiles; p.n_wtiles = h.n_wtiles;
    p.dirs = h.dirs_d; p.F = h.Fg_d; p.Ff = h.Ffg_d; p.fl = h.flg_d;   // tables in units of one grid step
    p.acc = h.acc_d;
    grid_params(h, p);
    RAD_CUDA(&h, launch_eval_grid(h, p, s));
    h.launches += 1;
    h.g_acc_valid = true;
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
    if (cfg->flags & ~(RAD_FLAG_DETERMINISTIC | RAD_FLAG_FORCE_GENERAL | RAD_FLAG_OVERLAP_STEPS | RAD_FLAG_FAST_GRIDDED |
                       RAD_FLAG_PRECISE))
        return fail(nullptr, RAD_ERR_INVALID_ARG, "unknown flag bits");
    if (cfg->n_regions < 0) return fail(nullptr, RAD_ERR_INVALID_ARG, "n_regions must be >= 0");
    if (!std::isfinite(cfg->nyquist_factor) || cfg->nyquist_factor < 0.0)
        return fail(nullptr, RAD_ERR_INVALID_ARG, "nyquist_factor must be finite and >= 0");
    if (cfg->window_type < RAD_WINDOW_NONE || cfg->window_type > RAD_WINDOW_HAMMING)
        return fail(nullptr, RAD_ERR_INVALID_ARG, "unknown window_type");
    if (cfg->window_type != RAD_WINDOW_NONE)
        for (int c = 0; c < 3; ++c)
            if (!std::isfinite(cfg->window_origin[c]) || !std::isfinite(cfg->window_extent[c]))
                return fail(nullptr, RAD_ERR_INVALID_ARG, "window origin/extent must be finite");
    if (cfg->form_factor_type < RAD_FF_NONE || cfg->form_factor_type > RAD_FF_INCOHERENT || cfg->reserved0 != 0)
        return fail(nullptr, RAD_ERR_INVALID_ARG, "unknown form_factor_type (or reserved0 != 0)");
    if (cfg->form_factor_type != RAD_FF_NONE)
        for (int c = 0; c < 3; ++c)
            if (!std::isfinite(cfg->form_factor_size[c]) || cfg->form_factor_size[c] < 0.0)
                return fail(nullptr, RAD_ERR_INVALID_ARG, "form_factor_size must be finite and >= 0");
    for (int j = 0; j < cfg->n_omega; ++j) {
        const double w = cfg->omega[j];
        if (!std::isfinite(w) || !(w > 0.0) || (j > 0 && !(w > cfg->omega[j - 1])))
            return fail(nullptr, RAD_ERR_INVALID_ARG, "omega must be finite, > 0 and strictly increasing");
    }
    const bool fast = (cfg->flags & RAD_FLAG_FAST_GRIDDED) != 0;
    if (fast) {
        for (int c = 0; c < 3; ++c)
            if (!std::isfinite(cfg->fast_box_min[c]) || !std::isfinite(cfg->fast_box_max[c]) ||
                cfg->fast_box_max[c] < cfg->fast_box_min[c])
                return fail(nullptr, RAD_ERR_INVALID_ARG, "fast_box must be finite with min <= max");
        if (cfg->fast_step_max < cfg->fast_step_min)
            return fail(nullptr, RAD_ERR_INVALID_ARG, "fast_step_max < fast_step_min");
        if (!std::isfinite(cfg->fast_tolerance) || cfg->fast_tolerance < 0.0 || cfg->fast_tolerance >= 1.0)
            return fail(nullptr, RAD_ERR_INVALID_ARG, "fast_tolerance must be in [0, 1)");
        if (cfg->n_regions > 1 || cfg->nyquist_factor > 0.0 || cfg->form_factor_type != RAD_FF_NONE ||
            (cfg->flags & RAD_FLAG_DETERMINISTIC))
            return fail(nullptr, RAD_ERR_UNSUPPORTED,
                        "RAD_FLAG_FAST_GRIDDED: no regions, Nyquist limiter, form factor or deterministic mode");
    }
    const bool precise = (cfg->flags & RAD_FLAG_PRECISE) != 0;
    if (precise && (fast || cfg->nyquist_factor > 0.0 || cfg->form_factor_type == RAD_FF_GAUSSIAN ||
                    cfg->form_factor_type == RAD_FF_CIC))
        return fail(nullptr, RAD_ERR_UNSUPPORTED,
                    "RAD_FLAG_PRECISE: no Nyquist limiter, Gaussian / CIC form factor or RAD_FLAG_FAST_GRIDDED");
    rad_handle *hh = new (std::nothrow) rad_handle();
    if (!hh) return fail(nullptr, RAD_ERR_ALLOC, "out of host memory");
    Handle &h = hh->h;
    h.device = cfg->device; h.D = cfg->n_dir; h.W = cfg->n_omega;
    h.R = cfg->n_regions > 1 ? cfg->n_regions : 1;
    h.nyq_lim = kPi * cfg->nyquist_factor;
    h.win_type = cfg->window_type;
    for (int c = 0; c < 3; ++c) {
        h.win_o[c] = cfg->window_origin[c];
        h.win_il[c] = (h.win_type != RAD_WINDOW_NONE && cfg->window_extent[c] > 0.0) ? 1.0 / cfg->window_extent[c] : 0.0;
    }
    if (h.win_il[0] == 0.0 && h.win_il[1] == 0.0 && h.win_il[2] == 0.0) h.win_type = RAD_WINDOW_NONE;
    h.ff_type = cfg->form_factor_type;
    // F = 0 for every bin (RAD_FF_INCOHERENT): g = sqrt(w) is a per-particle weight -- no table, no per-update square
    // root, every kernel variant stays available
    h.ff_table = h.ff_type == RAD_FF_GAUSSIAN || h.ff_type == RAD_FF_CIC;
    h.dt = cfg->dt; h.t0 = cfg->t0;
    h.scale = cfg->scale == 0.0 ? default_scale() : cfg->scale;
    h.state_f64 = cfg->state_dtype == RAD_F64;
    h.deterministic = (cfg->flags & RAD_FLAG_DETERMINISTIC) != 0;
    h.overlap = (cfg->flags & RAD_FLAG_OVERLAP_STEPS) != 0;
    h.fast = fast;
    h.precise = precise;

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
    h.sdir[0] = recs[0]; h.sdir[1] = recs[h.D > 1 ? 1 : 0];
    // particle split: the plain general / uniform sweeps only (rad_kernels.cu SPLIT instantiations)
    choose_tile(h, h.nyq_lim == 0.0 && !h.ff_table && !h.fast && !h.precise);
    // Dyadic log grid (SURVEY.md section 8(f) NEXT-4 "dyadic log grids (integer bins/octave) allow
    // z(2w) = z(w)^2"): w_(j+b) = 2 w_j for an integer b = c * lw with lw in {4, 8, 16, 32}, c in {1, 2} ->
    // bins i and i + c of a thread's strip are an octave apart.  Among the admissible tile shapes the
    // widest one wins unless it pads more than choose_tile's own choice does.
    h.dyad_c = 0;
    if (!(cfg->flags & RAD_FLAG_FORCE_GENERAL) && h.nyq_lim == 0.0 && !h.fast && !h.ff_table && !h.precise && h.W >= 2) {
        int b = 0;
        for (int cand = 4; cand <= 64 && cand < h.W && b == 0; ++cand) {
            bool ok = true;
            for (int j = 0; j + cand < h.W && ok; ++j)
                ok = std::fabs(h.omega_h[j + cand] / (2.0 * h.omega_h[j]) - 1.0) <= 1e-12;
            if (ok) b = cand;
        }
        double best = -1.0;
        int best_lw = 0, best_c = 0, best_ps = 0;
        for (int lw = 32; lw >= 4; lw >>= 1)
            for (int c = 1; c <= 2; ++c) {
                if (b != c * lw) continue;
                int ps;
                const double eff = tile_efficiency(h, lw, &ps, false);   // the squaring chains run without the split
                if (eff > best + 1e-9) { best = eff; best_lw = lw; best_c = c; best_ps = ps; }
            }
        int ps0;
        if (best_lw && best >= 0.8 * tile_efficiency(h, h.lw, &ps0, true)) {
            // the squaring chains are worth ~1.3x: accept up to 20 % more padding than the free choice
            set_tile(h, best_lw, best_ps);
            h.dyad_c = best_c;
        }
    }
    // per-region detectors and the Nyquist limiter: bin-owner kernels only
    h.stream_nb = (h.R > 1 || h.nyq_lim > 0.0 || h.fast || h.precise) ? 0 : stream_shape(h.D, h.W, &h.stream_nd);
    // uniform grid?  w_j = w_0 + j dw to fp64 rounding -> rotation-recurrence kernel (a2')
    h.uniform = false;
    double uni_dw = 0.0;
    if (h.W >= 2 * h.strip && !(cfg->flags & RAD_FLAG_FORCE_GENERAL) && h.nyq_lim == 0.0 && !h.fast && !h.precise) {
        const double dw = (h.omega_h.back() - h.omega_h.front()) / (h.W - 1);
        bool uni = true;
        for (int j = 0; j < h.W && uni; ++j)
            uni = std::fabs(h.omega_h[j] - (h.omega_h[0] + j * dw)) <= 4e-16 * h.omega_h.back() * (1 + j);
        if (uni) {
            const double step = dw / (2.0 * kPi) / h.f_unit * h.lw;  // rotator frequency, f_unit units
            const double G = std::nearbyint(step);
            h.uniform = true;
            // step can exceed 2^32 (lw > W - 1): the integer phase only needs G mod 2^32 (exact,
            // F*T wraps mod one turn anyway); the fp32 copy multiplies the residual and stays unwrapped
            h.rot_G = (uint32_t)((uint64_t)G & 0xffffffffull); h.rot_Gf = (float)G; h.rot_gl = (float)(step - G);
            uni_dw = dw;
        }
    }
    // Nyquist limiter: closed-form guess of the cut-off bin on log-spaced / linear grids (checked against the
    // exact fp64 predicate on the device, rad_device.cuh nyquist_count); any other grid bisects
    h.nyq_mode = 0;
    if (h.nyq_lim > 0.0 && h.W >= 3) {
        const double w0 = h.omega_h.front(), q = h.omega_h[1] / w0, dw = h.omega_h[1] - w0;
        bool is_log = true, is_lin = true;
        for (int j = 1; j < h.W; ++j) {
            is_log = is_log && std::fabs(h.omega_h[j] / h.omega_h[j - 1] / q - 1.0) <= 1e-9;
            is_lin = is_lin && std::fabs((h.omega_h[j] - h.omega_h[j - 1]) / dw - 1.0) <= 1e-9;
        }
        if (is_log) {
            h.nyq_mode = 1; h.nyq_a = (float)(1.0 / std::log2(q)); h.nyq_b = (float)(h.nyq_lim / (h.dt * w0));
        } else if (is_lin) {
            h.nyq_mode = 2; h.nyq_a = (float)(h.nyq_lim / (h.dt * dw)); h.nyq_b = (float)(-w0 / dw);
        }
    }
    // Frequency tables.  Padded bins [W, w_pad) are never folded, but on a uniform grid a thread's
    // rotation chain is anchored at its MIDDLE bin, which may be a padded one while lower bins of
    // the strip are valid: there the tables continue the grid, w_j = w_0 + j dw (F mod 2^32 for the
    // integer phase, the fp32 copy unwrapped); on a general grid padded bins stay 0.
    std::vector<uint32_t> F(h.w_pad, 0u);
    std::vector<float> Ff(h.w_pad, 0.0f), fl(h.w_pad, 0.0f);
    for (int j = 0; j < (h.uniform ? h.w_pad : h.W); ++j) {
        const double om = j < h.W ? h.omega_h[j] : h.omega_h[0] + j * uni_dw;
        const double fu = om / (2.0 * kPi) / h.f_unit;
        const double Fi = std::nearbyint(fu);
        F[j] = (uint32_t)((uint64_t)Fi & 0xffffffffull);
        Ff[j] = (float)Fi;
        fl[j] = (float)(fu - Fi);
        if (j < 16 && j < h.W) { h.sF[j] = F[j]; h.sFf[j] = Ff[j]; h.sfl[j] = fl[j]; }
    }

    // macro-particle form factor (rad.h, reading FF1): F^2(n, w_j) per (direction, frequency), fp64 -> fp32
    if (h.ff_table) {
        h.F2_h.assign((size_t)h.D * h.w_pad, 0.0f);
        const double *sz = cfg->form_factor_size;
        for (int d = 0; d < h.D; ++d)
            for (int j = 0; j < h.W; ++j) {
                const double *n = &h.dirs_h[3 * d];
                const double om = h.omega_h[j];
                double Fv = 0.0;
                if (h.ff_type == RAD_FF_GAUSSIAN) {
                    double q = 0.0;
                    for (int c = 0; c < 3; ++c) { const double x = om * n[c] * sz[c] / kC; q += x * x; }
                    Fv = std::exp(-0.5 * q);
                } else if (h.ff_type == RAD_FF_CIC) {
                    Fv = 1.0;
                    for (int c = 0; c < 3; ++c) {
                        const double x = om * n[c] * sz[c] / (2.0 * kC);
                        const double sinc = x == 0.0 ? 1.0 : std::sin(x) / x;
                        Fv *= sinc * sinc;
                    }
                }
                h.F2_h[(size_t)d * h.w_pad + j] = (float)(Fv * Fv);
            }
    }

    // fast gridded path: kernel width from the tolerance, grid spacing h = pi / (2 w_max), per direction
    // the retarded-time interval that the box and the step window can reach, 1 / Phi(w_j)
    std::vector<double> g_s0;
    std::vector<double2> g_corr;
    std::vector<uint32_t> Fg;
    std::vector<float> Ffg, flg;
    if (h.fast) {
        const double eps = cfg->fast_tolerance > 0.0 ? cfg->fast_tolerance : 1e-6;
        int wd = (int)std::ceil(std::log10(1.0 / eps)) + 1;
        wd = std::min(12, std::max(4, wd + (wd & 1)));
        h.g_w = wd;
        h.g_beta = 2.30 * wd;
        const double h_tau = kPi / (2.0 * h.omega_h.back());
        h.g_hs = h_tau * h.f_unit * kTwo32;
        for (int c = 0; c < 3; ++c) { h.g_box_min[c] = cfg->fast_box_min[c]; h.g_box_max[c] = cfg->fast_box_max[c]; }
        h.g_step_min = cfg->fast_step_min; h.g_step_max = cfg->fast_step_max;
        const double t_lo = h.t0 + (double)h.g_step_min * h.dt, t_hi = h.t0 + (double)h.g_step_max * h.dt;
        g_s0.resize(h.D);
        long long M = 0;
        for (int d = 0; d < h.D; ++d) {
            double pmin = 0.0, pmax = 0.0;  // range of n.r over the box
            for (int c = 0; c < 3; ++c) {
                const double a = h.dirs_h[3 * d + c] * h.g_box_min[c], b = h.dirs_h[3 * d + c] * h.g_box_max[c];
                pmin += std::min(a, b); pmax += std::max(a, b);
            }
            const double tau_lo = t_lo - pmax / kC, tau_hi = t_hi - pmin / kC;
            g_s0[d] = std::floor(tau_lo / h_tau) - (0.5 * wd + 2.0);   // grid points sit at integer multiples of h
            M = std::max(M, (long long)std::ceil((tau_hi - tau_lo) / h_tau) + wd + 8);
        }
        M = (M + 63) / 64 * 64;
        if ((double)M * h.D * 32.0 > 64e9) {
            delete hh;
            return fail(nullptr, RAD_ERR_INVALID_ARG, "RAD_FLAG_FAST_GRIDDED: the box / window needs more than 64 GB of grid");
        }
        h.g_M = (int)M;
        // frequency tables of the evaluation sweep: f_j in units of 1 / (h 2^32) (<= 2^30: h f_max = 1/4)
        Fg.assign(h.w_pad, 0u); Ffg.assign(h.w_pad, 0.0f); flg.assign(h.w_pad, 0.0f);
        for (int j = 0; j < h.W; ++j) {
            const double fu = h.omega_h[j] / (2.0 * kPi) * h_tau * kTwo32;
            const double Fi = std::nearbyint(fu);
            Fg[j] = (uint32_t)Fi; Ffg[j] = (float)Fi; flg[j] = (float)(fu - Fi);
        }
        // Phi(w) = (wd/2) * integral_{-1}^{1} phi(x) cos(xi x) dx, xi = w h wd / 2; with x = sin(theta) the
        // integrand exp(beta (cos(theta) - 1)) cos(xi sin(theta)) cos(theta) is smooth: trapezoid rule
        g_corr.assign(h.w_pad, make_double2(0.0, 0.0));
        // bins of whole frequency tiles with w h >= 2.5e-3 are evaluated from first differences of the grid
        // (rad_kernels.cu, GRID staging): first such bin, rounded up to a tile boundary
        {
            const int tile = h.lw * h.strip;
            int j_first = h.W;
            for (int j = 0; j < h.W; ++j)
                if (h.omega_h[j] * h_tau >= 2.5e-3) { j_first = j; break; }
            h.g_jdiff = (j_first + tile - 1) / tile * tile;
        }
        const int nq = 4096;
        for (int j = 0; j < h.W; ++j) {
            const double xi = h.omega_h[j] * h_tau * 0.5 * wd;
            double acc = 0.0;
            for (int q = 0; q <= nq; ++q) {
                const double th = -0.5 * kPi + kPi * q / nq;
                const double f = std::exp(h.g_beta * (std::cos(th) - 1.0)) * std::cos(xi * std::sin(th)) * std::cos(th);
                acc += (q == 0 || q == nq) ? 0.5 * f : f;
            }
            const double inv_phi = 1.0 / (0.5 * wd * acc * (kPi / nq));
            // the evaluation sums first differences of the grid: divide by 1 - exp(i w h) =
            // 2 sin^2(theta/2) - i sin(theta), theta = w h (no cancellation at small theta)
            if (j >= h.g_jdiff) {
                const double th = h.omega_h[j] * h_tau, sh = std::sin(0.5 * th);
                const double re = 2.0 * sh * sh, im = -std::sin(th), n2 = re * re + im * im;
                g_corr[j] = make_double2(inv_phi * re / n2, -inv_phi * im / n2);
            } else {
                g_corr[j] = make_double2(inv_phi, 0.0);
            }
            // phase_sincos_grid centres the turn on 0 (frac - 1/2): every term carries exp(-i pi) = -1
            g_corr[j].x = -g_corr[j].x;
            g_corr[j].y = -g_corr[j].y;
        }
    }

    cudaError_t e = cudaSetDevice(h.device);
    if (e != cudaSuccess) { delete hh; return cuda_fail(nullptr, e, "cudaSetDevice"); }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, h.device);
    if (e != cudaSuccess) { delete hh; return cuda_fail(nullptr, e, "cudaGetDeviceProperties"); }
    h.sm_count = prop.multiProcessorCount;
    const size_t acc_bytes = (size_t)h.R * h.D * h.w_pad * 4 * sizeof(double);
    bool ok = cudaMalloc(&h.dirs_d, sizeof(DirRec) * h.D) == cudaSuccess &&
              cudaMalloc(&h.basis_d, sizeof(double) * 6 * h.D) == cudaSuccess &&
              cudaMalloc(&h.F_d, sizeof(uint32_t) * h.w_pad) == cudaSuccess &&
              cudaMalloc(&h.Ff_d, sizeof(float) * h.w_pad) == cudaSuccess &&
              cudaMalloc(&h.fl_d, sizeof(float) * h.w_pad) == cudaSuccess &&
              cudaMalloc(&h.acc_d, acc_bytes) == cudaSuccess &&
              (h.nyq_lim == 0.0 || cudaMalloc(&h.omega_d, sizeof(double) * h.W) == cudaSuccess) &&
              (h.F2_h.empty() || cudaMalloc(&h.F2_d, sizeof(float) * h.F2_h.size()) == cudaSuccess) &&
              (!h.fast || (cudaMalloc(&h.g_s0_d, sizeof(double) * h.D) == cudaSuccess &&
                           cudaMalloc(&h.g_corr_d, sizeof(double2) * h.w_pad) == cudaSuccess &&
                           cudaMalloc(&h.Fg_d, sizeof(uint32_t) * h.w_pad) == cudaSuccess &&
                           cudaMalloc(&h.Ffg_d, sizeof(float) * h.w_pad) == cudaSuccess &&
                           cudaMalloc(&h.flg_d, sizeof(float) * h.w_pad) == cudaSuccess &&
                           cudaMalloc(&h.g_delta_d, sizeof(float2) * 2 * (size_t)h.D * h.g_M) == cudaSuccess &&
                           cudaMalloc(&h.g_master_d, sizeof(double2) * (size_t)h.D * h.g_M) == cudaSuccess &&
                           cudaMalloc(&h.g_oob_d, sizeof(unsigned long long)) == cudaSuccess));
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
         (!h.fast || (cudaMemcpy(h.g_s0_d, g_s0.data(), sizeof(double) * h.D, cudaMemcpyHostToDevice) == cudaSuccess &&
                      cudaMemcpy(h.g_corr_d, g_corr.data(), sizeof(double2) * h.w_pad, cudaMemcpyHostToDevice) == cudaSuccess &&
                      cudaMemcpy(h.Fg_d, Fg.data(), sizeof(uint32_t) * h.w_pad, cudaMemcpyHostToDevice) == cudaSuccess &&
                      cudaMemcpy(h.Ffg_d, Ffg.data(), sizeof(float) * h.w_pad, cudaMemcpyHostToDevice) == cudaSuccess &&
                      cudaMemcpy(h.flg_d, flg.data(), sizeof(float) * h.w_pad, cudaMemcpyHostToDevice) == cudaSuccess &&
                      cudaMemset(h.g_delta_d, 0, sizeof(float2) * 2 * (size_t)h.D * h.g_M) == cudaSuccess &&
                      cudaMemset(h.g_master_d, 0, sizeof(double2) * (size_t)h.D * h.g_M) == cudaSuccess &&
                      cudaMemset(h.g_oob_d, 0, sizeof(unsigned long long)) == cudaSuccess)) &&
         (!h.F2_d || cudaMemcpy(h.F2_d, h.F2_h.data(), sizeof(float) * h.F2_h.size(), cudaMemcpyHostToDevice) == cudaSuccess) &&
         (!h.omega_d || cudaMemcpy(h.omega_d, h.omega_h.data(), sizeof(double) * h.W, cudaMemcpyHostToDevice) == cudaSuccess) &&
         cudaStreamCreateWithFlags(&h.copy_stream, cudaStreamNonBlocking) == cudaSuccess;
    for (int i = 0; ok && i < 2; ++i)
        ok = cudaEventCreateWithFlags(&h.copied[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&h.consumed[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {
        e = cudaGetLastError(); free_all(h); delete hh;
        return cuda_fail(nullptr, e, "table upload / stream set-up");
    }
    h.g_acc_valid = h.fast;  // an empty grid evaluates to the zeroed accumulator
    *out = hh;
    return RAD_OK;
}

rad_status rad_accumulate_step(rad_handle *hh, int64_t step_index, int64_t n_particles,
                               const void *rx, const void *ry, const void *rz, const void *bx,
                               const void *by, const void *bz, const void *bdx, const void *bdy,
                               const void *bdz, const void *w, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    if (h.R > 1) return fail(&h, RAD_ERR_INVALID_ARG, "per-region handle: use rad_accumulate_step_regions");
    if (n_particles < 0) return fail(&h, RAD_ERR_INVALID_ARG, "n_particles < 0");
    if (n_particles == 0) return RAD_OK;
    const void *arr[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
    for (const void *p : arr)
        if (!p) return fail(&h, RAD_ERR_INVALID_ARG, "NULL state array");
    return accumulate_device(h, step_index, n_particles, arr, (cudaStream_t)cuda_stream);
}

rad_status rad_accumulate_steps(rad_handle *hh, int64_t first_step_index, int32_t n_steps,
                                int64_t n_particles, int64_t step_stride, const void *rx, const void *ry,
                                const void *rz, const void *bx, const void *by, const void *bz,
                                const void *bdx, const void *bdy, const void *bdz, const void *w,
                                void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    if (h.R > 1) return fail(&h, RAD_ERR_UNSUPPORTED, "rad_accumulate_steps on a per-region handle");
    if (n_particles < 0 || n_steps < 0) return fail(&h, RAD_ERR_INVALID_ARG, "n_particles / n_steps < 0");
    if (n_steps > 1 && step_stride < n_particles)
        return fail(&h, RAD_ERR_INVALID_ARG, "step_stride < n_particles");
    if (n_particles == 0 || n_steps == 0) return RAD_OK;
    const void *arr[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
    for (const void *p : arr)
        if (!p) return fail(&h, RAD_ERR_INVALID_ARG, "NULL state array");
    return accumulate_device(h, first_step_index, n_particles, arr, (cudaStream_t)cuda_stream, nullptr, 0,
                             n_steps, step_stride);
}

static rad_status check_regions(Handle &h, int32_t n_regions, const int64_t *off);

rad_status rad_accumulate_steps_regions(rad_handle *hh, int64_t first_step_index, int32_t n_steps,
                                        int64_t step_stride, int32_t n_regions,
                                        const int64_t *region_offsets, const void *rx, const void *ry,
                                        const void *rz, const void *bx, const void *by, const void *bz,
                                        const void *bdx, const void *bdy, const void *bdz, const void *w,
                                        void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    st = check_regions(h, n_regions, region_offsets);
    if (st != RAD_OK) return st;
    if (n_steps < 0) return fail(&h, RAD_ERR_INVALID_ARG, "n_steps < 0");
    if (n_steps > 1 && step_stride < region_offsets[n_regions])
        return fail(&h, RAD_ERR_INVALID_ARG, "step_stride < region_offsets[n_regions]");
    const long long n = region_offsets[n_regions] - region_offsets[0];
    if (n == 0 || n_steps == 0) return RAD_OK;
    const void *arr[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
    for (const void *p : arr)
        if (!p) return fail(&h, RAD_ERR_INVALID_ARG, "NULL state array");
    if (h.R == 1) {  // one region = the plain multi-step call on the sub-range
        const size_t esz = h.state_f64 ? 8 : 4;
        const void *sub[10];
        for (int i = 0; i < 10; ++i) sub[i] = (const char *)arr[i] + (size_t)region_offsets[0] * esz;
        return accumulate_device(h, first_step_index, n, sub, (cudaStream_t)cuda_stream, nullptr, 0, n_steps,
                                 step_stride);
    }
    return accumulate_device(h, first_step_index, region_offsets[n_regions], arr, (cudaStream_t)cuda_stream,
                             region_offsets, 0, n_steps, step_stride);
}

static rad_status check_regions(Handle &h, int32_t n_regions, const int64_t *off)
{
    if (n_regions != h.R) return fail(&h, RAD_ERR_INVALID_ARG, "n_regions differs from the handle's");
    if (!off) return fail(&h, RAD_ERR_INVALID_ARG, "region_offsets is NULL");
    if (off[0] < 0) return fail(&h, RAD_ERR_INVALID_ARG, "region_offsets[0] < 0");
    for (int r = 0; r < n_regions; ++r)
        if (off[r + 1] < off[r]) return fail(&h, RAD_ERR_INVALID_ARG, "region_offsets must be non-decreasing");
    return RAD_OK;
}

rad_status rad_accumulate_step_regions(rad_handle *hh, int64_t step_index, int32_t n_regions,
                                       const int64_t *region_offsets, const void *rx, const void *ry,
                                       const void *rz, const void *bx, const void *by, const void *bz,
                                       const void *bdx, const void *bdy, const void *bdz, const void *w,
                                       void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    st = check_regions(h, n_regions, region_offsets);
    if (st != RAD_OK) return st;
    const long long n = region_offsets[n_regions] - region_offsets[0];
    if (n == 0) return RAD_OK;
    const void *arr[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
    for (const void *p : arr)
        if (!p) return fail(&h, RAD_ERR_INVALID_ARG, "NULL state array");
    if (h.R == 1) {  // one region = the plain call on the sub-range [offsets[0], offsets[1])
        const size_t esz = h.state_f64 ? 8 : 4;
        const void *sub[10];
        for (int i = 0; i < 10; ++i) sub[i] = (const char *)arr[i] + (size_t)region_offsets[0] * esz;
        return accumulate_device(h, step_index, n, sub, (cudaStream_t)cuda_stream);
    }
    // the kernels index the caller's arrays directly: offsets stay absolute (base 0)
    return accumulate_device(h, step_index, region_offsets[n_regions], arr, (cudaStream_t)cuda_stream,
                             region_offsets, 0);
}

// HOST state: elements [first, first + n_particles) of the 10 arrays go through the handle's
// double-buffered device staging; region_off (optional) are the caller's absolute offsets.
static rad_status accumulate_host(Handle &h, int64_t step_index, long long first, int64_t n_particles,
                                  const void *const arr[10], const int64_t *region_off, cudaStream_t s)
{
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
        RAD_CUDA(&h, cudaMemcpyAsync(dst, (const char *)arr[i] + (size_t)first * esz,
                                     (size_t)n_particles * esz, cudaMemcpyHostToDevice, h.copy_stream));
        dev[i] = dst;
    }
    RAD_CUDA(&h, cudaEventRecord(h.copied[b], h.copy_stream));
    RAD_CUDA(&h, cudaStreamWaitEvent(s, h.copied[b], 0));
    rad_status st = accumulate_device(h, step_index, n_particles, dev, s, region_off, first);
    if (st != RAD_OK) return st;
    RAD_CUDA(&h, cudaEventRecord(h.consumed[b], s));
    h.consumed_valid[b] = true;
    return RAD_OK;
}

rad_status rad_accumulate_step_host(rad_handle *hh, int64_t step_index, int64_t n_particles,
                                    const void *rx, const void *ry, const void *rz, const void *bx,
                                    const void *by, const void *bz, const void *bdx, const void *bdy,
                                    const void *bdz, const void *w, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    if (h.R > 1) return fail(&h, RAD_ERR_INVALID_ARG, "per-region handle: use rad_accumulate_step_regions_host");
    if (n_particles < 0) return fail(&h, RAD_ERR_INVALID_ARG, "n_particles < 0");
    if (n_particles == 0) return RAD_OK;
    const void *arr[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
    for (const void *p : arr)
        if (!p) return fail(&h, RAD_ERR_INVALID_ARG, "NULL state array");
    return accumulate_host(h, step_index, 0, n_particles, arr, nullptr, (cudaStream_t)cuda_stream);
}

rad_status rad_accumulate_step_regions_host(rad_handle *hh, int64_t step_index, int32_t n_regions,
                                            const int64_t *region_offsets, const void *rx,
                                            const void *ry, const void *rz, const void *bx,
                                            const void *by, const void *bz, const void *bdx,
                                            const void *bdy, const void *bdz, const void *w,
                                            void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    st = check_regions(h, n_regions, region_offsets);
    if (st != RAD_OK) return st;
    const long long n = region_offsets[n_regions] - region_offsets[0];
    if (n == 0) return RAD_OK;
    const void *arr[10] = {rx, ry, rz, bx, by, bz, bdx, bdy, bdz, w};
    for (const void *p : arr)
        if (!p) return fail(&h, RAD_ERR_INVALID_ARG, "NULL state array");
    return accumulate_host(h, step_index, region_offsets[0], n, arr, h.R == 1 ? nullptr : region_offsets,
                           (cudaStream_t)cuda_stream);
}

}  // extern "C" (a template cannot have C linkage)

template <typename Launch>
static rad_status deliver(Handle &h, double *out, int out_on_device, size_t bytes, cudaStream_t s, Launch launch)
{
    if (!out) return fail(&h, RAD_ERR_INVALID_ARG, "out is NULL");
    if (out_on_device < RAD_OUT_HOST || out_on_device > RAD_OUT_HOST_ASYNC)
        return fail(&h, RAD_ERR_INVALID_ARG, "out_on_device must be RAD_OUT_HOST, RAD_OUT_DEVICE or RAD_OUT_HOST_ASYNC");
    if (h.fast) {  // approximate fast path: the accumulator is evaluated from the retarded-time grids on demand
        rad_status st_ = evaluate_gridded(h, s);
        if (st_ != RAD_OK) return st_;
        if (out_on_device == RAD_OUT_HOST) {  // the synchronous form also reports terms that missed the grid
            unsigned long long lost = 0;
            RAD_CUDA(&h, cudaMemcpyAsync(&lost, h.g_oob_d, sizeof(lost), cudaMemcpyDeviceToHost, s));
            RAD_CUDA(&h, cudaStreamSynchronize(s));
            if (lost)
                return fail(&h, RAD_ERR_STATE, std::to_string(lost) + " (particle, direction) terms fell outside "
                            "the fast_box / step window given at rad_create and were not deposited");
        }
    }
    if (out_on_device == RAD_OUT_DEVICE) {
        RAD_CUDA(&h, launch(h, out, s));
        h.launches += 1;
        return RAD_OK;
    }
    rad_status st = ensure_out(h, bytes);
    if (st != RAD_OK) return st;
    RAD_CUDA(&h, launch(h, h.out_d, s));
    h.launches += 1;
    RAD_CUDA(&h, cudaMemcpyAsync(out, h.out_d, bytes, cudaMemcpyDeviceToHost, s));
    if (out_on_device != RAD_OUT_HOST_ASYNC) RAD_CUDA(&h, cudaStreamSynchronize(s));
    return RAD_OK;
}

extern "C" {

rad_status rad_spectrum(rad_handle *hh, double *out, int out_on_device, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    return deliver(hh->h, out, out_on_device, (size_t)hh->h.R * hh->h.D * hh->h.W * sizeof(double),
                   (cudaStream_t)cuda_stream, launch_spectrum);
}

rad_status rad_spectrum_total(rad_handle *hh, double *out, int out_on_device, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    return deliver(hh->h, out, out_on_device, (size_t)hh->h.D * hh->h.W * sizeof(double),
                   (cudaStream_t)cuda_stream, launch_spectrum_total);
}

rad_status rad_amplitude(rad_handle *hh, double *out, int out_on_device, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    return deliver(hh->h, out, out_on_device, (size_t)hh->h.R * hh->h.D * hh->h.W * 6 * sizeof(double),
                   (cudaStream_t)cuda_stream, launch_amplitude);
}

rad_status rad_add_amplitude(rad_handle *hh, const double *amp_device, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    if (!amp_device) return fail(&hh->h, RAD_ERR_INVALID_ARG, "amp_device is NULL");
    if (hh->h.fast) return fail(&hh->h, RAD_ERR_UNSUPPORTED, "rad_add_amplitude on a RAD_FLAG_FAST_GRIDDED handle");
    RAD_CUDA(&hh->h, launch_add_amplitude(hh->h, amp_device, (cudaStream_t)cuda_stream));
    hh->h.launches += 1;
    return RAD_OK;
}

rad_status rad_export_accumulator(rad_handle *hh, double *out_device, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    if (!out_device) return fail(&h, RAD_ERR_INVALID_ARG, "out_device is NULL");
    if (h.fast) return fail(&h, RAD_ERR_UNSUPPORTED, "rad_export_accumulator on a RAD_FLAG_FAST_GRIDDED handle");
    // rows of W*4 doubles out of the padded [R*D][w_pad][4] accumulator; a memcpy keeps its full
    // stream dependencies under RAD_FLAG_OVERLAP_STEPS (it runs after every fold queued before)
    const size_t row = (size_t)h.W * 4 * sizeof(double);
    RAD_CUDA(&h, cudaMemcpy2DAsync(out_device, row, h.acc_d, (size_t)h.w_pad * 4 * sizeof(double), row,
                                   (size_t)h.R * h.D, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    return RAD_OK;
}

rad_status rad_import_accumulator(rad_handle *hh, const double *amp4_device, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    if (!amp4_device) return fail(&hh->h, RAD_ERR_INVALID_ARG, "amp4_device is NULL");
    if (hh->h.fast) return fail(&hh->h, RAD_ERR_UNSUPPORTED, "rad_import_accumulator on a RAD_FLAG_FAST_GRIDDED handle");
    RAD_CUDA(&hh->h, launch_import_accumulator(hh->h, amp4_device, (cudaStream_t)cuda_stream));
    hh->h.launches += 1;
    return RAD_OK;
}

rad_status rad_spectrum_of(rad_handle *hh, const double *amp4_device, double *out, int out_on_device,
                           void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    if (!amp4_device) return fail(&hh->h, RAD_ERR_INVALID_ARG, "amp4_device is NULL");
    return deliver(hh->h, out, out_on_device, (size_t)hh->h.R * hh->h.D * hh->h.W * sizeof(double),
                   (cudaStream_t)cuda_stream, [amp4_device](const Handle &h, double *o, cudaStream_t s) {
                       return launch_spectrum_of(h, amp4_device, o, s);
                   });
}

rad_status rad_reset(rad_handle *hh, void *cuda_stream)
{
    DeviceGuard guard;
    rad_status st = check_handle(hh, guard);
    if (st != RAD_OK) return st;
    Handle &h = hh->h;
    RAD_CUDA(&h, cudaMemsetAsync(h.acc_d, 0, (size_t)h.R * h.D * h.w_pad * 4 * sizeof(double),
                                 (cudaStream_t)cuda_stream));
    if (h.fast) {
        cudaStream_t s = (cudaStream_t)cuda_stream;
        RAD_CUDA(&h, cudaMemsetAsync(h.g_delta_d, 0, sizeof(float2) * 2 * (size_t)h.D * h.g_M, s));
        RAD_CUDA(&h, cudaMemsetAsync(h.g_master_d, 0, sizeof(double2) * (size_t)h.D * h.g_M, s));
        RAD_CUDA(&h, cudaMemsetAsync(h.g_oob_d, 0, sizeof(unsigned long long), s));
        h.g_pending = 0;
        h.g_acc_valid = true;
    }
    return RAD_OK;
}

void rad_destroy(rad_handle *hh)
{
    if (!hh) return;
    {
        DeviceGuard guard;
        if (guard.enter(hh->h.device) == cudaSuccess) {
            cudaDeviceSynchronize();
            free_all(hh->h);
        }
        cudaGetLastError();
    }
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

const char *rad_version(void) { return "rad-b200 0.4 (sm_100a)"; }

}  // extern "C"
