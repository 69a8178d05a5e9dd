// rad_internal.h -- host/device shared declarations of the CUDA path (NOT part of the ABI).
//
// Notation follows BASELINE.json north_star / SURVEY.md section 8: N particles, D directions n,
// W frequencies w_j = 2 pi f_j, A(n, w_j) complex amplitude, S = scale |A|^2.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "rad.h"

namespace rad {

constexpr double kC = 299792458.0;             // m/s
constexpr double kTwo32 = 4294967296.0;        // 2^32
constexpr int kWarpsPerBlock = 4;              // one warp per SM sub-partition
constexpr int kThreads = 32 * kWarpsPerBlock;
constexpr int kBatch = 32;                     // particles staged per warp batch (one per lane)
// general kernel, hybrid sincos: bins (of the 8-bin strip) per even / odd particle of a batch
// that take the FMA-pipe polynomial instead of the XU pipe (0 = pure MUFU).  Measured on B200
// (cfg 1 / cfg 2, % of R_gen): (0,0) 85.4 / 88.6, (0,1) 88.3 / 91.3, (0,2) 87.1 / 89.6,
// (1,1) 84.7 / 87.5, (1,2) 88.4 / 90.8, (0,3) 84.0 / 86.6, (2,2) 81.6 / 84.0; cfg 3d (8 lanes
// along frequency): 82.5 -> 84.6.  Frozen at (0,1) for every tile shape.
constexpr int kPolyEven = 0, kPolyOdd = 1;
constexpr int kStrip = 8;                      // frequency bins per thread (register strip)
constexpr int kMinBlocks = 4;                  // resident blocks per SM the kernels are bounded for

// Per direction (device table).  k = n * (f_unit 2^32 / c): the dot product k.r is the
// light-travel delay n.r/c measured in units of 2^-32 "unit turns" (phase).
struct DirRec {
    double kx, ky, kz;     // fp64: phase path
    double nx, ny, nz;     // fp64 unit vector: Doppler factor d = 1 - n.beta
    float nfx, nfy, nfz;   // fp32 copy for n.betadot
    float e1x, e1y, e1z;   // transverse orthonormal basis, e1 x e2 = n (A is _|_ n exactly)
    float e2x, e2y, e2z;
    float pad[3];
};
static_assert(sizeof(DirRec) == 96, "DirRec layout");

// One unit of particle work of a per-region or multi-step call: particles [k0, k0+len) of one
// region, at time step (first step of the call) + step.
struct ChunkRec {
    long long k0;
    int len;
    int region;
    int step;
    int pad;
};
static_assert(sizeof(ChunkRec) == 24, "ChunkRec layout");

// Everything the accumulate kernels need, passed by value.
struct AccumParams {
    const void *st[10];    // rx ry rz bx by bz bdx bdy bdz w (DEVICE, float or double)
    long long n_particles;
    int chunk;             // particles per chunk (multiple of kBatch); chunk c = [c*chunk, ...)
    int n_chunks;          // a warp task = (warp tile, chunk); n_tasks = n_wtiles * n_chunks
    const ChunkRec *chunks; // per-region / multi-step calls: [n_chunks] chunk table (DEVICE), else NULL
    int n_dir, n_omega;    // D, W
    int w_pad;             // W padded to the frequency tile
    int n_ftiles;          // frequency tiles per direction group
    int n_wtiles;          // warp tiles = direction groups * n_ftiles
    int psplit;            // particle split: 2^psplit lane groups of a warp share one direction (0: off)
    const DirRec *dirs;    // [D]
    const uint32_t *F;     // [w_pad] integer part of f_j / f_unit
    const float *Ff;       // [w_pad] (float)F_j
    const float *fl;       // [w_pad] f_j / f_unit - F_j  in [-0.5, 0.5]
    const float *F2;       // form factor: [D][w_pad] F^2(n, w_j) (rad.h, reading FF1), NULL: off
    int w_sqrt;            // 1: the amplitude weight of a particle is sqrt(w) (RAD_FF_INCOHERENT: F = 0, g = sqrt(w) per particle)
    double ts32;           // (t0 + step dt) f_unit 2^32
    double dts32;          // dt f_unit 2^32: multi-step calls, chunk time = ts32 + chunk.step * dts32
    float dt;              // quadrature weight
    double nyq_lim;        // pi * nyquist_factor, 0: limiter off
    int nyq_mode;          // cut-off guess: 0 none (bisection), 1 log grid, 2 linear grid
    float nyq_a, nyq_b;    // log: guess = nyq_a * log2(nyq_b / d); linear: guess = nyq_a / d + nyq_b
    double dt64;           // dt in fp64 (limiter comparison)
    const double *omega64; // [W] fp64 angular frequencies (limiter comparison)
    int win_type;          // RAD_WINDOW_*; 0: none
    double win_o[3];       // window box origin
    double win_il[3];      // 1 / extent, 0: axis not windowed
    double *acc;           // [D][w_pad][4]: A1.re A1.im A2.re A2.im (transverse components)
    double *partial;       // deterministic mode: [n_chunks][D][w_pad][4], else NULL
    // streaming variant only: per-frequency constants and the (<= 2) direction records in the
    // parameter constant bank (operands come straight from c[0][..]: no loads, no registers)
    uint32_t sF[16];
    float sFf[16], sfl[16];
    float sF2[16];         // form factor: F^2 of bin b = d * WB + j
    DirRec sdir[2];
    // fast gridded path (rad_gridded.cu; rad.h RAD_FLAG_FAST_GRIDDED): per direction a uniform grid in
    // retarded time, point m at tau = (g_s0[dir] + m) h, h = g_hs in s32 units (s32 = tau f_unit 2^32)
    float2 *g_delta;             // [D][2][g_M] fp32 (A1, A2) deposits since the last fold: chunks starting at
                                 // even points, and chunks starting at odd points (stored one point to the left)
    const double2 *g_master;     // [D][g_M] fp64 grid (evaluation reads it)
    const double *g_s0;          // [D] index of grid point 0 in units of h: tau_m = (g_s0[n] + m) h (integers)
    const double2 *g_corr;       // [w_pad] complex 1 / (Phi(w_j) (1 - exp(i w_j h))): deconvolution of the
                                 // spreading kernel and of the first differences the evaluation sums
    double g_hs, g_ihs;          // grid spacing in s32 units and its inverse
    int g_M;                     // grid points per direction (even)
    int g_jdiff;                 // evaluation: frequency tiles starting at bins >= g_jdiff sum first differences
    float g_beta2;               // ES kernel exponent beta * log2(e)
    unsigned long long *g_oob;   // terms that fell outside the grid
    int dir0, dir1;              // spreading: directions [dir0, dir1) of this launch
    // uniform-grid variant only: LW*(f_1 - f_0)/f_unit = rot_G + rot_gl (integer + fraction)
    uint32_t rot_G;
    float rot_Gf, rot_gl;
};

struct Handle;

// Kernel launch, optionally with programmatic stream serialization (RAD_FLAG_OVERLAP_STEPS):
// the grid may start while its predecessor in the stream drains; the kernels call
// dev::pdl_wait() before they touch memory that earlier work writes.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                 bool overlap, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = overlap ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// kernels/launchers (rad_kernels.cu, rad_finalize.cu)
cudaError_t launch_accumulate(const Handle &h, const AccumParams &p, bool state_f64,
                              cudaStream_t s, int *n_launches, const char **variant);
cudaError_t launch_accumulate_stream(const Handle &h, const AccumParams &p, bool state_f64, int grid,
                                     cudaStream_t s);
int stream_tile_particles(int nb, bool state_f64);
int stream_blocks_per_sm(int nb);
int stream_shape(int D, int W, int *nd);
cudaError_t launch_spread(const Handle &h, const AccumParams &p, bool state_f64, cudaStream_t s);
cudaError_t launch_grid_fold(const Handle &h, cudaStream_t s);
cudaError_t launch_eval_grid(const Handle &h, const AccumParams &p, cudaStream_t s);
cudaError_t launch_spectrum(const Handle &h, double *out_dev, cudaStream_t s);
cudaError_t launch_amplitude(const Handle &h, double *out_dev, cudaStream_t s);
cudaError_t launch_add_amplitude(const Handle &h, const double *amp_dev, cudaStream_t s);
cudaError_t launch_reduce_partials(const Handle &h, const double *partial, int n_chunks,
                                   const int *region_chunk_start, cudaStream_t s);
cudaError_t launch_spectrum_total(const Handle &h, double *out_dev, cudaStream_t s);
cudaError_t launch_spectrum_of(const Handle &h, const double *amp4_dev, double *out_dev, cudaStream_t s);
cudaError_t launch_import_accumulator(const Handle &h, const double *amp4_dev, cudaStream_t s);

struct Handle {
    int device = 0;
    int D = 0, W = 0, w_pad = 0;
    int R = 1;                            // per-region detectors: acc is [R][D][w_pad][4]
    int lw = 32, strip = kStrip;          // lanes along frequency, bins per lane
    int n_ftiles = 0, n_wtiles = 0;
    int psplit = 0;                       // log2 of the lane groups per direction (few-direction detectors)
    int stream_nd = 1;
    int stream_nb = 0;               // > 0: D*W <= 16 -> particle-streaming kernel with 8 or 16 bins/thread
    double dt = 0, t0 = 0, scale = 0, f_unit = 0;
    double nyq_lim = 0;              // pi * nyquist_factor
    int nyq_mode = 0;                // closed-form cut-off guess for log / linear grids (rad_device.cuh nyquist_count)
    float nyq_a = 0, nyq_b = 0;
    double *omega_d = nullptr;       // [W] fp64 (Nyquist limiter only)
    int win_type = 0;
    double win_o[3] = {0, 0, 0}, win_il[3] = {0, 0, 0};
    bool state_f64 = false, deterministic = false, uniform = false;
    bool overlap = false;            // RAD_FLAG_OVERLAP_STEPS
    bool precise = false;            // RAD_FLAG_PRECISE: all-polynomial sincos on the general-grid kernel
    int dyad_c = 0;                  // > 0: dyadic log grid, w_(j + dyad_c*lw) = 2 w_j -> squaring chains (rad_kernels.cu DY)
    uint32_t rot_G = 0;              // uniform grid: rotator frequency LW*df in f_unit units
    float rot_Gf = 0, rot_gl = 0;
    int sm_count = 148;
    std::vector<double> dirs_h;      // normalised [D][3]
    std::vector<double> omega_h;
    uint32_t sF[16] = {0};           // streaming shapes: first 16 frequency constants (host copy)
    float sFf[16] = {0}, sfl[16] = {0};
    DirRec sdir[2] = {};             // streaming shapes: the direction records (host copy)
    DirRec *dirs_d = nullptr;
    double *basis_d = nullptr;       // [D][6] fp64 e1, e2 (amplitude export/import)
    uint32_t *F_d = nullptr;
    float *Ff_d = nullptr, *fl_d = nullptr;
    int ff_type = 0;                 // RAD_FF_*
    bool ff_table = false;           // Gaussian / CIC shape: per-update weight from the F^2 table (incoherent: sqrt(w) per particle)
    float *F2_d = nullptr;           // form factor on: [D][w_pad] F^2(n, w_j)
    std::vector<float> F2_h;         // host copy (streaming shapes pass it in the parameter bank)
    double *acc_d = nullptr;         // [D][w_pad][4]
    double *partial_d = nullptr;     // deterministic workspace
    size_t partial_bytes = 0;
    // host-state staging (rad_accumulate_step_host): two device buffers, copy stream
    void *stage_d[2] = {nullptr, nullptr};
    size_t stage_bytes[2] = {0, 0};
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t copied[2] = {nullptr, nullptr}, consumed[2] = {nullptr, nullptr};
    bool consumed_valid[2] = {false, false};
    int stage_next = 0;
    // per-region calls: chunk table (pinned host copy + device copy), rebuilt when the
    // caller's offsets or the chunk size change
    std::vector<long long> reg_offsets;   // offsets of the table currently on the device
    int reg_chunk = 0, reg_n_chunks = 0, reg_steps = 1;
    long long reg_stride = 0;
    long long tap_n = -1;                 // tapered plain-call table on the device: its n and chunk
    int tap_chunk = 0;
    int stp_steps = 0, stp_chunk = 0;     // multi-step table on the device (reg_chunk == -2): its shape
    long long stp_n = -1, stp_stride = 0;
    ChunkRec *chunks_h = nullptr, *chunks_d = nullptr;   // [reg_cap]
    int *reg_cstart_h = nullptr, *reg_cstart_d = nullptr; // [R+1] first chunk of each region
    size_t reg_cap = 0;
    cudaEvent_t reg_uploaded = nullptr;
    // fast gridded path (RAD_FLAG_FAST_GRIDDED)
    bool fast = false;
    int g_w = 0, g_M = 0;            // kernel width (grid points, even), grid points per direction
    int g_jdiff = 0;                 // first bin of the frequency tiles evaluated from first differences
    double g_hs = 0, g_beta = 0;     // grid spacing in s32 units, ES kernel parameter
    double g_box_min[3] = {0, 0, 0}, g_box_max[3] = {0, 0, 0};
    long long g_step_min = 0, g_step_max = 0;
    double *g_s0_d = nullptr;
    double2 *g_corr_d = nullptr;
    uint32_t *Fg_d = nullptr;        // frequency tables of the evaluation sweep, in units of 1 / (h 2^32)
    float *Ffg_d = nullptr, *flg_d = nullptr;
    float2 *g_delta_d = nullptr;
    double2 *g_master_d = nullptr;
    unsigned long long *g_oob_d = nullptr;
    int g_pending = 0;               // accumulate calls since the last fold of delta into master
    bool g_acc_valid = false;        // acc_d holds the evaluation of the current grid
    double *out_d = nullptr;         // scratch for HOST-destination results
    size_t out_bytes = 0;
    int64_t launches = 0;
    const char *variant = "none";
    bool broken = false;
    std::string err;
};

}  // namespace rad
