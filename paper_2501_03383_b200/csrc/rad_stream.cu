// rad_stream.cu -- particle-streaming accumulate kernel ("particle owner" mapping) for detectors
// with very few bins (D*W <= 16, e.g. config 4b: 1 direction x 8 frequencies), where the 40 B
// of state per particle feed only a handful of updates and HBM bandwidth binds
// (BASELINE.json configs[4] "streamed from HBM each step").
//
// Mapping: a thread owns particles (4 per 1024-particle tile) and keeps ALL bins' fp32 partial
// amplitudes in registers; blocks are persistent and walk the tiles with stride gridDim.x.
// Staging (the "per-step particle-staging kernel ... staged via TMA", BASELINE.json north_star):
// one elected thread issues ten 1-D bulk async copies (cp.async.bulk, SASS UBLKCP) per tile
// into a two-stage shared-memory ring, completion signalled on an mbarrier (expect_tx), so
// the copy of tile i+1 runs under the arithmetic of tile i.  Unaligned arrays or a ragged
// last tile fall back to coalesced ld.global.nc.  At the end the partials go through
// warp-shuffle reductions, a shared-memory cross-warp sum and one fp64 atomic per value
// per block (or the deterministic workspace).
#include "rad_device.cuh"
#include "rad_internal.h"

namespace rad {

namespace {

using namespace dev;

// Shape of the ring, frozen from the round-1 sweeps.
constexpr int kSThreads = 256;
constexpr int kSStages = 2;
constexpr int kSUnroll = 4;
constexpr int kSMinBlocks = 2;
constexpr int kSTileBytes = 4096;  // per array per stage -> 1024 fp32 / 512 fp64 particles

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

template <typename ST, bool WIN>
__device__ __forceinline__ Particle make_particle(ST rx, ST ry, ST rz, ST bx, ST by, ST bz, ST dx,
                                                  ST dy, ST dz, ST w, const AccumParams &P)
{
    Particle p;
    p.rx = to_f64(rx); p.ry = to_f64(ry); p.rz = to_f64(rz);
    p.bx = to_f64(bx); p.by = to_f64(by); p.bz = to_f64(bz);
    p.bfx = (float)bx; p.bfy = (float)by; p.bfz = (float)bz;
    p.bdx = (float)dx; p.bdy = (float)dy; p.bdz = (float)dz;
    p.wdt = (float)w * P.dt;
    if (WIN) p.wdt *= window_weight(P, p.rx, p.ry, p.rz);
    return p;
}

// NB bins per thread = ND directions x WB frequencies (compile time; W is padded to WB with
// zero-frequency bins that are discarded).  Per-bin frequency constants come straight from the
// kernel-parameter constant bank (P.sF/sFf/sfl), not from registers.
// WIN: spatial window compiled in (kept out of the default instantiation: the streaming kernel
// is latency bound and loses 3 % to the extra per-particle code even when the window is off)
template <typename ST, int NB, int ND, bool WIN>
__global__ void __launch_bounds__(kSThreads, NB <= 8 ? kSMinBlocks : 1) rad_accum_stream(const AccumParams P, const int use_bulk)
{
    constexpr int TILE = kSTileBytes / (int)sizeof(ST);  // particles per tile
    constexpr int PPT = TILE / kSThreads;                 // particles per thread per tile
    constexpr int WB = NB / ND;
    static_assert(PPT >= 1 && WB * ND == NB, "tile/bin shape");
    extern __shared__ __align__(128) unsigned char s_raw[];
    __shared__ __align__(8) uint64_t s_full[kSStages];
    __shared__ float s_red[kSThreads / 32][NB * 4];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    pdl_trigger();
    float acc[NB][4];
#pragma unroll
    for (int b = 0; b < NB; ++b) acc[b][0] = acc[b][1] = acc[b][2] = acc[b][3] = 0.0f;

    const long long N = P.n_particles;
    const long long n_tiles = (N + TILE - 1) / TILE;
    if (tid == 0) {
        for (int s = 0; s < kSStages; ++s) mbar_init(&s_full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto tile_bulk = [&](long long t) -> bool {  // full tile (16-B multiple) and aligned arrays
        return use_bulk && (t + 1) * TILE <= N;
    };
    auto issue = [&](long long t, int stage) {  // thread 0 only
        mbar_expect_tx(&s_full[stage], 10u * kSTileBytes);
#pragma unroll
        for (int a = 0; a < 10; ++a)
            bulk_g2s(s_raw + ((size_t)stage * 10 + a) * kSTileBytes,
                     reinterpret_cast<const ST *>(P.st[a]) + t * TILE, kSTileBytes, &s_full[stage]);
    };

    // prologue: fill kSStages-1 stages ahead
    const long long t0 = blockIdx.x, dtile = gridDim.x;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kSStages - 1; ++s) {
            const long long tp = t0 + s * dtile;
            if (tp < n_tiles && tile_bulk(tp)) issue(tp, s);
        }
    }
    uint32_t phase_bits = 0;  // bit s: parity the next wait on stage s expects
    int stage = 0;
    for (long long t = t0; t < n_tiles; t += dtile) {
        // stage (stage-1) mod kSStages was read in the previous iteration; its barrier is behind us
        const long long tn = t + (kSStages - 1) * dtile;
        const int sn = stage == 0 ? kSStages - 1 : stage - 1;
        if (tid == 0 && tn < n_tiles && tile_bulk(tn)) issue(tn, sn);
        const bool bulk = tile_bulk(t);
        if (bulk) {
            mbar_wait(&s_full[stage], (phase_bits >> stage) & 1u);
            phase_bits ^= 1u << stage;
        }
        const ST *sm = reinterpret_cast<const ST *>(s_raw + (size_t)stage * 10 * kSTileBytes);
#pragma unroll kSUnroll
        for (int pp = 0; pp < PPT; ++pp) {
            const int kl = tid + pp * kSThreads;
            const long long k = t * TILE + kl;
            Particle p;
            if (bulk) {
                p = make_particle<ST, WIN>(sm[0 * TILE + kl], sm[1 * TILE + kl], sm[2 * TILE + kl],
                                      sm[3 * TILE + kl], sm[4 * TILE + kl], sm[5 * TILE + kl],
                                      sm[6 * TILE + kl], sm[7 * TILE + kl], sm[8 * TILE + kl],
                                      sm[9 * TILE + kl], P);
            } else {
                p = load_particle<ST, WIN>(P, k, k < N);
            }
#pragma unroll
            for (int d = 0; d < ND; ++d) {
                float4 r4;
                float sf;
                stage_record(p, P.sdir[d], P.ts32, r4, sf);  // a1 (direction record: constant bank)
#pragma unroll
                for (int j = 0; j < WB; ++j) {  // a2
                    const int b = d * WB + j;
                    float sn2, cs2;
                    phase_sincos(P.sF[j], P.sFf[j], P.sfl[j], __float_as_uint(r4.x), r4.y, sf, sn2, cs2);
                    acc[b][0] = fmaf(r4.z, cs2, acc[b][0]);
                    acc[b][1] = fmaf(r4.z, sn2, acc[b][1]);
                    acc[b][2] = fmaf(r4.w, cs2, acc[b][2]);
                    acc[b][3] = fmaf(r4.w, sn2, acc[b][3]);
                }
            }
        }
        __syncthreads();  // this stage may be refilled by the next iteration's issue
        stage = stage + 1 == kSStages ? 0 : stage + 1;
    }

    // a3: warp-shuffle reduction, cross-warp sum in shared memory, one fp64 add per value
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            float v = acc[b][c];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) s_red[warp][b * 4 + c] = v;
        }
    __syncthreads();
    pdl_wait();  // the accumulator belongs to earlier work until here
    if (tid < NB * 4) {
        const int b = tid >> 2, c = tid & 3;
        const int d = b / WB, j = b - d * WB;
        if (d < P.n_dir && j < P.n_omega) {
            double v = 0.0;
#pragma unroll
            for (int wp = 0; wp < kSThreads / 32; ++wp) v += (double)s_red[wp][tid];
            const size_t off = ((size_t)d * P.w_pad + j) * 4 + c;
            if (P.partial)
                P.partial[(size_t)blockIdx.x * P.n_dir * P.w_pad * 4 + off] = v;
            else
                atomicAdd(P.acc + off, v);
        }
    }
}

template <typename ST, int NB, int ND, bool WIN>
cudaError_t launch_stream_w(const AccumParams &p, int grid, cudaStream_t s, bool overlap)
{
    const size_t smem = (size_t)kSStages * 10 * kSTileBytes;
    // per device and per template instance; the call is a cheap host-side set, so no caching
    cudaError_t e = cudaFuncSetAttribute(rad_accum_stream<ST, NB, ND, WIN>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int use_bulk = 1;
    for (int a = 0; a < 10; ++a)
        if (reinterpret_cast<uintptr_t>(p.st[a]) & 15) use_bulk = 0;
    return launch_kernel(rad_accum_stream<ST, NB, ND, WIN>, dim3(grid), dim3(kSThreads), smem, s, overlap, p, use_bulk);
}

template <typename ST, int NB, int ND>
cudaError_t launch_stream_t(const AccumParams &p, int grid, cudaStream_t s, bool overlap)
{
    return p.win_type != RAD_WINDOW_NONE ? launch_stream_w<ST, NB, ND, true>(p, grid, s, overlap)
                                         : launch_stream_w<ST, NB, ND, false>(p, grid, s, overlap);
}

template <typename ST>
cudaError_t dispatch_stream(const Handle &h, const AccumParams &p, int grid, cudaStream_t s)
{
    if (h.stream_nb == 8) return h.stream_nd == 1 ? launch_stream_t<ST, 8, 1>(p, grid, s, h.overlap) : launch_stream_t<ST, 8, 2>(p, grid, s, h.overlap);
    return h.stream_nd == 1 ? launch_stream_t<ST, 16, 1>(p, grid, s, h.overlap) : launch_stream_t<ST, 16, 2>(p, grid, s, h.overlap);
}

}  // namespace

int stream_tile_particles(bool state_f64) { return kSTileBytes / (state_f64 ? 8 : 4); }
int stream_blocks_per_sm(int nb) { return nb <= 8 ? kSMinBlocks : 1; }

// Shapes served: ND in {1, 2} directions x WB = NB/ND frequencies, NB in {8, 16}.
// Returns NB (and *nd), or 0 if this detector shape is not a streaming shape.
int stream_shape(int D, int W, int *nd)
{
    for (int nb = 8; nb <= 16; nb *= 2)
        for (int d = 1; d <= 2; ++d)
            if (D <= d && W <= nb / d) { *nd = d; return nb; }
    return 0;
}

// grid = number of persistent blocks (also the number of deterministic partial slots)
cudaError_t launch_accumulate_stream(const Handle &h, const AccumParams &p, bool state_f64, int grid,
                                     cudaStream_t s)
{
    return state_f64 ? dispatch_stream<double>(h, p, grid, s) : dispatch_stream<float>(h, p, grid, s);
}

}  // namespace rad
