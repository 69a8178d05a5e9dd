// rad_stream.cu -- particle-streaming accumulate kernel ("particle owner" mapping) for detectors
// with very few bins (D*W <= 16, e.g. config 4b: 1 direction x 8 frequencies), where the 40 B
// of state per particle feed only a handful of updates and HBM bandwidth binds
// (BASELINE.json configs[4] "streamed from HBM each step").
//
// Mapping: a lane owns particles and keeps ALL bins' fp32 partial amplitudes in registers.
// Every WARP runs its own copy pipeline -- no block-level barrier anywhere in the loop (round 1's
// per-tile __syncthreads cost 0.75 stall cycles per issued instruction at 16 warps per SM):
//   * one persistent block of 20 warps per SM; the warps work through "warp tiles" of 32 x PPT
//     particles (PPT = 16 B / sizeof(state element): 4 fp32 or 2 fp64 particles per lane) drawn
//     from the block's tile counter in shared memory (work stealing within the SM; static
//     round-robin shares in deterministic mode);
//   * staging (the "per-step particle-staging kernel ... staged via TMA" of BASELINE.json
//     north_star): lane 0 issues ten 512-byte 1-D bulk async copies (cp.async.bulk, SASS UBLKCP)
//     per warp tile into the warp's own two-stage shared-memory ring (2 x 5 KB), completion
//     signalled on the warp's own mbarrier (expect_tx);
//   * a lane reads its PPT consecutive particles of each array with ONE 16-byte shared-memory
//     load (10 LDS.128 per warp tile instead of 40 LDS.32); at the top of a turn -- after a
//     __syncwarp -- lane 0 refills the stage read in the previous turn with the next tile, which
//     arrives under this turn's arithmetic (20 warps x 5 KB in flight per SM, ~3x the 35 KB that
//     latency x bandwidth asks for).
// The ragged tail (N mod 32*PPT particles) and arrays that are not 16-byte aligned go through
// coalesced ld.global.nc, one particle per lane.  At the end the partials go through warp-shuffle
// reductions, a shared-memory cross-warp sum and one fp64 atomic per value per block (or the
// deterministic workspace).
//
// Per update the four accumulate FMAs are two packed fma.rn.f32x2 (A1 and A2 each times the
// (cos, sin) pair): the kernel is co-limited by instruction issue (~200 instructions per particle
// against 40 B of HBM traffic), so halving the accumulate instructions matters more than the
// lower per-instruction rate of the packed form.
#include "rad_device.cuh"
#include "rad_internal.h"

namespace rad {

namespace {

using namespace dev;

// Shape of the pipeline: ONE block per SM, so that the warps of an SM can
// share a tile counter in shared memory.
constexpr int kSStages = 2;
constexpr int kSArrayBytes = 512;           // per array per stage per warp: 32 lanes x 16 B
constexpr int kSStageBytes = 10 * kSArrayBytes;
// warps per block, each with its own 10 KB ring: 20 (200 KB of rings, <= 102 registers) for <= 8
// bins per thread, 12 for 16 bins per thread (168 registers)
__host__ __device__ constexpr int stream_warps(int nb) { return nb <= 8 ? 20 : 12; }

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

// one lane of the (converged) warp; with warp-uniform operands the copy instructions that follow
// are issued from the uniform datapath without a per-lane address loop
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}" : "=r"(pred));
    return pred != 0;
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
    p.w = (float)w;
    p.ww = fmaf(p.w, p.w, -p.w);
    p.wdt = (WIN && P.F2) ? P.dt : (P.w_sqrt ? __fsqrt_rn(p.w) : p.w) * P.dt;  // form factor table on: the weight enters per update (ff_weight)
    if (WIN) p.wdt *= window_weight(P, p.rx, p.ry, p.rz);
    return p;
}

// 16 bytes of state = PPT consecutive particles of one array
template <typename ST> struct Vec16;
template <> struct Vec16<float> {
    float4 v;
    __device__ __forceinline__ float get(int i) const { return i == 0 ? v.x : i == 1 ? v.y : i == 2 ? v.z : v.w; }
};
template <> struct Vec16<double> {
    double2 v;
    __device__ __forceinline__ double get(int i) const { return i == 0 ? v.x : v.y; }
};

// a1 + a2 for one particle: all bins of all (<= 2) directions
template <int NB, int ND, bool WIN>
__device__ __forceinline__ void accumulate_particle(const AccumParams &P, const Particle &p,
                                                    unsigned long long (&acc01)[NB], unsigned long long (&acc23)[NB])
{
    constexpr int WB = NB / ND;
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        float4 r4;
        float sf;
        stage_record(p, P.sdir[d], P.ts32, r4, sf);  // a1 (direction record: constant bank)
        const unsigned long long a1 = pack2(r4.z, r4.z), a2 = pack2(r4.w, r4.w);
#pragma unroll
        for (int j = 0; j < WB; ++j) {  // a2
            float sn, cs;
            phase_sincos(P.sF[j], P.sFf[j], P.sfl[j], __float_as_uint(r4.x), r4.y, sf, sn, cs);
            if (WIN && P.F2) {  // macro-particle form factor (rad.h, reading FF1)
                const float g = ff_weight(p.w, p.ww, P.sF2[d * WB + j]);
                sn *= g;
                cs *= g;
            }
            const unsigned long long z = pack2(cs, sn);
            fma2(acc01[d * WB + j], a1, z);  // (Re, Im) A1 += a1 (cos, sin)
            fma2(acc23[d * WB + j], a2, z);  // (Re, Im) A2 += a2 (cos, sin)
        }
    }
}

// NB bins per thread = ND directions x WB frequencies (compile time; W is padded to WB with
// zero-frequency bins that are discarded).  Per-bin frequency constants come straight from the
// kernel-parameter constant bank (P.sF/sFf/sfl), not from registers.
// WIN: spatial window and macro-particle form factor compiled in (kept out of the default
// instantiation: the streaming kernel loses 3 % to the extra per-particle code even when both are off)
template <typename ST, int NB, int ND, bool WIN>
__global__ void __launch_bounds__(32 * stream_warps(NB), 1) rad_accum_stream(const AccumParams P, const int use_bulk)
{
    constexpr int kSWarps = stream_warps(NB);
    constexpr int PPT = 16 / (int)sizeof(ST);  // particles per lane per warp tile
    constexpr int WTILE = 32 * PPT;            // particles per warp tile
    constexpr int WB = NB / ND;
    static_assert(WB * ND == NB && kSStages == 2, "bin shape / two-stage ring");
    extern __shared__ __align__(128) unsigned char s_raw[];  // [kSWarps][kSStages][10][512 B]
    __shared__ __align__(8) uint64_t s_full[kSWarps][kSStages];
    __shared__ float s_red[kSWarps][NB * 4];
    __shared__ int s_next;  // dynamic schedule: next tile of this block

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);  // warp-uniform to the compiler: uniform-datapath addresses
    pdl_trigger();
    unsigned long long acc01[NB], acc23[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) acc01[b] = acc23[b] = 0ull;

    const long long N = P.n_particles;
    const long long n_full = use_bulk ? N / WTILE : 0;  // warp tiles that go through the bulk-copy ring
    const long long gw = (long long)blockIdx.x * kSWarps + warp, GW = (long long)gridDim.x * kSWarps;
    unsigned char *ring = s_raw + (size_t)warp * kSStages * kSStageBytes;
    uint64_t *full = s_full[warp];

    if (tid == 0) s_next = 0;
    if (elect_one()) {
#pragma unroll
        for (int s = 0; s < kSStages; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();  // the one block barrier before the loop (tile counter, barriers)

    auto issue = [&](long long t, int stage) {  // one elected lane: ten 512-byte copies, one barrier
        mbar_expect_tx(&full[stage], (uint32_t)kSStageBytes);
#pragma unroll
        for (int a = 0; a < 10; ++a)
            bulk_g2s(ring + (size_t)stage * kSStageBytes + a * kSArrayBytes,
                     reinterpret_cast<const ST *>(P.st[a]) + t * WTILE, kSArrayBytes, &full[stage]);
    };

    // Which tiles a warp works on.  The tiles are dealt to the blocks round robin (block b owns
    // tiles b, b + gridDim.x, ...); within the block (= within the SM) the warps DRAW the block's
    // tiles from a shared-memory counter, one draw ahead of the copy it feeds.  The warp schedulers
    // are not fair (measured: with equal static shares the favoured warps of an SM finish early and
    // the rest crawl on alone -- 14.5 of 20 resident warps active on average); with a counter the
    // fast warps simply take more tiles and all end together.  (A single global counter serialises
    // in L2: 131 072 draws took 0.3 ms.)  Deterministic mode (P.partial != NULL) keeps static
    // round-robin shares, whose partial sums do not depend on timing.
    const bool dynamic = P.partial == nullptr;
    const long long n_mine = n_full > blockIdx.x ? (n_full - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;  // tiles of this block
    int n_drawn = 0;  // static schedule: tiles this warp has drawn so far
    constexpr long long kNoTile = 0x7fffffffffffffffLL;
    auto draw = [&]() -> long long {  // lane 0 only -> block-local tile index
        if (dynamic) return (long long)atomicAdd(&s_next, 1);
        return warp + (long long)(n_drawn++) * kSWarps;
    };
    auto tile_of = [&](long long k) { return (long long)blockIdx.x + k * (long long)gridDim.x; };
    long long t_a = kNoTile, t_b = kNoTile;
    if (lane == 0) {
        t_a = draw();
        if (t_a < n_mine) t_b = draw();
    }
    long long cur = __shfl_sync(0xffffffffu, t_a, 0);
    if (cur < n_mine && elect_one()) issue(tile_of(cur), 0);  // prologue: the first tile
    uint32_t parity = 0;  // bit s: parity the next wait on stage s expects
    int stage = 0;
    while (cur < n_mine) {
        // the other stage was read in the previous turn (its values are consumed): refill it with
        // the next tile, which then arrives under this turn's arithmetic
        __syncwarp();
        const int other = stage ^ 1;
        const long long nxt = __shfl_sync(0xffffffffu, t_b, 0);  // drawn one turn ago
        if (lane == 0) t_b = nxt < n_mine ? draw() : kNoTile;     // for the turn after the next
        if (nxt < n_mine && elect_one()) issue(tile_of(nxt), other);
        mbar_wait(&full[stage], (parity >> stage) & 1u);
        parity ^= 1u << stage;
        const unsigned char *src = ring + (size_t)stage * kSStageBytes + lane * 16;
        Vec16<ST> v[10];
#pragma unroll
        for (int a = 0; a < 10; ++a) v[a].v = *reinterpret_cast<const decltype(v[a].v) *>(src + a * kSArrayBytes);
#pragma unroll
        for (int pp = 0; pp < PPT; ++pp) {
            const Particle p = make_particle<ST, WIN>(v[0].get(pp), v[1].get(pp), v[2].get(pp), v[3].get(pp),
                                                      v[4].get(pp), v[5].get(pp), v[6].get(pp), v[7].get(pp),
                                                      v[8].get(pp), v[9].get(pp), P);
            accumulate_particle<NB, ND, WIN>(P, p, acc01, acc23);
        }
        cur = nxt;
        stage = other;
    }
    // ragged tail / unaligned arrays: plain coalesced loads, one particle per lane
    for (long long k = n_full * WTILE + gw * 32 + lane; k < N; k += GW * 32) {
        const Particle p = load_particle<ST, WIN>(P, k, true, WIN && P.F2);
        accumulate_particle<NB, ND, WIN>(P, p, acc01, acc23);
    }

    // a3: warp-shuffle reduction, cross-warp sum in shared memory, one fp64 add per value
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        float v4[4];
        unpack2(acc01[b], v4[0], v4[1]);
        unpack2(acc23[b], v4[2], v4[3]);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            float v = v4[c];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) s_red[warp][b * 4 + c] = v;
        }
    }
    __syncthreads();
    pdl_wait();  // the accumulator belongs to earlier work until here
    if (tid < NB * 4) {
        const int b = tid >> 2, c = tid & 3;
        const int d = b / WB, j = b - d * WB;
        if (d < P.n_dir && j < P.n_omega) {
            double v = 0.0;
#pragma unroll
            for (int wp = 0; wp < kSWarps; ++wp) v += (double)s_red[wp][tid];
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
    const size_t smem = (size_t)stream_warps(NB) * kSStages * kSStageBytes;
    // per device and per template instance; the call is a cheap host-side set, so no caching
    cudaError_t e = cudaFuncSetAttribute(rad_accum_stream<ST, NB, ND, WIN>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int use_bulk = 1;  // bulk copies need 16-byte aligned sources
    for (int a = 0; a < 10; ++a)
        if (reinterpret_cast<uintptr_t>(p.st[a]) & 15) use_bulk = 0;
    return launch_kernel(rad_accum_stream<ST, NB, ND, WIN>, dim3(grid), dim3(32 * stream_warps(NB)), smem, s, overlap, p, use_bulk);
}

template <typename ST, int NB, int ND>
cudaError_t launch_stream_t(const AccumParams &p, int grid, cudaStream_t s, bool overlap)
{
    return (p.win_type != RAD_WINDOW_NONE || p.F2) ? launch_stream_w<ST, NB, ND, true>(p, grid, s, overlap)
                                         : launch_stream_w<ST, NB, ND, false>(p, grid, s, overlap);
}

template <typename ST>
cudaError_t dispatch_stream(const Handle &h, const AccumParams &p, int grid, cudaStream_t s)
{
    if (h.stream_nb == 8) return h.stream_nd == 1 ? launch_stream_t<ST, 8, 1>(p, grid, s, h.overlap) : launch_stream_t<ST, 8, 2>(p, grid, s, h.overlap);
    return h.stream_nd == 1 ? launch_stream_t<ST, 16, 1>(p, grid, s, h.overlap) : launch_stream_t<ST, 16, 2>(p, grid, s, h.overlap);
}

}  // namespace

// particles per block per turn of the persistent loop (host side: grid sizing)
int stream_tile_particles(int nb, bool state_f64) { return stream_warps(nb) * 32 * (state_f64 ? 2 : 4); }
int stream_blocks_per_sm(int) { return 1; }

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
