// rad_ubench.cu -- pipe microbenchmarks behind the ALU rooflines of bench.py (SURVEY.md section 7
// step 4, section 8(d): "microbenchmark all three pipes on the box").  Built as its own small
// library, librad_ubench.so; NOT part of librad.so or of the ABI in include/rad.h.
//
// Every kind runs 8 independent dependency chains per thread (dependent-free at the warp level
// once >= 4 warps per scheduler are resident), ITERS x 8 operations per thread, and reports
//   per_clk_sm = thread-level results per SM clock per SM, from clock64() inside the kernel
//                (independent of the clock frequency): per SM, the results of all warps that ran
//                there / (latest end - earliest start over those warps), averaged over the SMs
//                (a single warp's own duration would overstate the rate: the warp scheduler is
//                not fair, early warps finish while late ones are still running), and
//   gops       = 1e-9 x thread-level results per second of the whole GPU, from CUDA events.
// The roofline denominators derived from them:
//   general grid   R_gen = sincos pairs/clk/SM (kind SINCOS) x SMs x clock      [nominal 8]
//   uniform grid   R_lin = FFMA/clk/SM (kind FFMA) / 8 x SMs x clock            [nominal 16]
// Kinds FFMA / FFMA2 keep two of their three operands loop-invariant (operand-reuse cache hits);
// FFMA_VAR / FFMA2_VAR / FFMA2_BCAST read three DIFFERENT, changing registers per instruction and
// measure what the register file feeds the FMA pipe without reuse (about 2 register reads per lane
// per clock: 75 FFMA, 85 packed FMA per clock per SM) -- the regime of the uniform-grid sweep, whose
// rotations and accumulates have few repeated operands.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int kIters = 2048;
constexpr int kChains = 8;
constexpr int kThreads = 256;
constexpr int kMaxSmid = 1024;  // %smid values are not guaranteed contiguous: generous table

enum Kind {
    K_FFMA = 0,      // fma.rn.f32, three register operands
    K_FFMA_IMM = 1,  // fma.rn.f32 with immediate multiplier/addend
    K_FFMA2 = 2,     // fma.rn.f32x2 (two FMAs per instruction): counts INSTRUCTIONS
    K_MUFU_SIN = 3,  // sin.approx.ftz.f32 = FMUL.RZ + MUFU.SIN
    K_SINCOS = 4,    // sin + cos of the same argument (FMUL.RZ, two MUFU, one FADD): counts PAIRS
    K_MUFU_EX2 = 5,  // ex2.approx.ftz.f32 = MUFU.EX2 alone
    K_DFMA = 6,      // fma.rn.f64
    K_F2F_64_32 = 7, // cvt.rn.f32.f64 (+ FADD + DADD to keep the chain alive)
    K_F2F_32_64 = 8, // cvt.f64.f32 (+ DADD)
    K_IMAD = 9,      // mad.lo.u32
    K_FFMA2_VAR = 10,   // fma.rn.f32x2 whose three operands are all different, changing registers: INSTRUCTIONS
    K_FFMA2_BCAST = 11, // fma.rn.f32x2 with one operand a broadcast scalar (SASS Rn.F32), as the uniform-grid sweep issues it
    K_FFMA_VAR = 12,    // fma.rn.f32 whose three operands are all different, changing registers
    K_RED_V4 = 13,      // red.global.add.v4.f32 (16-byte vector reduction), runs of 4 consecutive chunks at scattered places of a 64 MB, L2-resident
                        // buffer: the rate at which L2 takes the reductions of the fast gridded path's spreading kernel
    K_COUNT = 14
};

template <int KIND>
__global__ void __launch_bounds__(kThreads) pipe_kernel(float *out, float a, float b, long long *clk)
{
    // clk: [3][kMaxSmid] = earliest start, latest end, number of warps, per SM (%smid)
    float x[kChains];
    unsigned long long y[kChains];
    double z[kChains];
    unsigned w[kChains];
    float c[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) {
        x[i] = threadIdx.x * 1e-3f + i;
        y[i] = ((unsigned long long)__float_as_uint(x[i]) << 32) | __float_as_uint(x[i] + 1.0f);
        z[i] = x[i];
        w[i] = threadIdx.x + i;
        c[i] = 0.0f;
    }
    const unsigned long long a2 = ((unsigned long long)__float_as_uint(a) << 32) | __float_as_uint(a);
    const unsigned long long b2 = ((unsigned long long)__float_as_uint(b) << 32) | __float_as_uint(b);
    const long long t0 = clock64();
    // unrolled 4x: with one 8-operation pass per trip the loop's own IADD3 / ISETP / BRA take 3 of 11 issue
    // slots and cap every one-instruction kind at 93 per clock per SM (round-2 figures: FFMA 85.8)
#pragma unroll 4
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < kChains; ++i) {
            if (KIND == K_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
            if (KIND == K_FFMA_IMM) x[i] = fmaf(x[i], 1.0001f, 0.5f);
            if (KIND == K_FFMA2) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(y[i]) : "l"(a2), "l"(b2));
            if (KIND == K_MUFU_SIN) asm volatile("sin.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
            if (KIND == K_SINCOS) {
                float s, k;
                __sincosf(x[i], &s, &k);
                x[i] = s;
                c[i] += k;  // the cosine is consumed every iteration (one FADD on the FMA pipe)
            }
            if (KIND == K_MUFU_EX2) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
            if (KIND == K_DFMA) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(z[i]) : "d"(1.0000001), "d"(0.5));
            if (KIND == K_F2F_64_32) {
                float f;
                asm volatile("cvt.rn.f32.f64 %0, %1;" : "=f"(f) : "d"(z[i]));
                x[i] += f;
                z[i] += 1.0;
            }
            if (KIND == K_F2F_32_64) {
                double d;
                asm volatile("cvt.f64.f32 %0, %1;" : "=d"(d) : "f"(x[i]));
                z[i] += d;
            }
            if (KIND == K_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(w[i]) : "r"(__float_as_uint(a)), "r"(__float_as_uint(b)));
            if (KIND == K_FFMA2_VAR)
                asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(y[i]) : "l"(y[(i + 3) & 7]), "l"(y[(i + 5) & 7]));
            if (KIND == K_FFMA2_BCAST) {
                unsigned long long bc;
                asm volatile("mov.b64 %0, {%1, %1};" : "=l"(bc) : "f"(x[(i + 1) & 7]));
                asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(y[i]) : "l"(bc), "l"(y[(i + 5) & 7]));
            }
            if (KIND == K_FFMA_VAR)
                asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(x[i]) : "f"(x[(i + 3) & 7]), "f"(x[(i + 5) & 7]));
        }
    }
    const long long t1 = clock64();
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += x[i] + c[i] + (float)(y[i] >> 32) + (float)z[i] + (float)w[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
    if ((threadIdx.x & 31) == 0) {
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        if (smid < kMaxSmid) {
            atomicMin(clk + smid, t0);
            atomicMax(clk + kMaxSmid + smid, t1);
            atomicAdd(reinterpret_cast<unsigned long long *>(clk + 2 * kMaxSmid + smid), 1ull);
        }
    }
}

// 16-byte vector reductions to pseudo-random 16-byte-aligned places of buf[n_chunks] (n_chunks a power of two)
__global__ void __launch_bounds__(kThreads) red_kernel(float4 *buf, unsigned n_mask, long long *clk)
{
    unsigned x = (blockIdx.x * kThreads + threadIdx.x) * 2654435761u + 12345u;
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters / 4; ++it) {
#pragma unroll
        for (int i = 0; i < kChains; i += 4) {  // runs of four consecutive chunks from a random chunk, as the spreading kernel issues them
            x = x * 1664525u + 1013904223u;
            float4 *q = buf + ((x >> 7) & n_mask);
#pragma unroll
            for (int c = 0; c < 4; ++c)
                asm volatile("red.global.v4.f32.add [%0], {%1, %1, %1, %1};" ::"l"(q + c), "f"(1.0f) : "memory");
        }
    }
    const long long t1 = clock64();
    if ((threadIdx.x & 31) == 0) {
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        if (smid < kMaxSmid) {
            atomicMin(clk + smid, t0);
            atomicMax(clk + kMaxSmid + smid, t1);
            atomicAdd(reinterpret_cast<unsigned long long *>(clk + 2 * kMaxSmid + smid), 1ull);
        }
    }
}

template <int KIND>
int run_kind(int n_sm, int blocks_per_sm, int reps, double *per_clk_sm, double *gops)
{
    const int grid = n_sm * blocks_per_sm;
    float *out = nullptr;
    long long *clk = nullptr;
    constexpr unsigned kRedChunks = 1u << 22;  // x 16 B = 64 MB
    const int iters = KIND == K_RED_V4 ? kIters / 4 : kIters;
    if (cudaMalloc(&out, KIND == K_RED_V4 ? (size_t)(kRedChunks + 4) * 16 : (size_t)grid * kThreads * sizeof(float)) != cudaSuccess) return 1;
    if (KIND == K_RED_V4) cudaMemset(out, 0, (size_t)kRedChunks * 16);
    auto launch = [&]() {
        if (KIND == K_RED_V4) red_kernel<<<grid, kThreads>>>(reinterpret_cast<float4 *>(out), kRedChunks - 1, clk);
        else pipe_kernel<KIND><<<grid, kThreads>>>(out, 1.0001f, 0.5f, clk);
    };
    const size_t clk_bytes = (size_t)3 * kMaxSmid * sizeof(long long);
    if (cudaMalloc(&clk, clk_bytes) != cudaSuccess) { cudaFree(out); return 1; }
    long long *h = new long long[3 * kMaxSmid];
    auto reset_clk = [&]() {
        for (int i = 0; i < kMaxSmid; ++i) { h[i] = 0x7fffffffffffffffLL; h[kMaxSmid + i] = 0; h[2 * kMaxSmid + i] = 0; }
        cudaMemcpy(clk, h, clk_bytes, cudaMemcpyHostToDevice);
    };
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    reset_clk();
    for (int r = 0; r < 2; ++r) launch();  // warm-up
    cudaDeviceSynchronize();
    reset_clk();
    launch();  // the launch the per-SM cycle windows are read from
    int rc = cudaDeviceSynchronize() == cudaSuccess ? 0 : 2;
    if (cudaMemcpy(h, clk, clk_bytes, cudaMemcpyDeviceToHost) != cudaSuccess) rc = 2;
    cudaEventRecord(e0);
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(e1);
    if (cudaDeviceSynchronize() != cudaSuccess) rc = 2;
    float ms = 0.0f;
    cudaEventElapsedTime(&ms, e0, e1);
    double rate = 0.0;
    int used = 0;
    for (int i = 0; i < kMaxSmid; ++i) {
        const double warps = (double)h[2 * kMaxSmid + i], cyc = (double)(h[kMaxSmid + i] - h[i]);
        if (warps > 0.0 && cyc > 0.0) { rate += warps * 32.0 * iters * kChains / cyc; ++used; }
    }
    delete[] h;
    const double ops_per_sm = (double)iters * kChains * kThreads * blocks_per_sm;  // thread-level results
    *per_clk_sm = used ? rate / used : 0.0;
    *gops = ms > 0.0f ? ops_per_sm * n_sm * reps / (ms * 1e-3) / 1e9 : 0.0;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    cudaFree(clk);
    return rc;
}

}  // namespace

extern "C" {

// Number of kinds and their names (static storage).
__attribute__((visibility("default"))) int rad_ubench_kinds(void) { return K_COUNT; }

__attribute__((visibility("default"))) const char *rad_ubench_name(int kind)
{
    static const char *names[K_COUNT] = {"ffma", "ffma_imm", "ffma2_instr", "mufu_sin", "sincos_pairs",
                                         "mufu_ex2", "dfma", "f2f_f32_from_f64", "f2f_f64_from_f32", "imad",
                                         "ffma2_var_instr", "ffma2_bcast_instr", "ffma_var", "red_v4_f32"};
    return kind >= 0 && kind < K_COUNT ? names[kind] : "?";
}

// Runs one kind on `device` with blocks_per_sm resident 256-thread blocks per SM, `reps` timed
// launches.  HOST outputs: per_clk_sm (from clock64) and gops (from CUDA events).
// Returns 0, 1 (bad argument / allocation) or 2 (CUDA error).
__attribute__((visibility("default"))) int rad_ubench_run(int device, int kind, int blocks_per_sm, int reps,
                                                          double *per_clk_sm, double *gops)
{
    if (!per_clk_sm || !gops || blocks_per_sm < 1 || blocks_per_sm > 8 || reps < 1) return 1;
    if (cudaSetDevice(device) != cudaSuccess) return 2;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return 2;
    const int n_sm = prop.multiProcessorCount;
    switch (kind) {
        case K_FFMA: return run_kind<K_FFMA>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_FFMA_IMM: return run_kind<K_FFMA_IMM>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_FFMA2: return run_kind<K_FFMA2>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_MUFU_SIN: return run_kind<K_MUFU_SIN>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_SINCOS: return run_kind<K_SINCOS>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_MUFU_EX2: return run_kind<K_MUFU_EX2>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_DFMA: return run_kind<K_DFMA>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_F2F_64_32: return run_kind<K_F2F_64_32>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_F2F_32_64: return run_kind<K_F2F_32_64>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_IMAD: return run_kind<K_IMAD>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_FFMA2_VAR: return run_kind<K_FFMA2_VAR>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_FFMA2_BCAST: return run_kind<K_FFMA2_BCAST>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_FFMA_VAR: return run_kind<K_FFMA_VAR>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
        case K_RED_V4: return run_kind<K_RED_V4>(n_sm, blocks_per_sm, reps, per_clk_sm, gops);
    }
    return 1;
}

}  // extern "C"
