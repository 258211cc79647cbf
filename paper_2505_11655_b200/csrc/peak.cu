// libile: FP64 peak probes ("the build must measure the real FP64 FMA peak with a
// register-resident FMA-chain micro-benchmark").  Two kernels with no memory traffic: independent
// DFMA chains on the FP64 ALUs, and independent DMMA.8x8x4 chains on the FP64 tensor pipe.  The
// roofline of the fused lnL kernel is quoted against the larger of the two measured rates.
#include "common.cuh"

#define PK_CHAINS 8

__global__ void __launch_bounds__(256) dfma_chain_kernel(int iters, double seed, double* out) {
    double a[PK_CHAINS];
#pragma unroll
    for (int c = 0; c < PK_CHAINS; c++) a[c] = seed + c + threadIdx.x * 1e-9;
    const double m = 1.0 - 1e-9, b = 1e-9;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int r = 0; r < 8; r++)
#pragma unroll
            for (int c = 0; c < PK_CHAINS; c++) a[c] = fma(a[c], m, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < PK_CHAINS; c++) s += a[c];
    if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chain live
}

__global__ void __launch_bounds__(256) dmma_chain_kernel(int iters, double seed, double* out) {
    double d0[PK_CHAINS], d1[PK_CHAINS];
#pragma unroll
    for (int c = 0; c < PK_CHAINS; c++) { d0[c] = seed + c; d1[c] = seed - c; }
    const double a = 1e-9 * (threadIdx.x & 3), b = 1.0 + 1e-9 * (threadIdx.x >> 2);
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int c = 0; c < PK_CHAINS; c++)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(d0[c]), "+d"(d1[c]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < PK_CHAINS; c++) s += d0[c] + d1[c];
    if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// mode 0: DFMA chains (2 flop per thread-instruction); mode 1: DMMA m8n8k4 (512 flop per warp-
// instruction).  Runs on the context's stream, synchronises, returns TFLOP/s of the best of 3 runs.
extern "C" int ile_fp64_peak(ile_ctx* ctx, int mode, double* tflops) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (!tflops || mode < 0 || mode > 1) return ile_fail(ctx, ILE_EINVAL, "fp64_peak: mode 0 (DFMA) or 1 (DMMA)");
    const int blocks = ctx->sm_count * 8, threads = 256, iters = mode == 0 ? 4096 : 2048;
    void* scratch = nullptr;
    int rc = ile_scratch(ctx, (size_t)blocks * threads * 8, &scratch);
    if (rc) return rc;
    cudaEvent_t e0, e1;
    ILE_CUDA(ctx, cudaEventCreate(&e0));
    ILE_CUDA(ctx, cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 4; rep++) {
        ILE_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        if (mode == 0) dfma_chain_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, 1.0, (double*)scratch);
        else dmma_chain_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, 1.0, (double*)scratch);
        ILE_LAUNCH_CHECK(ctx);
        ILE_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
        ILE_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        ILE_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        const double flop = mode == 0 ? (double)blocks * threads * iters * 8.0 * PK_CHAINS * 2.0
                                      : (double)blocks * (threads / 32) * iters * 4.0 * PK_CHAINS * 512.0;
        const double tf = flop / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tflops = best;
    return ILE_OK;
}

// ---------------------------------------------------------------- int8 tensor-path probe (tcgen05.mma kind::i8)
// The MMA schedule of the fused lnL kernel (lnl_split.cu) with nothing around it: per round 33 MMAs of 128 x 32 x 32,
// A from tensor memory, B from shared memory (no-swizzle K-major descriptors), six accumulators, issued either k-step major
// (the kernel's order: consecutive MMAs go to different accumulators) or sum major (dependent chains back to back).
// Operands are whatever the memories hold: the rate does not depend on the values.  One CTA per SM.
#include "sm100_ptx.cuh"

__global__ void __launch_bounds__(64, 1) int8_mma_probe_kernel(int rounds, int sum_major) {
    extern __shared__ __align__(1024) unsigned char probe_smem[];
    __shared__ uint64_t bar;
    __shared__ uint32_t tbase;
    const int w = threadIdx.x >> 5;
    if (w == 0) tmem_alloc512(&tbase);
    if (threadIdx.x == 32) {
        mbar_init(&bar, 1);
        mbar_init_fence();
    }
    for (int q = threadIdx.x; q < 4 * 2432 / 16; q += blockDim.x) reinterpret_cast<int4*>(probe_smem)[q] = make_int4(q, q * 3, q * 5, q * 7);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tbase;
    if (w == 1) {
        const bool el = elect_one();
        const uint32_t idesc = umma_idesc_s8_m128(32);
        const uint64_t b0 = umma_desc_kmajor_noswizzle(smem_u32(probe_smem), 128, 2432);
        for (int r = 0; r < rounds; r++) {
            if (el) {
                if (!sum_major) {
#pragma unroll
                    for (int t = 0; t < 9; t++)
#pragma unroll
                        for (int s = 0; s < 6; s++) {
                            const int Ks = s == 0 ? 64 : s == 1 ? 96 : s == 2 ? 160 : s == 3 ? 192 : s == 4 ? 256 : 288;
                            if (32 * t < Ks) umma_i8_ts(tmem + 256 + 32 * s, tmem + 8 * t, b0 + (uint64_t)(((3 * (5 - s) + 2 * t) * 128) >> 4), idesc, t > 0 ? 1u : 0u);
                        }
                } else {
#pragma unroll
                    for (int s = 0; s < 6; s++)
#pragma unroll
                        for (int t = 0; t < 9; t++) {
                            const int Ks = s == 0 ? 64 : s == 1 ? 96 : s == 2 ? 160 : s == 3 ? 192 : s == 4 ? 256 : 288;
                            if (32 * t < Ks) umma_i8_ts(tmem + 256 + 32 * s, tmem + 8 * t, b0 + (uint64_t)(((3 * (5 - s) + 2 * t) * 128) >> 4), idesc, t > 0 ? 1u : 0u);
                        }
                }
            }
            __syncwarp();
        }
        if (el) umma_commit(&bar);
        mbar_wait(&bar, 0);
    }
    tc_fence_before();
    __syncthreads();
    if (w == 0) tmem_free512(tmem);
}

// mode 0: k-step-major issue (the fused kernel's), 1: sum-major.  *tops (host) = int8 multiply-adds x 2 per second of the whole
// GPU, best of three; synchronises.
extern "C" int ile_int8_mma_peak(ile_ctx* ctx, int mode, double* tops) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);
    if (!tops || mode < 0 || mode > 1) return ile_fail(ctx, ILE_EINVAL, "int8_mma_peak: mode 0 (k-step major) or 1 (sum major)");
    const int rounds = 2000, smem = 4 * 2432 + 1024;
    cudaEvent_t e0, e1;
    ILE_CUDA(ctx, cudaEventCreate(&e0));
    ILE_CUDA(ctx, cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 4; rep++) {
        ILE_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        int8_mma_probe_kernel<<<ctx->sm_count, 64, smem, ctx->stream>>>(rounds, mode);
        ILE_LAUNCH_CHECK(ctx);
        ILE_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
        ILE_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        ILE_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        const double ops = (double)ctx->sm_count * rounds * 33.0 * 128.0 * 32.0 * 32.0 * 2.0;
        const double t = ops / (ms * 1e-3) / 1e12;
        if (rep > 0 && t > best) best = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tops = best;
    return ILE_OK;
}
