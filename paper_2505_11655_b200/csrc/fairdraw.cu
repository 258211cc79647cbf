// libile: fair draws from weighted samples (reading G39).
// Fixed-point weights q_i = qfix(ln w_i - max) (the integrators' uint64 weights), exact inclusive
// prefix sums (three-kernel scan), M positions (systematic: one uniform; independent: one uniform
// per draw, Philox counter (j, iter)), binary search.  Compiled with -fmad=false: bit-exact.
#include "integ.cuh"

#define FD_TILE 2048
#define FD_THREADS 256

__global__ void __launch_bounds__(256) fd_max_kernel(int N, const double* __restrict__ lnw, unsigned long long* m_ord) {
    unsigned long long mx = 0ull;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const double w = lnw[i];
        if (is_finite_d(w)) {
            const unsigned long long o = ord_from_double(w);
            mx = o > mx ? o : mx;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long v = __shfl_xor_sync(0xffffffffu, mx, o);
        mx = v > mx ? v : mx;
    }
    if ((threadIdx.x & 31) == 0 && mx) atomicMax(m_ord, mx);
}

__device__ __forceinline__ unsigned long long fd_q(const double* __restrict__ lnw, long long i, int N, double m, bool any) {
    if (i >= N || !any) return 0ull;
    const double w = lnw[i];
    return is_finite_d(w) ? qfix_dev(__dsub_rn(w, m)) : 0ull;
}

// block b sums its tile of q
__global__ void __launch_bounds__(FD_THREADS) fd_blocksum_kernel(int N, const double* __restrict__ lnw, const unsigned long long* __restrict__ m_ord,
                                                                 unsigned long long* __restrict__ blk) {
    const bool any = *m_ord != 0ull;
    const double m = double_from_ord(*m_ord);
    const long long base = (long long)blockIdx.x * FD_TILE;
    unsigned long long s = 0;
    for (int r = 0; r < FD_TILE / FD_THREADS; r++) s += fd_q(lnw, base + r * FD_THREADS + threadIdx.x, N, m, any);
    __shared__ unsigned long long sh[FD_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int w = 0; w < FD_THREADS / 32; w++) t += sh[w];
        blk[blockIdx.x] = t;
    }
}

// exclusive scan of the block sums (one block); total -> blk[nblocks]
__global__ void __launch_bounds__(1024) fd_scan_kernel(int nblocks, unsigned long long* __restrict__ blk) {
    __shared__ unsigned long long part[1024];
    const int t = threadIdx.x;
    const int per = (nblocks + 1023) / 1024;
    const int b0 = min(t * per, nblocks), b1 = min(b0 + per, nblocks);
    unsigned long long s = 0;
    for (int b = b0; b < b1; b++) s += blk[b];
    part[t] = s;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
        const unsigned long long add = t >= o ? part[t - o] : 0ull;
        __syncthreads();
        part[t] += add;
        __syncthreads();
    }
    unsigned long long run = part[t] - s;
    for (int b = b0; b < b1; b++) {
        const unsigned long long c = blk[b];
        blk[b] = run;
        run += c;
    }
    if (t == 1023) blk[nblocks] = part[1023];
}

// inclusive prefix sums S[i]; thread t owns FD_TILE / FD_THREADS consecutive samples
__global__ void __launch_bounds__(FD_THREADS) fd_prefix_kernel(int N, const double* __restrict__ lnw, const unsigned long long* __restrict__ m_ord,
                                                               const unsigned long long* __restrict__ blk, unsigned long long* __restrict__ S) {
    const bool any = *m_ord != 0ull;
    const double m = double_from_ord(*m_ord);
    constexpr int PER = FD_TILE / FD_THREADS;
    const long long i0 = (long long)blockIdx.x * FD_TILE + (long long)threadIdx.x * PER;
    unsigned long long q[PER], s = 0;
#pragma unroll
    for (int r = 0; r < PER; r++) { q[r] = fd_q(lnw, i0 + r, N, m, any); s += q[r]; }
    __shared__ unsigned long long sc[FD_THREADS];
    sc[threadIdx.x] = s;
    __syncthreads();
    for (int o = 1; o < FD_THREADS; o <<= 1) {
        const unsigned long long add = threadIdx.x >= o ? sc[threadIdx.x - o] : 0ull;
        __syncthreads();
        sc[threadIdx.x] += add;
        __syncthreads();
    }
    unsigned long long run = blk[blockIdx.x] + sc[threadIdx.x] - s;
#pragma unroll
    for (int r = 0; r < PER; r++) {
        run += q[r];
        if (i0 + r < N) S[i0 + r] = run;
    }
}

__global__ void __launch_bounds__(256) fd_draw_kernel(int N, int M, unsigned long long seed, unsigned int iter, int mode,
                                                      const unsigned long long* __restrict__ S, const unsigned long long* __restrict__ total,
                                                      long long* __restrict__ idx) {
    const long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (j >= M) return;
    const unsigned long long T = *total;
    if (T == 0ull) {
        idx[j] = -1;
        return;
    }
    double ua, ub, pos;
    if (mode == 0) {                                   // systematic: one uniform, equally spaced positions
        philox_pair(seed, 0ull, iter, 0u, &ua, &ub);
        pos = __ddiv_rn(__dadd_rn((double)j, ua), (double)M);
    } else {                                           // independent draws
        philox_pair(seed, (unsigned long long)j, iter, 0u, &ua, &ub);
        pos = ua;
    }
    unsigned long long r = (unsigned long long)floor(__dmul_rn(pos, __ull2double_rn(T)));
    if (r > T - 1) r = T - 1;
    long long lo = 0, hi = N;                          // first i with S[i] > r
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (S[mid] > r) hi = mid; else lo = mid + 1;
    }
    idx[j] = lo;
}

// M fair draws (with replacement, probability proportional to w) from N log-weights: device
// pointers lnw [N], idx [M] (int64; -1 everywhere when no sample has positive weight).
// mode 0 = systematic resampling, 1 = independent draws.  Asynchronous on the context's stream.
extern "C" int ile_fair_draw(ile_ctx* ctx, int N, const double* lnw, int M, uint64_t seed, uint64_t iter, int mode, int64_t* idx) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (N < 1 || M < 1 || !lnw || !idx || mode < 0 || mode > 1) return ile_fail(ctx, ILE_EINVAL, "fair_draw: bad argument");
    const int nblocks = (N + FD_TILE - 1) / FD_TILE;
    void* scratch = nullptr;
    int rc = ile_scratch(ctx, (size_t)N * 8 + ((size_t)nblocks + 2) * 8 + 256, &scratch);
    if (rc) return rc;
    unsigned long long* S = (unsigned long long*)scratch;
    unsigned long long* blk = S + N;
    unsigned long long* m_ord = blk + nblocks + 1;
    ILE_CUDA(ctx, cudaMemsetAsync(m_ord, 0, 8, ctx->stream));
    int g = ctx->sm_count * 4 < (N + 255) / 256 ? ctx->sm_count * 4 : (N + 255) / 256;
    fd_max_kernel<<<g, 256, 0, ctx->stream>>>(N, lnw, m_ord);
    ILE_LAUNCH_CHECK(ctx);
    fd_blocksum_kernel<<<nblocks, FD_THREADS, 0, ctx->stream>>>(N, lnw, m_ord, blk);
    ILE_LAUNCH_CHECK(ctx);
    fd_scan_kernel<<<1, 1024, 0, ctx->stream>>>(nblocks, blk);
    ILE_LAUNCH_CHECK(ctx);
    fd_prefix_kernel<<<nblocks, FD_THREADS, 0, ctx->stream>>>(N, lnw, m_ord, blk, S);
    ILE_LAUNCH_CHECK(ctx);
    fd_draw_kernel<<<(M + 255) / 256, 256, 0, ctx->stream>>>(N, M, seed, (unsigned int)iter, mode, S, blk + nblocks, (long long*)idx);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}
