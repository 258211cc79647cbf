// libile: device-resident stable LSD radix sort (see radix_sort.cuh).  Three kernels per 8-bit
// pass: per-block digit histogram into a [digit][block] table, an exclusive scan of every digit's row
// (one block per digit, row totals aside), and a stable scatter that ranks keys inside a warp with
// __match_any_sync and adds the scan of the 256 row totals itself.
#include "radix_sort.cuh"

__device__ __forceinline__ int rs_passes(int bits) { return bits <= 0 ? 0 : (bits + 7) >> 3; }

// which ping-pong buffer holds the data before pass p (inactive passes do not move it)
__device__ __forceinline__ int rs_src(int p, int npass) { return (p < npass ? p : npass) & 1; }

__global__ void __launch_bounds__(RS_THREADS) rs_hist_kernel(int p, const long long* __restrict__ n_dev, const int* __restrict__ bits_dev,
                                                             const uint64_t* __restrict__ k0, const uint64_t* __restrict__ k1,
                                                             uint32_t* __restrict__ hist, int max_blocks) {
    const int npass = rs_passes(*bits_dev);
    if (p >= npass) return;
    const long long n = *n_dev;
    const long long base = (long long)blockIdx.x * RS_TILE;
    if (base >= n) return;
    __shared__ uint32_t sh[256];
    sh[threadIdx.x] = 0;
    __syncthreads();
    const uint64_t* src = rs_src(p, npass) ? k1 : k0;
    const int shift = 8 * p;
    uint64_t keys[RS_TILE / RS_THREADS];
#pragma unroll
    for (int r = 0; r < RS_TILE / RS_THREADS; r++) {
        const long long i = base + r * RS_THREADS + threadIdx.x;
        keys[r] = i < n ? src[i] : 0ull;
    }
#pragma unroll
    for (int r = 0; r < RS_TILE / RS_THREADS; r++) {
        const bool act = base + r * RS_THREADS + threadIdx.x < n;
        const int dg = act ? (int)((keys[r] >> shift) & 0xffu) : 256;
        const unsigned m = __match_any_sync(0xffffffffu, dg);
        if (act && (threadIdx.x & 31) == __ffs(m) - 1) atomicAdd(&sh[dg], (uint32_t)__popc(m));
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * max_blocks + blockIdx.x] = sh[threadIdx.x];      // [digit][block]
}

// exclusive scan of digit blockIdx.x's counts over the blocks, in place; the row total goes to hist[256 max_blocks + digit]
__global__ void __launch_bounds__(256) rs_scan_kernel(int p, const long long* __restrict__ n_dev, const int* __restrict__ bits_dev,
                                                      uint32_t* __restrict__ hist, int max_blocks) {
    const int npass = rs_passes(*bits_dev);
    if (p >= npass) return;
    const long long n = *n_dev;
    const int nblocks = (int)((n + RS_TILE - 1) / RS_TILE);
    uint32_t* row = hist + (size_t)blockIdx.x * max_blocks;
    __shared__ uint32_t part[256];
    const int t = threadIdx.x;
    const int per = (nblocks + 255) >> 8;
    const int b0 = min(t * per, nblocks), b1 = min(b0 + per, nblocks);
    uint32_t s = 0;
    for (int b = b0; b < b1; b++) s += row[b];
    part[t] = s;
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {
        const uint32_t add = (t >= o) ? part[t - o] : 0;
        __syncthreads();
        part[t] += add;
        __syncthreads();
    }
    uint32_t run = part[t] - s;
    for (int b = b0; b < b1; b++) {
        const uint32_t c = row[b];
        row[b] = run;
        run += c;
    }
    if (t == 255) hist[(size_t)256 * max_blocks + blockIdx.x] = part[255];
}

template <bool HAS_VAL>
__global__ void __launch_bounds__(RS_THREADS) rs_scatter_kernel(int p, const long long* __restrict__ n_dev, const int* __restrict__ bits_dev,
                                                                uint64_t* __restrict__ k0, uint32_t* __restrict__ v0,
                                                                uint64_t* __restrict__ k1, uint32_t* __restrict__ v1,
                                                                const uint32_t* __restrict__ hist, int max_blocks) {
    const int npass = rs_passes(*bits_dev);
    if (p >= npass) return;
    const long long n = *n_dev;
    const long long base = (long long)blockIdx.x * RS_TILE;
    if (base >= n) return;
    __shared__ uint32_t wh[RS_THREADS / 32][257];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int q = threadIdx.x; q < (RS_THREADS / 32) * 257; q += RS_THREADS) (&wh[0][0])[q] = 0;
    __syncthreads();
    const bool s = rs_src(p, npass);
    const uint64_t* ksrc = s ? k1 : k0;
    uint64_t* kdst = s ? k0 : k1;
    const uint32_t* vsrc = s ? v1 : v0;
    uint32_t* vdst = s ? v0 : v1;
    const int shift = 8 * p;
    constexpr int ROUNDS = RS_TILE / RS_THREADS;      // rounds per warp; warp w owns keys [w*ROUNDS*32, ...)
    const long long wbase = base + (long long)w * ROUNDS * 32;
    // the warp's keys (and payloads) are read once, all loads in flight together, and stay in registers for both phases
    uint64_t keys[ROUNDS];
    uint32_t vals[ROUNDS];
#pragma unroll
    for (int r = 0; r < ROUNDS; r++) {
        const long long i = wbase + r * 32 + lane;
        keys[r] = i < n ? ksrc[i] : 0ull;
        if (HAS_VAL) vals[r] = i < n ? vsrc[i] : 0u;
    }
    // phase A: per-warp digit counts
#pragma unroll
    for (int r = 0; r < ROUNDS; r++) {
        const bool act = wbase + r * 32 + lane < n;
        const int dg = act ? (int)((keys[r] >> shift) & 0xffu) : 256;
        const unsigned m = __match_any_sync(0xffffffffu, dg);
        if (lane == __ffs(m) - 1) wh[w][dg] += (uint32_t)__popc(m);
        __syncwarp();
    }
    __syncthreads();
    // phase B: turn the counts into start offsets (digits below + this digit in earlier blocks + earlier warps)
    {
        __shared__ uint32_t dsum[256];
        const int dg = threadIdx.x;
        const uint32_t tot = hist[(size_t)256 * max_blocks + dg];
        dsum[dg] = tot;
        __syncthreads();
        for (int o = 1; o < 256; o <<= 1) {
            const uint32_t add = (dg >= o) ? dsum[dg - o] : 0;
            __syncthreads();
            dsum[dg] += add;
            __syncthreads();
        }
        uint32_t run = dsum[dg] - tot + hist[(size_t)dg * max_blocks + blockIdx.x];
        for (int ww = 0; ww < RS_THREADS / 32; ww++) {
            uint32_t c = wh[ww][dg];
            wh[ww][dg] = run;
            run += c;
        }
    }
    __syncthreads();
    // phase C: stable rank and scatter
#pragma unroll
    for (int r = 0; r < ROUNDS; r++) {
        const bool act = wbase + r * 32 + lane < n;
        const uint64_t key = keys[r];
        const int dg = act ? (int)((key >> shift) & 0xffu) : 256;
        const unsigned m = __match_any_sync(0xffffffffu, dg);
        const uint32_t pos = wh[w][dg] + (uint32_t)__popc(m & ((1u << lane) - 1u));
        __syncwarp();
        if (lane == __ffs(m) - 1) wh[w][dg] += (uint32_t)__popc(m);
        __syncwarp();
        if (act) {
            kdst[pos] = key;
            if (HAS_VAL) vdst[pos] = vals[r];
        }
    }
}

// result is in buffer (npass & 1): copy back into (k0, v0) when that is buffer 1
template <bool HAS_VAL>
__global__ void rs_finish_kernel(const long long* __restrict__ n_dev, const int* __restrict__ bits_dev, uint64_t* __restrict__ k0,
                                 uint32_t* __restrict__ v0, const uint64_t* __restrict__ k1, const uint32_t* __restrict__ v1, int max_passes) {
    int npass = rs_passes(*bits_dev);
    if (npass > max_passes) npass = max_passes;
    if (!(npass & 1)) return;
    const long long n = *n_dev;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        k0[i] = k1[i];
        if (HAS_VAL) v0[i] = v1[i];
    }
}

size_t radix_sort_scratch_bytes(int max_n) {
    size_t blocks = ((size_t)max_n + RS_TILE - 1) / RS_TILE;
    if (blocks < 1) blocks = 1;
    return (256 * blocks + 256) * sizeof(uint32_t);
}

int radix_sort_device(ile_ctx* ctx, int max_n, const long long* n_dev, const int* bits_dev, uint64_t* k0, uint32_t* v0, uint64_t* k1,
                      uint32_t* v1, void* scratch, int max_passes) {
    if (max_n < 1) return ILE_OK;
    if (max_passes > RS_MAX_PASSES) max_passes = RS_MAX_PASSES;
    const int blocks = (max_n + RS_TILE - 1) / RS_TILE;
    uint32_t* hist = (uint32_t*)scratch;
    const bool has_val = v0 != nullptr;
    for (int p = 0; p < max_passes; p++) {
        rs_hist_kernel<<<blocks, RS_THREADS, 0, ctx->stream>>>(p, n_dev, bits_dev, k0, k1, hist, blocks);
        ILE_LAUNCH_CHECK(ctx);
        rs_scan_kernel<<<256, 256, 0, ctx->stream>>>(p, n_dev, bits_dev, hist, blocks);
        ILE_LAUNCH_CHECK(ctx);
        if (has_val) rs_scatter_kernel<true><<<blocks, RS_THREADS, 0, ctx->stream>>>(p, n_dev, bits_dev, k0, v0, k1, v1, hist, blocks);
        else rs_scatter_kernel<false><<<blocks, RS_THREADS, 0, ctx->stream>>>(p, n_dev, bits_dev, k0, v0, k1, v1, hist, blocks);
        ILE_LAUNCH_CHECK(ctx);
    }
    int g = blocks < ctx->sm_count * 4 ? blocks : ctx->sm_count * 4;
    if (has_val) rs_finish_kernel<true><<<g, 256, 0, ctx->stream>>>(n_dev, bits_dev, k0, v0, k1, v1, max_passes);
    else rs_finish_kernel<false><<<g, 256, 0, ctx->stream>>>(n_dev, bits_dev, k0, v0, k1, v1, max_passes);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}
