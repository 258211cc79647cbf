// libile: step 7, Monte Carlo weight reduction (Eq. 8, 9, 14-16): ln I, variance, n_eff, n_ESS.
// Two kernels: per-block online log-sum-exp partials (warp shuffle -> block), then one block that
// combines the partials and writes the ile_result (and folds it into the cumulative estimate).
#include "common.cuh"

struct RedPart {
    double m, s1, s2;
    unsigned long long bad;
};

__device__ __forceinline__ void lse_merge(double& m, double& s1, double& s2, double m2, double a1, double a2) {
    if (m2 == neg_inf()) return;
    if (m == neg_inf()) { m = m2; s1 = a1; s2 = a2; return; }
    if (m2 > m) {
        double e = exp(m - m2);
        s1 = s1 * e + a1;
        s2 = s2 * e * e + a2;
        m = m2;
    } else {
        double e = exp(m2 - m);
        s1 += a1 * e;
        s2 += a2 * e * e;
    }
}

__device__ __forceinline__ void block_lse(double& m, double& s1, double& s2, unsigned long long& bad, RedPart* sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        double m2 = __shfl_xor_sync(0xffffffffu, m, o), a1 = __shfl_xor_sync(0xffffffffu, s1, o), a2 = __shfl_xor_sync(0xffffffffu, s2, o);
        bad += __shfl_xor_sync(0xffffffffu, bad, o);
        lse_merge(m, s1, s2, m2, a1, a2);
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if (lane == 0) { sh[w].m = m; sh[w].s1 = s1; sh[w].s2 = s2; sh[w].bad = bad; }
    __syncthreads();
    if (w == 0) {
        m = lane < nw ? sh[lane].m : neg_inf();
        s1 = lane < nw ? sh[lane].s1 : 0.0;
        s2 = lane < nw ? sh[lane].s2 : 0.0;
        bad = lane < nw ? sh[lane].bad : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            double m2 = __shfl_xor_sync(0xffffffffu, m, o), a1 = __shfl_xor_sync(0xffffffffu, s1, o), a2 = __shfl_xor_sync(0xffffffffu, s2, o);
            bad += __shfl_xor_sync(0xffffffffu, bad, o);
            lse_merge(m, s1, s2, m2, a1, a2);
        }
    }
}

__global__ void __launch_bounds__(256) reduce_partial_kernel(int N, const double* __restrict__ lnw, RedPart* __restrict__ part) {
    __shared__ RedPart sh[8];
    double m = neg_inf(), s1 = 0.0, s2 = 0.0;
    unsigned long long bad = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        double v = lnw[i];
        if (v != v || v == pos_inf()) { bad++; continue; }
        if (v == neg_inf()) continue;
        if (v > m) {
            double e = exp(m - v);      // exp(-inf) = 0 the first time
            s1 = s1 * e + 1.0;
            s2 = s2 * e * e + 1.0;
            m = v;
        } else {
            double e = exp(v - m);
            s1 += e;
            s2 += e * e;
        }
    }
    block_lse(m, s1, s2, bad, sh);
    if (threadIdx.x == 0) { part[blockIdx.x].m = m; part[blockIdx.x].s1 = s1; part[blockIdx.x].s2 = s2; part[blockIdx.x].bad = bad; }
}

__device__ void fill_estimate(double m, double s1, double s2, double n, double* ln_int, double* relvar, double* neff, double* ness) {
    if (m == neg_inf() || !(s1 > 0.0)) {
        *ln_int = neg_inf(); *relvar = pos_inf(); *neff = 0.0; *ness = 0.0;
        return;
    }
    *ln_int = m + log(s1) - log(n);
    *neff = s1;
    *ness = s1 * s1 / s2;
    *relvar = s2 / (s1 * s1) - 1.0 / n;
}

__global__ void __launch_bounds__(256) reduce_final_kernel(int nparts, const RedPart* __restrict__ part, int N, ile_result* out, int accumulate) {
    __shared__ RedPart sh[8];
    double m = neg_inf(), s1 = 0.0, s2 = 0.0;
    unsigned long long bad = 0;
    for (int i = threadIdx.x; i < nparts; i += blockDim.x) {
        lse_merge(m, s1, s2, part[i].m, part[i].s1, part[i].s2);
        bad += part[i].bad;
    }
    block_lse(m, s1, s2, bad, sh);
    if (threadIdx.x == 0) {
        ile_result r = *out;
        fill_estimate(m, s1, s2, (double)N, &r.ln_integral, &r.rel_variance, &r.n_eff, &r.n_ess);
        r.ln_w_max = m; r.S1 = s1; r.S2 = s2;
        r.n_samples = (unsigned long long)N;
        r.n_nonfinite = bad;
        double cm = neg_inf(), c1 = 0.0, c2 = 0.0;
        unsigned long long cn = 0;
        if (accumulate) { cm = r.cum_ln_w_max; c1 = r.cum_S1; c2 = r.cum_S2; cn = r.cum_n_samples; if (cn == 0) cm = neg_inf(); }
        lse_merge(cm, c1, c2, m, s1, s2);
        cn += (unsigned long long)N;
        r.cum_ln_w_max = cm; r.cum_S1 = c1; r.cum_S2 = c2; r.cum_n_samples = cn;
        fill_estimate(cm, c1, c2, (double)cn, &r.cum_ln_integral, &r.cum_rel_variance, &r.cum_n_eff, &r.cum_n_ess);
        *out = r;
    }
}

// accumulate = 0: *out_dev is zeroed first (fresh result); 1: cumulative fields of *out_dev are
// carried forward (the caller pre-loaded them), per-iteration fields overwritten.
int ile_launch_reduce(ile_ctx* ctx, int N, const double* lnw, ile_result* out_dev, int accumulate) {
    if (N < 1 || !lnw || !out_dev) return ile_fail(ctx, ILE_EINVAL, "reduce: bad argument");
    int nblocks = (N + 256 * 8 - 1) / (256 * 8);
    if (nblocks > ctx->sm_count * 8) nblocks = ctx->sm_count * 8;
    void* scratch = nullptr;
    int rc = ile_scratch(ctx, (size_t)nblocks * sizeof(RedPart), &scratch);
    if (rc) return rc;
    if (!accumulate) ILE_CUDA(ctx, cudaMemsetAsync(out_dev, 0, sizeof(ile_result), ctx->stream));
    reduce_partial_kernel<<<nblocks, 256, 0, ctx->stream>>>(N, lnw, (RedPart*)scratch);
    ILE_LAUNCH_CHECK(ctx);
    reduce_final_kernel<<<1, 256, 0, ctx->stream>>>(nblocks, (const RedPart*)scratch, N, out_dev, accumulate);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

extern "C" int ile_reduce(ile_ctx* ctx, int N, const double* lnw, ile_result* out_dev) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    return ile_launch_reduce(ctx, N, lnw, out_dev, 0);
}

// ---------------------------------------------------------------- ile_reduce without allocation
// For callers that must not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the
// per-block partials live in a file-scope device array instead of the context's grow-only scratch.  Every GPU that
// loads the library holds the array (64 KB) until exit.  All calls on a device share it: calls that overlap on the GPU
// (two contexts, or two streams) race; calls on one stream do not.  Every partial a call reads was written by that
// call (block b writes entry b, the final kernel reads entries 0 .. nblocks - 1), so nothing has to start at zero and the
// contents the last call left behind are never seen.
#define RED_NOALLOC_MAX_BLOCKS 2048
#define RED_NOALLOC_MAX_DEVICES 64
static __device__ __align__(256) RedPart red_noalloc_part[RED_NOALLOC_MAX_BLOCKS];

// device address of the array on the current device; looked up once per device, with that device current
static int red_noalloc_address(ile_ctx* ctx, RedPart** out) {
    static RedPart* addr[RED_NOALLOC_MAX_DEVICES];            // zero-initialised: not looked up yet
    const int dev = ctx->device;
    if (dev < 0 || dev >= RED_NOALLOC_MAX_DEVICES) return ile_fail(ctx, ILE_EINVAL, "reduce_noalloc: device %d beyond %d", dev, RED_NOALLOC_MAX_DEVICES);
    if (!addr[dev]) {
        RedPart* p = nullptr;
        ILE_CUDA(ctx, cudaGetSymbolAddress((void**)&p, red_noalloc_part));     // the symbol's name is not a device address in host code
        if (!p) return ile_fail(ctx, ILE_ECUDA, "reduce_noalloc: no device address for the static scratch");
        addr[dev] = p;
    }
    *out = addr[dev];
    return ILE_OK;
}

extern "C" int ile_reduce_noalloc(ile_ctx* ctx, int N, const double* lnw, ile_result* out_dev) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);
    if (N < 1 || !lnw || !out_dev) return ile_fail(ctx, ILE_EINVAL, "reduce_noalloc: bad argument");
    if (N > ILE_REDUCE_NOALLOC_MAX_N)
        return ile_fail(ctx, ILE_EINVAL, "reduce_noalloc: N = %d exceeds the maximum %d of the allocation-free path (use ile_reduce)", N,
                        ILE_REDUCE_NOALLOC_MAX_N);
    RedPart* part = nullptr;
    int rc = red_noalloc_address(ctx, &part);
    if (rc) return rc;
    // the same grid as ile_reduce, capped by the array
    int nblocks = (N + 256 * 8 - 1) / (256 * 8);
    if (nblocks > ctx->sm_count * 8) nblocks = ctx->sm_count * 8;
    if (nblocks > RED_NOALLOC_MAX_BLOCKS) nblocks = RED_NOALLOC_MAX_BLOCKS;
    ILE_CUDA(ctx, cudaMemsetAsync(out_dev, 0, sizeof(ile_result), ctx->stream));
    reduce_partial_kernel<<<nblocks, 256, 0, ctx->stream>>>(N, lnw, part);
    ILE_LAUNCH_CHECK(ctx);
    reduce_final_kernel<<<1, 256, 0, ctx->stream>>>(nblocks, part, N, out_dev, 0);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}
