// libile: lifecycle and problem definition (host side of the C ABI in include/ile.h).
#include <stdarg.h>
#include <stdlib.h>
#include <vector>
#include "common.cuh"

int ile_fail(ile_ctx* ctx, int code, const char* fmt, ...) {
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

int ile_scratch(ile_ctx* ctx, size_t bytes, void** out) {
    if (bytes > ctx->scratch_bytes) {
        if (ctx->d_scratch) {
            ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
            ILE_CUDA(ctx, cudaFree(ctx->d_scratch));
            ctx->d_scratch = nullptr;
            ctx->scratch_bytes = 0;
        }
        size_t want = bytes + (bytes >> 2) + 4096;
        if (cudaMalloc(&ctx->d_scratch, want) != cudaSuccess) {
            cudaGetLastError();
            return ile_fail(ctx, ILE_ENOMEM, "scratch allocation of %zu bytes failed", want);
        }
        ctx->scratch_bytes = want;
    }
    *out = ctx->d_scratch;
    return ILE_OK;
}

uint64_t ile_launch_count(ile_ctx* ctx) { return ctx->launches; }

extern "C" uint64_t ile_kernel_launches(const ile_ctx* ctx) { return ctx ? ctx->launches : 0; }

// ---- device timing of the dominant kernel: cudaEvent pairs recorded on the context's stream
int ile_timing_begin(ile_ctx* ctx) {
    if (!ctx->timing_on) return -1;
    if (ctx->tev_used == ILE_TIMING_SLOTS && ile_timing_drain(ctx) != ILE_OK) return -1;
    const int slot = ctx->tev_used++;
    cudaEventRecord(ctx->tev[2 * slot], ctx->stream);
    return slot;
}
void ile_timing_end(ile_ctx* ctx, int slot) {
    if (slot >= 0) cudaEventRecord(ctx->tev[2 * slot + 1], ctx->stream);
}
int ile_timing_drain(ile_ctx* ctx) {
    if (!ctx->tev) return ILE_OK;
    for (int s = 0; s < ctx->tev_used; s++) {
        ILE_CUDA(ctx, cudaEventSynchronize(ctx->tev[2 * s + 1]));
        float ms = 0.f;
        ILE_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->tev[2 * s], ctx->tev[2 * s + 1]));
        ctx->t_ms_total += ms;
        ctx->t_count++;
    }
    ctx->tev_used = 0;
    return ILE_OK;
}
extern "C" int ile_kernel_timing(ile_ctx* ctx, int on) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    int rc = ile_timing_drain(ctx);
    if (rc) return rc;
    if (on && !ctx->tev) {
        ctx->tev = (cudaEvent_t*)calloc(2 * ILE_TIMING_SLOTS, sizeof(cudaEvent_t));
        if (!ctx->tev) return ile_fail(ctx, ILE_ENOMEM, "kernel_timing: out of host memory");
        for (int s = 0; s < 2 * ILE_TIMING_SLOTS; s++) ILE_CUDA(ctx, cudaEventCreate(&ctx->tev[s]));
    }
    ctx->timing_on = on ? 1 : 0;
    ctx->t_ms_total = 0.0;
    ctx->t_count = 0;
    return ILE_OK;
}
extern "C" int ile_kernel_time(ile_ctx* ctx, double* total_ms, uint64_t* launches) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    int rc = ile_timing_drain(ctx);
    if (rc) return rc;
    if (total_ms) *total_ms = ctx->t_ms_total;
    if (launches) *launches = ctx->t_count;
    return ILE_OK;
}

extern "C" const char* ile_version(void) { return "ile-b200 0.1 (sm_100a)"; }

extern "C" int ile_create(ile_ctx** out, int device, void* cuda_stream) {
    if (!out) return ILE_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return ILE_ECUDA;  // no CUDA device: there is no CPU fallback
    }
    ile_ctx* ctx = (ile_ctx*)calloc(1, sizeof(ile_ctx));
    if (!ctx) return ILE_ENOMEM;
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    if (cudaSetDevice(device) != cudaSuccess) {
        free(ctx);
        return ILE_ECUDA;
    }
    cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device);
    ctx->D_min = 1.0;
    ctx->D_max = 2.0;
    ctx->sky_sort = 1;
    ctx->lnl_split = 1;
    *out = ctx;
    return ILE_OK;
}

extern "C" int ile_destroy(ile_ctx* ctx) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    cudaFree(ctx->d_ylm);
    cudaFree(ctx->d_Qc);
    cudaFree(ctx->d_Qf);
    cudaFree(ctx->d_Qs);
    cudaFree(ctx->d_qeb);
    cudaFree(ctx->d_qhi);
    free(ctx->h_qeb);
    cudaFree(ctx->pc_buf);
    cudaFree(ctx->d_U);
    cudaFree(ctx->d_V);
    cudaFree(ctx->d_UVp);
    cudaFree(ctx->d_pairs);
    cudaFree(ctx->d_lnT);
    cudaFree(ctx->d_lnT4);
    cudaFree(ctx->d_scratch);
    if (ctx->tev) {
        for (int s = 0; s < 2 * ILE_TIMING_SLOTS; s++) cudaEventDestroy(ctx->tev[s]);
        free(ctx->tev);
    }
    free(ctx);
    return ILE_OK;
}

extern "C" const char* ile_last_error(const ile_ctx* ctx) { return ctx ? ctx->err : "null context"; }

extern "C" int ile_sync(ile_ctx* ctx) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ILE_CUDA(ctx, cudaGetLastError());
    return ILE_OK;
}

extern "C" int ile_set_lnL_variant(ile_ctx* ctx, int variant) {
    if (!ctx || variant < 0 || variant > 3) return ile_fail(ctx, ILE_EINVAL, "variant must be 0..3");
    ctx->variant = variant == 1 ? 1 : 0;
    ctx->lnl_split = variant == 0 ? 1 : 0;
    ctx->sky_sort = variant == 3 ? 0 : 1;
    return ILE_OK;
}

extern "C" int ile_set_network(ile_ctx* ctx, int K, const double* D, const double* pos_m, double gmst) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (K < 1 || K > ILE_MAX_K || !D || !pos_m) return ile_fail(ctx, ILE_EINVAL, "set_network: K in 1..%d", ILE_MAX_K);
    for (int k = 0; k < K; k++)
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                double x = D[k * 9 + a * 3 + b], y = D[k * 9 + b * 3 + a];
                if (!(fabs(x - y) <= 1e-12 * (fabs(x) + fabs(y) + 1e-300)) && x != y)
                    return ile_fail(ctx, ILE_EINVAL, "set_network: D[%d] is not symmetric", k);
            }
    if (ctx->have_quv && K != ctx->K) return ile_fail(ctx, ILE_ESTATE, "set_network: K differs from the loaded Q/U/V");
    ctx->K = K;
    ctx->gmst = gmst;
    ctx->max_delay = 0.0;
    for (int k = 0; k < K; k++) {
        memcpy(ctx->D[k], D + 9 * k, 9 * sizeof(double));
        memcpy(ctx->pos[k], pos_m + 3 * k, 3 * sizeof(double));
        double r = sqrt(pos_m[3 * k] * pos_m[3 * k] + pos_m[3 * k + 1] * pos_m[3 * k + 1] + pos_m[3 * k + 2] * pos_m[3 * k + 2]);
        if (r / ILE_C_LIGHT > ctx->max_delay) ctx->max_delay = r / ILE_C_LIGHT;
    }
    ctx->have_net = true;
    ctx->have_grid = false;  // the range check depends on the delays
    return ILE_OK;
}

// exact binomial / factorial in long double (l <= 8: all values < 2^53)
static long double fact_ld(int n) {
    long double f = 1.0L;
    for (int i = 2; i <= n; i++) f *= (long double)i;
    return f;
}
static long double binom_ld(int n, int k) {
    if (k < 0 || k > n) return 0.0L;
    return fact_ld(n) / (fact_ld(k) * fact_ld(n - k));
}

// Eq. (4): coefficient table of -2Y_lm as a polynomial in cos(theta/2), sin(theta/2)
// (Goldberg et al. 1967 closed form with s = -2).
extern "C" int ile_set_modes(ile_ctx* ctx, int M, const int* ell, const int* m) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (M < 1 || M > ILE_MAX_M || !ell || !m) return ile_fail(ctx, ILE_EINVAL, "set_modes: M in 1..%d", ILE_MAX_M);
    if (ctx->have_quv && M != ctx->M) return ile_fail(ctx, ILE_ESTATE, "set_modes: M differs from the loaded Q/U/V");
    YlmTable& T = ctx->h_ylm;
    memset(&T, 0, sizeof(T));
    T.M = M;
    const int s = -2;
    for (int i = 0; i < M; i++) {
        int l = ell[i], mm = m[i];
        if (l < 2 || l > ILE_MAX_L || abs(mm) > l) return ile_fail(ctx, ILE_EINVAL, "set_modes: mode %d = (%d,%d) unsupported", i, l, mm);
        for (int j = 0; j < i; j++)
            if (ell[j] == l && m[j] == mm) return ile_fail(ctx, ILE_EINVAL, "set_modes: duplicate mode (%d,%d)", l, mm);
        YlmMode& Y = T.mode[i];
        Y.m = mm;
        long double norm = sqrtl(fact_ld(l + mm) * fact_ld(l - mm) * (2 * l + 1) /
                                 (4.0L * 3.14159265358979323846264338327950288L * fact_ld(l + s) * fact_ld(l - s)));
        if ((l + mm - s) & 1) norm = -norm;
        int nt = 0;
        for (int r = 0; r <= l - s; r++) {
            int kk = r + s - mm;
            if (kk < 0 || kk > l + s) continue;
            long double c = binom_ld(l - s, r) * binom_ld(l + s, kk) * norm;
            if (r & 1) c = -c;
            if (nt >= ILE_YLM_MAX_TERMS) return ile_fail(ctx, ILE_EINVAL, "set_modes: too many terms");
            Y.coef[nt] = (double)c;
            Y.pc[nt] = 2 * r + s - mm;
            Y.ps[nt] = 2 * l - 2 * r - s + mm;
            if (Y.pc[nt] > T.max_pow) T.max_pow = Y.pc[nt];
            if (Y.ps[nt] > T.max_pow) T.max_pow = Y.ps[nt];
            nt++;
        }
        Y.nterms = nt;
        if (abs(mm) > T.max_abs_m) T.max_abs_m = abs(mm);
        ctx->ell[i] = l;
        ctx->m[i] = mm;
    }
    ctx->M = M;
    ctx->ylm_max_pow = T.max_pow;
    ctx->ylm_max_abs_m = T.max_abs_m;
    {   // pair list of the upper triangle, row by row
        std::vector<int2> pr;
        for (int a = 0; a < M; a++)
            for (int b = a; b < M; b++) pr.push_back(make_int2(a, b));
        cudaFree(ctx->d_pairs);
        ctx->d_pairs = nullptr;
        ctx->n_pairs = (int)pr.size();
        ILE_CUDA(ctx, cudaMalloc(&ctx->d_pairs, pr.size() * sizeof(int2)));
        ILE_CUDA(ctx, cudaMemcpy(ctx->d_pairs, pr.data(), pr.size() * sizeof(int2), cudaMemcpyHostToDevice));
    }
    if (!ctx->d_ylm) ILE_CUDA(ctx, cudaMalloc(&ctx->d_ylm, sizeof(YlmTable)));
    ILE_CUDA(ctx, cudaMemcpyAsync(ctx->d_ylm, &T, sizeof(YlmTable), cudaMemcpyHostToDevice, ctx->stream));
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->have_modes = true;
    return ILE_OK;
}

// ---------------------------------------------------------------- Q / U / V
// Repack Q [K][M][N_Q] complex -> tiled [K][N_Qpad][48]: one stored bin = 24 complex mode
// slots (zero padded), 8-double groups XOR-swizzled by bin parity so that the DMMA B-fragment
// LDS.128 of the fused kernel is bank-conflict free.
// Qf holds the same values fragment-major, [N_Qpad/2 bin pairs][6 k-step pairs][2 bins][8 columns]:
// the 8 bins x 4 lanes x 16 bytes of one DMMA B-fragment load are four whole 128-byte lines.
__global__ void repack_q_kernel(const double* __restrict__ Qc, double* __restrict__ Qf, int PK, int M, int N_Q,
                                int N_Qpad) {
    long long total = (long long)PK * N_Qpad * ILE_QT_ROW;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        int col = (int)(idx % ILE_QT_ROW);
        long long rest = idx / ILE_QT_ROW;
        int n = (int)(rest % N_Qpad);
        int pk = (int)(rest / N_Qpad);
        int r = col ^ ((n & 1) << 3);
        int mode = r >> 1, part = r & 1;
        double v = 0.0;
        if (mode < M && n < N_Q) v = Qc[(((long long)pk * M + mode) * N_Q + n) * 2 + part];
        Qf[(((long long)pk * N_Qpad + n) >> 1) * (2 * ILE_QT_ROW) + (r >> 3) * 16 + (n & 1) * 8 + (r & 7)] = v;
    }
}

__global__ void pack_uv_kernel(const double* __restrict__ U, const double* __restrict__ V, const int2* __restrict__ pairs, double* __restrict__ UVp,
                               int P, int K, int M, int n_pairs) {
    const long long total = (long long)P * n_pairs * K;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const int k = (int)(idx % K);
        const int pr = (int)((idx / K) % n_pairs);
        const int p = (int)(idx / ((long long)K * n_pairs));
        const int2 ab = pairs[pr];
        const double w = ab.x == ab.y ? 1.0 : 2.0;
        const size_t src = ((((size_t)p * K + k) * M + ab.x) * M + ab.y) * 2;
        double* o = UVp + (size_t)idx * 4;
        o[0] = w * U[src]; o[1] = w * U[src + 1]; o[2] = w * V[src]; o[3] = w * V[src + 1];
    }
}

// Device arrays of a Q/U/V set of P points and N_Q stored bins; a set of the same shape (the next intrinsic point of a
// run) reuses the allocations.  The resident set is invalid from here until the load completes.
int ile_quv_alloc(ile_ctx* ctx, int P, int N_Q) {
    const int K = ctx->K, M = ctx->M;
    const size_t nU = (size_t)P * K * M * M * 2, nQ = (size_t)P * K * M * N_Q * 2;
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const int N_Qpad = ((N_Q + 1) & ~1) + 256;
    size_t nQt = (size_t)P * K * N_Qpad * ILE_QT_ROW;
    // same shapes as the resident set (the next intrinsic point of a run): reuse the allocations
    const bool reuse = ctx->have_quv && ctx->P == P && ctx->N_Q == N_Q && ctx->quv_K == K && ctx->quv_M == M;
    ctx->have_quv = false;
    if (!reuse) {
        cudaFree(ctx->d_Qc); cudaFree(ctx->d_Qf); cudaFree(ctx->d_U); cudaFree(ctx->d_V); cudaFree(ctx->d_UVp);
        cudaFree(ctx->d_Qs); cudaFree(ctx->d_qeb); cudaFree(ctx->d_qhi); free(ctx->h_qeb);
        ctx->d_Qc = ctx->d_Qf = ctx->d_U = ctx->d_V = ctx->d_UVp = nullptr;
        ctx->d_Qs = nullptr; ctx->d_qeb = nullptr; ctx->d_qhi = nullptr;
        ctx->h_qeb = (int*)malloc((size_t)P * K * sizeof(int));
        if (cudaMalloc(&ctx->d_Qc, nQ * 8) != cudaSuccess || cudaMalloc(&ctx->d_Qf, nQt * 8) != cudaSuccess ||
            cudaMalloc(&ctx->d_U, nU * 8) != cudaSuccess || cudaMalloc(&ctx->d_V, nU * 8) != cudaSuccess ||
            cudaMalloc(&ctx->d_UVp, (size_t)P * ctx->n_pairs * K * 4 * 8) != cudaSuccess ||
            cudaMalloc(&ctx->d_Qs, ile_split_qs_bytes(P, K, N_Q)) != cudaSuccess || cudaMalloc(&ctx->d_qeb, (size_t)P * K * sizeof(int)) != cudaSuccess ||
            cudaMalloc(&ctx->d_qhi, (size_t)P * K * sizeof(int)) != cudaSuccess || !ctx->h_qeb) {
            cudaGetLastError();
            return ile_fail(ctx, ILE_ENOMEM, "load_quv: device allocation failed");
        }
    }
    return ILE_OK;
}

// trusted: U and V were made by ile_precompute_quv, whose last kernel writes the lower triangle from the upper by
// Eq. 17-18 - the symmetry check (and its copy to the host) is skipped
int ile_load_quv_impl(ile_ctx* ctx, int P, int N_Q, double fs, double t_Q0, const double* Q, const double* U, const double* V, double D_ref,
                      int src_is_device, bool trusted) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);
    if (!ctx->have_net || !ctx->have_modes) return ile_fail(ctx, ILE_ESTATE, "load_quv: set_network and set_modes first");
    if (P < 1 || N_Q < 4 || !(fs > 0) || !Q || !U || !V || !(D_ref > 0))
        return ile_fail(ctx, ILE_EINVAL, "load_quv: bad argument");
    if (ctx->M > ILE_QT_ROW / 2 - 2) return ile_fail(ctx, ILE_EINVAL, "load_quv: at most %d modes", ILE_QT_ROW / 2 - 2);
    const int K = ctx->K, M = ctx->M;
    size_t nU = (size_t)P * K * M * M * 2, nQ = (size_t)P * K * M * N_Q * 2;
    // symmetry check (Eq. 17-18) on the host
    std::vector<double> hU, hV;
    const double *pU = U, *pV = V;
    if (src_is_device && !trusted) {
        hU.resize(nU);
        hV.resize(nU);
        ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));      // producers of U, V on the context's (possibly non-blocking) stream
        ILE_CUDA(ctx, cudaMemcpy(hU.data(), U, nU * 8, cudaMemcpyDeviceToHost));
        ILE_CUDA(ctx, cudaMemcpy(hV.data(), V, nU * 8, cudaMemcpyDeviceToHost));
        pU = hU.data();
        pV = hV.data();
    }
    for (size_t pk = 0; pk < (trusted ? 0 : (size_t)P * K); pk++) {
        const double* u = pU + pk * M * M * 2;
        const double* v = pV + pk * M * M * 2;
        double scale = 0.0;
        for (int a = 0; a < M * M * 2; a++) scale = fmax(scale, fmax(fabs(u[a]), fabs(v[a])));
        double tol = 1e-12 * scale;
        for (int a = 0; a < M; a++)
            for (int b = 0; b < M; b++) {
                double ur = u[(a * M + b) * 2], ui = u[(a * M + b) * 2 + 1];
                double tr = u[(b * M + a) * 2], ti = u[(b * M + a) * 2 + 1];
                if (fabs(ur - tr) > tol || fabs(ui + ti) > tol)
                    return ile_fail(ctx, ILE_EINVAL, "load_quv: U[%zu] is not Hermitian at (%d,%d) (Eq. 17)", pk, a, b);
                double vr = v[(a * M + b) * 2], vi = v[(a * M + b) * 2 + 1];
                double wr = v[(b * M + a) * 2], wi = v[(b * M + a) * 2 + 1];
                if (fabs(vr - wr) > tol || fabs(vi - wi) > tol)
                    return ile_fail(ctx, ILE_EINVAL, "load_quv: V[%zu] is not symmetric at (%d,%d) (Eq. 18)", pk, a, b);
            }
    }
    if (Q != ctx->d_Qc) {                       // ile_precompute_quv has allocated and written the arrays themselves
        const int rc_alloc = ile_quv_alloc(ctx, P, N_Q);
        if (rc_alloc) return rc_alloc;
    }
    const int N_Qpad = ((N_Q + 1) & ~1) + 256;
    cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    if (Q != ctx->d_Qc) ILE_CUDA(ctx, cudaMemcpyAsync(ctx->d_Qc, Q, nQ * 8, kind, ctx->stream));
    if (U != ctx->d_U) ILE_CUDA(ctx, cudaMemcpyAsync(ctx->d_U, U, nU * 8, kind, ctx->stream));
    if (V != ctx->d_V) ILE_CUDA(ctx, cudaMemcpyAsync(ctx->d_V, V, nU * 8, kind, ctx->stream));
    ctx->qf_valid = 0;                          // the DMMA kernel's copy of Q is made when that kernel first runs (ile_ensure_qf)
    pack_uv_kernel<<<ctx->sm_count * 2, 256, 0, ctx->stream>>>(ctx->d_U, ctx->d_V, ctx->d_pairs, ctx->d_UVp, P, K, M, ctx->n_pairs);
    ILE_LAUNCH_CHECK(ctx);
    if (K <= 3 && M <= 24) {
        // signed 8-bit digit image of Q for the tcgen05 contraction (lnl_split.cu)
        int rc = ile_split_build_q(ctx, P, K, M, N_Q, ctx->d_Qc, ctx->d_Qs, ctx->d_qeb, ctx->d_qhi);
        if (rc) return rc;
        ILE_CUDA(ctx, cudaMemcpyAsync(ctx->h_qeb, ctx->d_qeb, (size_t)P * K * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    }
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->P = P; ctx->N_Q = N_Q; ctx->N_Qpad = N_Qpad; ctx->quv_K = K; ctx->quv_M = M; ctx->fs = fs; ctx->t_Q0 = t_Q0; ctx->D_ref = D_ref;
    ctx->have_quv = true;
    ctx->have_grid = false;
    return ILE_OK;
}

// The row-pair layout of Q that the DMMA kernel (lnl_fused2.cu) reads: built on first use, the default tcgen05 kernel
// reads the digit image instead.
int ile_ensure_qf(ile_ctx* ctx) {
    if (ctx->qf_valid) return ILE_OK;
    repack_q_kernel<<<ctx->sm_count * 8, 256, 0, ctx->stream>>>(ctx->d_Qc, ctx->d_Qf, ctx->P * ctx->quv_K, ctx->quv_M, ctx->N_Q, ctx->N_Qpad);
    ILE_LAUNCH_CHECK(ctx);
    ctx->qf_valid = 1;
    return ILE_OK;
}

extern "C" int ile_load_quv(ile_ctx* ctx, int P, int N_Q, double fs, double t_Q0, const double* Q, const double* U,
                            const double* V, double D_ref, int src_is_device) {
    return ile_load_quv_impl(ctx, P, N_Q, fs, t_Q0, Q, U, V, D_ref, src_is_device, false);
}

extern "C" int ile_set_time_grid(ile_ctx* ctx, double t_lo, double dt, int N_t, int interp) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (!ctx->have_quv) return ile_fail(ctx, ILE_ESTATE, "set_time_grid: load_quv first");
    if (N_t < 1 || !(dt > 0) || (interp != 0 && interp != 1)) return ile_fail(ctx, ILE_EINVAL, "set_time_grid: bad argument");
    double s = dt * ctx->fs;
    int stride = (int)llrint(s);
    if (stride < 1 || fabs(s - stride) > 1e-9) return ile_fail(ctx, ILE_EINVAL, "set_time_grid: dt*fs = %.12g is not a positive integer", s);
    // stored-bin coordinate of the earliest / latest access (G10: a set-up error, never a per-sample branch)
    double u_min = (t_lo - ctx->max_delay - ctx->t_Q0) * ctx->fs;
    double u_max = (t_lo + (N_t - 1) * dt + ctx->max_delay - ctx->t_Q0) * ctx->fs;
    if (u_min < 0.5 || u_max > (double)(ctx->N_Q - 2) - 0.5)
        return ile_fail(ctx, ILE_ERANGE, "set_time_grid: window [%.3f, %.3f] bins leaves the stored span [0, %d]", u_min, u_max, ctx->N_Q - 1);
    ctx->t_lo = t_lo; ctx->dt = dt; ctx->N_t = N_t; ctx->interp = interp; ctx->stride = stride;
    ctx->have_grid = true;
    return ILE_OK;
}

extern "C" int ile_set_prior(ile_ctx* ctx, double D_min, double D_max) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (!(D_min > 0) || !(D_max > D_min)) return ile_fail(ctx, ILE_EINVAL, "set_prior: need 0 < D_min < D_max");
    ctx->D_min = D_min; ctx->D_max = D_max; ctx->have_prior = true;
    return ILE_OK;
}

extern "C" int ile_load_distance_table(ile_ctx* ctx, int nA, int nB, double A_lo, double A_hi, double B_lo, double B_hi,
                                       const double* lnT) {
    if (!ctx) return ILE_EINVAL;
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (nA == 0) {
        cudaFree(ctx->d_lnT); ctx->d_lnT = nullptr; cudaFree(ctx->d_lnT4); ctx->d_lnT4 = nullptr; ctx->nA = ctx->nB = 0;
        return ILE_OK;
    }
    if (nA < 2 || nB < 2 || !(A_hi > A_lo) || !(B_hi > B_lo) || !lnT) return ile_fail(ctx, ILE_EINVAL, "load_distance_table: bad argument");
    cudaFree(ctx->d_lnT); ctx->d_lnT = nullptr;
    if (cudaMalloc(&ctx->d_lnT, (size_t)nA * nB * 8) != cudaSuccess) { cudaGetLastError(); return ile_fail(ctx, ILE_ENOMEM, "table allocation failed"); }
    ILE_CUDA(ctx, cudaMemcpy(ctx->d_lnT, lnT, (size_t)nA * nB * 8, cudaMemcpyHostToDevice));
    {   // cell copy for the fused kernel: the four corners of a bilinear lookup in one 32-byte sector
        std::vector<double> cells((size_t)(nA - 1) * (nB - 1) * 4);
        for (int b = 0; b < nB - 1; b++)
            for (int a = 0; a < nA - 1; a++) {
                double* c = &cells[((size_t)b * (nA - 1) + a) * 4];
                c[0] = lnT[(size_t)b * nA + a]; c[1] = lnT[(size_t)b * nA + a + 1];
                c[2] = lnT[(size_t)(b + 1) * nA + a]; c[3] = lnT[(size_t)(b + 1) * nA + a + 1];
            }
        cudaFree(ctx->d_lnT4); ctx->d_lnT4 = nullptr;
        if (cudaMalloc(&ctx->d_lnT4, cells.size() * 8) != cudaSuccess) { cudaGetLastError(); return ile_fail(ctx, ILE_ENOMEM, "table allocation failed"); }
        ILE_CUDA(ctx, cudaMemcpy(ctx->d_lnT4, cells.data(), cells.size() * 8, cudaMemcpyHostToDevice));
    }
    ctx->nA = nA; ctx->nB = nB; ctx->A_lo = A_lo; ctx->A_hi = A_hi; ctx->B_lo = B_lo; ctx->B_hi = B_hi;
    return ILE_OK;
}

int ile_fill_params(ile_ctx* ctx, int p, int d, LnlParams* L) {
    if (!ctx->have_net || !ctx->have_modes || !ctx->have_quv || !ctx->have_grid)
        return ile_fail(ctx, ILE_ESTATE, "lnL: network, modes, Q/U/V and time grid must be set first");
    if (p < 0 || p >= ctx->P) return ile_fail(ctx, ILE_EINVAL, "lnL: intrinsic point %d out of range [0,%d)", p, ctx->P);
    bool table = ctx->d_lnT != nullptr;
    if (d == 6 && !ctx->have_prior) return ile_fail(ctx, ILE_ESTATE, "lnL: set_prior (distance range) before evaluating with d = 6");
    if (!((d == 6 && !table) || (d == 5 && table)))
        return ile_fail(ctx, ILE_EINVAL, "lnL: d = %d does not match the distance-table state (6 without table, 5 with)", d);
    memset(L, 0, sizeof(*L));
    const int K = ctx->K, M = ctx->M;
    L->K = K; L->M = M; L->N_Q = ctx->N_Q; L->N_t = ctx->N_t; L->stride = ctx->stride; L->interp = ctx->interp;
    L->d = d; L->use_table = table ? 1 : 0; L->N_Qpad = ctx->N_Qpad;
    L->fs = ctx->fs; L->t_Q0 = ctx->t_Q0; L->t_lo = ctx->t_lo; L->dt = ctx->dt; L->D_ref = ctx->D_ref; L->gmst = ctx->gmst;
    memcpy(L->D, ctx->D, sizeof(ctx->D));
    memcpy(L->pos, ctx->pos, sizeof(ctx->pos));
    const double PI = 3.14159265358979323846;
    double lo[6] = {0.0, -1.0, 0.0, 0.0, -1.0, ctx->D_min}, hi[6] = {2 * PI, 1.0, PI, 2 * PI, 1.0, ctx->D_max};
    memcpy(L->lo, lo, sizeof(lo));
    memcpy(L->hi, hi, sizeof(hi));
    L->ln_prior_const = -log(2 * PI) - log(2.0) - log(PI) - log(2 * PI) - log(2.0);
    L->dist_norm = 3.0 / (ctx->D_max * ctx->D_max * ctx->D_max - ctx->D_min * ctx->D_min * ctx->D_min);
    L->ln_Nt = log((double)ctx->N_t);
    L->nA = ctx->nA; L->nB = ctx->nB; L->A_lo = ctx->A_lo; L->A_hi = ctx->A_hi; L->B_lo = ctx->B_lo; L->B_hi = ctx->B_hi;
    L->lnT = ctx->d_lnT;
    L->lnT4 = ctx->d_lnT4;
    L->Qc = ctx->d_Qc + (size_t)p * K * M * ctx->N_Q * 2;
    L->Qf = ctx->d_Qf + (size_t)p * K * ctx->N_Qpad * ILE_QT_ROW;
    L->U = ctx->d_U + (size_t)p * K * M * M * 2;
    L->V = ctx->d_V + (size_t)p * K * M * M * 2;
    L->ylm = ctx->d_ylm;
    L->pairs = ctx->d_pairs;
    L->n_pairs = ctx->n_pairs;
    L->UVp = ctx->d_UVp + (size_t)p * ctx->n_pairs * K * 4;
    L->Qs = nullptr;
    if (K <= 3 && M <= 24 && ctx->d_Qs) {
        L->NG8 = ile_split_ng8(ctx->N_Q);
        L->Qs = ctx->d_Qs + (size_t)p * K * L->NG8 * 2432;
        for (int k = 0; k < K; k++) L->qeb[k] = ctx->h_qeb[p * K + k];
        // rows of the triangle (row a has M - a pairs) to the four thread groups of a sample, longest row first to the
        // group with the least work so far; groups 0..K-1 start with the digit cutting of one detector, which costs about
        // as much as `head` pairs (measured: the kernel time is flat around these values)
        const int head = K == 1 ? 36 : K == 2 ? 26 : 20;
        int load[4] = {head, K > 1 ? head : 0, K > 2 ? head : 0, 0};
        for (int a = 0; a < M; a++) {
            int gmin = 0;
            for (int g = 1; g < 4; g++)
                if (load[g] < load[gmin]) gmin = g;
            L->tri_group[a] = (unsigned char)gmin;
            load[gmin] += M - a;
        }
    }
    return ILE_OK;
}
