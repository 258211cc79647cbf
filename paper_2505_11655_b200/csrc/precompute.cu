// libile: the inner products Q, U, V of Eq. (6a-c) on the device (PAPER.md:78-87,
// 337-345: "GPU-optimized ... overlaps for U, V, Q" is the paper's own wish).
//   w_k[j]      = 2 df / S_k(|f_j|) for |f_j| > f_low, else 0            (numpy FFT bin order)
//   U_k[a][b]   = sum_j w_k[j] conj(h_a[j]) h_b[j]                        (6b)
//   V_k[a][b]   = sum_j w_k[j] h_a[-j] h_b[j]                             (6c)
//   Q_k[a][n]   = sum_j w_k[j] conj(h_a[j]) d_k[j] exp(2 pi i j (n + n0) / N_f)   (6a), t_n = (n0 + n) / fs
// U, V: upper triangle, frequency slices staged in shared memory, deterministic two-stage sum.  Q: for power-of-two N_f <= 2^18 a four-step
// inverse FFT (column DFTs in registers, row FFTs in shared memory, only the stored window written);
// otherwise the definition (one thread per output time, twiddle advanced by complex rotation and
// re-seeded from an exact table every 32 bins).  Installed through ile_load_quv (symmetry check, repack).
#include "common.cuh"

#define PC_THREADS 256
#define PC_RESEED 32

__global__ void pc_weight_kernel(int K, int N_f, double df, double f_low, const double* __restrict__ S, double* __restrict__ w) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
    if (j >= N_f) return;
    const int ja = j <= N_f / 2 ? j : N_f - j;
    const double f = (double)ja * df;
    w[(size_t)k * N_f + j] = f > f_low ? 2.0 * df / S[(size_t)k * (N_f / 2 + 1) + ja] : 0.0;
}

__global__ void pc_twiddle_kernel(int N_f, double2* __restrict__ W) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N_f) return;
    double s, c;
    sincospi(2.0 * (double)m / (double)N_f, &s, &c);
    W[m] = make_double2(c, s);
}

// U and V, upper triangle.  Block (slice, p): frequency slice of point p in chunks of PC_CH bins staged in
// shared memory (h_m[j] and h_m[-j] for all modes, w_k[j]); thread = pair (a <= b), 4 K running sums;
// per-block partial sums go to part[p][slice][pair][k][4] and are added in slice order by pc_uv_finish_kernel
// (deterministic), which also fills the lower triangle by Eq. 17-18.
#define PC_CH 32
__global__ void __launch_bounds__(PC_THREADS) pc_uv_kernel(int M, int K, int N_f, int n_pairs, int chunks_per_block, const int2* __restrict__ pairs,
                                                           const double2* __restrict__ h, const double* __restrict__ w, double* __restrict__ part) {
    __shared__ double2 hs[ILE_MAX_M][PC_CH + 1], hm[ILE_MAX_M][PC_CH + 1];
    __shared__ double ws[ILE_MAX_K][PC_CH];
    const int p = blockIdx.y, tid = threadIdx.x;
    const double2* hp = h + (size_t)p * M * N_f;
    const bool act = tid < n_pairs;
    const int2 ab = act ? pairs[tid] : make_int2(0, 0);
    double acc[ILE_MAX_K][4];
#pragma unroll
    for (int k = 0; k < ILE_MAX_K; k++) acc[k][0] = acc[k][1] = acc[k][2] = acc[k][3] = 0.0;
    for (int cc = 0; cc < chunks_per_block; cc++) {
        const int j0 = (blockIdx.x * chunks_per_block + cc) * PC_CH;
        if (j0 >= N_f) break;
        __syncthreads();                                              // the previous chunk is consumed
        for (int q = tid; q < K * PC_CH; q += PC_THREADS) {
            const int k = q / PC_CH, jj = q % PC_CH;
            ws[k][jj] = j0 + jj < N_f ? w[(size_t)k * N_f + j0 + jj] : 0.0;
        }
        // chunks outside the band carry no weight
        if (!__syncthreads_or(tid < K * PC_CH && ws[tid / PC_CH][tid % PC_CH] != 0.0)) continue;
        for (int q = tid; q < M * PC_CH; q += PC_THREADS) {
            const int m = q / PC_CH, jj = q % PC_CH, j = j0 + jj;
            const bool in = j < N_f;
            hs[m][jj] = in ? hp[(size_t)m * N_f + j] : make_double2(0.0, 0.0);
            hm[m][jj] = in ? hp[(size_t)m * N_f + (j == 0 ? 0 : N_f - j)] : make_double2(0.0, 0.0);
        }
        __syncthreads();
        if (act) {
#pragma unroll 4
            for (int jj = 0; jj < PC_CH; jj++) {
                const double2 x = hs[ab.x][jj], y = hs[ab.y][jj], xm = hm[ab.x][jj];
                const double cr = x.x * y.x + x.y * y.y, ci = x.x * y.y - x.y * y.x;          // conj(x) y
                const double vr = xm.x * y.x - xm.y * y.y, vi = xm.x * y.y + xm.y * y.x;      // x(-f) y
#pragma unroll
                for (int k = 0; k < ILE_MAX_K; k++)
                    if (k < K) {
                        const double wj = ws[k][jj];
                        acc[k][0] += wj * cr; acc[k][1] += wj * ci; acc[k][2] += wj * vr; acc[k][3] += wj * vi;
                    }
            }
        }
    }
    if (act) {
        double* o = part + ((((size_t)p * gridDim.x + blockIdx.x) * n_pairs + tid) * K) * 4;
        for (int k = 0; k < K; k++) {
            o[4 * k + 0] = acc[k][0]; o[4 * k + 1] = acc[k][1]; o[4 * k + 2] = acc[k][2]; o[4 * k + 3] = acc[k][3];
        }
    }
}

__global__ void pc_uv_finish_kernel(int P, int M, int K, int n_pairs, int slices, const int2* __restrict__ pairs, const double* __restrict__ part,
                                    double2* __restrict__ U, double2* __restrict__ V) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= P * n_pairs * K) return;
    const int k = idx % K, pr = (idx / K) % n_pairs, p = idx / (K * n_pairs);
    double t[4] = {0.0, 0.0, 0.0, 0.0};
    for (int sl = 0; sl < slices; sl++) {
        const double* o = part + ((((size_t)p * slices + sl) * n_pairs + pr) * K + k) * 4;
        for (int e = 0; e < 4; e++) t[e] += o[e];
    }
    const int2 ab = pairs[pr];
    const size_t base = ((size_t)p * K + k) * M * M;
    U[base + ab.x * M + ab.y] = make_double2(t[0], t[1]);
    V[base + ab.x * M + ab.y] = make_double2(t[2], t[3]);
    if (ab.x != ab.y) {
        U[base + ab.y * M + ab.x] = make_double2(t[0], -t[1]);      // U Hermitian (Eq. 17)
        V[base + ab.y * M + ab.x] = make_double2(t[2], t[3]);       // V symmetric (Eq. 18)
    }
}

// x_{k,a}[j] = w_k[j] conj(h_a[j]) d_k[j]  (shared by all output times)
__global__ void pc_prod_kernel(int M, int K, int N_f, const double2* __restrict__ h, const double2* __restrict__ d, const double* __restrict__ w,
                               double2* __restrict__ x) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, ka = blockIdx.y, p = blockIdx.z;
    if (j >= N_f) return;
    const int k = ka / M, a = ka % M;
    const double wj = w[(size_t)k * N_f + j];
    const double2 hh = h[((size_t)p * M + a) * N_f + j], dd = d[(size_t)k * N_f + j];
    x[((size_t)p * K * M + ka) * N_f + j] = make_double2(wj * (hh.x * dd.x + hh.y * dd.y), wj * (hh.x * dd.y - hh.y * dd.x));
}

// grid (ceil(N_Q / 128), K*M, P): thread = output time n; Q[n] = sum_j x[j] W^{j (n + n0)}
__global__ void __launch_bounds__(128) pc_q_kernel(int N_f, int N_Q, int n0, const double2* __restrict__ x, const double2* __restrict__ W,
                                                   const double* __restrict__ w, int M, double2* __restrict__ Q) {
    __shared__ double2 xs[PC_RESEED * 8];
    const int n = blockIdx.x * 128 + threadIdx.x, ka = blockIdx.y, p = blockIdx.z, KM = gridDim.y;
    const double2* xp = x + ((size_t)p * KM + ka) * N_f;
    long long step = ((long long)n + n0) % N_f;
    if (step < 0) step += N_f;
    const double2 rot = W[step];
    double qr = 0.0, qi = 0.0;
    for (int j0 = 0; j0 < N_f; j0 += PC_RESEED * 8) {
        __syncthreads();
        for (int q = threadIdx.x; q < PC_RESEED * 8; q += 128) xs[q] = j0 + q < N_f ? xp[j0 + q] : make_double2(0.0, 0.0);
        __syncthreads();
#pragma unroll 1
        for (int g = 0; g < 8; g++) {
            const int jb = j0 + g * PC_RESEED;
            if (jb >= N_f) break;
            double2 tw = W[(int)(((long long)jb * step) % N_f)];       // exact re-seed
#pragma unroll
            for (int q = 0; q < PC_RESEED; q++) {
                const double2 v = xs[g * PC_RESEED + q];
                qr += v.x * tw.x - v.y * tw.y;
                qi += v.x * tw.y + v.y * tw.x;
                const double tr = tw.x * rot.x - tw.y * rot.y;
                tw.y = tw.x * rot.y + tw.y * rot.x;
                tw.x = tr;
            }
        }
    }
    if (n < N_Q) Q[((size_t)p * KM + ka) * N_Q + n] = make_double2(qr, qi);
}

// ---------------------------------------------------------------- power-of-two N_f: four-step inverse FFT
// N_f = N1 N2, j = j1 + N1 j2, n = n1 N2 + n2:
//   W_N^{jn} = W_N1^{j1 n1} W_N^{j1 n2} W_N2^{j2 n2}
// pc_fft_cols: thread = (series, j1): x[j1 + N1 j2] = w conj(h) d formed on the fly (coalesced over j1), the
//   N2-point DFT over j2 by its definition, times the twiddle W_N^{j1 n2}           -> B[series][n2][j1]
// pc_fft_rows: CTA = (n2, series): N1-point decimation-in-frequency FFT in shared memory, two radix-2 stages per pass (natural
//   order in, bit-reversed out), then only the outputs n = n1 N2 + n2 that fall in the stored window
//   [n0, n0 + N_Q) are written.  Every twiddle is an exact entry of the sincospi table W.
template <int N2>
__global__ void __launch_bounds__(256) pc_fft_cols_kernel(int M, int K, int N_f, int N1, const double2* __restrict__ h,
                                                          const double2* __restrict__ d, const double* __restrict__ w,
                                                          const double2* __restrict__ W, double2* __restrict__ B) {
    __shared__ double2 w2[N2];
    const int j1 = blockIdx.x * 256 + threadIdx.x, ka = blockIdx.y, p = blockIdx.z;
    const int k = ka / M, a = ka % M;
    if (threadIdx.x < N2) w2[threadIdx.x] = W[(size_t)threadIdx.x * (N_f / N2)];
    __syncthreads();
    if (j1 >= N1) return;
    double2 x[N2];
#pragma unroll
    for (int j2 = 0; j2 < N2; j2++) {
        const int j = j1 + N1 * j2;
        const double wj = w[(size_t)k * N_f + j];
        const double2 hh = h[((size_t)p * M + a) * N_f + j], dd = d[(size_t)k * N_f + j];
        x[j2] = make_double2(wj * (hh.x * dd.x + hh.y * dd.y), wj * (hh.x * dd.y - hh.y * dd.x));
    }
    double2* Bp = B + ((size_t)p * K * M + ka) * N_f;
#pragma unroll 1
    for (int n2 = 0; n2 < N2; n2++) {
        double sr = 0.0, si = 0.0;
#pragma unroll
        for (int j2 = 0; j2 < N2; j2++) {
            const double2 t = w2[(j2 * n2) & (N2 - 1)];
            sr += x[j2].x * t.x - x[j2].y * t.y;
            si += x[j2].x * t.y + x[j2].y * t.x;
        }
        const double2 t = W[(j1 * n2) & (N_f - 1)];
        Bp[(size_t)n2 * N1 + j1] = make_double2(sr * t.x - si * t.y, sr * t.y + si * t.x);
    }
}

__global__ void __launch_bounds__(256) pc_fft_rows_kernel(int N_f, int N1, int log2N1, int N2, int N_Q, int n0m, const double2* __restrict__ B,
                                                          const double2* __restrict__ W, double2* __restrict__ Q) {
    extern __shared__ double2 sm[];
    const int n2 = blockIdx.x, s = blockIdx.y;
    const double2* Bp = B + ((size_t)s * N2 + n2) * N1;
    for (int i = threadIdx.x; i < N1; i += 256) sm[i] = Bp[i];
    __syncthreads();
    // two radix-2 stages per pass (halves H and H/2 on the elements p, p + H/2, p + H, p + 3H/2):
    // W_2H^(p + H/2) = i W_2H^p, so a pass needs two table twiddles; a last single stage if log2 N1 is odd
    int H = N1 >> 1, ts = N_f / N1, stages = log2N1;
    while (stages >= 2) {
        const int q = H >> 1;
        for (int t = threadIdx.x; t < (N1 >> 2); t += 256) {
            const int pos = t & (q - 1), i0 = ((t - pos) << 2) + pos;
            const double2 x0 = sm[i0], x1 = sm[i0 + q], x2 = sm[i0 + 2 * q], x3 = sm[i0 + 3 * q];
            const double2 w1 = W[(size_t)pos * ts], w2 = W[(size_t)pos * 2 * ts];
            const double2 y0 = make_double2(x0.x + x2.x, x0.y + x2.y), y1 = make_double2(x1.x + x3.x, x1.y + x3.y);
            const double ar = x0.x - x2.x, ai = x0.y - x2.y, br = x1.x - x3.x, bi = x1.y - x3.y;
            const double2 y2 = make_double2(ar * w1.x - ai * w1.y, ar * w1.y + ai * w1.x);
            const double2 y3 = make_double2(-(br * w1.y + bi * w1.x), br * w1.x - bi * w1.y);      // (x1 - x3) i w1
            const double cr = y0.x - y1.x, ci = y0.y - y1.y, dr = y2.x - y3.x, di = y2.y - y3.y;
            sm[i0] = make_double2(y0.x + y1.x, y0.y + y1.y);
            sm[i0 + q] = make_double2(cr * w2.x - ci * w2.y, cr * w2.y + ci * w2.x);
            sm[i0 + 2 * q] = make_double2(y2.x + y3.x, y2.y + y3.y);
            sm[i0 + 3 * q] = make_double2(dr * w2.x - di * w2.y, dr * w2.y + di * w2.x);
        }
        __syncthreads();
        H >>= 2;
        ts <<= 2;
        stages -= 2;
    }
    if (stages == 1) {                                   // H == 1: last butterflies, twiddle 1
        for (int t = threadIdx.x; t < (N1 >> 1); t += 256) {
            const double2 u = sm[2 * t], v = sm[2 * t + 1];
            sm[2 * t] = make_double2(u.x + v.x, u.y + v.y);
            sm[2 * t + 1] = make_double2(u.x - v.x, u.y - v.y);
        }
        __syncthreads();
    }
    // window bins t with (n0m + t) mod N2 == n2
    int t0 = (n2 - n0m) % N2;
    if (t0 < 0) t0 += N2;
    for (int t = t0 + threadIdx.x * N2; t < N_Q; t += 256 * N2) {
        const int n = (n0m + t) & (N_f - 1), n1 = n / N2;
        Q[(size_t)s * N_Q + t] = sm[__brev((unsigned)n1) >> (32 - log2N1)];
    }
}

template <int N2>
static void launch_fft_cols(int P, int M, int K, int N_f, int N1, const double2* h, const double2* d, const double* w, const double2* W, double2* B,
                            cudaStream_t st) {
    pc_fft_cols_kernel<N2><<<dim3((N1 + 255) / 256, K * M, P), 256, 0, st>>>(M, K, N_f, N1, h, d, w, W, B);
}

// Eq. (6a-c) for P intrinsic points from frequency-domain inputs (device pointers, numpy FFT bin
// order): h [P][M][N_f][2] mode spectra, d [K][N_f][2] data spectra, S [K][N_f/2+1] one-sided PSDs
// over |f|.  fs = N_f df; the stored window starts at t_Q0 (t_Q0 fs must be an integer) and has N_Q
// bins.  The result replaces the context's Q/U/V exactly as ile_load_quv would.
extern "C" int ile_precompute_quv(ile_ctx* ctx, int P, int N_f, double df, double f_low, const double* h, const double* d, const double* S,
                                  double t_Q0, int N_Q, double D_ref) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);
    if (!ctx->have_net || !ctx->have_modes) return ile_fail(ctx, ILE_ESTATE, "precompute_quv: set_network and set_modes first");
    if (P < 1 || N_f < 8 || (N_f & 1) || !(df > 0) || !h || !d || !S || N_Q < 4 || N_Q > N_f || !(D_ref > 0))
        return ile_fail(ctx, ILE_EINVAL, "precompute_quv: bad argument");
    const double fs = (double)N_f * df;
    const double n0d = t_Q0 * fs;
    const long long n0 = llrint(n0d);
    if (fabs(n0d - (double)n0) > 1e-6) return ile_fail(ctx, ILE_EINVAL, "precompute_quv: t_Q0 * fs = %.9g is not an integer", n0d);
    const int K = ctx->K, M = ctx->M, n_pairs = ctx->n_pairs;
    if (n_pairs > PC_THREADS || K * PC_CH > PC_THREADS) return ile_fail(ctx, ILE_EINVAL, "precompute_quv: at most 22 modes");
    const size_t nQ = (size_t)P * K * M * N_Q, nU = (size_t)P * K * M * M, nX = (size_t)P * K * M * N_f;
    // frequency slices per point: enough blocks for two waves, at least one chunk each
    const int chunks = (N_f + PC_CH - 1) / PC_CH;
    int slices = (2 * ctx->sm_count + P - 1) / P;
    if (slices > chunks) slices = chunks;
    const int cpb = (chunks + slices - 1) / slices;
    slices = (chunks + cpb - 1) / cpb;
    const size_t nPart = (size_t)P * slices * n_pairs * K * 4;
    // one grow-only scratch allocation: w | W | x | Q | U | V | part  (256-byte aligned pieces)
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t o_w = 0, o_W = o_w + al((size_t)K * N_f * 8), o_x = o_W + al((size_t)N_f * 16), o_Q = o_x + al(nX * 16),
                 o_U = o_Q + al(nQ * 16), o_V = o_U + al(nU * 16), o_p = o_V + al(nU * 16), total = o_p + al(nPart * 8);
    if (total > ctx->pc_bytes) {
        cudaStreamSynchronize(ctx->stream);
        cudaFree(ctx->pc_buf);
        ctx->pc_buf = nullptr;
        ctx->pc_bytes = 0;
        if (cudaMalloc(&ctx->pc_buf, total) != cudaSuccess) {
            cudaGetLastError();
            return ile_fail(ctx, ILE_ENOMEM, "precompute_quv: device allocation of %zu bytes failed", total);
        }
        ctx->pc_bytes = total;
    }
    char* buf = (char*)ctx->pc_buf;
    double* w = (double*)(buf + o_w);
    double2 *W = (double2*)(buf + o_W), *x = (double2*)(buf + o_x), *Q = (double2*)(buf + o_Q), *U = (double2*)(buf + o_U),
            *V = (double2*)(buf + o_V);
    double* part = (double*)(buf + o_p);
    cudaStream_t st = ctx->stream;
    pc_weight_kernel<<<dim3((N_f + 255) / 256, K), 256, 0, st>>>(K, N_f, df, f_low, S, w);
    pc_twiddle_kernel<<<(N_f + 255) / 256, 256, 0, st>>>(N_f, W);
    pc_uv_kernel<<<dim3(slices, P), PC_THREADS, 0, st>>>(M, K, N_f, n_pairs, cpb, ctx->d_pairs, (const double2*)h, w, part);
    pc_uv_finish_kernel<<<(P * n_pairs * K + 255) / 256, 256, 0, st>>>(P, M, K, n_pairs, slices, ctx->d_pairs, part, U, V);
    if ((N_f & (N_f - 1)) == 0 && N_f <= (1 << 18)) {                       // four-step FFT; x serves as B
        const int N1 = N_f <= 4096 ? N_f : (N_f <= 4096 * 32 ? 4096 : 8192), N2 = N_f / N1;
        int log2N1 = 0;
        while ((1 << log2N1) < N1) log2N1++;
        const double2 *hh = (const double2*)h, *dd = (const double2*)d;
        switch (N2) {
            case 1: launch_fft_cols<1>(P, M, K, N_f, N1, hh, dd, w, W, x, st); break;
            case 2: launch_fft_cols<2>(P, M, K, N_f, N1, hh, dd, w, W, x, st); break;
            case 4: launch_fft_cols<4>(P, M, K, N_f, N1, hh, dd, w, W, x, st); break;
            case 8: launch_fft_cols<8>(P, M, K, N_f, N1, hh, dd, w, W, x, st); break;
            case 16: launch_fft_cols<16>(P, M, K, N_f, N1, hh, dd, w, W, x, st); break;
            default: launch_fft_cols<32>(P, M, K, N_f, N1, hh, dd, w, W, x, st); break;
        }
        const size_t smem = (size_t)N1 * sizeof(double2);
        cudaFuncSetAttribute(pc_fft_rows_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        long long n0m = n0 % N_f;
        if (n0m < 0) n0m += N_f;
        pc_fft_rows_kernel<<<dim3(N2, P * K * M), 256, smem, st>>>(N_f, N1, log2N1, N2, N_Q, (int)n0m, x, W, Q);
    } else {
        pc_prod_kernel<<<dim3((N_f + 255) / 256, K * M, P), 256, 0, st>>>(M, K, N_f, (const double2*)h, (const double2*)d, w, x);
        pc_q_kernel<<<dim3((N_Q + 127) / 128, K * M, P), 128, 0, st>>>(N_f, N_Q, (int)n0, x, W, w, M, Q);
    }
    ctx->launches += 6;
    ILE_LAUNCH_CHECK(ctx);
    ILE_CUDA(ctx, cudaStreamSynchronize(st));          // ile_load_quv reads U and V back for its symmetry check
    return ile_load_quv(ctx, P, N_Q, fs, (double)n0 / fs, (const double*)Q, (const double*)U, (const double*)V, D_ref, 1);
}

// Copies the resident Q/U/V of intrinsic point p to host arrays (caller layout of ile_load_quv).
extern "C" int ile_get_quv(ile_ctx* ctx, int p, double* Q, double* U, double* V) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context\'s device, whatever the caller\'s current one
    if (!ctx->have_quv) return ile_fail(ctx, ILE_ESTATE, "get_quv: nothing loaded");
    if (p < 0 || p >= ctx->P) return ile_fail(ctx, ILE_EINVAL, "get_quv: point out of range");
    const size_t nQ = (size_t)ctx->K * ctx->M * ctx->N_Q * 2, nU = (size_t)ctx->K * ctx->M * ctx->M * 2;
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (Q) ILE_CUDA(ctx, cudaMemcpy(Q, ctx->d_Qc + (size_t)p * nQ, nQ * 8, cudaMemcpyDeviceToHost));
    if (U) ILE_CUDA(ctx, cudaMemcpy(U, ctx->d_U + (size_t)p * nU, nU * 8, cudaMemcpyDeviceToHost));
    if (V) ILE_CUDA(ctx, cudaMemcpy(V, ctx->d_V + (size_t)p * nU, nU * 8, cudaMemcpyDeviceToHost));
    return ILE_OK;
}
