// libile: the inner products Q, U, V of Eq. (6a-c) on the device (PAPER.md:78-87,
// 337-345: "GPU-optimized ... overlaps for U, V, Q" is the paper's own wish).
//   w_k[j]      = 2 df / S_k(|f_j|) for |f_j| > f_low, else 0            (numpy FFT bin order)
//   U_k[a][b]   = sum_j w_k[j] conj(h_a[j]) h_b[j]                        (6b)
//   V_k[a][b]   = sum_j w_k[j] h_a[-j] h_b[j]                             (6c)
//   Q_k[a][n]   = sum_j w_k[j] conj(h_a[j]) d_k[j] exp(2 pi i j (n + n0) / N_f)   (6a), t_n = (n0 + n) / fs
// U, V: upper triangle, frequency slices staged in shared memory, deterministic two-stage sum.  Q: for power-of-two N_f and a stored
// window of at most 2048 bins an inverse FFT pruned to the window (decimated spectra transformed in shared memory, no
// intermediate in global memory); otherwise the definition (one thread per output time, twiddle advanced by complex
// rotation and re-seeded from an exact table every 32 bins).  Installed as ile_load_quv would (repack, digit image).
#include "common.cuh"
#include <cuda_pipeline.h>

#define PC_RESEED 32

__global__ void pc_weight_kernel(int K, int N_f, double df, double f_low, const double* __restrict__ S, const double2* __restrict__ d,
                                 double* __restrict__ w, double2* __restrict__ dw) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
    if (j >= N_f) return;
    const int ja = j <= N_f / 2 ? j : N_f - j;
    const double f = (double)ja * df;
    const double wj = f > f_low ? 2.0 * df / S[(size_t)k * (N_f / 2 + 1) + ja] : 0.0;
    w[(size_t)k * N_f + j] = wj;
    const double2 dd = d[(size_t)k * N_f + j];
    dw[(size_t)k * N_f + j] = make_double2(wj * dd.x, wj * dd.y);          // the weighted data spectrum of Eq. 6a
}

__global__ void pc_twiddle_kernel(int N_f, double2* __restrict__ W) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N_f) return;
    double s, c;
    sincospi(2.0 * (double)m / (double)N_f, &s, &c);
    W[m] = make_double2(c, s);
}

// U and V, upper triangle.  CTA (slice, p): the frequency slice of point p in chunks of UV_CH bins, triple-buffered in
// shared memory by asynchronous copies (h_m[j] and h_m[-j] for all modes, w_k[j]).  Thread = (2 x 2 tile of mode pairs,
// one of UV_SUB interleaved sub-slices of the chunk): 6 shared-memory loads feed 4 pairs x (8 + 12 K / 3) FP64 operations,
// 16 K running sums in registers.  The sub-slices are added in shared memory, the per-CTA partial sums part[p][slice][pair][k][4]
// in slice order by pc_uv_finish_kernel (deterministic), which also fills the lower triangle by Eq. 17-18.
#define UV_CH 64
#define UV_SUB 5
#define UV_NBUF 3
#define UV_SB (2 * UV_CH + 1)                  // stride of a mode pair's rows in 16-byte units (odd: no bank conflicts)
#define UV_MAXTHREADS(BIG) ((BIG) ? 416 : 352)  // 78 tiles (24 modes) or 66 (22 modes) x 5 sub-slices: 13 or 11 warps, close to even over 4 sub-partitions
template <int KK, bool BIG>
__global__ void __launch_bounds__(UV_MAXTHREADS(BIG), 1) pc_uv_kernel(int M, int N_f, int n_pairs, int chunks_per_block, const double2* __restrict__ h, const double* __restrict__ w,
                                                                 double* __restrict__ part) {
    extern __shared__ double2 uv_sm[];
    const int MB = (M + 1) >> 1, n_tiles = MB * (MB + 1) / 2;
    double2* hs = uv_sm;                                   // [UV_NBUF][MB][UV_CH][2]  (+1 per mode pair)
    double2* hm = hs + UV_NBUF * MB * UV_SB;               // the same at -f
    double* ws = reinterpret_cast<double*>(hm + UV_NBUF * MB * UV_SB);   // [UV_NBUF][KK][UV_CH]
    const int p = blockIdx.y, tid = threadIdx.x, nthr = blockDim.x;
    const double2* hp = h + (size_t)p * M * N_f;
    const int tile = tid % n_tiles, sub = tid / n_tiles;
    const bool act = sub < UV_SUB;
    int ta = 0, tb = 0;
    {
        int rem = tile;
        while (rem >= MB - ta) { rem -= MB - ta; ta++; }
        tb = ta + rem;
    }
    double acc[2][2][KK][4];
#pragma unroll
    for (int e = 0; e < 16 * KK; e++) (&acc[0][0][0][0])[e] = 0.0;
    // rows of a padding mode (odd M) stay zero in both buffers
    for (int q = tid; q < 2 * UV_NBUF * MB * UV_SB; q += nthr) hs[q] = make_double2(0.0, 0.0);
    __syncthreads();
    const int c_begin = blockIdx.x * chunks_per_block, c_end = min(c_begin + chunks_per_block, (N_f + UV_CH - 1) / UV_CH);
    auto stage = [&](int c, int buf) {
        const int j0 = c * UV_CH;
        double2* hsb = hs + buf * MB * UV_SB;
        double2* hmb = hm + buf * MB * UV_SB;
        for (int q = tid; q < M * UV_CH; q += nthr) {
            const int m = q / UV_CH, jj = q % UV_CH, j = j0 + jj;
            const int e = (m >> 1) * UV_SB + 2 * jj + (m & 1);
            if (j < N_f) {
                __pipeline_memcpy_async(&hsb[e], &hp[(size_t)m * N_f + j], 16);
                __pipeline_memcpy_async(&hmb[e], &hp[(size_t)m * N_f + (j == 0 ? 0 : N_f - j)], 16);
            } else {
                hsb[e] = make_double2(0.0, 0.0);
                hmb[e] = make_double2(0.0, 0.0);
            }
        }
        for (int q = tid; q < KK * UV_CH; q += nthr) {
            const int k = q / UV_CH, jj = q % UV_CH;
            if (j0 + jj < N_f) __pipeline_memcpy_async(&ws[(buf * KK + k) * UV_CH + jj], &w[(size_t)k * N_f + j0 + jj], 8);
            else ws[(buf * KK + k) * UV_CH + jj] = 0.0;
        }
        __pipeline_commit();
    };
    // three buffers: chunk c + 2 is requested right after the barrier of chunk c, into the buffer chunk c - 1 was read from
    // (every thread is past it), so one barrier per chunk suffices
    if (c_begin < c_end) stage(c_begin, 0);
    if (c_begin + 1 < c_end) stage(c_begin + 1, 1);
    for (int c = c_begin; c < c_end; c++) {
        const int buf = (c - c_begin) % UV_NBUF;
        if (c + 1 < c_end) __pipeline_wait_prior(1); else __pipeline_wait_prior(0);
        __syncthreads();
        if (c + 2 < c_end) stage(c + 2, (c + 2 - c_begin) % UV_NBUF);
        if (act) {
            const double2* xa = hs + (buf * MB + ta) * UV_SB;
            const double2* xm = hm + (buf * MB + ta) * UV_SB;
            const double2* yb = hs + (buf * MB + tb) * UV_SB;
            const double* wk = ws + buf * KK * UV_CH;
#pragma unroll 2
            for (int jj = sub; jj < UV_CH; jj += UV_SUB) {
                double2 x[2], xr[2], y[2];
                x[0] = xa[2 * jj]; x[1] = xa[2 * jj + 1];
                xr[0] = xm[2 * jj]; xr[1] = xm[2 * jj + 1];
                y[0] = yb[2 * jj]; y[1] = yb[2 * jj + 1];
                double wj[KK];
#pragma unroll
                for (int k = 0; k < KK; k++) wj[k] = wk[k * UV_CH + jj];
#pragma unroll
                for (int ia = 0; ia < 2; ia++)
#pragma unroll
                    for (int ib = 0; ib < 2; ib++) {
                        const double cr = x[ia].x * y[ib].x + x[ia].y * y[ib].y, ci = x[ia].x * y[ib].y - x[ia].y * y[ib].x;          // conj(x) y
                        const double vr = xr[ia].x * y[ib].x - xr[ia].y * y[ib].y, vi = xr[ia].x * y[ib].y + xr[ia].y * y[ib].x;      // x(-f) y
#pragma unroll
                        for (int k = 0; k < KK; k++) {
                            acc[ia][ib][k][0] += wj[k] * cr; acc[ia][ib][k][1] += wj[k] * ci;
                            acc[ia][ib][k][2] += wj[k] * vr; acc[ia][ib][k][3] += wj[k] * vi;
                        }
                    }
            }
        }
    }
    __syncthreads();                                                  // the staging buffers are free
    // the sub-slices of a tile meet in shared memory (sub-slice order), one partial per (slice, pair)
    double* red = reinterpret_cast<double*>(uv_sm);                  // [UV_SUB][n_tiles][16 KK], the staging buffers are idle
    if (act) {
#pragma unroll
        for (int e = 0; e < 16 * KK; e++) red[((size_t)sub * n_tiles + tile) * 16 * KK + e] = (&acc[0][0][0][0])[e];
    }
    __syncthreads();
    for (int q = tid; q < n_tiles * 4; q += nthr) {
        const int tl = q >> 2, ia = (q >> 1) & 1, ib = q & 1;
        int qa = 0, rem = tl;
        while (rem >= MB - qa) { rem -= MB - qa; qa++; }
        const int a = 2 * qa + ia, b = 2 * (qa + rem) + ib;
        if (a > b || b >= M) continue;
        const int pr = a * M - a * (a - 1) / 2 + (b - a);          // row-by-row list of the upper triangle (ile_set_modes)
        double* o = part + (((size_t)p * gridDim.x + blockIdx.x) * n_pairs + pr) * KK * 4;
        for (int e = 0; e < 4 * KK; e++) {
            double v = 0.0;
            for (int sb = 0; sb < UV_SUB; sb++) v += red[((size_t)sb * n_tiles + tl) * 16 * KK + (ia * 2 + ib) * 4 * KK + e];
            o[e] = v;
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

// ---------------------------------------------------------------- power-of-two N_f: FFT pruned to the stored window
// Only N_Q <= Mq = 2^q consecutive output times are stored.  With N_f = L Mq and j = L a + b:
//   Q[n] = sum_b W_N^{b n} Y_b[n mod Mq],   Y_b[r] = sum_a x[L a + b] W_Mq^{a r}
// i.e. L inverse FFTs of Mq points over the decimated spectra and one twiddled sum per stored bin: 2/3 of the
// butterflies of the full transform at N_f = 32 Mq, no intermediate in global memory, and the product
// x = w conj(h) d formed while loading.  CTA = one (point, mode, detector) series; PQ_BG decimated spectra at a time
// (contiguous 16 PQ_BG byte reads) go through shared memory: decimation-in-frequency passes of two radix-2 stages with
// twiddles shared by the PQ_BG transforms (exact entries of the sincospi table), bit-reversed output read in place.
#define PQ_THREADS 256
#define PQ_BG 4
// shared-memory index of element i of a transform: one 16-byte pad per 16 elements, so that a thread's 16 contiguous
// elements (register tail) and 8 consecutive elements (passes) both spread over the 8 bank groups
__device__ __forceinline__ int pq_pad(int i) { return i + (i >> 4); }
template <int NOUT>
__global__ void __launch_bounds__(PQ_THREADS, NOUT <= 4 ? 2 : 1) pc_q_pruned_kernel(int M, int K, int N_f, int Mq, int log2Mq, int N_Q, int n0m,
                                                                 const double2* __restrict__ h, const double2* __restrict__ dw,
                                                                 const double2* __restrict__ W, double2* __restrict__ Q) {
    extern __shared__ double2 pq_sm[];
    const int MqP = Mq + (Mq >> 4) + 2;        // stride between the PQ_BG transforms: 2 mod 8 bank groups apart
    double2* tw = pq_sm;                       // [Mq / 2]: W_Mq^m
    double2* xs = pq_sm + (Mq >> 1);           // [PQ_BG][MqP]
    const int tid = threadIdx.x, a_m = blockIdx.x / K, k = blockIdx.x % K, p = blockIdx.y;
    const int L = N_f / Mq;
    const double2* hp = h + ((size_t)p * M + a_m) * N_f;
    const double2* dp = dw + (size_t)k * N_f;
    for (int q = tid; q < (Mq >> 1); q += PQ_THREADS) tw[q] = W[(size_t)q * L];
    // this thread's outputs: the stored bins whose transform output lands at the natural positions tid + 256 u
    // (bit-reversed order of a decimation-in-frequency transform): t_out = (bitrev(pos) - n0) mod Mq, kept if < N_Q
    int t_out[NOUT], n_out[NOUT];
    double2 acc[NOUT], rot[NOUT];
#pragma unroll
    for (int u = 0; u < NOUT; u++) {
        acc[u] = make_double2(0.0, 0.0);
        const int pos = tid + PQ_THREADS * u;
        const int r = (int)(__brev((unsigned)pos) >> (32 - log2Mq));
        t_out[u] = pos < Mq ? ((r - n0m) & (Mq - 1)) : N_Q;
        n_out[u] = (n0m + t_out[u]) & (N_f - 1);
        rot[u] = W[n_out[u]];
    }
    const bool tail16 = (log2Mq & 1) == 0 && log2Mq >= 4 && (Mq >> 4) * PQ_BG <= PQ_THREADS * 4;
    for (int b0 = 0; b0 < L; b0 += PQ_BG) {
        __syncthreads();                                              // the previous group is consumed (and tw is written)
        // x = conj(h) (w d) for PQ_BG consecutive bins of every decimated index a: contiguous 16 PQ_BG byte runs
        for (int e = tid; e < PQ_BG * Mq; e += PQ_THREADS) {
            const int bb = e % PQ_BG, a = e / PQ_BG;
            double2 x = make_double2(0.0, 0.0);
            if (b0 + bb < L) {
                const size_t j = (size_t)L * a + b0 + bb;
                const double2 hh = hp[j], dd = dp[j];
                x = make_double2(hh.x * dd.x + hh.y * dd.y, hh.x * dd.y - hh.y * dd.x);
            }
            xs[bb * MqP + pq_pad(a)] = x;
        }
        __syncthreads();
        int H = Mq >> 1, ts = 1, stages = log2Mq;
        if (tail16 && stages >= 8) {
            // the first four stages (quarters Mq/4 and Mq/16) on 16 elements Mq/16 apart in registers: thread = (transform, offset)
            const int q2 = Mq >> 4;
            for (int it = tid; it < q2 * PQ_BG; it += PQ_THREADS) {
                const int i0 = it % q2;
                double2* sm = xs + (it / q2) * MqP;
                double2 v[16];
#pragma unroll
                for (int m = 0; m < 16; m++) v[m] = sm[pq_pad(i0 + q2 * m)];
#pragma unroll
                for (int c = 0; c < 4; c++) {                 // quarter Mq/4: elements c, c + 4, c + 8, c + 12
                    const int pos = i0 + q2 * c;
                    const double2 w1 = tw[pos], w2 = tw[2 * pos];
                    const double2 x0 = v[c], x1 = v[c + 4], x2 = v[c + 8], x3 = v[c + 12];
                    const double2 y0 = make_double2(x0.x + x2.x, x0.y + x2.y), y1 = make_double2(x1.x + x3.x, x1.y + x3.y);
                    const double ar = x0.x - x2.x, ai = x0.y - x2.y, br = x1.x - x3.x, bi = x1.y - x3.y;
                    const double2 y2 = make_double2(ar * w1.x - ai * w1.y, ar * w1.y + ai * w1.x);
                    const double2 y3 = make_double2(-(br * w1.y + bi * w1.x), br * w1.x - bi * w1.y);
                    const double cr = y0.x - y1.x, ci = y0.y - y1.y, dr = y2.x - y3.x, di = y2.y - y3.y;
                    v[c] = make_double2(y0.x + y1.x, y0.y + y1.y);
                    v[c + 4] = make_double2(cr * w2.x - ci * w2.y, cr * w2.y + ci * w2.x);
                    v[c + 8] = make_double2(y2.x + y3.x, y2.y + y3.y);
                    v[c + 12] = make_double2(dr * w2.x - di * w2.y, dr * w2.y + di * w2.x);
                }
                {
                    const double2 w1 = tw[4 * i0], w2 = tw[8 * i0];   // quarter Mq/16: elements 4 r .. 4 r + 3, one twiddle pair
#pragma unroll
                    for (int r = 0; r < 4; r++) {
                        const double2 x0 = v[4 * r], x1 = v[4 * r + 1], x2 = v[4 * r + 2], x3 = v[4 * r + 3];
                        const double2 y0 = make_double2(x0.x + x2.x, x0.y + x2.y), y1 = make_double2(x1.x + x3.x, x1.y + x3.y);
                        const double ar = x0.x - x2.x, ai = x0.y - x2.y, br = x1.x - x3.x, bi = x1.y - x3.y;
                        const double2 y2 = make_double2(ar * w1.x - ai * w1.y, ar * w1.y + ai * w1.x);
                        const double2 y3 = make_double2(-(br * w1.y + bi * w1.x), br * w1.x - bi * w1.y);
                        const double cr = y0.x - y1.x, ci = y0.y - y1.y, dr = y2.x - y3.x, di = y2.y - y3.y;
                        v[4 * r] = make_double2(y0.x + y1.x, y0.y + y1.y);
                        v[4 * r + 1] = make_double2(cr * w2.x - ci * w2.y, cr * w2.y + ci * w2.x);
                        v[4 * r + 2] = make_double2(y2.x + y3.x, y2.y + y3.y);
                        v[4 * r + 3] = make_double2(dr * w2.x - di * w2.y, dr * w2.y + di * w2.x);
                    }
                }
#pragma unroll
                for (int m = 0; m < 16; m++) sm[pq_pad(i0 + q2 * m)] = v[m];
            }
            __syncthreads();
            H >>= 4;
            ts <<= 4;
            stages -= 4;
        }
        while (stages >= 2 && !(tail16 && stages == 4)) {
            const int q = H >> 1;
            for (int t = tid; t < (Mq >> 2); t += PQ_THREADS) {
                const int pos = t & (q - 1), i0 = ((t - pos) << 2) + pos;
                const double2 w1 = tw[pos * ts], w2 = tw[pos * 2 * ts];
                const int e0 = pq_pad(i0), e1 = pq_pad(i0 + q), e2 = pq_pad(i0 + 2 * q), e3 = pq_pad(i0 + 3 * q);
#pragma unroll
                for (int bb = 0; bb < PQ_BG; bb++) {
                    double2* sm = xs + bb * MqP;
                    const double2 x0 = sm[e0], x1 = sm[e1], x2 = sm[e2], x3 = sm[e3];
                    const double2 y0 = make_double2(x0.x + x2.x, x0.y + x2.y), y1 = make_double2(x1.x + x3.x, x1.y + x3.y);
                    const double ar = x0.x - x2.x, ai = x0.y - x2.y, br = x1.x - x3.x, bi = x1.y - x3.y;
                    const double2 y2 = make_double2(ar * w1.x - ai * w1.y, ar * w1.y + ai * w1.x);
                    const double2 y3 = make_double2(-(br * w1.y + bi * w1.x), br * w1.x - bi * w1.y);      // (x1 - x3) i w1
                    const double cr = y0.x - y1.x, ci = y0.y - y1.y, dr = y2.x - y3.x, di = y2.y - y3.y;
                    sm[e0] = make_double2(y0.x + y1.x, y0.y + y1.y);
                    sm[e1] = make_double2(cr * w2.x - ci * w2.y, cr * w2.y + ci * w2.x);
                    sm[e2] = make_double2(y2.x + y3.x, y2.y + y3.y);
                    sm[e3] = make_double2(dr * w2.x - di * w2.y, dr * w2.y + di * w2.x);
                }
            }
            __syncthreads();
            H >>= 2;
            ts <<= 2;
            stages -= 2;
        }
        if (tail16) {
            // the last four stages on 16 contiguous elements in registers: thread = (transform, block of 16)
            const int nblk = Mq >> 4;
            for (int it = tid; it < nblk * PQ_BG; it += PQ_THREADS) {
                double2* sm = xs + (it / nblk) * MqP + pq_pad((it % nblk) << 4);
                double2 v[16];
#pragma unroll
                for (int e = 0; e < 16; e++) v[e] = sm[e];
                // stages with halves 8 and 4 (quarter q = 4): twiddles W_16^pos, W_8^pos
#pragma unroll
                for (int pos = 0; pos < 4; pos++) {
                    const double2 w1 = tw[pos * (Mq >> 4)], w2 = tw[pos * (Mq >> 3)];
                    const double2 x0 = v[pos], x1 = v[pos + 4], x2 = v[pos + 8], x3 = v[pos + 12];
                    const double2 y0 = make_double2(x0.x + x2.x, x0.y + x2.y), y1 = make_double2(x1.x + x3.x, x1.y + x3.y);
                    const double ar = x0.x - x2.x, ai = x0.y - x2.y, br = x1.x - x3.x, bi = x1.y - x3.y;
                    const double2 y2 = make_double2(ar * w1.x - ai * w1.y, ar * w1.y + ai * w1.x);
                    const double2 y3 = make_double2(-(br * w1.y + bi * w1.x), br * w1.x - bi * w1.y);
                    const double cr = y0.x - y1.x, ci = y0.y - y1.y, dr = y2.x - y3.x, di = y2.y - y3.y;
                    v[pos] = make_double2(y0.x + y1.x, y0.y + y1.y);
                    v[pos + 4] = make_double2(cr * w2.x - ci * w2.y, cr * w2.y + ci * w2.x);
                    v[pos + 8] = make_double2(y2.x + y3.x, y2.y + y3.y);
                    v[pos + 12] = make_double2(dr * w2.x - di * w2.y, dr * w2.y + di * w2.x);
                }
                // stages with halves 2 and 1 (quarter q = 1): twiddle 1, and i on the odd difference
#pragma unroll
                for (int g4 = 0; g4 < 4; g4++) {
                    const double2 x0 = v[4 * g4], x1 = v[4 * g4 + 1], x2 = v[4 * g4 + 2], x3 = v[4 * g4 + 3];
                    const double2 y0 = make_double2(x0.x + x2.x, x0.y + x2.y), y1 = make_double2(x1.x + x3.x, x1.y + x3.y);
                    const double2 y2 = make_double2(x0.x - x2.x, x0.y - x2.y);
                    const double2 y3 = make_double2(-(x1.y - x3.y), x1.x - x3.x);                          // (x1 - x3) i
                    v[4 * g4] = make_double2(y0.x + y1.x, y0.y + y1.y);
                    v[4 * g4 + 1] = make_double2(y0.x - y1.x, y0.y - y1.y);
                    v[4 * g4 + 2] = make_double2(y2.x + y3.x, y2.y + y3.y);
                    v[4 * g4 + 3] = make_double2(y2.x - y3.x, y2.y - y3.y);
                }
#pragma unroll
                for (int e = 0; e < 16; e++) sm[e] = v[e];
            }
            __syncthreads();
        } else if (stages == 1) {                            // H == 1: last butterflies, twiddle 1
            for (int t = tid; t < (Mq >> 1); t += PQ_THREADS) {
                const int e0 = pq_pad(2 * t), e1 = pq_pad(2 * t + 1);
#pragma unroll
                for (int bb = 0; bb < PQ_BG; bb++) {
                    double2* sm = xs + bb * MqP;
                    const double2 u = sm[e0], v = sm[e1];
                    sm[e0] = make_double2(u.x + v.x, u.y + v.y);
                    sm[e1] = make_double2(u.x - v.x, u.y - v.y);
                }
            }
            __syncthreads();
        }
#pragma unroll
        for (int u = 0; u < NOUT; u++) {
            if (t_out[u] < N_Q) {
                const int e = pq_pad(tid + PQ_THREADS * u);
                // W_N^{(b0 + bb) n}: an exact table entry for bb = 0, then PQ_BG - 1 rotations by W_N^n
                double2 f = W[(int)(((long long)b0 * n_out[u]) & (N_f - 1))];
#pragma unroll
                for (int bb = 0; bb < PQ_BG; bb++) {
                    const double2 y = xs[bb * MqP + e];
                    acc[u].x += y.x * f.x - y.y * f.y;
                    acc[u].y += y.x * f.y + y.y * f.x;
                    const double fr = f.x * rot[u].x - f.y * rot[u].y;
                    f.y = f.x * rot[u].y + f.y * rot[u].x;
                    f.x = fr;
                }
            }
        }
    }
    double2* Qp = Q + (((size_t)p * K + k) * M + a_m) * N_Q;
#pragma unroll
    for (int u = 0; u < NOUT; u++)
        if (t_out[u] < N_Q) Qp[t_out[u]] = acc[u];
}

template <int NOUT>
static void launch_q_pruned(int P, int M, int K, int N_f, int Mq, int log2Mq, int N_Q, int n0m, const double2* h, const double2* dw,
                            const double2* W, double2* Q, cudaStream_t st) {
    const size_t smem = ((size_t)(Mq >> 1) + (size_t)PQ_BG * (Mq + (Mq >> 4) + 2)) * sizeof(double2);
    cudaFuncSetAttribute(pc_q_pruned_kernel<NOUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    pc_q_pruned_kernel<NOUT><<<dim3(M * K, P), PQ_THREADS, smem, st>>>(M, K, N_f, Mq, log2Mq, N_Q, n0m, h, dw, W, Q);
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
    if (M > ILE_QT_ROW / 2 - 2 || K > 4)                       // the limit of ile_load_quv, which installs the result
        return ile_fail(ctx, ILE_EINVAL, "precompute_quv: at most %d modes and 4 detectors", ILE_QT_ROW / 2 - 2);
    int Mq = 4, log2Mq = 2;
    while (Mq < N_Q) { Mq <<= 1; log2Mq++; }
    const bool pruned = (N_f & (N_f - 1)) == 0 && Mq <= 2048 && Mq <= N_f;
    const size_t nX = pruned ? 0 : (size_t)P * K * M * N_f;
    // frequency slices per point: two CTAs per SM in all, at least one chunk each; UV_SUB partial sums per slice
    const int chunks = (N_f + UV_CH - 1) / UV_CH;
    int slices = 2 * ctx->sm_count / P;
    if (slices < 1) slices = 1;
    if (slices > chunks) slices = chunks;
    const int cpb = (chunks + slices - 1) / slices;
    slices = (chunks + cpb - 1) / cpb;
    const int nsl = slices;
    const size_t nPart = (size_t)P * nsl * n_pairs * K * 4;
    // one grow-only scratch allocation: W | w | w d | x | part  (256-byte aligned pieces)
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t o_W = 0, o_w = o_W + al((size_t)N_f * 16), o_dw = o_w + al((size_t)K * N_f * 8), o_x = o_dw + al((size_t)K * N_f * 16), o_p = o_x + al(nX * 16),
                 total = o_p + al(nPart * 8);
    if (total > ctx->pc_bytes) {
        cudaStreamSynchronize(ctx->stream);
        cudaFree(ctx->pc_buf);
        ctx->pc_buf = nullptr;
        ctx->pc_bytes = 0;
        ctx->pc_W_nf = 0;
        if (cudaMalloc(&ctx->pc_buf, total) != cudaSuccess) {
            cudaGetLastError();
            return ile_fail(ctx, ILE_ENOMEM, "precompute_quv: device allocation of %zu bytes failed", total);
        }
        ctx->pc_bytes = total;
    }
    // the results go straight into the context's arrays
    {
        const int rc = ile_quv_alloc(ctx, P, N_Q);
        if (rc) return rc;
    }
    char* buf = (char*)ctx->pc_buf;
    double* w = (double*)(buf + o_w);
    double2 *W = (double2*)(buf + o_W), *x = (double2*)(buf + o_x), *Q = (double2*)ctx->d_Qc, *U = (double2*)ctx->d_U, *V = (double2*)ctx->d_V;
    double* part = (double*)(buf + o_p);
    double2* dwp = (double2*)(buf + o_dw);
    cudaStream_t st = ctx->stream;
    pc_weight_kernel<<<dim3((N_f + 255) / 256, K), 256, 0, st>>>(K, N_f, df, f_low, S, (const double2*)d, w, dwp);
    if (ctx->pc_W_nf != N_f) {                                             // the table survives in the scratch between calls
        pc_twiddle_kernel<<<(N_f + 255) / 256, 256, 0, st>>>(N_f, W);
        ctx->pc_W_nf = N_f;
    }
    {
        const int MB = (M + 1) / 2, uv_threads = (MB * (MB + 1) / 2 * UV_SUB + 31) / 32 * 32;
        const size_t uv_stage = (size_t)2 * UV_NBUF * MB * UV_SB * sizeof(double2) + (size_t)UV_NBUF * K * UV_CH * sizeof(double);
        const size_t uv_red = (size_t)UV_SUB * (MB * (MB + 1) / 2) * 16 * K * sizeof(double);
        const size_t uv_smem = uv_stage > uv_red ? uv_stage : uv_red;
        const double2* hh = (const double2*)h;
#define UV_CASE(KK_)                                                                                                        \
    case KK_:                                                                                                               \
        if (uv_threads > 352) {                                                                                             \
            ILE_CUDA(ctx, cudaFuncSetAttribute(pc_uv_kernel<KK_, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)uv_smem));  \
            pc_uv_kernel<KK_, true><<<dim3(slices, P), uv_threads, uv_smem, st>>>(M, N_f, n_pairs, cpb, hh, w, part);       \
        } else {                                                                                                            \
            ILE_CUDA(ctx, cudaFuncSetAttribute(pc_uv_kernel<KK_, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)uv_smem)); \
            pc_uv_kernel<KK_, false><<<dim3(slices, P), uv_threads, uv_smem, st>>>(M, N_f, n_pairs, cpb, hh, w, part);      \
        }                                                                                                                   \
        break;
        switch (K) { UV_CASE(1) UV_CASE(2) UV_CASE(3) UV_CASE(4) }
#undef UV_CASE
    }
    pc_uv_finish_kernel<<<(P * n_pairs * K + 255) / 256, 256, 0, st>>>(P, M, K, n_pairs, nsl, ctx->d_pairs, part, U, V);
    if (pruned) {                                                           // FFT pruned to the window: no intermediate
        long long n0m = n0 % N_f;
        if (n0m < 0) n0m += N_f;
        const double2* hh = (const double2*)h;
        const int nout = (Mq + PQ_THREADS - 1) / PQ_THREADS;
        switch (nout) {
            case 1: launch_q_pruned<1>(P, M, K, N_f, Mq, log2Mq, N_Q, (int)n0m, hh, dwp, W, Q, st); break;
            case 2: launch_q_pruned<2>(P, M, K, N_f, Mq, log2Mq, N_Q, (int)n0m, hh, dwp, W, Q, st); break;
            case 4: launch_q_pruned<4>(P, M, K, N_f, Mq, log2Mq, N_Q, (int)n0m, hh, dwp, W, Q, st); break;
            default: launch_q_pruned<8>(P, M, K, N_f, Mq, log2Mq, N_Q, (int)n0m, hh, dwp, W, Q, st); break;
        }
    } else {
        pc_prod_kernel<<<dim3((N_f + 255) / 256, K * M, P), 256, 0, st>>>(M, K, N_f, (const double2*)h, (const double2*)d, w, x);
        pc_q_kernel<<<dim3((N_Q + 127) / 128, K * M, P), 128, 0, st>>>(N_f, N_Q, (int)n0, x, W, w, M, Q);
    }
    ctx->launches += 6;
    ILE_LAUNCH_CHECK(ctx);
    return ile_load_quv_impl(ctx, P, N_Q, fs, (double)n0 / fs, (const double*)Q, (const double*)U, (const double*)V, D_ref, 1, true);
}

// Copies the resident Q/U/V of intrinsic point p to host arrays (caller layout of ile_load_quv).
extern "C" int ile_get_quv(ile_ctx* ctx, int p, double* Q, double* U, double* V) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (!ctx->have_quv) return ile_fail(ctx, ILE_ESTATE, "get_quv: nothing loaded");
    if (p < 0 || p >= ctx->P) return ile_fail(ctx, ILE_EINVAL, "get_quv: point out of range");
    const size_t nQ = (size_t)ctx->K * ctx->M * ctx->N_Q * 2, nU = (size_t)ctx->K * ctx->M * ctx->M * 2;
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (Q) ILE_CUDA(ctx, cudaMemcpy(Q, ctx->d_Qc + (size_t)p * nQ, nQ * 8, cudaMemcpyDeviceToHost));
    if (U) ILE_CUDA(ctx, cudaMemcpy(U, ctx->d_U + (size_t)p * nU, nU * 8, cudaMemcpyDeviceToHost));
    if (V) ILE_CUDA(ctx, cudaMemcpy(V, ctx->d_V + (size_t)p * nU, nU * 8, cudaMemcpyDeviceToHost));
    return ILE_OK;
}
