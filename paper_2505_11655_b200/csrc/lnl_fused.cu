// libile: the fused lnL path, B200-native.
//
//   prep kernel   (steps 1-4)  one thread per sample, in sky-sorted order: F_k, tau_k, Y_lm, x, the
//                              U/V quadratic term B -> a 12 KB Y tile per 32 samples + 16 doubles
//   fused kernel  (steps 5-6)  one CTA per 32-sample tile.  S_k[i][n] = sum_r coef_k[i][r] Q_k[r][n]
//                              is a dense real GEMM (K-dim 2M) on the FP64 tensor pipe (DMMA.8x8x4);
//                              Q windows are TMA bulk-copied into shared memory; the per-sample,
//                              per-detector arrival-time shift and the linear interpolation are
//                              applied when the epilogue reads S from a shared-memory ring; time
//                              marginalisation is a warp-level log-sum-exp (one warp per sample).
// DESIGN.md section 6 derives the tiling and the roofline.
#include "common.cuh"
#include "likelihood_dev.cuh"
#include "radix_sort.cuh"

#define FT_TS 32          // samples per CTA
#define FT_THREADS 256
#define FT_RING 80        // S ring length in stored bins
#define FT_SROW 88        // S row stride (== 8 mod 16: conflict-free 128-bit fragment stores)
#define FT_NEW 64         // new stored bins per phase (phase 0: FT_RING)
#define FT_CAP 15         // largest per-sample offset above the tile base handled in one round
#define FT_YM 24          // mode slots in the Y tile
#define FT_REC 16         // doubles per sample record

// ---------------------------------------------------------------- sky sort
// The fused kernel handles a tile of 32 samples in one round when, for every detector, their
// first-bin indices n_k = floor(u_k) lie within FT_CAP of the tile minimum.  n_k depends on the
// sky position only, so samples are ordered by the cell (n_k >> 3)_k of their delays: one key
// per sample, radix-sorted on the device with the sample index as payload (-> perm).
#define SKY_CELL_SHIFT 3
__global__ void __launch_bounds__(256) sky_key_kernel(LnlParams P, int N, const double* __restrict__ z, int n_min, int cell_bits,
                                                      unsigned long long* __restrict__ key, unsigned int* __restrict__ val, long long* n_dev,
                                                      int* bits_dev) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        *n_dev = N;
        *bits_dev = cell_bits * P.K + 1;
    }
    if (i >= N) return;
    const double ra = z[i], sd = z[(size_t)N + i];
    bool ok = true;
    for (int c = 0; c < P.d; c++) {
        const double v = z[(size_t)c * N + i];
        ok = ok && (v >= P.lo[c]) && (v < P.hi[c]);
    }
    unsigned long long k = 1ull << (cell_bits * P.K);      // out-of-box samples last
    if (ok) {
        const double cd = sqrt(fmax((1.0 - sd) * (1.0 + sd), 0.0));
        double sg, cg;
        sincos(P.gmst - ra, &sg, &cg);
        const double n0 = cd * cg, n1 = -cd * sg, n2 = sd;
        k = 0;
        for (int kk = 0; kk < P.K; kk++) {
            const double tau = -(P.pos[kk][0] * n0 + P.pos[kk][1] * n1 + P.pos[kk][2] * n2) / ILE_C_LIGHT;
            double u = (P.t_lo + tau - P.t_Q0) * P.fs;
            if (!P.interp) u = floor(u + 0.5);
            int cell = ((int)floor(u) - n_min) >> SKY_CELL_SHIFT;
            cell = max(0, min(cell, (1 << cell_bits) - 1));
            k = (k << cell_bits) | (unsigned long long)cell;
        }
    }
    key[i] = k;
    val[i] = (unsigned int)i;
}

// ---------------------------------------------------------------- prep kernel
// rec[t][0..3]=Re F_k, [4..7]=Im F_k (F = F+ - iFx), [8..11]=u_k (stored-bin coordinate of grid
// time 0 at detector k), [12]=x, [13]=B, [14]=valid, [15]=ln prior.
// ytile[t/32][m][t%32] = (Re, Im) Y_m, zero for m >= M.
__global__ void __launch_bounds__(128) lnl_prep_kernel(LnlParams P, int N, int Npad, const double* __restrict__ z, const int* __restrict__ perm,
                                                       double* __restrict__ rec, double2* __restrict__ ytile, double* __restrict__ ln_prior) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Npad) return;
    double2* yt = ytile + (size_t)(t / FT_TS) * FT_YM * FT_TS + (t % FT_TS);
    double* r = rec + (size_t)t * FT_REC;
    bool valid = false;
    SampleIn s;
    int i = -1;
    if (t < N) {
        i = perm ? perm[t] : t;
        s = sample_from_z(P, z, N, i);
        valid = s.valid;
        if (ln_prior) ln_prior[i] = valid ? ln_prior_dev(P, s) : neg_inf();
    }
    if (!valid) {
        for (int m = 0; m < FT_YM; m++) yt[m * FT_TS] = make_double2(0.0, 0.0);
        for (int q = 0; q < FT_REC; q++) r[q] = 0.0;
        return;
    }
    double Fp[ILE_MAX_K], Fx[ILE_MAX_K], tau[ILE_MAX_K], Yr[ILE_MAX_M], Yi[ILE_MAX_M];
    antenna_dev(P, s, Fp, Fx, tau);
    ylm_dev(P.ylm, s.ch, s.sh, -s.phi_ref, [&](int m, double yr, double yi) { Yr[m] = yr; Yi[m] = yi; });
    // quadratic term with the Eq. 17-18 symmetries: upper triangle only
    const int M = P.M;
    double B = 0.0;
    {
        double uu[ILE_MAX_K], vr[ILE_MAX_K], vi[ILE_MAX_K];
        for (int k = 0; k < P.K; k++) uu[k] = vr[k] = vi[k] = 0.0;
        for (int a = 0; a < M; a++)
            for (int b = a; b < M; b++) {
                double w = (a == b) ? 1.0 : 2.0;
                double pr = w * (Yr[a] * Yr[b] + Yi[a] * Yi[b]), pi = w * (Yr[a] * Yi[b] - Yi[a] * Yr[b]);   // conj(y_a) y_b
                double qr = w * (Yr[a] * Yr[b] - Yi[a] * Yi[b]), qi = w * (Yr[a] * Yi[b] + Yi[a] * Yr[b]);   // y_a y_b
                for (int k = 0; k < P.K; k++) {
                    const double2 u = __ldg((const double2*)(P.U + ((size_t)k * M * M + a * M + b) * 2));
                    const double2 v = __ldg((const double2*)(P.V + ((size_t)k * M * M + a * M + b) * 2));
                    uu[k] += u.x * pr - u.y * pi;
                    vr[k] += v.x * qr - v.y * qi;
                    vi[k] += v.x * qi + v.y * qr;
                }
            }
        for (int k = 0; k < P.K; k++) {
            double fr = Fp[k], fi = -Fx[k];
            B += (fr * fr + fi * fi) * uu[k] + ((fr * fr - fi * fi) * vr[k] - 2.0 * fr * fi * vi[k]);
        }
        B *= 0.25;
    }
    for (int m = 0; m < FT_YM; m++) yt[m * FT_TS] = (m < M) ? make_double2(Yr[m], Yi[m]) : make_double2(0.0, 0.0);
    for (int k = 0; k < ILE_MAX_K; k++) {
        double u = 0.0;
        if (k < P.K) {
            u = (P.t_lo + tau[k] - P.t_Q0) * P.fs;
            if (!P.interp) u = floor(u + 0.5);
        }
        r[k] = k < P.K ? Fp[k] : 0.0;
        r[4 + k] = k < P.K ? -Fx[k] : 0.0;
        r[8 + k] = u;
    }
    r[12] = P.use_table ? 1.0 : P.D_ref / s.dist;
    r[13] = B;
    r[14] = 1.0;
    r[15] = 0.0;
}

// ---------------------------------------------------------------- prep kernel without the quadratic term
// Steps 1-3 only (antenna, delays, harmonics, x, ln prior): one thread per sample, Y_m stored
// straight into the tile (no per-thread arrays).  The U/V quadratic term B (step 4) is computed by
// the fused kernel's prologue, where 8 threads share each sample.  rec[13] = 0 here.
__global__ void __launch_bounds__(128) lnl_prep3_kernel(LnlParams P, int N, int Npad, int scr_doubles, const double* __restrict__ z,
                                                        const int* __restrict__ perm, double* __restrict__ rec, double2* __restrict__ ytile,
                                                        double* __restrict__ ln_prior) {
    // shared memory: the harmonics' per-thread power and phase tables, then a copy of the mode table
    extern __shared__ __align__(16) double prep_scr[];
    YlmTable* tab = reinterpret_cast<YlmTable*>(prep_scr + scr_doubles);
    {
        const int4* src = reinterpret_cast<const int4*>(P.ylm);
        int4* dst = reinterpret_cast<int4*>(tab);
        const int n16 = (int)((offsetof(YlmTable, mode) + (size_t)P.M * sizeof(YlmMode) + 15) / 16);
        for (int q = threadIdx.x; q < n16; q += blockDim.x) dst[q] = src[q];
    }
    __syncthreads();
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Npad) return;
    double2* yt = ytile + (size_t)(t / FT_TS) * FT_YM * FT_TS + (t % FT_TS);
    double* r = rec + (size_t)t * FT_REC;
    bool valid = false;
    SampleIn s;
    if (t < N) {
        const int i = perm ? perm[t] : t;
        s = sample_from_z(P, z, N, i);
        valid = s.valid;
        if (ln_prior) ln_prior[i] = valid ? ln_prior_dev(P, s) : neg_inf();
    }
    if (!valid) {
        for (int m = 0; m < FT_YM; m++) yt[m * FT_TS] = make_double2(0.0, 0.0);
        for (int q = 0; q < FT_REC; q += 2) *reinterpret_cast<double2*>(r + q) = make_double2(0.0, 0.0);
        return;
    }
    double Fp[ILE_MAX_K], Fx[ILE_MAX_K], tau[ILE_MAX_K];
    antenna_dev(P, s, Fp, Fx, tau);
    ylm_dev_smem(tab, s.ch, s.sh, -s.phi_ref, prep_scr + threadIdx.x, blockDim.x, [&](int m, double yr, double yi) { yt[m * FT_TS] = make_double2(yr, yi); });
    for (int m = P.M; m < FT_YM; m++) yt[m * FT_TS] = make_double2(0.0, 0.0);
    double u[ILE_MAX_K];
#pragma unroll
    for (int k = 0; k < ILE_MAX_K; k++) {
        u[k] = 0.0;
        if (k < P.K) {
            u[k] = (P.t_lo + tau[k] - P.t_Q0) * P.fs;
            if (!P.interp) u[k] = floor(u[k] + 0.5);
        } else {
            Fp[k] = Fx[k] = 0.0;
        }
    }
    double2* r2 = reinterpret_cast<double2*>(r);
    r2[0] = make_double2(Fp[0], Fp[1]);
    r2[1] = make_double2(Fp[2], Fp[3]);
    r2[2] = make_double2(-Fx[0], -Fx[1]);
    r2[3] = make_double2(-Fx[2], -Fx[3]);
    r2[4] = make_double2(u[0], u[1]);
    r2[5] = make_double2(u[2], u[3]);
    r2[6] = make_double2(P.use_table ? 1.0 : P.D_ref / s.dist, 0.0);
    r2[7] = make_double2(1.0, 0.0);
}

// ---------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" ::"r"(
            smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// TMA 1-D bulk copy global -> shared, completion on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// FP64 tensor-core MMA, D(8x8) += A(8x4) * B(4x8)  (SASS: DMMA.8x8x4)
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

struct FusedSmem {
    double Q[3][FT_RING][ILE_QT_ROW];   // staged Q windows, one per detector        92,160 B
    double S[3][FT_TS][FT_SROW];        // S_k[sample][ring bin]                       67,584 B
    double2 Y[FT_YM][FT_TS];            // Y_m per sample                              12,288 B
    double rec[FT_TS][FT_REC];          //                                              4,096 B
    double frac[3][FT_TS];
    int n[3][FT_TS];
    int base[4];
    int part[FT_TS];
    int done[FT_TS];
    int n_part, n_left;
    unsigned long long bar;
};

// ---------------------------------------------------------------- fused kernel
template <int NPAIR, bool SINGLE>
__global__ void __launch_bounds__(FT_THREADS, 1)
lnl_fused_kernel(LnlParams P, int N, const double* __restrict__ rec, const double2* __restrict__ ytile, const int* __restrict__ perm,
                 double* __restrict__ lnL) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    FusedSmem& sm = *reinterpret_cast<FusedSmem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int tile = blockIdx.x;
    const int K = P.K, stride = P.stride, N_t = P.N_t;

    // ---- stage the tile's records and Y table
    {
        const double* src = rec + (size_t)tile * FT_TS * FT_REC;
        for (int q = tid; q < FT_TS * FT_REC; q += FT_THREADS) (&sm.rec[0][0])[q] = src[q];
        const double2* ys = ytile + (size_t)tile * FT_YM * FT_TS;
        for (int q = tid; q < FT_YM * FT_TS; q += FT_THREADS) (&sm.Y[0][0])[q] = ys[q];
        if (tid == 0) mbar_init((uint64_t*)&sm.bar, 1);
    }
    __syncthreads();
    if (tid < FT_TS) {
        bool valid = sm.rec[tid][14] != 0.0;
        sm.done[tid] = valid ? 0 : 1;
        for (int k = 0; k < K; k++) {
            double u = sm.rec[tid][8 + k];
            double fl = floor(u);
            sm.n[k][tid] = (int)fl;
            sm.frac[k][tid] = u - fl;
        }
        if (!valid) {
            int t = tile * FT_TS + tid;
            if (t < N) lnL[perm ? perm[t] : t] = neg_inf();
        }
    }
    uint32_t bar_parity = 0;
    const int half = w >> 2;           // which 16 samples this warp multiplies
    const int c = lane & 3, rq = lane >> 2;

    for (;;) {   // rounds: normally one; more only when the tile's delay spread exceeds FT_CAP
        __syncthreads();
        if (w == 0) {
            int dn = sm.done[lane];
            int base[3];
            for (int k = 0; k < K; k++) {
                int v = dn ? 0x7fffffff : sm.n[k][lane];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, o));
                base[k] = v & ~1;
            }
            bool q = !dn;
            for (int k = 0; k < K; k++) q = q && (sm.n[k][lane] - base[k] <= FT_CAP);
            unsigned mask = __ballot_sync(0xffffffffu, q);
            unsigned left = __ballot_sync(0xffffffffu, !dn);
            if (left != 0 && mask == 0) {   // pivot on the first unfinished sample: always progresses
                int piv = __ffs(left) - 1;
                for (int k = 0; k < K; k++) base[k] = sm.n[k][piv] & ~1;
                q = !dn;
                for (int k = 0; k < K; k++) q = q && (sm.n[k][lane] >= base[k]) && (sm.n[k][lane] - base[k] <= FT_CAP);
                mask = __ballot_sync(0xffffffffu, q);
            }
            sm.part[lane] = q ? 1 : 0;
            if (lane == 0) {
                for (int k = 0; k < K; k++) sm.base[k] = base[k];
                sm.n_part = __popc(mask);
                sm.n_left = __popc(left);
            }
        }
        __syncthreads();
        if (sm.n_left == 0) break;

        // running log-sum-exp state of this warp's 4 samples (lane-partial sums, warp-uniform max)
        double run_m[4], run_s[4];
#pragma unroll
        for (int q = 0; q < 4; q++) { run_m[q] = neg_inf(); run_s[q] = 0.0; }

        const int last_bin = stride * (N_t - 1) + 1 + FT_CAP;   // highest stored bin (relative to base) any sample reads
        int c_lo = 0, j0 = 0;
        // first copy
        int ntiles = min(FT_RING / 8, (last_bin + 1 - c_lo + 7) / 8);
        if (tid == 0) {
            mbar_expect_tx((uint64_t*)&sm.bar, (uint32_t)(K * ntiles * 8 * ILE_QT_ROW * 8));
            for (int k = 0; k < K; k++)
                bulk_g2s(&sm.Q[k][0][0], P.Qt + ((size_t)k * P.N_Qpad + sm.base[k] + c_lo) * ILE_QT_ROW, (uint32_t)(ntiles * 8 * ILE_QT_ROW * 8),
                         (uint64_t*)&sm.bar);
        }
        for (int phase = 0;; phase++) {
            const int c_hi = c_lo + ntiles * 8;
            int j1 = (c_hi - 1 - FT_CAP - 1) / stride + 1;      // outputs whose reads are all below c_hi
            if (j1 > N_t) j1 = N_t;
            mbar_wait((uint64_t*)&sm.bar, bar_parity);
            bar_parity ^= 1;

            // ---------------- MMA: S_k[16 samples][8 bins] tiles on the FP64 tensor pipe
            {
                const int nunits = K * ntiles;
                int cur_k = -1;
                double a[2][2 * NPAIR + (SINGLE ? 1 : 0)];
                for (int u = (w & 3); u < nunits; u += 4) {
                    const int k = u / ntiles, t = u - k * ntiles;
                    if (k != cur_k) {
                        cur_k = k;
#pragma unroll
                        for (int g = 0; g < 2; g++) {
                            const int s = 16 * half + 8 * g + rq;
                            const double fr = sm.rec[s][k], fi = sm.rec[s][4 + k];
#pragma unroll
                            for (int p = 0; p < NPAIR; p++) {
                                const double2 y = sm.Y[4 * p + c][s];
                                a[g][2 * p] = fr * y.x - fi * y.y;       // Re(F Y)
                                a[g][2 * p + 1] = fr * y.y + fi * y.x;   // Im(F Y)
                            }
                            if (SINGLE) {
                                const double2 y = sm.Y[4 * NPAIR + (c >> 1)][s];
                                a[g][2 * NPAIR] = (c & 1) ? fr * y.y + fi * y.x : fr * y.x - fi * y.y;
                            }
                        }
                    }
                    const int row = 8 * t + rq;
                    const int swz = (row & 1) << 3;
                    const double* qrow = &sm.Q[k][row][0];
                    double b[2 * NPAIR + (SINGLE ? 1 : 0)];
#pragma unroll
                    for (int p = 0; p < NPAIR; p++) {
                        const double2 v = *reinterpret_cast<const double2*>(qrow + ((8 * p + 2 * c) ^ swz));
                        b[2 * p] = v.x;
                        b[2 * p + 1] = v.y;
                    }
                    if (SINGLE) b[2 * NPAIR] = qrow[(8 * NPAIR + c) ^ swz];
                    double d00 = 0.0, d01 = 0.0, d10 = 0.0, d11 = 0.0;
#pragma unroll
                    for (int q = 0; q < 2 * NPAIR + (SINGLE ? 1 : 0); q++) {
                        dmma(d00, d01, a[0][q], b[q]);
                        dmma(d10, d11, a[1][q], b[q]);
                    }
                    const int col = (c_lo + 8 * t) % FT_RING + 2 * c;
                    *reinterpret_cast<double2*>(&sm.S[k][16 * half + rq][col]) = make_double2(d00, d01);
                    *reinterpret_cast<double2*>(&sm.S[k][16 * half + 8 + rq][col]) = make_double2(d10, d11);
                }
            }
            __syncthreads();   // S complete; Q buffers free

            // ---------------- prefetch the next phase's Q windows while the epilogue runs
            const bool more = j1 < N_t;
            int next_lo = c_hi, next_tiles = 0;
            if (more) {
                next_tiles = min(FT_NEW / 8, (last_bin + 1 - next_lo + 7) / 8);
                if (tid == 0) {
                    mbar_expect_tx((uint64_t*)&sm.bar, (uint32_t)(K * next_tiles * 8 * ILE_QT_ROW * 8));
                    for (int k = 0; k < K; k++)
                        bulk_g2s(&sm.Q[k][0][0], P.Qt + ((size_t)k * P.N_Qpad + sm.base[k] + next_lo) * ILE_QT_ROW,
                                 (uint32_t)(next_tiles * 8 * ILE_QT_ROW * 8), (uint64_t*)&sm.bar);
                }
            }

            // ---------------- epilogue: shift + interpolate + sum detectors + log-sum-exp over time
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const int s = 4 * w + q;
                if (!sm.part[s]) continue;
                const double x = sm.rec[s][12], Bq = sm.rec[s][13];
                double v[2];
                double vmax = neg_inf();
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const int jj = j0 + lane + 32 * e;
                    v[e] = neg_inf();
                    if (jj < j1) {
                        double A = 0.0;
                        for (int k = 0; k < K; k++) {
                            const int b0 = sm.n[k][s] - sm.base[k] + stride * jj;
                            const int r0 = b0 % FT_RING;
                            const int r1 = (r0 + 1 == FT_RING) ? 0 : r0 + 1;
                            const double f = sm.frac[k][s];
                            A += (1.0 - f) * sm.S[k][s][r0] + f * sm.S[k][s][r1];
                        }
                        v[e] = P.use_table ? table_lookup(P, A, Bq) : x * A - x * x * Bq;
                        vmax = fmax(vmax, v[e]);
                    }
                }
                vmax = warp_max(vmax);
                if (vmax > run_m[q]) {
                    run_s[q] *= exp(run_m[q] - vmax);     // exp(-inf) = 0 on the first tile
                    run_m[q] = vmax;
                }
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const double dlt = v[e] - run_m[q];
                    if (dlt > -745.0) run_s[q] += exp(dlt);
                }
            }
            if (!more) break;
            j0 = j1;
            c_lo = next_lo;
            ntiles = next_tiles;
            __syncthreads();   // ring reads done before the next phase overwrites old bins
        }
        // ---------------- finalise this round's samples
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const int s = 4 * w + q;
            if (!sm.part[s]) continue;
            const double tot = warp_sum(run_s[q]);
            if (lane == 0) {
                const int t = tile * FT_TS + s;
                if (t < N) lnL[perm ? perm[t] : t] = run_m[q] + log(tot) - log((double)N_t);
                sm.done[s] = 1;
            }
        }
    }
}

// ---------------------------------------------------------------- launch
template <int NPAIR, bool SINGLE>
static int launch_fused_t(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL) {
    static bool configured = false;
    const int smem = (int)sizeof(FusedSmem);
    if (!configured) {
        ILE_CUDA(ctx, cudaFuncSetAttribute(lnl_fused_kernel<NPAIR, SINGLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        configured = true;
    }
    const int tiles = (N + FT_TS - 1) / FT_TS;
    const int slot = ile_timing_begin(ctx);
    lnl_fused_kernel<NPAIR, SINGLE><<<tiles, FT_THREADS, smem, ctx->stream>>>(P, N, rec, yt, perm, lnL);
    ile_timing_end(ctx, slot);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

int ile_launch_lnL_plain_z(ile_ctx* ctx, const LnlParams& P, int N, const double* z, double* lnL, double* ln_prior);
int ile_launch_fused2(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL, bool quad);
int ile_launch_fused3(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL, bool quad);

int ile_launch_lnL_fused(ile_ctx* ctx, const LnlParams& P, int N, const double* z, const int* perm, double* lnL, double* ln_prior) {
    if (P.K > 3 || 2 * P.M > ILE_QT_ROW) return ile_launch_lnL_plain_z(ctx, P, N, z, lnL, ln_prior);
    const int tiles = (N + 63) / 64 * 2;                       // 32-sample sub-tiles, padded to whole 64-sample tiles
    const size_t rec_bytes = ((size_t)tiles * FT_TS * FT_REC * sizeof(double) + 255) / 256 * 256;
    const size_t y_bytes = ((size_t)tiles * FT_YM * FT_TS * sizeof(double2) + 255) / 256 * 256;
    const size_t key_bytes = ((size_t)N * 8 + 255) / 256 * 256, val_bytes = ((size_t)N * 4 + 255) / 256 * 256;
    const size_t sort_bytes = (radix_sort_scratch_bytes(N) + 255) / 256 * 256;
    const bool sort = perm == nullptr && ctx->sky_sort && N > FT_TS;
    void* scratch = nullptr;
    int rc = ile_scratch(ctx, rec_bytes + y_bytes + (sort ? 2 * key_bytes + 2 * val_bytes + sort_bytes + 256 : 0), &scratch);
    if (rc) return rc;
    char* base = (char*)scratch;
    double* rec = (double*)base;
    double2* yt = (double2*)(base + rec_bytes);
    if (sort) {
        char* sb = base + rec_bytes + y_bytes;
        unsigned long long* k0 = (unsigned long long*)sb;
        unsigned long long* k1 = (unsigned long long*)(sb + key_bytes);
        unsigned int* v0 = (unsigned int*)(sb + 2 * key_bytes);
        unsigned int* v1 = (unsigned int*)(sb + 2 * key_bytes + val_bytes);
        void* hist = sb + 2 * key_bytes + 2 * val_bytes;
        long long* n_dev = (long long*)(sb + 2 * key_bytes + 2 * val_bytes + sort_bytes);
        int* bits_dev = (int*)(n_dev + 1);
        // cells of 2^SKY_CELL_SHIFT stored bins over the range of delays the network allows
        const int n_min = (int)floor((P.t_lo - ctx->max_delay - P.t_Q0) * P.fs) - 1;
        const int n_max = (int)floor((P.t_lo + ctx->max_delay - P.t_Q0) * P.fs) + 1;
        int cell_bits = 1;
        while ((1 << cell_bits) <= ((n_max - n_min) >> SKY_CELL_SHIFT)) cell_bits++;
        sky_key_kernel<<<(N + 255) / 256, 256, 0, ctx->stream>>>(P, N, z, n_min, cell_bits, k0, v0, n_dev, bits_dev);
        ILE_LAUNCH_CHECK(ctx);
        rc = radix_sort_device(ctx, N, n_dev, bits_dev, (uint64_t*)k0, v0, (uint64_t*)k1, v1, hist, (cell_bits * P.K + 1 + 7) / 8);
        if (rc) return rc;
        perm = (const int*)v0;
    }
    // the second-generation fused kernel computes the quadratic term itself (prologue)
    const int n2_ = 2 * P.M, np_ = n2_ / 8, rem_ = n2_ % 8;
    const bool gen2 = !ctx->fused_gen1 && rem_ >= 1 && rem_ <= 4 && ((P.K == 3 && np_ == 5) || (P.K == 2 && np_ == 1));
    if (gen2 && !ctx->prep_gen1) {
        // shared-memory scratch of the harmonics: (2 (max_pow + 1) + 2 (max_abs_m + 1)) doubles per thread
        // ... and a copy of the mode table
        const int scr_d = (2 * (ctx->ylm_max_pow + 1) + 2 * (ctx->ylm_max_abs_m + 1)) * 128;
        const size_t scr = (size_t)scr_d * sizeof(double) + sizeof(YlmTable) + 16;
        lnl_prep3_kernel<<<(tiles * FT_TS + 127) / 128, 128, scr, ctx->stream>>>(P, N, tiles * FT_TS, scr_d, z, perm, rec, yt, ln_prior);
    } else {
        lnl_prep_kernel<<<(tiles * FT_TS + 127) / 128, 128, 0, ctx->stream>>>(P, N, tiles * FT_TS, z, perm, rec, yt, ln_prior);
    }
    ILE_LAUNCH_CHECK(ctx);
    if (!ctx->fused_gen1) {
        rc = ctx->fused_gen3 ? ile_launch_fused3(ctx, P, N, rec, yt, perm, lnL, gen2 && !ctx->prep_gen1)
                             : ile_launch_fused2(ctx, P, N, rec, yt, perm, lnL, gen2 && !ctx->prep_gen1);
        if (rc != 1) return rc;                              // 1: shape not instantiated -> first generation
    }
    const int n2 = 2 * P.M, np = n2 / 8, rem = n2 % 8;
    if (np == 5 && rem >= 1 && rem <= 4) return launch_fused_t<5, true>(ctx, P, N, rec, yt, perm, lnL);
    if (np == 1 && rem >= 1 && rem <= 4) return launch_fused_t<1, true>(ctx, P, N, rec, yt, perm, lnL);
    return launch_fused_t<6, false>(ctx, P, N, rec, yt, perm, lnL);
}
