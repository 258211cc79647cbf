// libile: fused lnL kernel, second generation.  Design notes in DESIGN.md
// section 6; the measurements behind it (profiles/r1_pipes.md): on sm_100a a dependent DMMA.8x8x4
// issues every ~150 cycles while the pipe accepts one every 16, and DFMA shares that FP64 datapath.
// Hence: >= 8 independent accumulator chains per warp in the contraction, and an epilogue with as
// few FP64 instructions per (sample, time bin) as the arithmetic allows.
//
//   one CTA = 64 samples (delay-cell sorted), 8 warps, one CTA per SM
//   contraction   S_k[s][n] = sum_r coef_k[s][r] Q_k[r][n]  (coef = x Re/Im(F_k Y_m), K-dim 2M):
//                 unit = (detector k, 8 stored bins) x all 64 samples = 8 independent DMMA chains;
//                 A fragments (coef) from shared memory in fragment order, B fragments (Q) straight
//                 from global/L2 into registers, prefetched one unit ahead; D -> S ring in smem
//   epilogue      one warp per sample row, lanes along time: per-sample delay shift + linear
//                 interpolation (2 FMA per detector), ln L(t_j) = A_j - x^2 B, streaming log-sum-exp
//                 with a lazily raised reference and a 13-instruction exp
#include "common.cuh"
#include "likelihood_dev.cuh"

#define F2_TS 64
#define F2_THREADS 256
#define F2_WARPS 8
#define F2_RING 80        // S ring length in stored bins
#define F2_SROW 88        // S row stride (== 8 mod 16: conflict-free 128-bit fragment stores)
#define F2_NEW 64         // new stored bins per phase (phase 0: F2_RING)
#define F2_CAP 15         // largest per-sample offset above the tile base handled in one round
#define F2_YM 24          // mode slots in the prep kernel's Y tile (32-sample sub-tiles)
#define F2_REC 16
#define F2_NP 6           // k-step pairs allocated per detector in the A-fragment table

struct Fused2Smem {
    double S[3][F2_TS][F2_SROW];             // 135,168 B
    double2 A[3][F2_NP][8][32];              //  73,728 B  [k][k-step pair][row block][lane]
    double rec[F2_TS][F2_REC];               //   8,192 B
    double w1[3][F2_TS];                     // interpolation fraction f
    int n[3][F2_TS];
    int base[4];
    int part[F2_TS];
    int done[F2_TS];
    int n_part, n_left;
};

__device__ __forceinline__ void dmma2(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// exp(d) for d in (-40, 31]: k = rint(d log2 e) by the magic-number add, r = d - k ln2,
// degree-10 Taylor polynomial (|r| <= 0.3466: truncation < 2.3e-13 relative), scaled by 2^k through
// the exponent field.  13 FP64 instructions; the tolerance budget is DESIGN.md section 6.
__device__ __forceinline__ double exp_small(double d) {
    const double t = fma(d, 1.4426950408889634, 6755399441055744.0);
    const int k = __double2loint(t);
    const double kf = t - 6755399441055744.0;
    double r = fma(kf, -6.93147180369123816490e-01, d);
    r = fma(kf, -1.90821492927058770002e-10, r);
    double p = 1.0 / 3628800.0;
    p = fma(p, r, 1.0 / 362880.0);
    p = fma(p, r, 1.0 / 40320.0);
    p = fma(p, r, 1.0 / 5040.0);
    p = fma(p, r, 1.0 / 720.0);
    p = fma(p, r, 1.0 / 120.0);
    p = fma(p, r, 1.0 / 24.0);
    p = fma(p, r, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}

template <int NPAIR, bool SINGLE, bool TABLE>
__global__ void __launch_bounds__(F2_THREADS, 1)
lnl_fused2_kernel(LnlParams P, int N, const double* __restrict__ rec, const double2* __restrict__ ytile, const int* __restrict__ perm,
                  double* __restrict__ lnL) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Fused2Smem& sm = *reinterpret_cast<Fused2Smem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int tile = blockIdx.x;
    const int K = P.K, stride = P.stride, N_t = P.N_t;
    const int c = lane & 3, rq = lane >> 2;

    // ---- stage the tile's records
    {
        const double* src = rec + (size_t)tile * F2_TS * F2_REC;
        for (int q = tid; q < F2_TS * F2_REC; q += F2_THREADS) (&sm.rec[0][0])[q] = src[q];
    }
    __syncthreads();
    if (tid < F2_TS) {
        const bool valid = sm.rec[tid][14] != 0.0;
        sm.done[tid] = valid ? 0 : 1;
        for (int k = 0; k < K; k++) {
            const double u = sm.rec[tid][8 + k];
            const double fl = floor(u);
            sm.n[k][tid] = (int)fl;
            sm.w1[k][tid] = u - fl;
        }
        if (!valid) {
            const int t = tile * F2_TS + tid;
            if (t < N) lnL[perm ? perm[t] : t] = neg_inf();
        }
    }
    // ---- coefficient fragments: A[k][p][rb][lane] = x (Re, Im)(F_k Y_m), sample 8 rb + lane/4,
    //      mode m = 4 p + lane%4; the trailing half k-step (SINGLE) holds Re or Im of mode
    //      4 NPAIR + (lane%4)/2 in .x
    {
        const int NPT = NPAIR + (SINGLE ? 1 : 0);
        for (int q = tid; q < K * NPT * 8 * 32; q += F2_THREADS) {
            const int ln = q & 31, rb = (q >> 5) & 7, p = (q >> 8) % NPT, k = (q >> 8) / NPT;
            const int s = 8 * rb + (ln >> 2), cc = ln & 3;
            const double x = sm.rec[s][12], fr = x * sm.rec[s][k], fi = x * sm.rec[s][4 + k];
            const double2* yt = ytile + ((size_t)(2 * tile + (s >> 5)) * F2_YM) * 32 + (s & 31);
            double2 a;
            if (p < NPAIR) {
                const double2 y = yt[(4 * p + cc) * 32];
                a = make_double2(fr * y.x - fi * y.y, fr * y.y + fi * y.x);
            } else {
                const double2 y = yt[(4 * NPAIR + (cc >> 1)) * 32];
                a = make_double2((cc & 1) ? fr * y.y + fi * y.x : fr * y.x - fi * y.y, 0.0);
            }
            sm.A[k][p][rb][ln] = a;
        }
    }

    for (;;) {   // rounds: normally one; more only when the tile's delay spread exceeds F2_CAP
        __syncthreads();
        if (tid < 32) {
            int base[3];
            bool q0, q1;
            const int dn0 = sm.done[lane], dn1 = sm.done[lane + 32];
            for (int k = 0; k < K; k++) {
                int v = min(dn0 ? 0x7fffffff : sm.n[k][lane], dn1 ? 0x7fffffff : sm.n[k][lane + 32]);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, o));
                base[k] = v & ~1;
            }
            q0 = !dn0;
            q1 = !dn1;
            for (int k = 0; k < K; k++) {
                q0 = q0 && (sm.n[k][lane] - base[k] <= F2_CAP);
                q1 = q1 && (sm.n[k][lane + 32] - base[k] <= F2_CAP);
            }
            unsigned m0 = __ballot_sync(0xffffffffu, q0), m1 = __ballot_sync(0xffffffffu, q1);
            const unsigned l0 = __ballot_sync(0xffffffffu, !dn0), l1 = __ballot_sync(0xffffffffu, !dn1);
            if ((l0 | l1) != 0 && (m0 | m1) == 0) {   // pivot on the first unfinished sample: always progresses
                const int piv = l0 ? __ffs(l0) - 1 : 32 + __ffs(l1) - 1;
                for (int k = 0; k < K; k++) base[k] = sm.n[k][piv] & ~1;
                q0 = !dn0;
                q1 = !dn1;
                for (int k = 0; k < K; k++) {
                    q0 = q0 && (sm.n[k][lane] >= base[k]) && (sm.n[k][lane] - base[k] <= F2_CAP);
                    q1 = q1 && (sm.n[k][lane + 32] >= base[k]) && (sm.n[k][lane + 32] - base[k] <= F2_CAP);
                }
                m0 = __ballot_sync(0xffffffffu, q0);
                m1 = __ballot_sync(0xffffffffu, q1);
            }
            sm.part[lane] = q0 ? 1 : 0;
            sm.part[lane + 32] = q1 ? 1 : 0;
            if (lane == 0) {
                for (int k = 0; k < K; k++) sm.base[k] = base[k];
                sm.n_part = __popc(m0) + __popc(m1);
                sm.n_left = __popc(l0) + __popc(l1);
            }
        }
        __syncthreads();
        if (sm.n_left == 0) break;

        // per-sample epilogue state of this warp's 8 rows: reference m (warp-uniform), lane-partial sum
        double run_m[8], run_s[8];
#pragma unroll
        for (int q = 0; q < 8; q++) { run_m[q] = -1.0e300; run_s[q] = 0.0; }

        const int last_bin = stride * (N_t - 1) + 1 + F2_CAP;   // highest stored bin (relative to base) any sample reads
        int c_lo = 0, j0 = 0;
        int ntiles = min(F2_RING / 8, (last_bin + 1 - c_lo + 7) / 8);
        for (int phase = 0;; phase++) {
            const int c_hi = c_lo + ntiles * 8;
            int j1 = (c_hi - 1 - F2_CAP - 1) / stride + 1;      // outputs whose reads are all below c_hi
            if (j1 > N_t) j1 = N_t;

            // ---------------- contraction: unit = (k, 8 bins) x 64 samples, 8 DMMA chains per warp
            {
                const int nunits = K * ntiles;
                double2 bn[NPAIR];
                double bs = 0.0;
                auto load_b = [&](int u) {
                    const int k = u / ntiles, t = u - k * ntiles;
                    const int row = sm.base[k] + c_lo + 8 * t + rq;
                    const int swz = (row & 1) << 3;
                    const double* qrow = P.Qt + ((size_t)k * P.N_Qpad + row) * ILE_QT_ROW;
#pragma unroll
                    for (int p = 0; p < NPAIR; p++) bn[p] = __ldg(reinterpret_cast<const double2*>(qrow + ((8 * p + 2 * c) ^ swz)));
                    if (SINGLE) bs = __ldg(qrow + ((8 * NPAIR + c) ^ swz));
                };
                int u = w;
                if (u < nunits) load_b(u);
                for (; u < nunits; u += F2_WARPS) {
                    const int k = u / ntiles, t = u - k * ntiles;
                    double2 b[NPAIR];
#pragma unroll
                    for (int p = 0; p < NPAIR; p++) b[p] = bn[p];
                    const double bsc = bs;
                    if (u + F2_WARPS < nunits) load_b(u + F2_WARPS);
                    double d[8][2];
#pragma unroll
                    for (int rb = 0; rb < 8; rb++) d[rb][0] = d[rb][1] = 0.0;
#pragma unroll
                    for (int p = 0; p < NPAIR; p++) {
#pragma unroll
                        for (int rb = 0; rb < 8; rb++) {
                            const double2 a = sm.A[k][p][rb][lane];
                            dmma2(d[rb][0], d[rb][1], a.x, b[p].x);
                            dmma2(d[rb][0], d[rb][1], a.y, b[p].y);
                        }
                    }
                    if (SINGLE) {
#pragma unroll
                        for (int rb = 0; rb < 8; rb++) {
                            const double a = sm.A[k][NPAIR][rb][lane].x;
                            dmma2(d[rb][0], d[rb][1], a, bsc);
                        }
                    }
                    const int col = (c_lo + 8 * t) % F2_RING + 2 * c;
#pragma unroll
                    for (int rb = 0; rb < 8; rb++)
                        *reinterpret_cast<double2*>(&sm.S[k][8 * rb + rq][col]) = make_double2(d[rb][0], d[rb][1]);
                }
            }
            __syncthreads();   // S complete for bins < c_hi

            // ---------------- epilogue: shift + interpolate + sum detectors + streaming log-sum-exp
#pragma unroll
            for (int q = 0; q < 8; q++) {
                const int s = 8 * w + q;
                if (!sm.part[s]) continue;
                const double Bq = sm.rec[s][13], x = sm.rec[s][12];
                const double cB = TABLE ? 0.0 : x * x * Bq;
                double f1[3], f0[3];
                int off[3];
                for (int k = 0; k < K; k++) {
                    f1[k] = sm.w1[k][s];
                    f0[k] = 1.0 - f1[k];
                    off[k] = sm.n[k][s] - sm.base[k];
                }
                for (int jb = j0; jb < j1; jb += 32) {
                    const int jj = jb + lane;
                    double v = neg_inf();
                    if (jj < j1) {
                        double A = -cB;
                        for (int k = 0; k < K; k++) {
                            const int b0 = off[k] + stride * jj;
                            const int r0 = b0 % F2_RING;
                            const int r1 = (r0 + 1 == F2_RING) ? 0 : r0 + 1;
                            A = fma(f0[k], sm.S[k][s][r0], A);
                            A = fma(f1[k], sm.S[k][s][r1], A);
                        }
                        v = TABLE ? table_lookup(P, A, Bq) : A;
                    }
                    double dl = v - run_m[q];
                    if (__any_sync(0xffffffffu, dl > 30.0)) {      // raise the reference (rare)
                        const double mx = warp_max(v);
                        run_s[q] *= exp(run_m[q] - mx);
                        run_m[q] = mx;
                        dl = v - mx;
                    }
                    if (dl > -40.0) run_s[q] += exp_small(dl);
                }
            }
            if (j1 >= N_t) break;
            j0 = j1;
            c_lo = c_hi;
            ntiles = min(F2_NEW / 8, (last_bin + 1 - c_lo + 7) / 8);
            __syncthreads();   // ring reads done before the next phase overwrites old bins
        }
        // ---------------- finalise this round's samples
#pragma unroll
        for (int q = 0; q < 8; q++) {
            const int s = 8 * w + q;
            if (!sm.part[s]) continue;
            const double tot = warp_sum(run_s[q]);
            if (lane == 0) {
                const int t = tile * F2_TS + s;
                if (t < N) lnL[perm ? perm[t] : t] = run_m[q] + log(tot) - log((double)N_t);
                sm.done[s] = 1;
            }
        }
    }
}

template <int NPAIR, bool SINGLE, bool TABLE>
static int launch_fused2_t(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL) {
    static bool configured = false;
    const int smem = (int)sizeof(Fused2Smem);
    if (!configured) {
        ILE_CUDA(ctx, cudaFuncSetAttribute(lnl_fused2_kernel<NPAIR, SINGLE, TABLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        configured = true;
    }
    const int tiles = (N + F2_TS - 1) / F2_TS;
    const int slot = ile_timing_begin(ctx);
    lnl_fused2_kernel<NPAIR, SINGLE, TABLE><<<tiles, F2_THREADS, smem, ctx->stream>>>(P, N, rec, yt, perm, lnL);
    ile_timing_end(ctx, slot);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

// rec / yt as written by lnl_prep_kernel for ceil(N/64)*64 padded samples
int ile_launch_fused2(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL) {
    const int n2 = 2 * P.M, np = n2 / 8, rem = n2 % 8;
    const bool tb = P.use_table != 0;
    if (np == 5 && rem >= 1 && rem <= 4)
        return tb ? launch_fused2_t<5, true, true>(ctx, P, N, rec, yt, perm, lnL) : launch_fused2_t<5, true, false>(ctx, P, N, rec, yt, perm, lnL);
    if (np == 1 && rem >= 1 && rem <= 4)
        return tb ? launch_fused2_t<1, true, true>(ctx, P, N, rec, yt, perm, lnL) : launch_fused2_t<1, true, false>(ctx, P, N, rec, yt, perm, lnL);
    return tb ? launch_fused2_t<6, false, true>(ctx, P, N, rec, yt, perm, lnL) : launch_fused2_t<6, false, false>(ctx, P, N, rec, yt, perm, lnL);
}
