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

#define F2_THREADS 256
#define F2_WARPS 8
#define F2_RING 80        // S ring length in stored bins
#define F2_SROW 88        // S row stride (== 8 mod 16: conflict-free 128-bit fragment stores)
#define F2_NEW 64         // new stored bins per phase (phase 0: F2_RING)
#define F2_CAP 15         // largest per-sample offset above the tile base handled in one round
#define F2_YM 24          // mode slots in the prep kernel's Y tile (32-sample sub-tiles)
#define F2_REC 16
#ifndef F2_G
#define F2_G 4
#endif
#define F2_NP 6           // k-step pairs allocated per detector in the A-fragment table

// RB = row blocks of 8 samples per CTA: 8 (64 samples, one CTA per SM) or 4 (32 samples, two per SM)
template <int K, int RB>
struct Fused2Smem {
    double S[K][8 * RB][F2_SROW];            // S_k[sample][ring bin]
    double2 A[K][F2_NP][RB][32];             // coefficient fragments [k][k-step pair][row block][lane]
    double rec[8 * RB][F2_REC];
    double w1[K][8 * RB];                    // interpolation fraction f
    int n[K][8 * RB];
    int base[4];
    int part[8 * RB];
    int done[8 * RB];
    int n_part, n_left;
    double2 ew[8 * RB][K];                   // epilogue constants per sample: (1 - f_k, f_k)
    double2 ec[8 * RB];                      // (x^2 B, B)
    int eoff[8 * RB][4];                     // n_k - base_k, clamped to [0, F2_CAP]
};

__device__ __forceinline__ void dmma2(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// exp(d) for d in (-690, 31]: k = rint(d log2 e) by the magic-number add, r = d - k ln2,
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


template <int K, int RB, int NPAIR, bool SINGLE, bool TABLE, bool STRIDE1>
__global__ void __launch_bounds__(F2_THREADS, (RB == 4 ? 2 : 1))
lnl_fused2_kernel(LnlParams P, int N, const double* __restrict__ rec, const double2* __restrict__ ytile, const int* __restrict__ perm,
                  double* __restrict__ lnL) {
    constexpr int TS = 8 * RB;        // samples per CTA
    constexpr int SPW = RB;           // sample rows per warp in the epilogue
    constexpr int NPT = NPAIR + (SINGLE ? 1 : 0);
    constexpr int G = F2_G < SPW ? F2_G : SPW;   // sample rows in flight per warp in the epilogue
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Fused2Smem<K, RB>& sm = *reinterpret_cast<Fused2Smem<K, RB>*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int tile = blockIdx.x;
    const int stride = STRIDE1 ? 1 : P.stride, N_t = P.N_t;
    const int c = lane & 3, rq = lane >> 2;

    // ---- stage the tile's records
    {
        const double* src = rec + (size_t)tile * TS * F2_REC;
        for (int q = tid; q < TS * F2_REC; q += F2_THREADS) (&sm.rec[0][0])[q] = src[q];
    }
    __syncthreads();
    if (tid < TS) {
        const bool valid = sm.rec[tid][14] != 0.0;
        sm.done[tid] = valid ? 0 : 1;
#pragma unroll
        for (int k = 0; k < K; k++) {
            const double u = sm.rec[tid][8 + k];
            const double fl = floor(u);
            sm.n[k][tid] = (int)fl;
            sm.w1[k][tid] = u - fl;
        }
        if (!valid) {
            const int t = tile * TS + tid;
            if (t < N) lnL[perm ? perm[t] : t] = neg_inf();
        }
    }
    // ---- coefficient fragments: A[k][p][rb][lane] = x (Re, Im)(F_k Y_m), sample 8 rb + lane/4,
    //      mode m = 4 p + lane%4; the trailing half k-step (SINGLE) holds Re or Im of mode
    //      4 NPAIR + (lane%4)/2 in .x
    for (int q = tid; q < K * NPT * RB * 32; q += F2_THREADS) {
        const int ln = q & 31, rb = (q >> 5) & (RB - 1), pk = q / (32 * RB), p = pk % NPT, k = pk / NPT;
        const int s = 8 * rb + (ln >> 2), cc = ln & 3;
        const int t = tile * TS + s;
        const double x = sm.rec[s][12], fr = x * sm.rec[s][k], fi = x * sm.rec[s][4 + k];
        const double2* yt = ytile + ((size_t)(t >> 5) * F2_YM) * 32 + (t & 31);
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

    for (;;) {   // rounds: normally one; more only when the tile's delay spread exceeds F2_CAP
        __syncthreads();
        if (tid < 32) {
            constexpr int NS = TS / 32;       // samples per lane
            int base[K];
            int dn[NS];
            bool qq[NS];
#pragma unroll
            for (int h = 0; h < NS; h++) dn[h] = sm.done[lane + 32 * h];
#pragma unroll
            for (int k = 0; k < K; k++) {
                int v = 0x7fffffff;
#pragma unroll
                for (int h = 0; h < NS; h++) v = min(v, dn[h] ? 0x7fffffff : sm.n[k][lane + 32 * h]);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, o));
                base[k] = v & ~1;
            }
            unsigned any_q = 0, left = 0;
            int first_left = -1;
#pragma unroll
            for (int h = 0; h < NS; h++) {
                qq[h] = !dn[h];
#pragma unroll
                for (int k = 0; k < K; k++) qq[h] = qq[h] && (sm.n[k][lane + 32 * h] - base[k] <= F2_CAP);
                any_q |= __ballot_sync(0xffffffffu, qq[h]);
                const unsigned l = __ballot_sync(0xffffffffu, !dn[h]);
                if (l && first_left < 0) first_left = 32 * h + __ffs(l) - 1;
                left |= l;
            }
            if (left != 0 && any_q == 0) {   // pivot on the first unfinished sample: always progresses
#pragma unroll
                for (int k = 0; k < K; k++) base[k] = sm.n[k][first_left] & ~1;
#pragma unroll
                for (int h = 0; h < NS; h++) {
                    qq[h] = !dn[h];
#pragma unroll
                    for (int k = 0; k < K; k++)
                        qq[h] = qq[h] && (sm.n[k][lane + 32 * h] >= base[k]) && (sm.n[k][lane + 32 * h] - base[k] <= F2_CAP);
                }
            }
#pragma unroll
            for (int h = 0; h < NS; h++) sm.part[lane + 32 * h] = qq[h] ? 1 : 0;
            if (lane == 0) {
#pragma unroll
                for (int k = 0; k < K; k++) sm.base[k] = base[k];
                sm.n_left = __popc(left);
            }
            unsigned np_ = 0;
#pragma unroll
            for (int h = 0; h < NS; h++) np_ += __popc(__ballot_sync(0xffffffffu, qq[h]));
            if (lane == 0) sm.n_part = (int)np_;
        }
        __syncthreads();
        if (sm.n_left == 0) break;
        const bool last_round = sm.n_part == sm.n_left;   // every unfinished sample takes part: no re-check needed

        // epilogue constants of this warp's own rows (written and read by the same warp)
        if (lane < SPW) {
            const int s = SPW * w + lane;
            const double x = sm.rec[s][12], Bs = sm.rec[s][13];
            sm.ec[s] = make_double2(TABLE ? 0.0 : x * x * Bs, Bs);
#pragma unroll
            for (int k = 0; k < K; k++) {
                const double f = sm.w1[k][s];
                sm.ew[s][k] = make_double2(1.0 - f, f);
                sm.eoff[s][k] = min(max(sm.n[k][s] - sm.base[k], 0), F2_CAP);
            }
        }
        __syncwarp();
        // per-sample epilogue state of this warp's rows: reference m (warp-uniform), lane-partial sum
        double run_m[SPW], run_s[SPW];
#pragma unroll
        for (int q = 0; q < SPW; q++) { run_m[q] = -1.0e300; run_s[q] = 0.0; }

        const int last_bin = stride * (N_t - 1) + 1 + F2_CAP;   // highest stored bin (relative to base) any sample reads
        int c_lo = 0, j0 = 0;
        int ntiles = min(F2_RING / 8, (last_bin + 1 - c_lo + 7) / 8);
        for (;;) {
            const int c_hi = c_lo + ntiles * 8;
            int j1 = (c_hi - 1 - F2_CAP - 1) / stride + 1;      // outputs whose reads are all below c_hi
            if (j1 > N_t) j1 = N_t;

            // ---------------- contraction: unit = (k, 8 bins) x TS samples, RB DMMA chains per warp.
            // Q fragments of the next unit are loaded into the other register set while this one
            // is multiplied (two units per trip: no register copies).
            {
                const int nunits = K * ntiles;
                auto unit_kt = [&](int u, int& k, int& t) {
                    k = (u >= ntiles ? 1 : 0) + (u >= 2 * ntiles ? 1 : 0);
                    t = u - k * ntiles;
                };
                auto load_b = [&](int u, double2 (&b)[NPAIR], double& bs) {
                    int k, t;
                    unit_kt(u, k, t);
                    const int row = sm.base[k] + c_lo + 8 * t + rq;
                    const int swz = (row & 1) << 3;
                    const double* qrow = P.Qt + ((size_t)k * P.N_Qpad + row) * ILE_QT_ROW;
#pragma unroll
                    for (int p = 0; p < NPAIR; p++) b[p] = __ldg(reinterpret_cast<const double2*>(qrow + ((8 * p + 2 * c) ^ swz)));
                    if (SINGLE) bs = __ldg(qrow + ((8 * NPAIR + c) ^ swz));
                };
                auto compute = [&](int u, const double2 (&b)[NPAIR], const double bs) {
                    int k, t;
                    unit_kt(u, k, t);
                    // two accumulators per row block (the .x and .y halves of each k-step pair):
                    // 2 RB independent DMMA chains per warp
                    double d[RB][2], e[RB][2];
#pragma unroll
                    for (int rb = 0; rb < RB; rb++) d[rb][0] = d[rb][1] = e[rb][0] = e[rb][1] = 0.0;
                    const double2* Ak = &sm.A[k][0][0][lane];
#pragma unroll
                    for (int p = 0; p < NPAIR; p++) {
                        double2 a[RB];
#pragma unroll
                        for (int rb = 0; rb < RB; rb++) a[rb] = Ak[(p * RB + rb) * 32];
#pragma unroll
                        for (int rb = 0; rb < RB; rb++) dmma2(d[rb][0], d[rb][1], a[rb].x, b[p].x);
#pragma unroll
                        for (int rb = 0; rb < RB; rb++) dmma2(e[rb][0], e[rb][1], a[rb].y, b[p].y);
                    }
                    if (SINGLE) {
#pragma unroll
                        for (int rb = 0; rb < RB; rb++) dmma2(d[rb][0], d[rb][1], Ak[(NPAIR * RB + rb) * 32].x, bs);
                    }
#pragma unroll
                    for (int rb = 0; rb < RB; rb++) { d[rb][0] += e[rb][0]; d[rb][1] += e[rb][1]; }
                    int cr = c_lo + 8 * t;
                    cr -= (cr / F2_RING) * F2_RING;
                    double* srow = &sm.S[k][rq][cr + 2 * c];
#pragma unroll
                    for (int rb = 0; rb < RB; rb++) *reinterpret_cast<double2*>(srow + rb * 8 * F2_SROW) = make_double2(d[rb][0], d[rb][1]);
                    if (cr == 0 && c == 0) {      // ring column F2_RING mirrors column 0: the epilogue reads [r], [r+1] unwrapped
#pragma unroll
                        for (int rb = 0; rb < RB; rb++) srow[rb * 8 * F2_SROW + F2_RING] = d[rb][0];
                    }
                };
                double2 b0[NPAIR], b1[NPAIR];
                double s0 = 0.0, s1 = 0.0;
#ifdef F2_DBG_NOMMA
                int u = nunits;
#else
                int u = w;
#endif
                if (u < nunits) load_b(u, b0, s0);
                while (u < nunits) {
                    if (u + F2_WARPS < nunits) load_b(u + F2_WARPS, b1, s1);
                    compute(u, b0, s0);
                    u += F2_WARPS;
                    if (u >= nunits) break;
                    if (u + F2_WARPS < nunits) load_b(u + F2_WARPS, b0, s0);
                    compute(u, b1, s1);
                    u += F2_WARPS;
                }
            }
            __syncthreads();   // S complete for bins < c_hi

            // ---------------- epilogue: shift + interpolate + sum detectors + streaming log-sum-exp.
            // G sample rows in flight per warp (independent dependency chains); rows that do not
            // take part in this round are computed on clamped offsets and discarded.
            {
                int j0m = stride * j0;
                j0m -= (j0m / F2_RING) * F2_RING;
#pragma unroll
                for (int g0 = 0; g0 < SPW; g0 += G) {
                    double2 wk[G][K], cb[G];
                    int r[G][K];                   // ring column of this lane's first tap
                    const double* Srow[G];
#pragma unroll
                    for (int i = 0; i < G; i++) {
                        const int s = SPW * w + g0 + i;
                        cb[i] = sm.ec[s];
                        Srow[i] = &sm.S[0][s][0];
                        const int4 o4 = *reinterpret_cast<const int4*>(&sm.eoff[s][0]);
                        const int off[4] = {o4.x, o4.y, o4.z, o4.w};
#pragma unroll
                        for (int k = 0; k < K; k++) {
                            wk[i][k] = sm.ew[s][k];
                            int rr = off[k] + j0m;
                            if (rr >= F2_RING) rr -= F2_RING;
                            if (STRIDE1) {
                                rr += lane;
                                if (rr >= F2_RING) rr -= F2_RING;
                            }
                            r[i][k] = rr;
                        }
                    }
#ifdef F2_DBG_NOEPI
                    for (int jb = j0; jb < j0; jb += 32) {
#else
                    for (int jb = j0; jb < j1; jb += 32) {
#endif
                        const bool act = jb + lane < j1;
                        double v[G];
#pragma unroll
                        for (int i = 0; i < G; i++) {
                            double A = -cb[i].x;
#pragma unroll
                            for (int k = 0; k < K; k++) {
                                int r0;
                                if (STRIDE1) {
                                    r0 = r[i][k];
                                    const int nx = r0 + 32;
                                    r[i][k] = nx >= F2_RING ? nx - F2_RING : nx;
                                } else {
                                    r0 = (r[i][k] + stride * (jb - j0 + lane)) % F2_RING;
                                }
                                const double* row = Srow[i] + k * (TS * F2_SROW) + r0;
                                A = fma(wk[i][k].x, row[0], A);
                                A = fma(wk[i][k].y, row[1], A);
                            }
                            if (TABLE) A = table_lookup(P, A, cb[i].y);
                            v[i] = act ? A : neg_inf();
                        }
#pragma unroll
                        for (int i = 0; i < G; i++) {
                            double dl = v[i] - run_m[g0 + i];
                            if (__any_sync(0xffffffffu, dl > 30.0)) {      // raise the reference (rare)
                                // new reference >= max_lane v, found on the ordered high words with
                                // one REDUX; it need not be the exact maximum
                                const int h = __double2hiint(v[i]);
                                const int key = __reduce_max_sync(0xffffffffu, h ^ ((h >> 31) & 0x7fffffff));
                                const int hm = key ^ ((key >> 31) & 0x7fffffff);
                                const double mx = __hiloint2double(hm, hm < 0 ? 0 : -1);
                                const double dm = run_m[g0 + i] - mx;
                                // the running sum may hold terms up to e^30 above its reference: rescale it
                                // exactly (exp_small is valid down to the underflow of 2^k)
                                run_s[g0 + i] = dm > -690.0 ? run_s[g0 + i] * exp_small(dm) : 0.0;
                                run_m[g0 + i] = mx;
                                dl = v[i] - mx;
                            }
                            if (dl > -40.0) run_s[g0 + i] += exp_small(dl);
                        }
                    }
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
        for (int q = 0; q < SPW; q++) {
            const int s = SPW * w + q;
            const double tot = warp_sum(run_s[q]);
            if (lane == 0 && sm.part[s]) {
                const int t = tile * TS + s;
                if (t < N) lnL[perm ? perm[t] : t] = run_m[q] + log(tot) - log((double)N_t);
                sm.done[s] = 1;
            }
        }
        if (last_round) break;
    }
}

template <int K, int RB, int NPAIR, bool SINGLE, bool TABLE, bool STRIDE1>
static int launch_fused2_t(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL) {
    static bool configured = false;
    const int smem = (int)sizeof(Fused2Smem<K, RB>);
    if (!configured) {
        ILE_CUDA(ctx, cudaFuncSetAttribute(lnl_fused2_kernel<K, RB, NPAIR, SINGLE, TABLE, STRIDE1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        configured = true;
    }
    const int tiles = (N + 8 * RB - 1) / (8 * RB);
    const int slot = ile_timing_begin(ctx);
    lnl_fused2_kernel<K, RB, NPAIR, SINGLE, TABLE, STRIDE1><<<tiles, F2_THREADS, smem, ctx->stream>>>(P, N, rec, yt, perm, lnL);
    ile_timing_end(ctx, slot);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

template <int K, int RB, int NPAIR, bool SINGLE>
static int launch_fused2_k(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL) {
    const bool tb = P.use_table != 0, s1 = P.stride == 1;
    if (tb) return s1 ? launch_fused2_t<K, RB, NPAIR, SINGLE, true, true>(ctx, P, N, rec, yt, perm, lnL)
                      : launch_fused2_t<K, RB, NPAIR, SINGLE, true, false>(ctx, P, N, rec, yt, perm, lnL);
    return s1 ? launch_fused2_t<K, RB, NPAIR, SINGLE, false, true>(ctx, P, N, rec, yt, perm, lnL)
              : launch_fused2_t<K, RB, NPAIR, SINGLE, false, false>(ctx, P, N, rec, yt, perm, lnL);
}

// rec / yt as written by lnl_prep_kernel for ceil(N/64)*64 padded samples.  Returns 1 when the
// shape has no instantiation (the caller falls back to the first-generation kernel).
int ile_launch_fused2(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL) {
    const int n2 = 2 * P.M, np = n2 / 8, rem = n2 % 8;
    const int rb = ctx->fused_rb == 8 ? 8 : 4;
    if (P.K == 3 && np == 5 && rem >= 1 && rem <= 4)
        return rb == 4 ? launch_fused2_k<3, 4, 5, true>(ctx, P, N, rec, yt, perm, lnL) : launch_fused2_k<3, 8, 5, true>(ctx, P, N, rec, yt, perm, lnL);
    if (P.K == 2 && np == 1 && rem >= 1 && rem <= 4)
        return rb == 4 ? launch_fused2_k<2, 4, 1, true>(ctx, P, N, rec, yt, perm, lnL) : launch_fused2_k<2, 8, 1, true>(ctx, P, N, rec, yt, perm, lnL);
    return 1;
}
