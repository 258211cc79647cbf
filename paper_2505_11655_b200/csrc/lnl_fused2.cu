// libile: fused lnL kernel.  Design notes in DESIGN.md section 6; the
// measurements behind it are in profiles/r1_pipes.md: on sm_100a DMMA.8x8x4 and DFMA share one FP64
// datapath (37 TFLOP/s either way), a dependent DMMA waits on the one before it, and every operand
// fragment that is not register-resident costs 256 bytes of shared-memory/L1 wavefronts - the pipe
// that is as busy as the FP64 datapath in this kernel.  Hence: 8 independent accumulator chains per
// warp in the contraction; coefficient fragments read with conflict-free 128-bit loads, Q fragments
// from a fragment-major global copy (whole 128-byte lines); an epilogue that is branch-free
// straight-line code over 8 independent (sample, 32-bin) groups with as few FP64 instructions and
// shared-memory wavefronts per (sample, time bin) as the arithmetic allows.
//
//   one CTA = 32 samples (delay-cell sorted), 8 warps, two CTAs per SM
//   prologue      records, harmonics and the packed upper-triangle U/V staged by cp.async in the (still
//                 idle) S ring; coefficient fragments built in DMMA A-fragment order; step 4, the U/V
//                 quadratic term B: warp w walks a contiguous run of the upper triangle for all 32 samples
//   contraction   S_k[s][n] = sum_r coef_k[s][r] Q_k[r][n]  (coef = x Re/Im(F_k Y_m), K-dim 2M):
//                 phases of 64 new bins; in a full phase a warp owns a pair of 8-bin tiles and every
//                 coefficient fragment it reads from shared memory feeds two DMMAs (Q fragments stream
//                 from global/L2 two steps ahead); the tail phase runs units of (detector k, 8 bins)
//                 x 32 samples with the Q fragments loaded one unit ahead; D -> S ring in shared memory
//   epilogue      one warp per 4 sample rows, lanes along time: per-sample delay shift + linear
//                 interpolation (2 FMA per detector), ln L(t_j) = A_j - x^2 B (or the distance table),
//                 streaming log-sum-exp with a lazily raised reference and an 8-instruction table exp;
//                 range logic on the high words in the integer pipe
#include "common.cuh"
#include "likelihood_dev.cuh"
#include "exp_tab.cuh"

#define F2_THREADS 256
#define F2_WARPS 8
#define F2_TS 32          // samples per CTA
#define F2_RB 4           // row blocks of 8 samples
#define F2_SPW 4          // sample rows per warp in the epilogue
#define F2_RING 80        // S ring length in stored bins (+ column F2_RING mirroring column 0)
#define F2_SROW 88        // S row stride (== 8 mod 16: conflict-free 128-bit fragment stores)
#define F2_NEW 64         // new stored bins per phase
#define F2_CAP 15         // largest per-sample offset above the tile base handled in one round
#define F2_YM 24          // mode slots in the prep kernel's Y tile (32-sample sub-tiles)
#define F2_YS 34          // row stride of the staged Y tile in shared memory (conflict-free fragment-builder reads)
#define F2_REC 16
#define F2_RECS 17         // record row stride in shared memory (odd: lane = sample reads are conflict-free)
#define F2_NP 6           // k-step pairs allocated per detector in the A-fragment table
#define F2_UVMAX (300 * 3 * 2)   // packed U/V entries staged in shared memory (M <= 24: 300 pairs)
#define F2_NG 2           // 32-bin groups per phase (at most 64 outputs per phase)
#ifndef F2_LA
#define F2_LA 2            // steps the Q fragments of the tile-pair contraction are loaded ahead
#endif
#ifndef F2_NO_PAIRJOBS
#define F2_PAIRJOBS       // full phases: contraction by pairs of bin tiles (profiles/r1_pipes.md); -DF2_NO_PAIRJOBS for the A/B
#endif

template <int K>
struct Fused2Smem {
    double S[K][F2_TS][F2_SROW];             // S_k[sample][ring bin]
    double2 A[K][F2_NP][F2_RB][32];          // coefficient fragments [k][k-step pair][row block][lane]; the half k-step: [row block pair][lane]
    double rec[F2_TS][F2_RECS];
    double w1[K][F2_TS];                     // interpolation fraction f
    double2 ew[F2_TS][K];                    // epilogue constants per sample: (1 - f_k, f_k)
    double2 ec[F2_TS];                       // (x^2 B, B); distance-table mode: (row fraction, row index) of the lookup
    int eoff[F2_TS][4];                      // n_k - base_k, clamped to [0, F2_CAP]
    int n[K][F2_TS];
    int base[4];
    int part[F2_TS];
    int done[F2_TS];
    int n_part, n_left;
    double etab[64];                         // 2^(j/64), the table of exp_tab
    int cap;                                 // largest offset above the base among this round's samples
    int pad_;
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


// exp(d) for d in [-40, 31] in 8 FP64 instructions: k = rint(64 d / ln2) by the magic-number add,
// r = d - k ln2/64 (|r| <= 0.00542; the rounding of ln2/64 costs < 3e-15 for |d| <= 40),
// exp(d) = 2^(k >> 6) tab[k & 63] (1 + r (1 + r/2 + r^2/6 + r^3/24)): truncation r^5/120 < 4e-14 relative.
// tab = the shared-memory copy of f2_exp2_tab.
__device__ __forceinline__ double exp_tab(double d, const double* __restrict__ tab) {
    const double t = fma(d, 0x1.71547652b82fep+6, 6755399441055744.0);
    const int k = __double2loint(t);
    const double kf = t - 6755399441055744.0;
    const double r = fma(kf, -0x1.62e42fefa39efp-7, d);
    const double T = tab[k & 63];
    double p = fma(r, 1.0 / 24.0, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    const double e = fma(T * r, p, T);
    return __hiloint2double(__double2hiint(e) + ((k >> 6) << 20), __double2loint(e));
}

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}

// general round set-up (warp 0): tile base = even floor of the per-detector minimum first bin over
// the unfinished samples; a sample takes part when all its offsets are within F2_CAP; when none
// does, pivot on the first unfinished sample so that every round makes progress
template <int K>
__device__ __forceinline__ void round_setup(Fused2Smem<K>& sm, int lane) {
    int base[K];
    const int dn = sm.done[lane];
#pragma unroll
    for (int k = 0; k < K; k++) {
        int v = dn ? 0x7fffffff : sm.n[k][lane];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, o));
        base[k] = v & ~1;
    }
    bool q = !dn;
#pragma unroll
    for (int k = 0; k < K; k++) q = q && (sm.n[k][lane] - base[k] <= F2_CAP);
    unsigned mq = __ballot_sync(0xffffffffu, q);
    const unsigned left = __ballot_sync(0xffffffffu, !dn);
    if (left != 0 && mq == 0) {
        const int piv = __ffs(left) - 1;
#pragma unroll
        for (int k = 0; k < K; k++) base[k] = sm.n[k][piv] & ~1;
        q = !dn;
#pragma unroll
        for (int k = 0; k < K; k++) q = q && (sm.n[k][lane] >= base[k]) && (sm.n[k][lane] - base[k] <= F2_CAP);
        mq = __ballot_sync(0xffffffffu, q);
    }
    sm.part[lane] = q ? 1 : 0;
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) sm.base[k] = base[k];
        sm.n_part = __popc(mq);
        sm.n_left = __popc(left);
        sm.cap = 0;
    }
}

// epilogue constants of sample s for the current tile base
template <int K, bool TABLE>
__device__ __forceinline__ void sample_consts(Fused2Smem<K>& sm, const LnlParams& P, int s) {
    const double x = sm.rec[s][12], Bs = sm.rec[s][13];
    if (TABLE) {
        // distance table (G28): the B coordinate is per sample: row index and fraction of the clamped bilinear lookup
        double b = (Bs - P.B_lo) / (P.B_hi - P.B_lo) * (double)(P.nB - 1);
        b = fmin(fmax(b, 0.0), (double)(P.nB - 1));
        const int ib = min((int)floor(b), P.nB - 2);
        sm.ec[s] = make_double2(b - ib, (double)ib);
    } else {
        sm.ec[s] = make_double2(x * x * Bs, Bs);
    }
#pragma unroll
    for (int k = 0; k < K; k++) {
        const double f = sm.w1[k][s];
        sm.ew[s][k] = make_double2(1.0 - f, f);
        const int o = min(max(sm.n[k][s] - sm.base[k], 0), F2_CAP);
        sm.eoff[s][k] = o;
        if (sm.part[s]) atomicMax(&sm.cap, o);
    }
}

template <int K, int NPAIR, bool SINGLE, bool TABLE, bool STRIDE1>
__device__ __forceinline__ void tile_body(Fused2Smem<K>& sm, const int tid, const int tile, const LnlParams& P,
                                          const int N, const int quad, const double* __restrict__ rec, const double2* __restrict__ ytile,
                                          const int* __restrict__ perm, double* __restrict__ lnL) {
    constexpr int RB = F2_RB, TS = F2_TS, SPW = F2_SPW, NG = F2_NG;
    constexpr int NPT = NPAIR + (SINGLE ? 1 : 0);
    const int lane = tid & 31, w = tid >> 5;
    const int stride = STRIDE1 ? 1 : P.stride, N_t = P.N_t;
    const int c = lane & 3, rq = lane >> 2;
    const double tabA_s = TABLE ? (double)(P.nA - 1) / (P.A_hi - P.A_lo) : 0.0, tabA_o = -P.A_lo * tabA_s;   // column coordinate of the distance table
    double2* ysm = reinterpret_cast<double2*>(&sm.S[0][0][0]);              // [F2_YM][F2_YS] during the prologue
    double* qpart = reinterpret_cast<double*>(ysm + F2_YM * F2_YS);            // [8 warps][3 K][32] partial quadratic sums
    double* qred = qpart + F2_WARPS * 3 * K * 32;                           // [3 K][32] their sums
    double2* uvsm = reinterpret_cast<double2*>(qred + 3 * K * 32);          // packed U/V, up to F2_UVMAX entries

    // ---- stage the tile's records; tile base by shared-memory atomicMin
    {
        // all copies are 16-byte cp.async: every load of the tile is in flight at once and the
        // prologue pays one memory round trip (a load/store loop pays one per iteration)
        const double* src = rec + (size_t)tile * TS * F2_REC;
        for (int q = tid; q < TS * F2_REC; q += F2_THREADS) cp_async8(&sm.rec[q / F2_REC][q % F2_REC], src + q);
        // the tile's harmonics Y[m][s] (12 KB) are staged in the S ring, which is idle until phase 0
        const double2* ysrc = ytile + (size_t)tile * F2_YM * 32;
#pragma unroll
        for (int q = tid; q < F2_YM * 32; q += F2_THREADS) cp_async16(ysm + (q >> 5) * F2_YS + (q & 31), ysrc + q);
        // ... and so are the packed U/V matrices of this intrinsic point (16 B per pair, detector and matrix)
        if (quad) {
            const double2* usrc = reinterpret_cast<const double2*>(P.UVp);
            const int nuv = min(P.n_pairs * K * 2, F2_UVMAX);
            for (int q = tid; q < nuv; q += F2_THREADS) cp_async16(uvsm + q, usrc + q);
        }
        if (tid < 4) sm.base[tid] = 0x7ffffffe;
        if (tid == 4) sm.cap = 0;
        if (tid >= 64 && tid < 128) sm.etab[tid - 64] = f2_exp2_tab[tid - 64];
        asm volatile("cp.async.commit_group;\n cp.async.wait_group 0;" ::: "memory");
    }
    __syncthreads();
    bool valid = false;
    if (tid < TS) {
        valid = sm.rec[tid][14] != 0.0;
        sm.done[tid] = valid ? 0 : 1;
#pragma unroll
        for (int k = 0; k < K; k++) {
            const double u = sm.rec[tid][8 + k];
            const double fl = floor(u);
            const int nk = (int)fl;
            sm.n[k][tid] = nk;
            sm.w1[k][tid] = u - fl;
            if (valid) atomicMin(&sm.base[k], nk & ~1);
        }
        if (!valid) {
            const int t = tile * TS + tid;
            if (t < N) lnL[perm ? perm[t] : t] = neg_inf();
        }
    }
    // ---- coefficient fragments: A[k][p][rb][lane] = x (Re, Im)(F_k Y_m), sample 8 rb + lane/4,
    //      mode m = 4 p + lane%4; the trailing half k-step (SINGLE) holds Re or Im of mode
    //      4 NPAIR + (lane%4)/2 in .x.  Fully unrolled: all of a thread's Y loads are in flight at once.
    {
        // warp w: row block w % 4, k-step pairs w / 4, w / 4 + 2, ...; the sample's record entries are
        // loaded once per detector (record rows are 17 doubles apart: conflict-free)
        static_assert(F2_WARPS == 2 * RB, "fragment builder: 8 warps = 4 row blocks x 2");
        const int rb = w & (RB - 1), h = w >> 2;
        const int s = 8 * rb + (lane >> 2), cc = lane & 3;
        const double x = sm.rec[s][12];
#pragma unroll
        for (int k = 0; k < K; k++) {
            const double fr = x * sm.rec[s][k], fi = x * sm.rec[s][4 + k];
#pragma unroll
            for (int p = h; p < NPT; p += 2) {
                const int m = p < NPAIR ? 4 * p + cc : 4 * NPAIR + (cc >> 1);
                const double2 y = ysm[m * F2_YS + s];
                if (p < NPAIR) sm.A[k][p][rb][lane] = make_double2(fr * y.x - fi * y.y, fr * y.y + fi * y.x);
                else   // the half k-step: row blocks (0, 1) and (2, 3) share a double2, two 128-bit loads per unit
                    reinterpret_cast<double*>(&sm.A[k][NPAIR][0][0])[((rb >> 1) * 32 + lane) * 2 + (rb & 1)] =
                        (cc & 1) ? fr * y.y + fi * y.x : fr * y.x - fi * y.y;
            }
        }
    }
    // ---- step 4, the U/V quadratic term (Eq. 7 with the Eq. 17-18 symmetries): warp w sums the
    //      upper-triangle pairs w, w + 8, ... for all 32 samples (lane = sample; the packed matrix
    //      entries are warp-uniform loads); partial sums meet in shared memory
    if (quad) {
        double uu[K], vr[K], vi[K];
#pragma unroll
        for (int k = 0; k < K; k++) uu[k] = vr[k] = vi[k] = 0.0;
        // warp w takes the contiguous run [w npw, (w + 1) npw) of the row-by-row upper triangle
        // (pairs (a, b), a <= b): y_a stays in registers along a row, so a pair costs one
        // harmonic load and the warp-uniform matrix loads (the loop is shared-memory-bound otherwise)
        const int M = P.M, npw = (P.n_pairs + F2_WARPS - 1) / F2_WARPS;
        int pq = w * npw;
        const int pq_end = min(pq + npw, P.n_pairs);
        int a = 0, b = pq;
        while (a < M && b >= M - a) { b -= M - a; a++; }
        b += a;
        while (pq < pq_end) {
            const double2 ya = ysm[a * F2_YS + lane];
            const int cnt = min(M - b, pq_end - pq);
            const double2* uv = uvsm + pq * K * 2;
            const double2* yrow = ysm + b * F2_YS + lane;
#pragma unroll 4
            for (int i = 0; i < cnt; i++) {
                double2 u[K], v[K];
#pragma unroll
                for (int k = 0; k < K; k++) { u[k] = uv[i * K * 2 + 2 * k]; v[k] = uv[i * K * 2 + 2 * k + 1]; }
                const double2 yb = yrow[i * F2_YS];
                // conj(y_a) y_b = (pr, pi), y_a y_b = (qr, qi): 6 FP64 instructions, then 6 FMAs per detector
                const double t2 = ya.y * yb.y, t4 = ya.y * yb.x;
                const double pr = fma(ya.x, yb.x, t2), qr = fma(ya.x, yb.x, -t2), pi = fma(ya.x, yb.y, -t4), qi = fma(ya.x, yb.y, t4);
#pragma unroll
                for (int k = 0; k < K; k++) {
                    uu[k] = fma(-u[k].y, pi, fma(u[k].x, pr, uu[k]));
                    vr[k] = fma(-v[k].y, qi, fma(v[k].x, qr, vr[k]));
                    vi[k] = fma(v[k].y, qr, fma(v[k].x, qi, vi[k]));
                }
            }
            pq += cnt;
            a++;
            b = a;
        }
#pragma unroll
        for (int k = 0; k < K; k++) {
            qpart[(w * 3 * K + 3 * k + 0) * 32 + lane] = uu[k];
            qpart[(w * 3 * K + 3 * k + 1) * 32 + lane] = vr[k];
            qpart[(w * 3 * K + 3 * k + 2) * 32 + lane] = vi[k];
        }
    }
    const int n_valid = __syncthreads_count(valid);      // also publishes n, w1, base, A
    if (n_valid == 0) return;
    // the 8 partial sums of each of the 3 K quadratic-form components are added by all warps (8 components
    // at a time): left to warp 0 alone it is a serial chain of ~100 FP64 instructions queueing behind the
    // other CTA's DMMAs while 7 warps wait at the next barrier
    if (quad) {
        for (int v = w; v < 3 * K; v += F2_WARPS) {
            double t[F2_WARPS];
#pragma unroll
            for (int ww = 0; ww < F2_WARPS; ww++) t[ww] = qpart[(ww * 3 * K + v) * 32 + lane];
            double acc = t[0];
#pragma unroll
            for (int ww = 1; ww < F2_WARPS; ww++) acc += t[ww];
            qred[v * 32 + lane] = acc;
        }
        __syncthreads();
    }
    // ---- round 0: who fits within F2_CAP of the base (normally everybody)
    bool part0 = false;
    if (tid < TS) {
        part0 = valid;
#pragma unroll
        for (int k = 0; k < K; k++) part0 = part0 && (sm.n[k][tid] - sm.base[k] <= F2_CAP);
        sm.part[tid] = part0 ? 1 : 0;
        if (quad) {
            double B = 0.0;
#pragma unroll
            for (int k = 0; k < K; k++) {
                const double uu = qred[(3 * k + 0) * 32 + tid], vr = qred[(3 * k + 1) * 32 + tid], vi = qred[(3 * k + 2) * 32 + tid];
                const double fr = sm.rec[tid][k], fi = sm.rec[tid][4 + k];
                B += (fr * fr + fi * fi) * uu + ((fr * fr - fi * fi) * vr - 2.0 * fr * fi * vi);
            }
            sm.rec[tid][13] = 0.25 * B;
        }
        sample_consts<K, TABLE>(sm, P, tid);
    }
    const int n_part0 = __syncthreads_count(part0);
    bool last_round = n_part0 == n_valid;
    bool need_setup = n_part0 == 0;                       // nobody fits: the general set-up pivots

    for (int round = 0;; round++) {   // rounds: normally one; more only when the tile's delay spread exceeds F2_CAP
        if (round > 0 || need_setup) {
            __syncthreads();
            if (tid < 32) round_setup<K>(sm, lane);
            __syncthreads();
            if (sm.n_left == 0) break;
            last_round = sm.n_part == sm.n_left;
            if (tid < TS) sample_consts<K, TABLE>(sm, P, tid);
            __syncthreads();
            need_setup = false;
        }
        // per-sample epilogue state of this warp's rows: reference m (warp-uniform), lane-partial sum
        double run_m[SPW], run_s[SPW];
#pragma unroll
        for (int q = 0; q < SPW; q++) { run_m[q] = -1.0e300; run_s[q] = 0.0; }

        // cap: the largest offset of a sample of this round above the base (<= F2_CAP; small after the sort);
        // the last bins of the window are only computed as far as some sample reads them
        const int cap = STRIDE1 ? sm.cap : F2_CAP;
        const int last_bin = stride * (N_t - 1) + 1 + cap;      // highest stored bin (relative to base) any sample reads
        int c_lo = 0, j0 = 0;
#ifdef F2_PAIRJOBS
        int ntiles = min(F2_NEW / 8, (last_bin + 1 - c_lo + 7) / 8);   // every full phase is 4 tile pairs
#else
        int ntiles = min(F2_RING / 8, (last_bin + 1 - c_lo + 7) / 8);
#endif
        for (;;) {
            const int c_hi = c_lo + ntiles * 8;
            int j1 = (c_hi - 1 - cap - 1) / stride + 1;         // outputs whose reads are all below c_hi ...
            j1 = min(min(j1, j0 + 32 * NG), N_t);               // ... as many as one epilogue pass takes
            {
#ifdef F2_PAIRJOBS
            // ---------------- contraction of a full phase (8 bin tiles): warp (q, h) = (w % 4, w / 4) owns the pair of
                // tiles (2 q, 2 q + 1) and, for K = 3, the work (detector h, all 4 row blocks) + (detector 2, row
                // blocks 2 h and 2 h + 1); every coefficient fragment read from shared memory feeds two DMMAs
                if (ntiles == 8)
                {
                    static_assert(K == 2 || K == 3, "contraction job split is written for two or three detectors");
                    const int q = w & 3, h = w >> 2;
                    if (2 * q < ntiles) {
                        constexpr int NSTEP = NPAIR + (SINGLE ? 1 : 0);
                        constexpr int NPART = K == 3 ? 2 : 1;
                        constexpr int NG_ = NPART * NSTEP;
                        const int t0 = 2 * q;
                        const bool two = t0 + 1 < ntiles;                 // the last phase may end on a single tile
                        const int t1 = two ? t0 + 1 : t0;
                        const double* qp[NPART][2];
#pragma unroll
                        for (int part = 0; part < NPART; part++) {
                            const int k = part == 0 ? h : 2;
#pragma unroll
                            for (int nt = 0; nt < 2; nt++) {
                                const int row = sm.base[k] + c_lo + 8 * (nt ? t1 : t0) + rq;
                                qp[part][nt] = P.Qf + (((size_t)k * P.N_Qpad + row) >> 1) * (2 * ILE_QT_ROW) + (row & 1) * 8;
                            }
                        }
                        double2 bb[F2_LA + 1][2];
                        auto issue = [&](const int g) {
                            const int part = g / NSTEP, st = g % NSTEP;
#pragma unroll
                            for (int nt = 0; nt < 2; nt++) {
                                if (st < NPAIR) bb[g % (F2_LA + 1)][nt] = __ldg(reinterpret_cast<const double2*>(qp[part][nt] + 16 * st + 2 * c));
                                else bb[g % (F2_LA + 1)][nt].x = __ldg(qp[part][nt] + 16 * NPAIR + c);
                            }
                        };
                        issue(0);
                        if (NG_ > 1 && F2_LA > 1) issue(1);
                        double acc[RB][2][2];
#pragma unroll
                        for (int g = 0; g < NG_; g++) {
                            if (g + F2_LA < NG_) issue(g + F2_LA);
                            const int part = g / NSTEP, st = g % NSTEP;
                            const int k = part == 0 ? h : 2;
                            const int nrb = part == 0 ? RB : RB / 2, rb0 = part == 0 ? 0 : 2 * h;
                            if (st == 0) {
#pragma unroll
                                for (int r = 0; r < RB; r++) acc[r][0][0] = acc[r][0][1] = acc[r][1][0] = acc[r][1][1] = 0.0;
                            }
                            const double2* Ak = &sm.A[k][0][0][lane];
                            if (st < NPAIR) {
                                double2 a[RB];
#pragma unroll
                                for (int r = 0; r < RB; r++)
                                    if (r < nrb) a[r] = Ak[(st * RB + rb0 + r) * 32];
#pragma unroll
                                for (int r = 0; r < RB; r++)
                                    if (r < nrb) {
                                        dmma2(acc[r][0][0], acc[r][0][1], a[r].x, bb[g % (F2_LA + 1)][0].x);
                                        dmma2(acc[r][1][0], acc[r][1][1], a[r].x, bb[g % (F2_LA + 1)][1].x);
                                    }
#pragma unroll
                                for (int r = 0; r < RB; r++)
                                    if (r < nrb) {
                                        dmma2(acc[r][0][0], acc[r][0][1], a[r].y, bb[g % (F2_LA + 1)][0].y);
                                        dmma2(acc[r][1][0], acc[r][1][1], a[r].y, bb[g % (F2_LA + 1)][1].y);
                                    }
                            } else {
#pragma unroll
                                for (int r = 0; r < RB; r += 2)
                                    if (r < nrb) {
                                        const double2 as = Ak[(NPAIR * RB + ((rb0 + r) >> 1)) * 32];
                                        dmma2(acc[r][0][0], acc[r][0][1], as.x, bb[g % (F2_LA + 1)][0].x);
                                        dmma2(acc[r][1][0], acc[r][1][1], as.x, bb[g % (F2_LA + 1)][1].x);
                                        dmma2(acc[r + 1][0][0], acc[r + 1][0][1], as.y, bb[g % (F2_LA + 1)][0].x);
                                        dmma2(acc[r + 1][1][0], acc[r + 1][1][1], as.y, bb[g % (F2_LA + 1)][1].x);
                                    }
                            }
                            if (st == NSTEP - 1) {
#pragma unroll
                                for (int nt = 0; nt < 2; nt++) {
                                    if (nt == 1 && !two) break;
                                    int cr = c_lo + 8 * (nt ? t1 : t0);
                                    cr -= (cr / F2_RING) * F2_RING;
                                    double* srow = &sm.S[k][8 * rb0 + rq][cr + 2 * c];
#pragma unroll
                                    for (int r = 0; r < RB; r++)
                                        if (r < nrb) *reinterpret_cast<double2*>(srow + r * 8 * F2_SROW) = make_double2(acc[r][nt][0], acc[r][nt][1]);
                                    if (cr == 0 && c == 0) {      // ring column F2_RING mirrors column 0: the epilogue reads [r], [r+1] unwrapped
#pragma unroll
                                        for (int r = 0; r < RB; r++)
                                            if (r < nrb) srow[r * 8 * F2_SROW + F2_RING] = acc[r][nt][0];
                                    }
                                }
                            }
                        }
                    }
                }

                else
#endif
            // ---------------- contraction: unit = (k, 8 bins) x 32 samples.  Q fragments of the next
                // unit are loaded into the other register set while this one is multiplied.
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
                        // fragment-major Q: bin pair block of 96 doubles, 16 per k-step pair, 8 per bin
                        const double* qrow = P.Qf + (((size_t)k * P.N_Qpad + row) >> 1) * (2 * ILE_QT_ROW) + (row & 1) * 8;
#pragma unroll
                        for (int p = 0; p < NPAIR; p++) b[p] = __ldg(reinterpret_cast<const double2*>(qrow + 16 * p + 2 * c));
                        if (SINGLE) bs = __ldg(qrow + 16 * NPAIR + c);
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
                            const double2 bp = b[p];
                            double2 a[RB];
#pragma unroll
                            for (int rb = 0; rb < RB; rb++) a[rb] = Ak[(p * RB + rb) * 32];
#pragma unroll
                            for (int rb = 0; rb < RB; rb++) dmma2(d[rb][0], d[rb][1], a[rb].x, bp.x);
#pragma unroll
                            for (int rb = 0; rb < RB; rb++) dmma2(e[rb][0], e[rb][1], a[rb].y, bp.y);
                        }
                        if (SINGLE) {
#pragma unroll
                            for (int rb = 0; rb < RB; rb += 2) {
                                const double2 as = Ak[(NPAIR * RB + (rb >> 1)) * 32];
                                dmma2(d[rb][0], d[rb][1], as.x, bs);
                                dmma2(d[rb + 1][0], d[rb + 1][1], as.y, bs);
                            }
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
                    int u = w;
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
    }
            __syncthreads();   // S complete for bins < c_hi
            // ---------------- epilogue: shift + interpolate + sum detectors, then a streaming
            // log-sum-exp.  Straight-line code over SPW x NG independent (sample row, 32-bin group)
            // chains; rows that do not take part in this round run on clamped offsets and are discarded.
            {
                int j0m = stride * j0;
                j0m -= (j0m / F2_RING) * F2_RING;
                const int jl0 = j0m + lane;                       // STRIDE1: ring bin of this lane's first output, before the sample offset
                bool inr[NG];                                     // output j0 + 32 gi + lane exists
#pragma unroll
                for (int gi = 0; gi < NG; gi++) inr[gi] = j0 + 32 * gi + lane < j1;
                // v: the values; (dh, dlo): high and low words of v - reference, the high word of a
                // missing output set to that of -inf.  All range logic runs on the high words in the
                // integer pipe: the FP64 pipe and the issue slots are what this loop is short of.
                double v[SPW][NG];
                int dh[SPW][NG], dlo[SPW][NG];
                bool need = false;
#pragma unroll
                for (int i = 0; i < SPW; i++) {
                    const int s = SPW * w + i;
                    const double2 cb = sm.ec[s];
                    const int4 o4 = *reinterpret_cast<const int4*>(&sm.eoff[s][0]);
                    const int off[4] = {o4.x, o4.y, o4.z, o4.w};
                    double2 wk[K];
                    int r[K];
#pragma unroll
                    for (int k = 0; k < K; k++) {
                        wk[k] = sm.ew[s][k];
                        if (STRIDE1) {
                            const unsigned rr = off[k] + jl0;                      // < 15 + 80 + 31: one wrap
                            r[k] = (int)min(rr, rr - F2_RING);
                        } else {
                            int rr = off[k] + j0m;
                            if (rr >= F2_RING) rr -= F2_RING;
                            r[k] = rr;
                        }
                    }
                    const double* Srow = &sm.S[0][s][0];
#pragma unroll
                    for (int gi = 0; gi < NG; gi++) {
                        double A = TABLE ? 0.0 : -cb.x;
#pragma unroll
                        for (int k = 0; k < K; k++) {
                            int r0;
                            if (STRIDE1) {
                                const unsigned rr = r[k] + 32 * gi;                // < 80 + 32: one wrap
                                r0 = gi == 0 ? r[k] : (int)min(rr, rr - F2_RING);
                            } else {
                                r0 = (r[k] + stride * (32 * gi + lane)) % F2_RING;
                            }
                            const double* row = Srow + k * (TS * F2_SROW) + r0;
                            A = fma(wk[k].x, row[0], A);
                            A = fma(wk[k].y, row[1], A);
                        }
                        if (TABLE) {
                            // lnT(A, B), bilinear and clamped: the row (cb.y) and its fraction (cb.x) are the sample's,
                            // the column coordinate one FMA (no division per bin), each lerp a subtraction and an FMA
                            double a = fma(A, tabA_s, tabA_o);
                            a = fmin(fmax(a, 0.0), (double)(P.nA - 1));
                            const int ia = min((int)a, P.nA - 2);
                            const double fa = a - (double)ia;
                            const double* T0 = P.lnT + (size_t)(int)cb.y * P.nA + ia;
                            const double t00 = __ldg(T0), t01 = __ldg(T0 + 1), t10 = __ldg(T0 + P.nA), t11 = __ldg(T0 + P.nA + 1);
                            const double t0 = fma(fa, t01 - t00, t00), t1 = fma(fa, t11 - t10, t10);
                            A = fma(cb.x, t1 - t0, t0);
                        }
                        v[i][gi] = A;
                        const double dl = A - run_m[i];
                        dh[i][gi] = inr[gi] ? __double2hiint(dl) : (int)0xFFF00000;
                        dlo[i][gi] = __double2loint(dl);
                        need = need || (dh[i][gi] >= 0x403E0000);                  // dl >= 30 (or NaN)
                    }
                }
                // raise the references where a new value is more than e^30 above (rare)
                if (__any_sync(0xffffffffu, need)) {
#pragma unroll
                    for (int i = 0; i < SPW; i++) {
                        double vm = neg_inf();
#pragma unroll
                        for (int gi = 0; gi < NG; gi++) vm = fmax(vm, inr[gi] ? v[i][gi] : neg_inf());
                        if (__any_sync(0xffffffffu, vm - run_m[i] >= 30.0)) {
                            // new reference >= max over lanes, found on the ordered high words with
                            // one REDUX; it need not be the exact maximum
                            const int h = __double2hiint(vm);
                            const int key = __reduce_max_sync(0xffffffffu, h ^ ((h >> 31) & 0x7fffffff));
                            const int hm = key ^ ((key >> 31) & 0x7fffffff);
                            const double mx = __hiloint2double(hm, hm < 0 ? 0 : -1);
                            const double dm = run_m[i] - mx;
                            // the running sum may hold terms up to e^30 above its reference: rescale exactly
                            run_s[i] = dm > -690.0 ? run_s[i] * exp_small(dm) : 0.0;
                            run_m[i] = mx;
#pragma unroll
                            for (int gi = 0; gi < NG; gi++) {
                                const double dl = v[i][gi] - mx;
                                dh[i][gi] = inr[gi] ? __double2hiint(dl) : (int)0xFFF00000;
                                dlo[i][gi] = __double2loint(dl);
                            }
                        }
                    }
                }
#pragma unroll
                for (int i = 0; i < SPW; i++)
#pragma unroll
                    for (int gi = 0; gi < NG; gi++) {
                        // terms below e^-40 of the reference (and missing outputs) are clamped to e^-40:
                        // dl <= -40 <=> high word >= 0xC0440000 as unsigned; one integer min.  The
                        // (N_t + 64) e^-40 < 3e-15 this adds to a sum >= 1 is in the tolerance budget.
                        const unsigned hc = min((unsigned)dh[i][gi], 0xC0440000u);
                        run_s[i] += exp_tab(__hiloint2double((int)hc, dlo[i][gi]), sm.etab);
                    }
            }
            if (j1 >= N_t) break;
            j0 = j1;
            c_lo = c_hi;
            ntiles = min(F2_NEW / 8, (last_bin + 1 - c_lo + 7) / 8);
            __syncthreads();   // ring reads done before the next phase overwrites old bins
        }
        // ---------------- finalise this round's samples: lane q < SPW writes sample row q
        {
            double my_m = run_m[0], my_t = warp_sum(run_s[0]);
#pragma unroll
            for (int q = 1; q < SPW; q++) {
                const double t = warp_sum(run_s[q]);
                if (lane == q) { my_m = run_m[q]; my_t = t; }
            }
            if (lane < SPW) {
                const int s = SPW * w + lane;
                if (sm.part[s]) {
                    const int t = tile * TS + s;
                    if (t < N) lnL[perm ? perm[t] : t] = my_m + log(my_t) - P.ln_Nt;
                    sm.done[s] = 1;
                }
            }
        }
        if (last_round) break;
    }
}


template <int K, int NPAIR, bool SINGLE, bool TABLE, bool STRIDE1>
__global__ void __launch_bounds__(F2_THREADS, 2)
lnl_fused2_kernel(LnlParams P, int N, int quad, const double* __restrict__ rec, const double2* __restrict__ ytile,
                  const int* __restrict__ perm, double* __restrict__ lnL) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Fused2Smem<K>& sm = *reinterpret_cast<Fused2Smem<K>*>(smem_raw);
    tile_body<K, NPAIR, SINGLE, TABLE, STRIDE1>(sm, threadIdx.x, blockIdx.x, P, N, quad, rec, ytile, perm, lnL);
}

template <int K, int NPAIR, bool SINGLE, bool TABLE, bool STRIDE1>
static int launch_fused2_t(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL, bool quad) {
    const int smem = (int)sizeof(Fused2Smem<K>);
    // per device, cheap: set on every launch (a per-process flag would miss a second device)
    ILE_CUDA(ctx, cudaFuncSetAttribute(lnl_fused2_kernel<K, NPAIR, SINGLE, TABLE, STRIDE1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    const int tiles = (N + F2_TS - 1) / F2_TS;
    const int slot = ile_timing_begin(ctx);
    lnl_fused2_kernel<K, NPAIR, SINGLE, TABLE, STRIDE1><<<tiles, F2_THREADS, smem, ctx->stream>>>(P, N, quad ? 1 : 0, rec, yt, perm, lnL);
    ile_timing_end(ctx, slot);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

template <int K, int NPAIR, bool SINGLE>
static int launch_fused2_k(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL, bool quad) {
    const bool tb = P.use_table != 0, s1 = P.stride == 1;
    if (tb) return s1 ? launch_fused2_t<K, NPAIR, SINGLE, true, true>(ctx, P, N, rec, yt, perm, lnL, quad)
                      : launch_fused2_t<K, NPAIR, SINGLE, true, false>(ctx, P, N, rec, yt, perm, lnL, quad);
    return s1 ? launch_fused2_t<K, NPAIR, SINGLE, false, true>(ctx, P, N, rec, yt, perm, lnL, quad)
              : launch_fused2_t<K, NPAIR, SINGLE, false, false>(ctx, P, N, rec, yt, perm, lnL, quad);
}

// rec / yt as written by lnl_prep_kernel (quad = false) or lnl_prep3_kernel (quad = true: the
// quadratic term is computed here) for ceil(N/64)*64 padded samples.  Returns 1 when the
// shape has no instantiation (the caller falls back to the plain kernel).
int ile_launch_fused2(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL, bool quad) {
    const int n2 = 2 * P.M, np = n2 / 8, rem = n2 % 8;
    if (P.K == 3 && np == 5 && rem >= 1 && rem <= 4) return launch_fused2_k<3, 5, true>(ctx, P, N, rec, yt, perm, lnL, quad);
    if (P.K == 2 && np == 1 && rem >= 1 && rem <= 4) return launch_fused2_k<2, 1, true>(ctx, P, N, rec, yt, perm, lnL, quad);
    return 1;
}

