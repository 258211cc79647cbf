// libile: fused lnL kernel on the Blackwell tensor path.
//
// Step 5 of the hot path, S_k[i][n] = sum_r coef_k[i][r] Q_k[r][n] (Eq. 7's Re[(F Y)^* Q] on the
// (time) x (extrinsic) array), is a dense real contraction with K-dimension 2M <= 48.  FP64 has no tcgen05 kind, so
// the contraction is done EXACTLY in integers instead: both operands are scaled by a power of two (per sample and
// detector for the coefficients, per intrinsic point and detector for Q), rounded to 47-bit integers and cut into
// six signed 8-bit digits, C = sum_a c_a 256^(5-a), Qi = sum_b q_b 256^(5-b).  Then
//     C Qi = sum_s 256^(10-s) acc_s,   acc_s = sum_{a+b=s} sum_r c_a[r] q_b[r]
// and each acc_s is one tcgen05.mma kind::i8 accumulation (int32, |acc_s| < 6 * 42 * 2^14: no overflow, no
// rounding) with the digit pairs of equal weight stacked along K.  Sums s <= 5 are kept (21 digit pairs); the
// dropped pairs are below 2^-43 of max|coef| max|Q| (DESIGN.md section 6 derives the bound against the 1e-9
// tolerance).  The six accumulators are recombined in FP64 by the epilogue.
//
//   operand A (coefficients): [c_0 | c_1 | ... | c_5], 48 bytes per digit block (2M <= 42 used), written to tensor
//              memory by the thread that owns the sample (tcgen05.st); stationary for the whole tile
//   operand B (Q digits): per stored bin 304 bytes [q_5 | q_4 | ... | q_0 | 16 zero bytes], built once per intrinsic
//              point at ile_load_quv in the K-major no-swizzle core-matrix layout, so that a 32-bin chunk is one
//              contiguous 9728-byte TMA bulk copy; sum s reads the view that starts at block 5 - s, which pairs
//              c_a with q_{s-a} (descriptor start addresses move in 16-byte steps)
//   tile       up to 128 samples of one delay cell (16 stored bins per detector) = the 128 lanes of tensor memory
//   work item  (32-bin chunk, detector): 33 MMAs of 128 x 32 x 32 into one set of six accumulators (192 columns), freed
//              as soon as the math warps have loaded it
//   warps      0-15: four threads per sample (group = warp / 4, lane quarter = warp % 4 = the tensor-memory lanes the warp
//              can reach): steps 1-2, harmonics, coefficients and digits (by detector), the U/V quadratic term (step 4, by
//              rows of the triangle); then per item accumulators -> 64-bit integer -> FP64 (8 bins per thread), interpolation
//              weights, accumulation of A_j = sum_k S_k(t_j + tau_k) into a thread-private column of a 64-row shared-memory
//              ring (the per-sample delay shift is an address offset), and the streaming log-sum-exp over complete time
//              bins (step 6, rows split over the four threads);  warp 16: TMA producer + MMA issuer
#include "common.cuh"
#include "likelihood_dev.cuh"
#include "radix_sort.cuh"
#include <type_traits>
#include "sm100_ptx.cuh"
#include "exp_tab.cuh"

#define SP_TS 128             // samples per tile
#define SP_NB 32              // stored bins per work item (MMA N)
#define SP_BLK 48             // bytes per digit block
#define SP_NCH 19             // 16-byte chunks per stored bin in the Q digit image (304 bytes)
#define SP_GRP (SP_NCH * 128) // bytes per group of 8 bins
#define SP_STAGE ((SP_NB / 8) * SP_GRP) // bytes per chunk of SP_NB bins
#define SP_NSTAGE 4
#define SP_RING 64            // rows (time bins) of the accumulation ring
#define SP_CAPMAX 24          // largest per-sample offset above the tile base
#define SP_CELL_SHIFT 4       // delay cells of 16 stored bins
#define SP_ACOLS 72           // tensor-memory columns of A per detector (288 bytes)
#define SP_DCOL 256           // first accumulator column; sum s at SP_DCOL + SP_NB s (one set: it is free again as soon as every warp has loaded its bins)
#define SP_G 4                // threads per sample (warp groups): digits by detector, bins, triangle rows, log-sum-exp rows
#define SP_MATH (SP_G * SP_TS)
#define SP_RAISE_HI 0x40800000   // high word of 512.0: the streaming log-sum-exp raises its reference beyond e^512
#define SP_REC 12               // doubles per sample record: z[0..5] (RA, sin Dec, psi, phi_ref, cos incl, D), u_k[0..2], padding
#define SP_THREADS (SP_MATH + 32)
#define SP_UVMAX (300 * 3 * 2)
#define SP_MAGIC 6755399441055744.0   // 1.5 * 2^52
#define SP_HOT 24               // distance table: first nodes of a sample's row pair kept (blended over B) in shared memory, one per row of sm.Y

struct SpTile {
    int start, cnt;           // sorted positions [start, start + cnt)
    int base[3];              // first stored bin of the tile's window per detector (multiple of 8)
    int cap;                  // largest offset n_k - base_k in the tile
    int nchunk;               // 16-bin chunks to contract
    int flags;                // 1: samples outside the prior box (lnL = -inf), 2: delay spread too large (NaN)
};

// ---------------------------------------------------------------- Q digits (ile_load_quv)
// biased exponent of max |Q| per (point, detector)
__global__ void sp_qmax_kernel(const double* __restrict__ Qc, int M, int N_Q, unsigned int* __restrict__ qhi) {
    const int pk = blockIdx.y;
    const double* src = Qc + (size_t)pk * M * N_Q * 2;
    const long long total = (long long)M * N_Q * 2;
    unsigned int mx = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x)
        mx = max(mx, (unsigned int)__double2hiint(src[i]) & 0x7fffffffu);
    mx = __reduce_max_sync(0xffffffffu, mx);
    if ((threadIdx.x & 31) == 0) atomicMax(&qhi[pk], mx);
}

// digits of rint(v), |v| < 2^46: c = sum_p d_p 256^p with d_p in [-128, 127]; lo = (d_0..d_3), hi bytes 0, 1 = d_4, d_5
__device__ __forceinline__ void sp_digits(double v, uint32_t& lo, uint32_t& hi) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v + SP_MAGIC);   // 0x4338000000000000 + rint(v)
    const unsigned long long c = (b + 0xBCC8808080808080ull) ^ 0x0000808080808080ull;
    lo = (uint32_t)c;
    hi = (uint32_t)(c >> 32);
}
// digit words of four values: w[a] = digit of weight 256^(5-a) of (v0, v1, v2, v3), one per byte
__device__ __forceinline__ void sp_digit_words(const uint32_t (&lo)[4], const uint32_t (&hi)[4], uint32_t (&w)[6]) {
    const uint32_t a01 = __byte_perm(lo[0], lo[1], 0x5140), b01 = __byte_perm(lo[0], lo[1], 0x7362);
    const uint32_t a23 = __byte_perm(lo[2], lo[3], 0x5140), b23 = __byte_perm(lo[2], lo[3], 0x7362);
    const uint32_t h01 = __byte_perm(hi[0], hi[1], 0x5140), h23 = __byte_perm(hi[2], hi[3], 0x5140);
    w[5] = __byte_perm(a01, a23, 0x5410);
    w[4] = __byte_perm(a01, a23, 0x7632);
    w[3] = __byte_perm(b01, b23, 0x5410);
    w[2] = __byte_perm(b01, b23, 0x7632);
    w[1] = __byte_perm(h01, h23, 0x5410);
    w[0] = __byte_perm(h01, h23, 0x7632);
}

// one thread per (point-detector, stored bin, group of four reals r = 4 q .. 4 q + 3, r = 2 mode + part)
__global__ void sp_qslice_kernel(const double* __restrict__ Qc, int PK, int M, int N_Q, int NG8, const unsigned int* __restrict__ qhi,
                                 int* __restrict__ qeb, unsigned char* __restrict__ Qs) {
    const long long total = (long long)PK * NG8 * 8 * 12;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const int q = (int)(idx % 12);
        const long long rest = idx / 12;
        const int n = (int)(rest % (NG8 * 8));
        const int pk = (int)(rest / (NG8 * 8));
        const int eb = min(max((int)(qhi[pk] >> 20), 200), 1800);
        if (n == 0 && q == 0) qeb[pk] = eb;
        const double sc = __hiloint2double((2091 - eb) << 20, 0);            // 2^(45 - (eb - 1023))
        uint32_t lo[4], hi[4], w[6];
#pragma unroll
        for (int r = 0; r < 4; r++) {
            const int rr = 4 * q + r, mode = rr >> 1, part = rr & 1;
            double v = 0.0;
            if (mode < M && n < N_Q) v = Qc[(((size_t)pk * M + mode) * N_Q + n) * 2 + part];
            sp_digits(v * sc, lo[r], hi[r]);
        }
        sp_digit_words(lo, hi, w);
        unsigned char* row = Qs + ((size_t)pk * NG8 + (n >> 3)) * SP_GRP + (n & 7) * 16;
#pragma unroll
        for (int b = 0; b < 6; b++) {
            const int off = SP_BLK * (5 - b) + 4 * q;                         // block 5 - b holds digit b
            *reinterpret_cast<uint32_t*>(row + (off >> 4) * 128 + (off & 15)) = w[b];
        }
    }
}

size_t ile_split_qs_bytes(int P, int K, int N_Q) { return (size_t)P * K * ((N_Q + 64 + 7) / 8) * SP_GRP; }
int ile_split_ng8(int N_Q) { return (N_Q + 64 + 7) / 8; }

int ile_split_build_q(ile_ctx* ctx, int P, int K, int M, int N_Q, const double* d_Qc, unsigned char* d_Qs, int* d_qeb, unsigned int* d_qhi) {
    const int NG8 = ile_split_ng8(N_Q);
    ILE_CUDA(ctx, cudaMemsetAsync(d_Qs, 0, ile_split_qs_bytes(P, K, N_Q), ctx->stream));
    ILE_CUDA(ctx, cudaMemsetAsync(d_qhi, 0, (size_t)P * K * sizeof(unsigned int), ctx->stream));
    sp_qmax_kernel<<<dim3(32, P * K), 256, 0, ctx->stream>>>(d_Qc, M, N_Q, d_qhi);
    ILE_LAUNCH_CHECK(ctx);
    sp_qslice_kernel<<<ctx->sm_count * 8, 256, 0, ctx->stream>>>(d_Qc, P * K, M, N_Q, NG8, d_qhi, d_qeb, d_Qs);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

// ---------------------------------------------------------------- delay-cell keys and tiles
__global__ void __launch_bounds__(256) sp_key_kernel(LnlParams P, int N, const double* __restrict__ z, int n_min, int cell_bits,
                                                     unsigned long long* __restrict__ key, unsigned int* __restrict__ val, double* __restrict__ rec,
                                                     long long* n_dev, int* bits_dev, int* ntiles_dev) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        *n_dev = N;
        *bits_dev = cell_bits * P.K + 1;
        ntiles_dev[0] = 0;                                 // tile count, run count
        ntiles_dev[1] = 0;
    }
    __shared__ double srec[256 * (SP_REC + 1)];
    if (i < N) {
        // the sample's record: coordinates (coalesced reads, one array per coordinate) and below its u_k, 96 bytes = three
        // whole 32-byte sectors, so that the fused kernel's gather through the sort permutation fetches nothing it does not use
        double zc[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 1.0}, uo[3] = {0.0, 0.0, 0.0};
#pragma unroll
        for (int c = 0; c < 6; c++)
            if (c < P.d) zc[c] = z[(size_t)c * N + i];          // six independent loads in flight
        const double ra = zc[0], sd = zc[1];
        bool ok = true;
        if (!P.box_trusted) {
#pragma unroll
            for (int c = 0; c < 6; c++)
                if (c < P.d) ok = ok && (zc[c] >= P.lo[c]) && (zc[c] < P.hi[c]);
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
                if (kk < 3) uo[kk] = u;                          // the fused kernel uses this very value
                int cell = ((int)floor(u) - n_min) >> SP_CELL_SHIFT;
                cell = max(0, min(cell, (1 << cell_bits) - 1));
                k = (k << cell_bits) | (unsigned long long)cell;
            }
        }
        key[i] = k;
        val[i] = (unsigned int)i;
        {
            double* r = &srec[threadIdx.x * (SP_REC + 1)];     // odd stride: conflict-free
    #pragma unroll
            for (int c = 0; c < 6; c++) r[c] = zc[c];
            r[6] = uo[0]; r[7] = uo[1]; r[8] = uo[2];
            r[9] = r[10] = r[11] = 0.0;
        }
    }
    // the block's records are contiguous in global memory: consecutive threads write consecutive doubles
    __syncthreads();
    const size_t first = (size_t)blockIdx.x * blockDim.x;
    const int nrec = (int)min((size_t)blockDim.x, (size_t)N - first);
    for (int q = threadIdx.x; q < nrec * SP_REC; q += blockDim.x) rec[first * SP_REC + q] = srec[(q / SP_REC) * (SP_REC + 1) + q % SP_REC];
}

// Tiles: the sorted order is cut at every cell change (run start) and every 128 samples after it.
// pass 1: run starts, appended in any order
__global__ void __launch_bounds__(256) sp_run_flag_kernel(int N, const unsigned long long* __restrict__ key, int* __restrict__ runs, int* nruns_dev) {
    const int pos = blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= N) return;
    if (pos == 0 || key[pos] != key[pos - 1]) runs[atomicAdd(nruns_dev, 1)] = pos;
}
// pass 2: one block per run: its end by binary search, then its tile starts
__global__ void __launch_bounds__(256) sp_run_tiles_kernel(int N, const unsigned long long* __restrict__ key, const int* __restrict__ runs,
                                                          const int* __restrict__ nruns_dev, int* __restrict__ tstart, int* ntiles_dev) {
    const int nruns = *nruns_dev;
    __shared__ int sh_first, sh_nt;
    for (int r = blockIdx.x; r < nruns; r += gridDim.x) {
        const int rs = runs[r];
        if (threadIdx.x == 0) {
            const unsigned long long k0 = key[rs];
            int lo = rs + 1, hi = N;                     // first position with a larger key
            while (lo < hi) {
                const int mid = (int)(((long long)lo + hi) >> 1);
                if (key[mid] > k0) hi = mid; else lo = mid + 1;
            }
            sh_nt = (lo - rs + SP_TS - 1) / SP_TS;
            sh_first = atomicAdd(ntiles_dev, sh_nt);
        }
        __syncthreads();
        for (int q = threadIdx.x; q < sh_nt; q += blockDim.x) tstart[sh_first + q] = rs + q * SP_TS;
        __syncthreads();
    }
}

// one warp per tile: extent; the window base per detector is the tile's delay cell (read off the key), so that every
// offset above it is at most 15 + 7 (cells of 16 bins on an 8-aligned grid) and no sample has to be looked at
__global__ void __launch_bounds__(256) sp_tile_info_kernel(LnlParams P, int N, int n_min, int cell_bits, const unsigned long long* __restrict__ key,
                                                           const int* __restrict__ tstart, const int* __restrict__ ntiles_dev, SpTile* __restrict__ tiles) {
    const int id = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (id >= *ntiles_dev) return;
    const int start = tstart[id];
    const unsigned long long k0 = key[start];
    int cnt = 0;
    bool open = true;
    for (int q = 0; q < SP_TS / 32; q++) {
        const int pos = start + 32 * q + lane;
        const bool mem = open && pos < N && key[pos] == k0;
        const unsigned b = __ballot_sync(0xffffffffu, mem);
        const int lead = b == 0xffffffffu ? 32 : __ffs(~b) - 1;      // members are a prefix
        cnt += lead;
        if (lead < 32) open = false;
    }
    SpTile t;
    t.start = start;
    t.cnt = cnt;
    t.flags = (k0 >> (cell_bits * P.K)) ? 1 : 0;
    t.cap = 0;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        t.base[k] = 0;
        if (k < P.K) {
            const int cell = (int)((k0 >> (cell_bits * (P.K - 1 - k))) & ((1ull << cell_bits) - 1ull));
            const int first = n_min + (cell << SP_CELL_SHIFT);          // first bin of the cell (n_min is a multiple of 8)
            t.base[k] = max(first, 0);
            t.cap = max(t.cap, first + (1 << SP_CELL_SHIFT) - 1 - t.base[k]);
        }
    }
    t.nchunk = t.flags ? 0 : (P.N_t + 1 + t.cap + SP_NB - 1) / SP_NB;
    if (lane == 0) tiles[id] = t;
}

// ---------------------------------------------------------------- the fused kernel
struct SplitSmem {
    unsigned char bst[SP_NSTAGE][SP_STAGE];   // Q digit chunks (TMA destination, MMA operand B)
    double ring[SP_RING][SP_TS];              // A_j accumulation: row = time bin mod 64, column = sample (thread-private)
    double2 Y[24][SP_TS];                     // harmonics of the tile, column = sample
    double2 uv[SP_UVMAX];                     // packed upper-triangle U/V of the intrinsic point
    double etab[64][16];                      // 2^(j/64), 16 copies: lane l reads copy l % 16 (conflict-free)
    double xch[2][3][SP_TS];                  // last bin of a chunk, from group 3 to group 0 of the next chunk (slot = chunk parity)
    double lse[SP_G][2][SP_TS];               // partial (reference, sum) of the four threads of a sample
    int eb[3][SP_TS];                         // biased exponent of max |coefficient| per detector
    double wgt[2][3][SP_TS];                  // interpolation weights of the sample's window per detector (scaled: unit of the integer contraction)
    int offs[3][SP_TS];                       // first stored bin of the sample's window above the tile's base, per detector
    YlmTable ytab;                            // term table of the harmonics (Eq. 4), copied once per CTA
    uint64_t a_full, d_full, d_empty, b_full[SP_NSTAGE], b_empty[SP_NSTAGE];
    uint32_t tmem_base;
};

// exp(d), d in [-40, 31]: 2^(k >> 6) tab[k & 63] (1 + r (1 + r/2 + r^2/6 + r^3/24)), k = rint(64 d / ln 2) (R2)
__device__ __forceinline__ double sp_exp_tab(double d, const double* __restrict__ tab_lane) {
    const double t = fma(d, 0x1.71547652b82fep+6, SP_MAGIC);
    const int k = __double2loint(t);
    const double kf = t - SP_MAGIC;
    const double r = fma(kf, -0x1.62e42fefa39efp-7, d);
    const double T = tab_lane[(k & 63) * 16];
    double p = fma(r, 1.0 / 24.0, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    const double e = fma(T * r, p, T);
    return __hiloint2double(__double2hiint(e) + ((k >> 6) << 20), __double2loint(e));
}
// exp(d) for d in (-690, 0]: degree-10 Taylor after range reduction (used only when a reference is raised)
__device__ __forceinline__ double sp_exp_small(double d) {
    const double t = fma(d, 1.4426950408889634, SP_MAGIC);
    const int k = __double2loint(t);
    const double kf = t - SP_MAGIC;
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

// V = sum_s acc_s 256^(5-s) = t0 2^32 + t1 2^16 + t2 with t = acc_even 256 + acc_odd (int32, no overflow), exact in 64-bit
// integers (|V| < 2^63), then one conversion (rounded to 53 bits: 2^-53 of |V|, far below the digits dropped)
__device__ __forceinline__ double sp_recombine(uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t a4, uint32_t a5) {
    const int t0 = (int)a0 * 256 + (int)a1, t1 = (int)a2 * 256 + (int)a3, t2 = (int)a4 * 256 + (int)a5;
    const long long wl = (long long)t1 * 65536LL + (long long)t2;
    const unsigned hi = (unsigned)(wl >> 32) + (unsigned)t0;                  // + t0 2^32: no carry into the low word
    return (double)(long long)(((unsigned long long)hi << 32) | (unsigned)wl);
}

// cursor over the work items (tile, chunk, detector) of this CTA, in the order both warp roles walk them
struct SpCursor {
    int t, c, k, nchunk;
    int base[3];
};
template <int K>
__device__ __forceinline__ void sp_cursor_load(SpCursor& cu, const SpTile* __restrict__ tiles, int ntiles, int step) {
    while (cu.t < ntiles) {
        const SpTile ti = tiles[cu.t];
        if (ti.nchunk > 0) {
            cu.nchunk = ti.nchunk;
#pragma unroll
            for (int k = 0; k < 3; k++) cu.base[k] = ti.base[k];
            cu.c = 0;
            cu.k = 0;
            return;
        }
        cu.t += step;
    }
    cu.nchunk = 0;
}
template <int K>
__device__ __forceinline__ void sp_cursor_next(SpCursor& cu, const SpTile* __restrict__ tiles, int ntiles, int step) {
    if (++cu.k < K) return;
    cu.k = 0;
    if (++cu.c < cu.nchunk) return;
    cu.t += step;
    sp_cursor_load<K>(cu, tiles, ntiles, step);
}

template <int K, bool TABLE>
__global__ void __launch_bounds__(SP_THREADS, 1)
lnl_split_kernel(LnlParams P, int N, const double* __restrict__ rec, const int* __restrict__ perm,
                 double* __restrict__ lnL, double* __restrict__ ln_prior, const SpTile* __restrict__ tiles, const int* __restrict__ ntiles_dev) {
    extern __shared__ __align__(1024) unsigned char sp_smem_raw[];
    SplitSmem& sm = *reinterpret_cast<SplitSmem*>(sp_smem_raw);
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int ntiles = *ntiles_dev;

    if (w == SP_MATH / 32) tmem_alloc512(&sm.tmem_base);
    if (tid == 0) {
        mbar_init(&sm.a_full, SP_MATH);
        mbar_init(&sm.d_full, 1);
        mbar_init(&sm.d_empty, SP_MATH);
        for (int s = 0; s < SP_NSTAGE; s++) { mbar_init(&sm.b_full[s], 1); mbar_init(&sm.b_empty[s], 1); }
        mbar_init_fence();
    }
    for (int q = tid; q < 64 * 16; q += SP_THREADS) sm.etab[q >> 4][q & 15] = f2_exp2_tab[q >> 4];
    {
        const int4* src = reinterpret_cast<const int4*>(P.ylm);
        int4* dst = reinterpret_cast<int4*>(&sm.ytab);
        for (int q = tid; q < (int)(sizeof(YlmTable) / 16); q += SP_THREADS) dst[q] = src[q];
    }
    {
        const double2* usrc = reinterpret_cast<const double2*>(P.UVp);
        const int nuv = min(P.n_pairs * K * 2, SP_UVMAX);
        for (int q = tid; q < nuv; q += SP_THREADS) sm.uv[q] = usrc[q];
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sm.tmem_base;

    if (w == SP_MATH / 32) {
        // ================================================================ producer: TMA loads and MMA issue
        const bool el = elect_one();
        const uint32_t idesc = umma_idesc_s8_m128(SP_NB);
        SpCursor L, Mc;
        L.t = Mc.t = blockIdx.x;
        sp_cursor_load<K>(L, tiles, ntiles, gridDim.x);
        sp_cursor_load<K>(Mc, tiles, ntiles, gridDim.x);
        unsigned nl = 0, nm = 0, tile_par = 0;
        while (Mc.nchunk > 0) {
            while (L.nchunk > 0 && nl < nm + (SP_NSTAGE - 1)) {
                const unsigned s = nl % SP_NSTAGE;
                if (nl >= SP_NSTAGE) mbar_wait(&sm.b_empty[s], ((nl / SP_NSTAGE) - 1) & 1);
                if (el) {
                    const unsigned char* src = P.Qs + ((size_t)L.k * P.NG8 + ((L.base[L.k] + SP_NB * L.c) >> 3)) * SP_GRP;
                    mbar_expect_tx(&sm.b_full[s], SP_STAGE);
                    bulk_g2s(sm.bst[s], src, SP_STAGE, &sm.b_full[s]);
                }
                nl++;
                sp_cursor_next<K>(L, tiles, ntiles, gridDim.x);
            }
            if (Mc.c == 0 && Mc.k == 0) {             // the tile's coefficient digits are in tensor memory
                mbar_wait(&sm.a_full, tile_par);
                tile_par ^= 1;
            }
            const unsigned s = nm % SP_NSTAGE;
            if (nm >= 1) mbar_wait(&sm.d_empty, (nm - 1) & 1);
            mbar_wait(&sm.b_full[s], (nm / SP_NSTAGE) & 1);
            tc_fence_after();
            if (el) {
                const uint64_t b0 = umma_desc_kmajor_noswizzle(smem_u32(sm.bst[s]), 128, SP_GRP);
                const uint32_t a0 = tmem + SP_ACOLS * Mc.k, d0 = tmem + SP_DCOL;
                // sum s reads K_s = 64, 96, 160, 192, 256, 288 bytes of A against the view of B starting at 16-byte chunk 3 (5 - s);
                // k-step major, so that consecutive MMAs go to different accumulators
#pragma unroll
                for (int t = 0; t < 9; t++) {
#pragma unroll
                    for (int sidx = 0; sidx < 6; sidx++) {
                        const int Ks = sidx == 0 ? 64 : sidx == 1 ? 96 : sidx == 2 ? 160 : sidx == 3 ? 192 : sidx == 4 ? 256 : 288;
                        if (32 * t < Ks) umma_i8_ts(d0 + SP_NB * sidx, a0 + 8 * t, b0 + (uint64_t)(((3 * (5 - sidx) + 2 * t) * 128) >> 4), idesc, t > 0 ? 1u : 0u);
                    }
                }
                umma_commit(&sm.b_empty[s]);
                umma_commit(&sm.d_full);
            }
            __syncwarp();
            nm++;
            sp_cursor_next<K>(Mc, tiles, ntiles, gridDim.x);
        }
    } else {
        // ================================================================ SP_G threads per sample
        // thread (g, i): sample i of the tile = tensor-memory lane i (warp % 4 is the lane quarter), group g = warp / 4.
        // The four threads of a sample split its work: detectors (digits), rows of the U/V triangle (step 4), bins of
        // every work item (4 each) and rows of the log-sum-exp.  They meet at a named barrier per lane quarter.
        const int g = w >> 2, qd = w & 3;
        const int i = 32 * qd + lane;
        const uint32_t tlane = tmem + ((uint32_t)(32 * qd) << 16);
        double* const rcol = &sm.ring[0][i];
        const double* const fx_col = &sm.lse[0][0][i];           // prologue: rows 0..2 Re F_k, 3..5 Im F_k, 6 x of sample i
        const double* const u_col = &sm.xch[0][0][i];            // prologue: rows 0..2 u_k
        const double* const etab = &sm.etab[0][lane & 15];
        const double tabA_s = TABLE ? (double)(P.nA - 1) / (P.A_hi - P.A_lo) : 0.0, tabA_o = -P.A_lo * tabA_s;
        auto qbar = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(1 + qd), "r"(32 * SP_G) : "memory"); };
        unsigned im = 0;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
            const SpTile ti = tiles[t];
            const int pos = ti.start + i;
            const bool member = i < ti.cnt;
            if (ti.nchunk == 0) {
                if (member && g == 0) {
                    lnL[perm[pos]] = (ti.flags & 2) ? __longlong_as_double(0x7ff8000000000000LL) : neg_inf();
                    if (ln_prior && (ti.flags & 1)) ln_prior[perm[pos]] = neg_inf();
                }
                continue;
            }
            const int N_t = P.N_t;
            // ---- steps 1-2 in place (no preparation kernel, no per-sample record in HBM).  The four threads of a sample
            //      share the work and meet in shared memory (arrays that are idle during the prologue): group 0 the antenna
            //      patterns F_k = F+ - i Fx, group 1 the powers of cos, sin(iota/2), group 2 the phases e^{i m phi}, group 3
            //      x = D_ref / D, ln prior and the stored-bin coordinates u_k of grid time 0 (from the key kernel: the very
            //      values the tile's window was built from).  Coordinates are gathered through the sort permutation.
            double fr[K], fi[K], w0[K], w1[K], x;
            int off[K];
            bool off_bad = false;
            {
                const size_t sidx = member ? (size_t)perm[pos] : 0;
                double* const shr = &sm.lse[0][0][i];                     // rows 0..2 Re F_k, 3..5 Im F_k, 6 x
                double* const shu = &sm.xch[0][0][i];                     // rows 0..2 u_k
                double* const scr = &sm.ring[0][i];                       // harmonics' tables: row q of table t at scr[(t0 + q) * SP_TS]
                const int mp = sm.ytab.max_pow, mm = sm.ytab.max_abs_m;
                double* const pc = scr;
                double* const ps = pc + (mp + 1) * SP_TS;
                double* const cm = ps + (mp + 1) * SP_TS;
                double* const sn = cm + (mm + 1) * SP_TS;
                if (g == 0) {
                    SampleIn sp;
                    sp.ra = 0.0; sp.sd = 0.0; sp.cd = 1.0; sp.psi = 0.0; sp.phi_ref = 0.0; sp.ch = 1.0; sp.sh = 0.0; sp.dist = 1.0; sp.valid = member;
                    if (member) {
                        const double2 r0 = __ldg(reinterpret_cast<const double2*>(rec + sidx * SP_REC));
                        sp.ra = r0.x;
                        sp.sd = r0.y;
                        sp.psi = __ldg(rec + sidx * SP_REC + 2);
                        sp.cd = sqrt(fmax((1.0 - sp.sd) * (1.0 + sp.sd), 0.0));
                    }
                    double Fp[ILE_MAX_K], Fx[ILE_MAX_K], tau[ILE_MAX_K];
                    antenna_dev(P, sp, Fp, Fx, tau);
#pragma unroll
                    for (int k = 0; k < K; k++) {
                        shr[k * SP_TS] = Fp[k];
                        shr[(3 + k) * SP_TS] = -Fx[k];
                    }
                } else if (g == 1) {
                    const double ci = member ? __ldg(rec + sidx * SP_REC + 4) : 1.0;
                    const double ch = sqrt(fmax(0.5 * (1.0 + ci), 0.0)), sh = sqrt(fmax(0.5 * (1.0 - ci), 0.0));
                    double a = 1.0, b = 1.0;
                    pc[0] = 1.0;
                    ps[0] = 1.0;
                    for (int q = 1; q <= mp; q++) {
                        a *= ch;
                        b *= sh;
                        pc[q * SP_TS] = a;
                        ps[q * SP_TS] = b;
                    }
                } else if (g == 2) {
                    const double phi = member ? -__ldg(rec + sidx * SP_REC + 3) : 0.0;   // -2Y_lm(iota, -phi_ref) (reading G7)
                    cm[0] = 1.0;
                    sn[0] = 0.0;
                    for (int q = 1; q <= mm; q++) {
                        double sq, cq;
                        sincos((double)q * phi, &sq, &cq);
                        cm[q * SP_TS] = cq;
                        sn[q * SP_TS] = sq;
                    }
                } else {
                    double xs = 0.0;
                    if (member) {
                        SampleIn sp;
                        sp.dist = P.d > 5 ? __ldg(rec + sidx * SP_REC + 5) : 1.0;
                        xs = TABLE ? 1.0 : P.D_ref / sp.dist;
                        if (ln_prior) ln_prior[sidx] = ln_prior_dev(P, sp);
                    }
                    shr[6 * SP_TS] = xs;
#pragma unroll
                    for (int k = 0; k < K; k++) shu[k * SP_TS] = member ? __ldg(rec + sidx * SP_REC + 6 + k) : (double)ti.base[k];
                }
                qbar();
                // ---- harmonics (Eq. 4): group g evaluates modes g, g + 4, ... from the tables
                const int M = sm.ytab.M;
                for (int m = g; m < 24; m += SP_G) {
                    double2 y = make_double2(0.0, 0.0);
                    if (m < M) {
                        const YlmMode& Ym = sm.ytab.mode[m];
                        double acc = 0.0;
                        for (int t = 0; t < Ym.nterms; t++) acc += Ym.coef[t] * pc[Ym.pc[t] * SP_TS] * ps[Ym.ps[t] * SP_TS];
                        const int am = Ym.m < 0 ? -Ym.m : Ym.m;
                        const double c = cm[am * SP_TS], sgn = Ym.m < 0 ? -sn[am * SP_TS] : sn[am * SP_TS];
                        y = make_double2(acc * c, acc * sgn);
                    }
                    sm.Y[m][i] = y;
                }
            }
            qbar();
            // ---- the next tile's records are gathered through the sort permutation (scattered 96-byte reads): ask for
            //      them now, so that its prologue finds them in L2 instead of waiting two dependent DRAM round trips
            if (t + (int)gridDim.x < ntiles) {
                const SpTile tn = tiles[t + gridDim.x];
                if (tn.nchunk > 0 && i < tn.cnt) {
                    const size_t sn_ = (size_t)perm[tn.start + i];
                    auto pf = [](const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); };
                    if (g < 3) pf(rec + sn_ * SP_REC + 4 * g);           // the record's three sectors
                }
            }
            // ---- step 3 (group k does detector k): coefficients x F_k Y_m -> six signed 8-bit digits -> tensor memory (operand A)
#pragma unroll
            for (int k = 0; k < K; k++) {
                if (k != g) continue;
                const double xk = fx_col[6 * SP_TS];                               // x, F_k from step 1 (read again after step 4: registers)
                const double xr = xk * fx_col[k * SP_TS], xi = xk * fx_col[(3 + k) * SP_TS];
                int mh = 0;
#pragma unroll 4
                for (int m = 0; m < 24; m++) {
                    const double2 y = sm.Y[m][i];
                    const double cr = xr * y.x - xi * y.y, ci = xr * y.y + xi * y.x;
                    mh = max(mh, max(__double2hiint(cr) & 0x7fffffff, __double2hiint(ci) & 0x7fffffff));
                }
                const int eb = min(max(mh >> 20, 200), 1800);
                sm.eb[k][i] = eb;
                const double sc = __hiloint2double((2091 - eb) << 20, 0);         // 2^(45 - (eb - 1023)): |coef sc| < 2^46
                uint32_t col[6][12];
#pragma unroll
                for (int q = 0; q < 12; q++) {
                    const double2 y0 = sm.Y[2 * q][i], y1 = sm.Y[2 * q + 1][i];
                    uint32_t lo[4], hi[4], wd[6];
                    sp_digits((xr * y0.x - xi * y0.y) * sc, lo[0], hi[0]);
                    sp_digits((xr * y0.y + xi * y0.x) * sc, lo[1], hi[1]);
                    sp_digits((xr * y1.x - xi * y1.y) * sc, lo[2], hi[2]);
                    sp_digits((xr * y1.y + xi * y1.x) * sc, lo[3], hi[3]);
                    sp_digit_words(lo, hi, wd);
#pragma unroll
                    for (int a = 0; a < 6; a++) col[a][q] = wd[a];
                }
#pragma unroll
                for (int gg = 0; gg < 9; gg++) {
                    uint32_t v[8];
#pragma unroll
                    for (int e = 0; e < 8; e++) v[e] = col[(8 * gg + e) / 12][(8 * gg + e) % 12];
                    tmem_st8(tlane + SP_ACOLS * k + 8 * gg, v);
                }
                tmem_wait_st();
            }
            tc_fence_before();
            mbar_arrive(&sm.a_full);
            // ---- step 4: B = 1/4 sum_k [ |F_k|^2 Re(y^H U_k y) + Re(F_k^2 y^T V_k y) ] over the upper triangle (Eq. 17-18).
            //      Group g walks the rows P.tri_group gives it (fewer pairs for the groups that cut digits above); the partial
            //      sums meet in the ring's memory.
            double* const qpart = &sm.ring[0][0];                // [SP_G][3 K][128], the ring is idle until the first work item
            {
                double uu[K], vr[K], vi[K];
#pragma unroll
                for (int k = 0; k < K; k++) uu[k] = vr[k] = vi[k] = 0.0;
                const int M = P.M;
                auto pair = [&](const double2 ya, const double2 yb, const double2* __restrict__ uq) {
                    const double t2 = ya.y * yb.y, t4 = ya.y * yb.x;
                    const double pr = fma(ya.x, yb.x, t2), qr = fma(ya.x, yb.x, -t2), pi = fma(ya.x, yb.y, -t4), qi = fma(ya.x, yb.y, t4);
#pragma unroll
                    for (int k = 0; k < K; k++) {
                        const double2 u = uq[2 * k], v = uq[2 * k + 1];
                        uu[k] = fma(-u.y, pi, fma(u.x, pr, uu[k]));
                        vr[k] = fma(-v.y, qi, fma(v.x, qr, vr[k]));
                        vi[k] = fma(v.y, qr, fma(v.x, qi, vi[k]));
                    }
                };
                for (int a = 0; a < M; a++) {
                    if (P.tri_group[a] != g) continue;
                    const double2 ya = sm.Y[a][i];
                    const double2* uv = sm.uv + (size_t)(a * M - (a * (a - 1)) / 2) * 2 * K;
                    int b = a;
                    if ((M - a) & 1) {                                   // odd row length: the diagonal pair alone
                        pair(ya, ya, uv);
                        uv += 2 * K;
                        b++;
                    }
                    for (; b < M; b += 2) {                              // two pairs per step, loads first
                        const double2 yb0 = sm.Y[b][i], yb1 = sm.Y[b + 1][i];
                        pair(ya, yb0, uv);
                        pair(ya, yb1, uv + 2 * K);
                        uv += 4 * K;
                    }
                }
#pragma unroll
                for (int k = 0; k < K; k++) {
                    qpart[((g * 3 * K) + 3 * k + 0) * SP_TS + i] = uu[k];
                    qpart[((g * 3 * K) + 3 * k + 1) * SP_TS + i] = vr[k];
                    qpart[((g * 3 * K) + 3 * k + 2) * SP_TS + i] = vi[k];
                }
            }
            qbar();
            // the sample's F_k, x and window offsets are picked up only now: step 4 above has the registers for its loads
            x = fx_col[6 * SP_TS];
#pragma unroll
            for (int k = 0; k < K; k++) {
                fr[k] = fx_col[k * SP_TS];
                fi[k] = fx_col[(3 + k) * SP_TS];
                const double u = u_col[k * SP_TS], fl = floor(u);
                w1[k] = u - fl;
                w0[k] = 1.0 - w1[k];
                off[k] = min(max((int)fl - ti.base[k], 0), SP_CAPMAX);
                off_bad = off_bad || ((int)fl - ti.base[k] != off[k]);      // outside the tile's window: cannot happen for a sample of this cell
            }
            double Bq = 0.0;
#pragma unroll
            for (int k = 0; k < K; k++) {
                double uu = 0.0, vr = 0.0, vi = 0.0;
#pragma unroll
                for (int gg = 0; gg < SP_G; gg++) {
                    uu += qpart[((gg * 3 * K) + 3 * k + 0) * SP_TS + i];
                    vr += qpart[((gg * 3 * K) + 3 * k + 1) * SP_TS + i];
                    vi += qpart[((gg * 3 * K) + 3 * k + 2) * SP_TS + i];
                }
                Bq += (fr[k] * fr[k] + fi[k] * fi[k]) * uu + ((fr[k] * fr[k] - fi[k] * fi[k]) * vr - 2.0 * fr[k] * fi[k] * vi);
                // 2^40 / (sc sq_k): the weight of the integer contraction, folded into the interpolation weights
                const double un = __hiloint2double(min(max(sm.eb[k][i] + P.qeb[k] - 1023 - 50, 1), 2046) << 20, 0);
                w0[k] *= un;
                w1[k] *= un;
                if (g == 0) {                                   // read back item by item: fifteen registers less across the work items
                    sm.wgt[0][k][i] = w0[k];
                    sm.wgt[1][k][i] = w1[k];
                    sm.offs[k][i] = off[k];
                }
            }
            Bq *= 0.25;
            // per-sample constants of the time marginalisation
            double init = -(x * x * Bq), tb_f = 0.0;
            const double* tb_row = nullptr;
            // the sample's hot part of the table: for the first nhot nodes q of its row pair, R_q = T(A_q, B) blended over B once
            // per sample (the B fraction is a constant of the sample) and the step to the next node, in sm.Y[q][i] - idle from
            // here to the next tile's harmonics, and entry [q][i] is touched by the four threads of sample i only (the quartets
            // of a tile are not in step with each other).  A_j is noise outside the few bins around the arrival time, so most
            // lookups fall below node nhot and take one shared-memory load instead of a 32-byte gather whose L1 misses stall
            // the whole batch for an L2 round trip.
            double2* const hot = &sm.Y[0][i];
            const int nhot = min(SP_HOT, P.nA - 2);              // not the last cell: a lookup there may lie past the table's edge (clamped in the other branch)
            if (TABLE) {
                double b = (Bq - P.B_lo) / (P.B_hi - P.B_lo) * (double)(P.nB - 1);
                b = fmin(fmax(b, 0.0), (double)(P.nB - 1));
                const int ib = min((int)floor(b), P.nB - 2);
                tb_f = b - ib;
                tb_row = P.lnT4 + (size_t)ib * (P.nA - 1) * 4;
                init = 0.0;
                double2 lo2[SP_HOT / SP_G], hi2[SP_HOT / SP_G];                                   // cell q = (T[ib][q], T[ib][q+1]), (T[ib+1][q], T[ib+1][q+1]): all loads in flight together
#pragma unroll
                for (int qq = 0; qq < SP_HOT / SP_G; qq++) {
                    const double2* c = reinterpret_cast<const double2*>(tb_row + 4 * max(min(g + SP_G * qq, nhot - 1), 0));
                    lo2[qq] = __ldg(c);
                    hi2[qq] = __ldg(c + 1);
                }
#pragma unroll
                for (int qq = 0; qq < SP_HOT / SP_G; qq++) {
                    const double R0 = fma(tb_f, hi2[qq].x - lo2[qq].x, lo2[qq].x), R1 = fma(tb_f, hi2[qq].y - lo2[qq].y, lo2[qq].y);
                    if (g + SP_G * qq < nhot) hot[(g + SP_G * qq) * SP_TS] = make_double2(R0, R1 - R0);
                }
            }
            qbar();                                              // partial sums read by everybody before the ring is initialised
#pragma unroll 4
            for (int r = g; r < SP_RING; r += SP_G) rcol[r * SP_TS] = init;
            if (g == 0) {
#pragma unroll
                for (int k = 0; k < K; k++) sm.xch[0][k][i] = sm.xch[1][k][i] = 0.0;
            }
            qbar();
            double run_m = -1.0e300, run_s = 0.0;
            int jdone = 0;

            // rows jdone + g, jdone + g + 4, ... below jend are complete: lnL(t_j) and this thread's share of the streaming
            // log-sum-exp (step 6); four rows per batch, loads first
            auto lse_batch = [&](const int j0, const int jend, auto fullc) {
                constexpr bool FULL = decltype(fullc)::value;          // all four rows below jend: no guards
                double v[4];
                double* pr[4];
#pragma unroll
                for (int e = 0; e < 4; e++) {
                    pr[e] = rcol + ((j0 + SP_G * e) & (SP_RING - 1)) * SP_TS;
                    v[e] = *pr[e];
                }
#pragma unroll
                for (int e = 0; e < 4; e++)
                    if (FULL || j0 + SP_G * e < jend) *pr[e] = init;
                bool need = false;
                double dl[4];
                if (TABLE) {
                    // node index and fraction of the four rows; a < 0 is clamped on the high word (to a denormal above 0:
                    // node 0, fraction 0 to rounding), the conversion saturates
                    int ia[4];
                    double fa[4];
                    bool cold = false;
#pragma unroll
                    for (int e = 0; e < 4; e++) {
                        double a = fma(v[e], tabA_s, tabA_o);
                        a = __hiloint2double(max(__double2hiint(a), 0), __double2loint(a));
                        ia[e] = min(__double2int_rz(a), P.nA - 2);
                        fa[e] = a - (double)ia[e];
                        cold = cold || ia[e] >= nhot;
                    }
                    if (!__any_sync(0xffffffffu, cold)) {
                        // every lane's four rows below node nhot: the sample's blended row in shared memory
                        double2 R[4];
#pragma unroll
                        for (int e = 0; e < 4; e++) R[e] = hot[ia[e] * SP_TS];
#pragma unroll
                        for (int e = 0; e < 4; e++) v[e] = fma(fa[e], R[e].y, R[e].x);
                    } else {
                        double2 lo2[4], hi2[4];
#pragma unroll
                        for (int e = 0; e < 4; e++) {
                            const double2* T0 = reinterpret_cast<const double2*>(tb_row + 4 * ia[e]);    // one 32-byte cell
                            lo2[e] = __ldg(T0);
                            hi2[e] = __ldg(T0 + 1);
                        }
#pragma unroll
                        for (int e = 0; e < 4; e++) {
                            // beyond the last node (ia = nA - 2, fraction above 1): clamped to the edge
                            const double f = __double2hiint(fa[e]) >= 0x3ff00000 ? 1.0 : fa[e];
                            const double t0 = fma(f, lo2[e].y - lo2[e].x, lo2[e].x), t1 = fma(f, hi2[e].y - hi2[e].x, hi2[e].x);
                            v[e] = fma(tb_f, t1 - t0, t0);
                        }
                    }
                }
#pragma unroll
                for (int e = 0; e < 4; e++) {
                    const double A = v[e];
                    v[e] = (FULL || j0 + SP_G * e < jend) ? A : neg_inf();
                    dl[e] = v[e] - run_m;
                    need = need || (__double2hiint(dl[e]) >= SP_RAISE_HI);   // dl >= 512 (or NaN): test on the high word
                }
                if (__any_sync(0xffffffffu, need)) {
                    // raise the reference to the largest new value (rare); the running sum is rescaled exactly
                    const double mx = fmax(fmax(v[0], v[1]), fmax(v[2], v[3]));
                    if (mx - run_m >= 512.0) {
                        const double dm = run_m - mx;
                        run_s = dm > -690.0 ? run_s * sp_exp_small(dm) : 0.0;
                        run_m = mx;
                    }
#pragma unroll
                    for (int e = 0; e < 4; e++) dl[e] = v[e] - run_m;
                }
                double part = 0.0;
#pragma unroll
                for (int e = 0; e < 4; e++) {
                    // terms below e^-40 of the reference (and rows past the end) are clamped to e^-40 (R2)
                    const unsigned hc = min((unsigned)__double2hiint(dl[e]), 0xC0440000u);
                    const double t = sp_exp_tab(__hiloint2double((int)hc, __double2loint(dl[e])), etab);
                    part = e == 0 ? t : part + t;
                }
                run_s += part;
            };
            auto lse_rows = [&](const int jend) {
                if (TABLE) {
                    // rows above the kept nodes (around the arrival time): ask for their cells now, so that the batches below
                    // find them in L1 instead of each waiting an L2 round trip
                    for (int j = jdone + g; j < jend; j += SP_G) {
                        const int ia = __double2int_rz(fma(rcol[(j & (SP_RING - 1)) * SP_TS], tabA_s, tabA_o));
                        if (ia >= nhot) {
                            unsigned dummy;
                            asm volatile("ld.global.nc.b32 %0, [%1];" : "=r"(dummy) : "l"(tb_row + 4 * min(ia, P.nA - 2)));
                        }
                    }
                }
                int j0 = jdone + g;
                for (; j0 + 3 * SP_G < jend; j0 += 4 * SP_G) lse_batch(j0, jend, std::true_type{});
                if (j0 < jend) lse_batch(j0, jend, std::false_type{});
                jdone = max(jdone, jend);
            };

            // ---- work items: accumulators -> FP64 -> interpolation -> ring; this thread takes bins 8 g .. 8 g + 7 of each item
            for (int c = 0; c < ti.nchunk; c++) {
                // rows of this chunk all inside [0, N_t) for every sample of the tile: no per-row guard
                const bool guard = !(SP_NB * c - 1 - ti.cap >= 0 && SP_NB * c + SP_NB - 2 < N_t);
#pragma unroll
                for (int k = 0; k < K; k++) {
                    const double w0k = sm.wgt[0][k][i], w1k = sm.wgt[1][k][i];
                    const int offk = sm.offs[k][i];
                    mbar_wait(&sm.d_full, im & 1);
                    tc_fence_after();
                    uint32_t acc[6][8], accp[6];
#pragma unroll
                    for (int s = 0; s < 6; s++) tmem_ld8(tlane + SP_DCOL + SP_NB * s + 8 * g, acc[s]);
                    if (g > 0) {
#pragma unroll
                        for (int s = 0; s < 6; s++) tmem_ld1(tlane + SP_DCOL + SP_NB * s + 8 * g - 1, accp[s]);
                    }
                    tmem_wait_ld();
                    tc_fence_before();
                    mbar_arrive(&sm.d_empty);                           // the accumulators are free for the next item's MMAs
                    im++;
                    // the bin before this thread's eight: the neighbour group's last (reloaded) or, for group 0, the last bin of
                    // the previous chunk, handed over by group 3 through shared memory (two slots: chunk parity)
                    double V[9];
                    if (g > 0) V[0] = sp_recombine(accp[0], accp[1], accp[2], accp[3], accp[4], accp[5]);
                    else V[0] = sm.xch[(c + 1) & 1][k][i];
#pragma unroll
                    for (int e = 0; e < 8; e++) V[e + 1] = sp_recombine(acc[0][e], acc[1][e], acc[2][e], acc[3][e], acc[4][e], acc[5][e]);
                    if (g == SP_G - 1) sm.xch[c & 1][k][i] = V[8];
                    const int j0 = SP_NB * c + 8 * g - 1 - offk;        // time bin of the pair (V[0], V[1])
                    if (guard) {
                        double rv[8];
                        double* pr[8];
                        bool ok[8];
#pragma unroll
                        for (int e = 0; e < 8; e++) {
                            ok[e] = (unsigned)(j0 + e) < (unsigned)N_t;
                            pr[e] = rcol + ((j0 + e) & (SP_RING - 1)) * SP_TS;
                            rv[e] = ok[e] ? *pr[e] : 0.0;
                        }
#pragma unroll
                        for (int e = 0; e < 8; e++) rv[e] = fma(w1k, V[e + 1], fma(w0k, V[e], rv[e]));
#pragma unroll
                        for (int e = 0; e < 8; e++)
                            if (ok[e]) *pr[e] = rv[e];
                    } else {
                        double rv[8];
                        double* pr[8];
#pragma unroll
                        for (int e = 0; e < 8; e++) {
                            pr[e] = rcol + ((j0 + e) & (SP_RING - 1)) * SP_TS;
                            rv[e] = *pr[e];
                        }
#pragma unroll
                        for (int e = 0; e < 8; e++) rv[e] = fma(w1k, V[e + 1], fma(w0k, V[e], rv[e]));
#pragma unroll
                        for (int e = 0; e < 8; e++) *pr[e] = rv[e];
                    }
                    qbar();                                             // the next item's rows overlap this one's (other detector, other offset)
                }
                lse_rows(min(N_t, SP_NB * c + SP_NB - 1 - ti.cap));
                qbar();                                                 // rows consumed before the next chunk wraps onto them
            }
            lse_rows(N_t);
            // ---- the four partial log-sum-exps of the sample
            sm.lse[g][0][i] = run_m;
            sm.lse[g][1][i] = run_s;
            qbar();
            if (g == 0 && member) {
                double mx = sm.lse[0][0][i];
#pragma unroll
                for (int gg = 1; gg < SP_G; gg++) mx = fmax(mx, sm.lse[gg][0][i]);
                double tot = 0.0;
#pragma unroll
                for (int gg = 0; gg < SP_G; gg++) tot += sm.lse[gg][1][i] * exp(sm.lse[gg][0][i] - mx);
                lnL[perm[pos]] = off_bad ? __longlong_as_double(0x7ff8000000000000LL) : mx + log(tot) - P.ln_Nt;
            }
            qbar();                                                     // the next tile's prologue reuses sm.lse
        }
    }
    tc_fence_before();
    __syncthreads();
    if (w == SP_MATH / 32) tmem_free512(tmem);
}

// ---------------------------------------------------------------- launch
template <int K, bool TABLE>
static int launch_split_t(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const int* perm, double* lnL,
                          double* ln_prior, const SpTile* tiles, const int* ntiles_dev) {
    const int smem = (int)sizeof(SplitSmem) + 1024;
    ILE_CUDA(ctx, cudaFuncSetAttribute(lnl_split_kernel<K, TABLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    const int slot = ile_timing_begin(ctx);
    lnl_split_kernel<K, TABLE><<<ctx->sm_count, SP_THREADS, smem, ctx->stream>>>(P, N, rec, perm, lnL, ln_prior, tiles, ntiles_dev);
    ile_timing_end(ctx, slot);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

bool ile_split_supported(const LnlParams& P) { return P.K >= 1 && P.K <= 3 && P.M <= 24 && P.stride == 1 && P.Qs != nullptr && P.n_pairs * P.K * 2 <= SP_UVMAX; }

// scratch layout helpers for the caller (ile_launch_lnL_fused): tile list capacity for N samples
int ile_split_max_tiles(int N, int cell_bits, int K) {
    const long long cells = (1ll << (cell_bits * K)) + 1;
    const long long t = (N + SP_TS - 1) / SP_TS + (cells < N ? cells : N) + 1;
    return (int)t;
}
size_t ile_split_tile_bytes(int max_tiles) { return ((size_t)max_tiles * (sizeof(SpTile) + 2 * sizeof(int)) + 255) / 256 * 256; }   // tiles, tile starts, run starts
size_t ile_split_rec_bytes(int N) { return (size_t)N * SP_REC * sizeof(double); }

int ile_split_cell_bits(int n_min, int n_max) {
    int cell_bits = 1;
    while ((1 << cell_bits) <= ((n_max - n_min) >> SP_CELL_SHIFT)) cell_bits++;
    return cell_bits;
}

int ile_launch_split_keys(ile_ctx* ctx, const LnlParams& P, int N, const double* z, int n_min, int cell_bits, unsigned long long* key,
                          unsigned int* val, double* rec, long long* n_dev, int* bits_dev, int* ntiles_dev) {
    sp_key_kernel<<<(N + 255) / 256, 256, 0, ctx->stream>>>(P, N, z, n_min, cell_bits, key, val, rec, n_dev, bits_dev, ntiles_dev);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

// key / perm = the sorted keys of sp_key_kernel and the sort permutation; rec = its sample records [N][SP_REC] (caller's order)
int ile_launch_split(ile_ctx* ctx, const LnlParams& P, int N, int n_min, int cell_bits, const unsigned long long* key, const double* rec,
                     const int* perm, double* lnL, double* ln_prior, int* tstart, SpTile* tiles, int* ntiles_dev) {
    const int max_tiles = ile_split_max_tiles(N, cell_bits, P.K);
    int* runs = tstart + max_tiles;                     // run starts; their count sits behind the tile count
    int* nruns_dev = ntiles_dev + 1;
    sp_run_flag_kernel<<<(N + 255) / 256, 256, 0, ctx->stream>>>(N, key, runs, nruns_dev);
    ILE_LAUNCH_CHECK(ctx);
    sp_run_tiles_kernel<<<ctx->sm_count * 2, 256, 0, ctx->stream>>>(N, key, runs, nruns_dev, tstart, ntiles_dev);
    ILE_LAUNCH_CHECK(ctx);
    sp_tile_info_kernel<<<(max_tiles * 32 + 255) / 256, 256, 0, ctx->stream>>>(P, N, n_min, cell_bits, key, tstart, ntiles_dev, tiles);
    ILE_LAUNCH_CHECK(ctx);
    const bool tb = P.use_table != 0;
#define SP_LAUNCH(K_, T_) launch_split_t<K_, T_>(ctx, P, N, rec, perm, lnL, ln_prior, tiles, ntiles_dev)
    if (P.K == 3) return tb ? SP_LAUNCH(3, true) : SP_LAUNCH(3, false);
    if (P.K == 2) return tb ? SP_LAUNCH(2, true) : SP_LAUNCH(2, false);
    return tb ? SP_LAUNCH(1, true) : SP_LAUNCH(1, false);
#undef SP_LAUNCH
}
