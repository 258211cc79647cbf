// libile: the fused lnL path, B200-native: launch sequence and the kernels in front of
// the fused kernel.
//
//   key + sort    samples are ordered by the cell of their per-detector arrival-time delays (a tile of the fused
//                 kernel then reads one window of Q per detector)
//   prep kernel   (steps 1-3)  one thread per sample, in sorted order: F_k, tau_k, Y_lm, x -> a Y tile per 32
//                 samples + a 16-double record
//   fused kernel  (steps 3-6)  lnl_split.cu (tcgen05, integer digits; the default) or lnl_fused2.cu (FP64 DMMA)
// DESIGN.md section 6 derives the tiling and the rooflines.
#include "common.cuh"
#include "likelihood_dev.cuh"
#include "radix_sort.cuh"

#define FT_TS 32          // samples per Y sub-tile
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

// ---------------------------------------------------------------- launch
int ile_launch_lnL_plain_z(ile_ctx* ctx, const LnlParams& P, int N, const double* z, double* lnL, double* ln_prior);
int ile_launch_fused2(ile_ctx* ctx, const LnlParams& P, int N, const double* rec, const double2* yt, const int* perm, double* lnL, bool quad);

int ile_launch_lnL_fused(ile_ctx* ctx, const LnlParams& P, int N, const double* z, const int* perm, double* lnL, double* ln_prior) {
    if (P.K > 3 || 2 * P.M > ILE_QT_ROW) return ile_launch_lnL_plain_z(ctx, P, N, z, lnL, ln_prior);
    // the tcgen05 path (lnl_split.cu) orders by cells of 16 bins, builds its tiles on the device and does steps 1-2 itself;
    // the DMMA path runs the preparation kernel into per-sample records and Y tiles first
    const bool split = ctx->lnl_split && perm == nullptr && ile_split_supported(P);
    const int tiles = (N + 63) / 64 * 2;                       // 32-sample sub-tiles, padded to whole 64-sample tiles
    const size_t rec_bytes = split ? 0 : ((size_t)tiles * FT_TS * FT_REC * sizeof(double) + 255) / 256 * 256;
    const size_t y_bytes = split ? 0 : ((size_t)tiles * FT_YM * FT_TS * sizeof(double2) + 255) / 256 * 256;
    const size_t uk_bytes = split ? (ile_split_rec_bytes(N) + 255) / 256 * 256 : 0;      // sample records of the tcgen05 path (coordinates + u_k)
    const size_t key_bytes = ((size_t)N * 8 + 255) / 256 * 256, val_bytes = ((size_t)N * 4 + 255) / 256 * 256;
    const size_t sort_bytes = (radix_sort_scratch_bytes(N) + 255) / 256 * 256;
    const bool sort = perm == nullptr && (split || (ctx->sky_sort && N > FT_TS));
    // cells of stored bins over the range of delays the network allows
    const int n_min = ((int)floor((P.t_lo - ctx->max_delay - P.t_Q0) * P.fs) - 1) & ~7;
    const int n_max = (int)floor((P.t_lo + ctx->max_delay - P.t_Q0) * P.fs) + 1;
    const int sp_bits = ile_split_cell_bits(n_min, n_max);
    const int sp_tiles = split ? ile_split_max_tiles(N, sp_bits, P.K) : 0;
    const size_t tile_bytes = split ? ile_split_tile_bytes(sp_tiles) : 0;
    void* scratch = nullptr;
    int rc = ile_scratch(ctx, rec_bytes + y_bytes + uk_bytes + (sort ? 2 * key_bytes + 2 * val_bytes + sort_bytes + 256 : 0) + tile_bytes, &scratch);
    if (rc) return rc;
    char* base = (char*)scratch;
    double* rec = (double*)base;
    double2* yt = (double2*)(base + rec_bytes);
    double* uk = (double*)(base + rec_bytes + y_bytes);
    unsigned long long* k0 = nullptr;
    int* ntiles_dev = nullptr;
    if (sort) {
        char* sb = base + rec_bytes + y_bytes + uk_bytes;
        k0 = (unsigned long long*)sb;
        unsigned long long* k1 = (unsigned long long*)(sb + key_bytes);
        unsigned int* v0 = (unsigned int*)(sb + 2 * key_bytes);
        unsigned int* v1 = (unsigned int*)(sb + 2 * key_bytes + val_bytes);
        void* hist = sb + 2 * key_bytes + 2 * val_bytes;
        long long* n_dev = (long long*)(sb + 2 * key_bytes + 2 * val_bytes + sort_bytes);
        int* bits_dev = (int*)(n_dev + 1);
        ntiles_dev = bits_dev + 1;
        int cell_bits = 1;
        if (split) {
            cell_bits = sp_bits;
            rc = ile_launch_split_keys(ctx, P, N, z, n_min, cell_bits, k0, v0, uk, n_dev, bits_dev, ntiles_dev);
            if (rc) return rc;
        } else {
            while ((1 << cell_bits) <= ((n_max - n_min) >> SKY_CELL_SHIFT)) cell_bits++;
            sky_key_kernel<<<(N + 255) / 256, 256, 0, ctx->stream>>>(P, N, z, n_min, cell_bits, k0, v0, n_dev, bits_dev);
            ILE_LAUNCH_CHECK(ctx);
        }
        rc = radix_sort_device(ctx, N, n_dev, bits_dev, (uint64_t*)k0, v0, (uint64_t*)k1, v1, hist, (cell_bits * P.K + 1 + 7) / 8);
        if (rc) return rc;
        perm = (const int*)v0;
    }
    if (split) {
        char* tb = base + rec_bytes + y_bytes + uk_bytes + 2 * key_bytes + 2 * val_bytes + sort_bytes + 256;
        SpTile* tl = (SpTile*)tb;
        int* tstart = (int*)(tb + (size_t)sp_tiles * 32);
        return ile_launch_split(ctx, P, N, n_min, sp_bits, k0, uk, perm, lnL, ln_prior, tstart, tl, ntiles_dev);
    }
    rc = ile_ensure_qf(ctx);
    if (rc) return rc;
    // shared-memory scratch of the harmonics: (2 (max_pow + 1) + 2 (max_abs_m + 1)) doubles per thread
    // ... and a copy of the mode table
    const int scr_d = (2 * (ctx->ylm_max_pow + 1) + 2 * (ctx->ylm_max_abs_m + 1)) * 128;
    const size_t scr = (size_t)scr_d * sizeof(double) + sizeof(YlmTable) + 16;
    lnl_prep3_kernel<<<(tiles * FT_TS + 127) / 128, 128, scr, ctx->stream>>>(P, N, tiles * FT_TS, scr_d, z, perm, rec, yt, ln_prior);
    ILE_LAUNCH_CHECK(ctx);
    rc = ile_launch_fused2(ctx, P, N, rec, yt, perm, lnL, true);
    if (rc != 1) return rc;
    return ile_launch_lnL_plain_z(ctx, P, N, z, lnL, ln_prior);   // shape without a fused instantiation
}
