// Internal declarations of the integrator kernels: device-side
// sampler state, the counter-based generator, the specified fixed-point exponential.
// The integrator translation units are compiled with -fmad=false: draws, bin indices,
// histograms and cell keys use only IEEE + - * / floor rint sqrt and comparisons, so they
// are reproducible bit for bit (reading G30).
#pragma once
#include "common.cuh"

#define AV_SEL_PASSES 12      // 8 digits of the ordered ln f key + 4 digits of the sample index

// ---------------------------------------------------------------- device-resident state
struct AvState {
    long long n;              // n_g: bins per dimension
    long long C;              // active cells
    long long N_min;          // kept samples of the last update
    double L_thr;             // ln f of the last kept sample
    double v;                 // C / n^d
    double ln_ps;             // -ln(v V0)
};

struct PortState {
    double W[ILE_MAX_MEMBERS];        // mixture weights of the contributing activated members (sum 1), 0 for the others
    int frozen[ILE_MAX_MEMBERS];      // 1: not trained on this batch (below 5 %, or not activated yet)
    int active[ILE_MAX_MEMBERS];      // activated set of the last draw
    int restarted, n_contrib;         // the weights were restarted uniform at the last draw; samples of contributing members
    long long alloc[ILE_MAX_MEMBERS];
    long long offset[ILE_MAX_MEMBERS + 1];
};

// one radix-select path over the composite key (ordered ln f descending, index ascending)
struct SelPath {
    unsigned long long prefix_key;
    unsigned int prefix_idx;
    int ndig;                 // digits fixed so far
    unsigned long long cum_metric, cum_count, target;
    int done, fail;
};

struct UpdScratch {           // per-update scalars
    unsigned long long m_ord;     // ordered bits of max ln w over the masked samples
    unsigned long long mn_ord;    // ordered bits of min ln p_s over the masked samples
    unsigned long long n_valid;
    unsigned long long total_q;
    int abort;                    // nothing to train on: leave the state unchanged
    unsigned int ticket;          // blocks of a select pass that have added their histogram (the last one fixes the digit)
    SelPath path[2];              // 0: weight-mass target (P_thr), 1: count target (N_min*)
    int use_path;                 // threshold path chosen: 0, 1, or 2 = keep every valid sample
    int n_bits;                   // significant bits of the new cell keys
    long long N_min, n_new, n_kept;
    unsigned long long R;         // sum of fixed-point 1/p_s over the kept samples
    unsigned long long max_skey;  // largest ordered key among the kept (-> L_thr)
    double v_new;
    long long n_heads;
};

struct SamplerDev {
    int kind;
    int nb;                   // AC: bins per dimension of this member
    // AC
    unsigned long long* H;    // [d][nb]
    double* pi;               // [d][nb]
    double* cdf;              // [d][nb+1]
    // AV
    AvState* av;
    unsigned long long* keys; // [cap] sorted unique
    // GMM: omega[C] | mu[C][d] | Sigma[C][d][d] | L[C][d][d]
    double* gmm;
};

struct IntegDev {
    int kind, d, n_members, nb, n_gmm;
    int box_trusted;          // 1: the batch was drawn by this integrator without a GMM member, so every sample lies in the box (no test, no read of z for it)
    double lo[ILE_MAX_D], hi[ILE_MAX_D], below_hi[ILE_MAX_D];
    double V0;
    unsigned long long seed;
    double eps, beta, P_thr;
    long long N_min_star, n_max;
    SamplerDev mem[ILE_MAX_MEMBERS];
    int first_iter[ILE_MAX_MEMBERS], silent[ILE_MAX_MEMBERS];   // portfolio options
    // GMM over a subset of the dimensions (reading G43): gd modelled dimensions gdim[0..gd), the other
    // d - gd dimensions udim[] are uniform over the box; ln_uvol = sum of ln(hi - lo) over them
    int gd, gdim[ILE_MAX_D], udim[ILE_MAX_D];
    double ln_uvol;
    PortState* port;
};

struct ile_integrator {
    ile_ctx* ctx;
    ile_integrator_opts o;
    IntegDev I;               // host copy of the by-value kernel argument
    long long cap;
    int last_N;
    bool drew;                // a batch is resident (portfolio allocation valid)
    // batch buffers [cap]
    double *z, *ln_ps, *lnL, *lnw, *ln_prior;
    // update scratch
    UpdScratch* us;
    unsigned long long *skey, *q, *kbuf0, *kbuf1;   // [cap]
    unsigned long long* sel_hist;                   // [2][2][256]
    unsigned int* blk_count;                        // unique: heads per block
    void* sort_scratch;
    double* gmm_part;                               // [C][blocks][28+] partial moments
    int gmm_blocks;
    double* port_part;                              // [members][blocks][3]
    int port_blocks;
    ile_result* res;                                // device: last iteration + cumulative
    void* arena;                                    // one allocation behind the small state
};

// ---------------------------------------------------------------- helpers
__device__ __forceinline__ unsigned long long ord_from_double(double f) {   // ascending order-preserving
    unsigned long long b = (unsigned long long)__double_as_longlong(f);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double double_from_ord(unsigned long long o) {
    unsigned long long b = (o >> 63) ? (o & 0x7fffffffffffffffull) : ~o;
    return __longlong_as_double((long long)b);
}
__device__ __forceinline__ bool is_finite_d(double v) { return fabs(v) < pos_inf(); }   // false for NaN

// Philox4x32-10 (Salmon et al. 2011); counter (i_lo, i_hi, g, s), key = seed
__device__ __forceinline__ void philox4x32_10(unsigned int c0, unsigned int c1, unsigned int c2, unsigned int c3, unsigned int k0,
                                              unsigned int k1, unsigned int* out) {
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const unsigned int hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const unsigned int hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const unsigned int n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
// uniforms 2s and 2s+1 of sample i at iteration g: u = (64 bits >> 11) * 2^-53, exact
__device__ __forceinline__ void philox_pair(unsigned long long seed, unsigned long long i, unsigned int g, unsigned int s, double* ua,
                                            double* ub) {
    unsigned int r[4];
    philox4x32_10((unsigned int)i, (unsigned int)(i >> 32), g, s, (unsigned int)seed, (unsigned int)(seed >> 32), r);
    const unsigned long long a = ((unsigned long long)r[1] << 32) | r[0], b = ((unsigned long long)r[3] << 32) | r[2];
    *ua = (double)(a >> 11) * 0x1.0p-53;
    *ub = (double)(b >> 11) * 0x1.0p-53;
}

// q = rint(sexp(t) 2^40), sexp the *specified* exponential:
// y = t log2(e); n = rint(y); f = y - n; zz = f ln2; degree-13 Taylor polynomial in Horner form
// with separate multiply and add; scaled by 2^n.  t > 0 is clamped; NaN and t < -29 give 0.
__device__ __forceinline__ unsigned long long qfix_dev(double t) {
    if (!(t >= -29.0)) return 0ull;
    if (t > 0.0) t = 0.0;
    const double y = __dmul_rn(t, 0x1.71547652b82fep+0);
    const double n = rint(y);
    const double f = __dsub_rn(y, n);
    const double zz = __dmul_rn(f, 0x1.62e42fefa39efp-1);
    double p = 1.0 / 6227020800.0;
    const double c[13] = {1.0 / 479001600.0, 1.0 / 39916800.0, 1.0 / 3628800.0, 1.0 / 362880.0, 1.0 / 40320.0, 1.0 / 5040.0, 1.0 / 720.0,
                          1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0, 1.0 / 2.0, 1.0, 1.0};
#pragma unroll
    for (int k = 0; k < 13; k++) p = __dadd_rn(__dmul_rn(p, zz), c[k]);
    return (unsigned long long)__double2ll_rn(ldexp(p, (int)n + 40));
}

// b = min(n-1, max(0, floor((z - lo) / (hi - lo) * n)))
__device__ __forceinline__ long long bin_index_dev(double z, double lo, double hi, long long n) {
    const double t = __dmul_rn(__ddiv_rn(__dsub_rn(z, lo), __dsub_rn(hi, lo)), (double)n);
    double b = floor(t);
    b = fmin(fmax(b, 0.0), (double)(n - 1));
    if (!(b == b)) b = 0.0;
    return (long long)b;
}

__device__ __forceinline__ bool in_box_dev(const IntegDev& I, const double* __restrict__ z, long long N, long long i) {
    if (I.box_trusted) return true;
    bool ok = true;
    for (int c = 0; c < I.d; c++) {
        const double v = z[(long long)c * N + i];
        ok = ok && (v >= I.lo[c]) && (v < I.hi[c]);
    }
    return ok;
}

__device__ __forceinline__ double pow_d_dev(long long n, int d) {
    double p = 1.0;
    for (int c = 0; c < d; c++) p = __dmul_rn(p, (double)n);
    return p;
}

__device__ __forceinline__ unsigned long long av_key_dev(const IntegDev& I, const double* __restrict__ z, long long N, long long i,
                                                         long long n) {
    unsigned long long key = 0, mul = 1;
    for (int c = 0; c < I.d; c++) {
        key += (unsigned long long)bin_index_dev(z[(long long)c * N + i], I.lo[c], I.hi[c], n) * mul;
        mul *= (unsigned long long)n;
    }
    return key;
}

// ---------------------------------------------------------------- GMM member in shared memory
// One copy per block of what every density evaluation reads, at fixed strides (so that the unrolled forward
// substitution addresses it with immediates): lndet[c] = sum_i ln L_c[i][i], lnom[c] = ln omega_c,
// inv[c][i] = 1 / L_c[i][i], mu[c][i], L[c][i][k]; 16 components x 8 dimensions.
#define GMS_LNDET 0
#define GMS_LNOM 16
#define GMS_INV 32
#define GMS_MU (32 + 128)
#define GMS_L (32 + 256)
#define GMS_DOUBLES (32 + 256 + 1024)
#define LN_TWO_PI 1.8378770664093453
__device__ __forceinline__ void gmm_load_shared(const IntegDev& I, const double* __restrict__ g, double* __restrict__ gs) {
    const int d = I.gd, C = I.n_gmm;
    const double* mu = g + C;
    const double* L = mu + C * d + C * d * d;
    for (int c = threadIdx.x; c < C; c += blockDim.x) {
        double lndet = 0.0;
        for (int i = 0; i < d; i++) {
            lndet = lndet + log(L[c * d * d + i * d + i]);
            gs[GMS_INV + 8 * c + i] = 1.0 / L[c * d * d + i * d + i];
        }
        gs[GMS_LNDET + c] = lndet;
        gs[GMS_LNOM + c] = log(g[c]);
    }
    for (int q = threadIdx.x; q < C * 64; q += blockDim.x) {
        const int c = q >> 6, i = (q >> 3) & 7, k = q & 7;
        gs[GMS_L + q] = (i < d && k < d) ? L[c * d * d + i * d + k] : 0.0;
        if (k == 0) gs[GMS_MU + 8 * c + i] = i < d ? mu[c * d + i] : 0.0;
    }
}
// e[c] = ln omega_c + ln N(zg; mu_c, Sigma_c) for every component (zg: the modelled coordinates, in the mixture's
// order); returns the largest
template <int D>
__device__ __forceinline__ double gmm_ln_comps(const IntegDev& I, const double* __restrict__ gs, const double* zg, double* e) {
    const int d = I.gd, C = I.n_gmm;
    const double cst = -0.5 * d * LN_TWO_PI;
    double mx = neg_inf();
    for (int c = 0; c < C; c++) {
        const double* Lc = gs + GMS_L + 64 * c;
        const double* mc = gs + GMS_MU + 8 * c;
        const double* ic = gs + GMS_INV + 8 * c;
        double y[D];
        double quad = 0.0;
#pragma unroll
        for (int i = 0; i < D; i++)
            if (i < d) {
                double s = zg[i] - mc[i];
#pragma unroll
                for (int k = 0; k < i; k++) s = s - Lc[i * 8 + k] * y[k];
                y[i] = s * ic[i];
                quad = quad + y[i] * y[i];
            }
        e[c] = -0.5 * quad - gs[GMS_LNDET + c] + cst + gs[GMS_LNOM + c];
        mx = fmax(mx, e[c]);
    }
    return mx;
}

// ---------------------------------------------------------------- cross-file entry points
int integ_launch_draw(ile_integrator* it, int N, unsigned int g, double* z, double* ln_ps);
int integ_launch_ln_pdf(ile_integrator* it, int N, const double* z, double* ln_ps);
int integ_launch_update(ile_integrator* it, int N, const double* z, const double* lnw, const double* ln_ps);
int integ_gmm_refresh(ile_integrator* it, int a);   // recompute the Cholesky factors of member a on the device
