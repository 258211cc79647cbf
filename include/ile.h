/*
 * ile.h -- C ABI of the B200-native ILE hot path (arxiv/paper_2505_11655, "Narrowing RIFT").
 *
 * One data-parallel path: the extrinsic-marginalised factored likelihood (PAPER.md:72-98,
 * Eq. 5/7) evaluated over Monte Carlo batches, plus the adaptive integrators that propose the
 * samples and reduce their weights (Eq. 8/9; Eq. 11-16).
 *
 * Conventions (all calls):
 *   - return 0 (ILE_OK) or a negative ile_status; no exceptions, no aborts, no partial writes
 *     on a parameter error; ile_last_error(ctx) gives a ctx-owned message.
 *   - "host" pointers are read on the CPU at call time; "device" pointers are device memory on
 *     the context's device and must stay valid until the work is complete (ile_sync or a
 *     stream/event wait by the caller).  The caller owns every buffer it passes; load/set calls
 *     copy into library-owned memory, so the caller may free immediately after they return.
 *   - all work is enqueued on the context's stream (a cudaStream_t passed as void*); calls are
 *     asynchronous unless they return host values (get_state, the *_host helpers).
 *   - a context is not thread-safe.  Every kernel runs on the GPU; there is no CPU fallback.
 *   - arrays are row-major in the index order written; complex values are (re, im) pairs of
 *     doubles; K detectors (k), M modes (m), N samples (i), N_t time bins (j), N_Q stored bins.
 */
#ifndef ILE_H_
#define ILE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ile_ctx ile_ctx;
typedef struct ile_integrator ile_integrator;

typedef enum {
    ILE_OK = 0,
    ILE_EINVAL = -1,  /* bad argument (NULL, size, asymmetric U/V, ...) */
    ILE_ESTATE = -2,  /* call order: network/modes/QUV/grid not yet set */
    ILE_ENOMEM = -3,
    ILE_ECUDA = -4,   /* a CUDA runtime call failed; see ile_last_error */
    ILE_ERANGE = -5   /* time grid + light-travel delays leave the stored Q span */
} ile_status;

#define ILE_MAX_K 4   /* detectors */
#define ILE_MAX_M 32  /* modes (l_max = 4 -> 21) */
#define ILE_MAX_D 8   /* integrator dimensions */
#define ILE_MAX_MEMBERS 8

enum { ILE_KIND_UNIFORM = 0, ILE_KIND_AC = 1, ILE_KIND_AV = 2, ILE_KIND_GMM = 3, ILE_KIND_PORTFOLIO = 4 };

/* Result of one integrator iteration (Eq. 8, 9, 14-16) and the cumulative estimate over all
 * iterations since create/reset (each sample keeping the p_s it was drawn from).  Lives in
 * device memory when written by the library (out_dev); plain-old-data, 8-byte aligned. */
typedef struct {
    double ln_integral;   /* ln[(1/N) sum w_i], w = L p / p_s            (Eq. 8)  */
    double rel_variance;  /* Var(w) / (N mean(w)^2) = 1/n_ess - 1/N      (population form) */
    double n_eff;         /* sum w / max w                               (Eq. 9)  */
    double n_ess;         /* (sum w)^2 / sum w^2                         (Eq. 16) */
    double ln_w_max;      /* max_i ln w_i over finite weights */
    double S1, S2;        /* sum exp(ln w - ln_w_max), sum exp(2 (ln w - ln_w_max)) */
    uint64_t n_samples;   /* N */
    uint64_t n_nonfinite; /* NaN / +inf log-weights (contribute 0) */
    /* AV (also the AV member of a portfolio); 0 otherwise */
    uint64_t n_cells;     /* C_g used for this iteration's draw */
    int64_t n_bins;       /* n_g per dimension */
    uint64_t N_min;       /* kept samples in this iteration's update */
    double ln_volume;     /* ln(v_g V_0) */
    double L_thr;         /* ln f of the last kept sample */
    /* PORTFOLIO: weights used for this iteration's draw; 0 otherwise */
    double W[ILE_MAX_MEMBERS];
    /* cumulative over iterations */
    double cum_ln_integral, cum_rel_variance, cum_n_eff, cum_n_ess, cum_ln_w_max, cum_S1, cum_S2;
    uint64_t cum_n_samples;
} ile_result;

typedef struct {
    int32_t kind;                  /* ILE_KIND_* */
    int32_t d;                     /* sampled dimensions: 6 = (RA, sin Dec, psi, phi_ref, cos incl, D),
                                      5 = the same without D (distance table loaded); for the
                                      generic draw/update use any 1..ILE_MAX_D */
    double lo[ILE_MAX_D], hi[ILE_MAX_D]; /* box in the flat-prior coordinates z */
    uint64_t seed;                 /* Philox key */
    int64_t max_batch;             /* capacity: largest N passed to draw/update/step/run */
    /* AC */
    int32_t n_bins;                /* bins per dimension (100) */
    int32_t pad0;
    double eps;                    /* uniform floor mixed into each marginal (0.1) */
    double beta;                   /* tempering exponent on the weights (1) */
    /* AV */
    double P_thr;                  /* enclosed probability target (0.999) */
    int64_t N_min_star;            /* fixed number of top points kept early on (4096) */
    /* GMM */
    int32_t n_gmm;                 /* components (8) */
    /* PORTFOLIO */
    int32_t n_members;
    int32_t member_kind[ILE_MAX_MEMBERS]; /* AC / AV / GMM / UNIFORM */
    /* "a list of N_s - 1 integers specifying the first iteration for which a given sampler is
     * activated within the portfolio" (entry 0 must be 0): before it the member gets no samples, has no term in p_s
     * and is not trained; N_s counts the activated members; the weights restart uniform when the set changes. */
    int32_t member_first_iter[ILE_MAX_MEMBERS];
    /* members that "contribute silently, only contributing training data for other samplers without
     * directly influencing the integral": a silent member draws N / N_active samples of every batch, has no term in
     * p_s and its samples (stored after the contributing members': silent members must be listed last) are left out
     * of the estimate (ile_result.n_samples counts the contributing ones); every trained member sees all N. */
    int32_t member_silent[ILE_MAX_MEMBERS];
    /* PAPER.md:297 "a list of options unique to each sampler realization": bins per dimension of an AC member,
     * 0 = n_bins (the paper's Fig. 7 portfolio: two AC members with 10 and 30 bins). */
    int32_t member_n_bins[ILE_MAX_MEMBERS];
    /* PAPER.md:107 "Gaussian mixture models ... for any user-specified subset of dimensions": bit c set = dimension c
     * is modelled by the mixture, the others are sampled uniformly; 0 = all d dimensions. */
    uint32_t gmm_dims_mask;
    int32_t pad1;
} ile_integrator_opts;

/* ------------------------------------------------------------------ lifecycle */
int ile_create(ile_ctx **out, int device, void *cuda_stream);
int ile_destroy(ile_ctx *ctx);
const char *ile_last_error(const ile_ctx *ctx);
int ile_sync(ile_ctx *ctx); /* waits for the stream; surfaces asynchronous CUDA errors */
const char *ile_version(void);

/* ------------------------------------------------------------------ measurement
 * Number of CUDA kernels this context has launched so far. */
uint64_t ile_kernel_launches(const ile_ctx *ctx);
/* on != 0: bracket every launch of the fused lnL kernel (the dominant kernel, steps 5-6) with
 * CUDA events on the context's stream and reset the totals; 0: stop.  ile_kernel_time waits for
 * the recorded events and returns the summed device time (ms) and the number of launches. */
int ile_kernel_timing(ile_ctx *ctx, int on);
int ile_kernel_time(ile_ctx *ctx, double *total_ms, uint64_t *launches);
/* Register-resident FP64 peak probe with no memory traffic: mode 0 = independent DFMA chains on
 * the FP64 ALUs, mode 1 = independent DMMA.8x8x4 chains on the FP64 tensor pipe.  Synchronises;
 * *tflops (host) receives the best of three timed runs. */
int ile_fp64_peak(ile_ctx *ctx, int mode, double *tflops);
/* Probe of the int8 tensor path the fused kernel's contraction runs on (tcgen05.mma kind::i8, 128 x 32 x 32, A from tensor
 * memory, B from shared memory, the kernel's 33-MMA schedule and nothing else): mode 0 = k-step-major issue (the kernel's),
 * 1 = sum-major.  Synchronises; *tops (host) receives int8 operations (2 per multiply-add) per second / 1e12, best of three. */
int ile_int8_mma_peak(ile_ctx *ctx, int mode, double *tops);

/* ------------------------------------------------------------------ problem definition (host pointers)
 * detector response functions and positions.  D[k] is the 3x3 response tensor
 * (symmetric; only that is checked), pos_m[k] the position in metres in the Earth-fixed frame,
 * gmst the Greenwich sidereal angle in radians. */
int ile_set_network(ile_ctx *ctx, int K, const double *D /*[K][3][3]*/, const double *pos_m /*[K][3]*/, double gmst);
/* PAPER.md:67-70 (Eq. 4): the (l, m) list; its order defines the mode index of Q, U, V. */
int ile_set_modes(ile_ctx *ctx, int M, const int *ell, const int *m);
/* PAPER.md:78-87 (Eq. 6a-c): Q_{k,lm}(t) on N_Q bins at rate fs starting at t_Q0 (geocentric
 * seconds), U, V mode-mode matrices, for P intrinsic points; D_ref in the distance unit of the
 * prior.  U = U^H and V = V^T are verified to 1e-12 relative (Eq. 17-18) -> ILE_EINVAL.  At most 22 modes
 * (l <= 4 gives 21; the packed Q layouts hold 24 complex columns, two of them padding) -> ILE_EINVAL.
 * src_is_device != 0: Q/U/V are device pointers (copied device-to-device). */
int ile_load_quv(ile_ctx *ctx, int P, int N_Q, double fs, double t_Q0,
                 const double *Q /*[P][K][M][N_Q][2]*/, const double *U /*[P][K][M][M][2]*/,
                 const double *V /*[P][K][M][M][2]*/, double D_ref, int src_is_device);
/* SURVEY 8(f) #1; the same Q, U, V computed on the device from
 * frequency-domain inputs (device pointers, numpy FFT bin order f_j = j df, j <= N_f/2, else
 * (j - N_f) df): h [P][M][N_f][2] mode spectra, d [K][N_f][2] data spectra, S [K][N_f/2+1]
 * one-sided PSDs over |f|; <a|b>_k = 2 sum_{|f| > f_low} df a*(f) b(f) / S_k(|f|).  fs = N_f df;
 * the stored window is t_n = t_Q0 + n / fs, n < N_Q (t_Q0 fs must be an integer).  Installs the
 * result like ile_load_quv (synchronises).  The inputs stay the caller's; scratch is one grow-only
 * device allocation owned by the context (freed by ile_destroy).  Errors: ILE_ESTATE before
 * set_network/set_modes, ILE_EINVAL for bad sizes, N_Q > N_f, t_Q0 off the sample grid or more
 * than 22 modes (the resident Q/U/V stay as they were), ILE_ENOMEM (of the scratch: the resident set
 * stays; of the result arrays: nothing is resident afterwards), ILE_ECUDA.  U and V come out Hermitian and
 * symmetric by construction (Eq. 17-18), so the install skips ile_load_quv's check.
 * ile_get_quv copies point p back to host arrays in ile_load_quv's layout (any of Q, U, V may be NULL). */
int ile_precompute_quv(ile_ctx *ctx, int P, int N_f, double df, double f_low, const double *h, const double *d,
                       const double *S, double t_Q0, int N_Q, double D_ref);
int ile_get_quv(ile_ctx *ctx, int p, double *Q, double *U, double *V);
/* Geocentric time grid t_j = t_lo + j dt, j < N_t, marginalised with a uniform prior
 * (PAPER.md:94, 547).  dt * fs must be a positive integer (native-spaced grid).  interp: 1 =
 * linear interpolation of Q between stored bins, 0 = nearest bin.  ILE_ERANGE unless
 * [t_lo - max|x_k|/c, t_hi + max|x_k|/c] lies inside the stored span (minus one bin). */
int ile_set_time_grid(ile_ctx *ctx, double t_lo, double dt, int N_t, int interp);
/* p(D) = 3 D^2 / (D_max^3 - D_min^3); angles isotropic (reading G13). */
int ile_set_prior(ile_ctx *ctx, double D_min, double D_max);
/* Distance marginalisation: lnT[b][a] on a regular grid A in [A_lo, A_hi],
 * B in [B_lo, B_hi]; bilinear, clamped.  Once loaded, lnL(t_j) = T(A_j, B) and d = 5.
 * nA = 0 unloads it. */
int ile_load_distance_table(ile_ctx *ctx, int nA, int nB, double A_lo, double A_hi, double B_lo,
                            double B_hi, const double *lnT /*[nB][nA] host*/);

/* ------------------------------------------------------------------ direct evaluation (device pointers, length N)
 * Step 1: antenna patterns and arrival-time delays tau_k = -x_k.n/c. */
int ile_antenna(ile_ctx *ctx, int N, const double *ra, const double *dec, const double *psi,
                double *Fp /*[K][N]*/, double *Fx /*[K][N]*/, double *tau /*[K][N]*/);
/* Step 2 (Eq. 4): -2Y_lm(incl, phi) for the mode list. */
int ile_ylm(ile_ctx *ctx, int N, const double *incl, const double *phi, double *Y /*[M][N][2]*/);
/* Steps 1-6 for intrinsic point p at the paper's angles (Eq. 7 + time marginalisation).
 * dist may be NULL when a distance table is loaded.  lnL_t (optional) receives lnL(t_j). */
int ile_lnL(ile_ctx *ctx, int p, int N, const double *ra, const double *dec, const double *psi,
            const double *phi_ref, const double *incl, const double *dist, double *lnL /*[N]*/,
            double *lnL_t /*[N][N_t] or NULL*/);
/* Same at integrator coordinates z = (RA, sin Dec, psi, phi_ref, cos incl[, D]), d = 5 or 6; the
 * kernel the integrators call.  Samples outside the prior box get lnL = -inf.  ln_prior
 * (optional) receives ln p(z).  ile_set_lnL_variant selects the kernel behind this call (and behind the
 * integrators): 0 = default: samples ordered by delay cell on the device, then the fused kernel whose contraction
 * (step 5) runs exactly, in signed 8-bit digits, on the Blackwell tensor cores (tcgen05, K <= 3 detectors, M <= 24
 * modes, time step of one stored bin; other shapes take variant 2); 1 = plain one-thread-per-sample kernel
 * (in-library cross-check); 2 = delay-cell ordering + the fused FP64 DMMA kernel; 3 = the DMMA kernel without the
 * ordering.  All variants meet the same tolerance; ILE_EINVAL for other values. */
int ile_lnL_z(ile_ctx *ctx, int p, int N, int d, const double *z /*[d][N]*/, double *lnL /*[N]*/,
              double *ln_prior /*[N] or NULL*/);
int ile_set_lnL_variant(ile_ctx *ctx, int variant);
/* Step 7 (Eq. 8, 9, 16): reduce N log-weights into *out_dev (device; cumulative fields reset). */
int ile_reduce(ile_ctx *ctx, int N, const double *lnw, ile_result *out_dev);
/* The same reduction for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): calls no cudaMalloc, cudaFree or allocating library routine.  Its per-block partial sums live in a
 * 64 KB file-scope device array (2048 partials of 32 bytes) that every GPU loading the library holds until exit.
 * N <= ILE_REDUCE_NOALLOC_MAX_N, else ILE_EINVAL with a message (ile_last_error) and nothing launched.  lnw [N] and
 * out_dev are device pointers owned by the caller, as for ile_reduce; the work is queued on the context's stream.  All
 * calls on a device share the array: calls that overlap on the GPU (two contexts, two streams) race; calls on one stream
 * are ordered and safe.  Nothing in the array has to start at zero: a call reads only what it wrote.  Results are
 * bit-identical to ile_reduce's (same kernels, same grid).  The first call on a device looks the array's address up
 * (cudaGetSymbolAddress, no allocation) and caches it per process: make that first call from one host thread. */
#define ILE_REDUCE_NOALLOC_MAX_N (1 << 24)
int ile_reduce_noalloc(ile_ctx *ctx, int N, const double *lnw, ile_result *out_dev);

/* ------------------------------------------------------------------ integrators (steps 8-11) */
int ile_integrator_opts_default(ile_integrator_opts *opts, int kind, int d);
int ile_integrator_create(ile_ctx *ctx, const ile_integrator_opts *opts, ile_integrator **out);
int ile_integrator_destroy(ile_integrator *it);
int ile_integrator_reset(ile_integrator *it); /* back to the iteration-0 state; clears cumulative */
/* Draw N samples for iteration `iter` (Philox counter (i, iter, stream), key = seed):
 * z [d][N] and ln p_s [N], both device. */
int ile_integrator_draw(ile_integrator *it, int N, uint64_t iter, double *z, double *ln_ps);
/* ln p_s at arbitrary points (device). */
int ile_integrator_ln_pdf(ile_integrator *it, int N, const double *z, double *ln_ps);
/* Teacher-forced training step on (z, ln w[, ln p_s]) (device).  ln_ps may be NULL for
 * UNIFORM / AC / GMM and for a standalone AV (its p_s is constant); a PORTFOLIO needs it and
 * must have drawn this batch (member allocation). */
int ile_integrator_update(ile_integrator *it, int N, const double *z, const double *lnw, const double *ln_ps);
/* One full iteration for intrinsic point p: draw, lnL, ln w = lnL + ln p - ln p_s, reduce into
 * *out_dev, update.  No host round-trip. */
int ile_integrator_step(ile_integrator *it, int p, int N, uint64_t iter, ile_result *out_dev);
/* p_count intrinsic points x n_iter iterations, enqueued back to back; the sampler is reset
 * between points.  out_dev [p_count][n_iter]. */
int ile_integrator_run(ile_integrator *it, int p_first, int p_count, int n_iter, int N, ile_result *out_dev);
/* The last batch's device buffers (valid until the next draw/step): z [d][N], ln_ps, lnL, lnw. */
int ile_integrator_last_batch(ile_integrator *it, const double **z, const double **ln_ps,
                              const double **lnL, const double **lnw);
/* Serialised sampler state (synchronises).  Call with buf = NULL to get the size in *bytes.
 * Layout (little endian, 8-byte aligned):
 *   header  int64 kind, d
 *   AC      int64 n_bins; uint64 H[d][n_bins]; double pi[d][n_bins]; double cdf[d][n_bins+1]
 *   AV      int64 n, C, N_min; double L_thr; uint64 keys[C]
 *   GMM     int64 n_comp, gd (modelled dimensions); double omega[C], mu[C][gd], Sigma[C][gd][gd], L[C][gd][gd]
 *   PORTF.  int64 n_members; double W[8]; int64 frozen[8]; int64 alloc[8]; int64 active[8];
 *           then per member: int64 bytes_m, followed by that member's blob (with header)
 *   UNIFORM nothing more */
int ile_integrator_get_state(ile_integrator *it, void *buf, size_t *bytes);
int ile_integrator_set_state(ile_integrator *it, const void *buf, size_t bytes);

/* ------------------------------------------------------------------ built-in test integrands
 * The paper's integrator test problems evaluated on the device, so that a whole AC / AV / portfolio
 * loop runs with no host round-trip on something with a known integral:
 *   ILE_F_GAUSSIAN_MIX  ln f = ln sum_c exp(ln_amp_c - |z - c_c|^2 / (2 sigma_c^2)), n_comp <= 4
 *                       (Fig. 6: two components, sigma = sqrt 2, centres (+-4, 0, 0));
 *                       par = per component { centre[ILE_MAX_D], sigma, ln_amp }
 *   ILE_F_ROSENBROCK    ln f = -sum_i [ (a - z_i)^2 + b (z_{i+1} - z_i^2)^2 ] / T (Fig. 3);
 *                       par = { a, b, T }
 * The integral is over the integrator's box with unit prior density: ln w = ln f - ln p_s. */
enum { ILE_F_GAUSSIAN_MIX = 0, ILE_F_ROSENBROCK = 1 };
typedef struct {
    int32_t kind, n_comp;
    double par[4 * (ILE_MAX_D + 2)];
} ile_integrand;
/* One iteration on integrand *f (host struct, copied): draw, ln f, reduce into *out_dev, update.
 * Works for any d in 1..ILE_MAX_D; needs no loaded problem.  ln f of the batch is left in the
 * lnL buffer of ile_integrator_last_batch. */
int ile_integrator_step_integrand(ile_integrator *it, const ile_integrand *f, int N, uint64_t iter, ile_result *out_dev);

/* ------------------------------------------------------------------ fair draws
 * "fairly drawing some (fixed) number of extrinsic parameters from the
 * underlying ILE Monte Carlo integral weighted samples".  M draws with replacement from N samples
 * with log-weights lnw (device): probability of sample i = w_i / sum w.  mode 0 = systematic
 * resampling (one uniform, equally spaced positions: every count within 1 of M w_i / sum w),
 * 1 = independent draws.  Uniforms: Philox counter (0 or j, iter), key = seed.  idx (device,
 * int64 [M]) receives the drawn sample indices, -1 everywhere if no weight is positive.  Exact:
 * fixed-point weights rint(exp(ln w - max) 2^40) and integer prefix sums. */
int ile_fair_draw(ile_ctx *ctx, int N, const double *lnw, int M, uint64_t seed, uint64_t iter, int mode, int64_t *idx);

#ifdef __cplusplus
}
#endif
#endif /* ILE_H_ */
