// libile: direct-evaluation entry points (steps 1-6) and the plain reference lnL kernel.
#include "common.cuh"
#include "likelihood_dev.cuh"

int ile_launch_lnL_fused(ile_ctx* ctx, const LnlParams& P, int N, const double* z, const int* perm, double* lnL, double* ln_prior);

// ---------------------------------------------------------------- step 1 / step 2 kernels
__global__ void antenna_kernel(LnlParams P, int N, const double* ra, const double* dec, const double* psi, double* Fp,
                               double* Fx, double* tau) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    SampleIn s = sample_from_angles(ra[i], dec[i], psi[i], 0.0, 0.0, 1.0);
    double fp[ILE_MAX_K], fx[ILE_MAX_K], t[ILE_MAX_K];
    antenna_dev(P, s, fp, fx, t);
    for (int k = 0; k < P.K; k++) {
        Fp[(size_t)k * N + i] = fp[k];
        Fx[(size_t)k * N + i] = fx[k];
        tau[(size_t)k * N + i] = t[k];
    }
}

__global__ void ylm_kernel(const YlmTable* T, int N, const double* incl, const double* phi, double* Y) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    double sh, ch;
    sincos(0.5 * incl[i], &sh, &ch);
    ylm_dev(T, ch, sh, phi[i], [&](int m, double yr, double yi) {
        Y[((size_t)m * N + i) * 2] = yr;
        Y[((size_t)m * N + i) * 2 + 1] = yi;
    });
}

// ---------------------------------------------------------------- plain reference kernel
// One thread per sample, loops in the order of Eq. 7: time bin j, detector k, mode m.  Reads Q
// from the caller's layout.  Slow; kept as the in-library cross-check and for lnL(t) dumps.
template <bool FROM_Z>
__global__ void lnL_plain_kernel(LnlParams P, int N, const double* a0, const double* a1, const double* a2, const double* a3,
                                 const double* a4, const double* a5, double* lnL, double* ln_prior, double* lnL_t) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    SampleIn s;
    if (FROM_Z) s = sample_from_z(P, a0, N, i);
    else s = sample_from_angles(a0[i], a1[i], a2[i], a3[i], a4[i], a5 ? a5[i] : 1.0);
    if (ln_prior) ln_prior[i] = s.valid ? ln_prior_dev(P, s) : neg_inf();
    if (!s.valid) {
        lnL[i] = neg_inf();
        return;
    }
    double Fp[ILE_MAX_K], Fx[ILE_MAX_K], tau[ILE_MAX_K], Yr[ILE_MAX_M], Yi[ILE_MAX_M];
    antenna_dev(P, s, Fp, Fx, tau);
    ylm_dev(P.ylm, s.ch, s.sh, -s.phi_ref, [&](int m, double yr, double yi) { Yr[m] = yr; Yi[m] = yi; });
    double B = quadratic_dev(P, Fp, Fx, Yr, Yi);
    double x = P.use_table ? 1.0 : P.D_ref / s.dist;
    double mx = neg_inf(), sum = 0.0;
    for (int j = 0; j < P.N_t; j++) {
        double tj = P.t_lo + j * P.dt;
        double A = 0.0;
        for (int k = 0; k < P.K; k++) {
            double u = (tj + tau[k] - P.t_Q0) * P.fs;
            double fl = P.interp ? floor(u) : floor(u + 0.5);
            double f = P.interp ? u - fl : 0.0;
            int n = (int)fl;
            double zr = 0.0, zi = 0.0;
            for (int m = 0; m < P.M; m++) {
                const double* q = P.Qc + (((size_t)k * P.M + m) * P.N_Q + n) * 2;
                double qr = (1.0 - f) * q[0] + f * q[2];
                double qi = (1.0 - f) * q[1] + f * q[3];
                zr += Yr[m] * qr + Yi[m] * qi;     // conj(Y) Q
                zi += Yr[m] * qi - Yi[m] * qr;
            }
            A += Fp[k] * zr - Fx[k] * zi;           // Re(conj(F) z), conj(F) = F+ + i Fx
        }
        double v = P.use_table ? table_lookup(P, A, B) : x * A - x * x * B;
        if (lnL_t) lnL_t[(size_t)i * P.N_t + j] = v;
        if (v > mx) {
            sum = sum * exp(mx - v) + 1.0;
            mx = v;
        } else {
            sum += exp(v - mx);
        }
    }
    lnL[i] = mx + log(sum) - log((double)P.N_t);
}

// ---------------------------------------------------------------- API
extern "C" int ile_antenna(ile_ctx* ctx, int N, const double* ra, const double* dec, const double* psi, double* Fp, double* Fx,
                           double* tau) {
    if (!ctx) return ILE_EINVAL;
    if (!ctx->have_net) return ile_fail(ctx, ILE_ESTATE, "antenna: set_network first");
    if (N < 0 || (N > 0 && (!ra || !dec || !psi || !Fp || !Fx || !tau))) return ile_fail(ctx, ILE_EINVAL, "antenna: bad argument");
    if (N == 0) return ILE_OK;
    LnlParams P;
    memset(&P, 0, sizeof(P));
    P.K = ctx->K;
    P.gmst = ctx->gmst;
    memcpy(P.D, ctx->D, sizeof(ctx->D));
    memcpy(P.pos, ctx->pos, sizeof(ctx->pos));
    antenna_kernel<<<(N + 127) / 128, 128, 0, ctx->stream>>>(P, N, ra, dec, psi, Fp, Fx, tau);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

extern "C" int ile_ylm(ile_ctx* ctx, int N, const double* incl, const double* phi, double* Y) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (!ctx->have_modes) return ile_fail(ctx, ILE_ESTATE, "ylm: set_modes first");
    if (N < 0 || (N > 0 && (!incl || !phi || !Y))) return ile_fail(ctx, ILE_EINVAL, "ylm: bad argument");
    if (N == 0) return ILE_OK;
    ylm_kernel<<<(N + 127) / 128, 128, 0, ctx->stream>>>(ctx->d_ylm, N, incl, phi, Y);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

extern "C" int ile_lnL(ile_ctx* ctx, int p, int N, const double* ra, const double* dec, const double* psi, const double* phi_ref,
                       const double* incl, const double* dist, double* lnL, double* lnL_t) {
    if (!ctx) return ILE_EINVAL;
    LnlParams P;
    int d = ctx->d_lnT ? 5 : 6;
    int rc = ile_fill_params(ctx, p, d, &P);
    if (rc) return rc;
    if (N < 0 || (N > 0 && (!ra || !dec || !psi || !phi_ref || !incl || !lnL))) return ile_fail(ctx, ILE_EINVAL, "lnL: bad argument");
    if (d == 6 && N > 0 && !dist) return ile_fail(ctx, ILE_EINVAL, "lnL: dist is required without a distance table");
    if (N == 0) return ILE_OK;
    lnL_plain_kernel<false><<<(N + 63) / 64, 64, 0, ctx->stream>>>(P, N, ra, dec, psi, phi_ref, incl, dist, lnL, nullptr, lnL_t);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

int ile_launch_lnL_plain_z(ile_ctx* ctx, const LnlParams& P, int N, const double* z, double* lnL, double* ln_prior) {
    lnL_plain_kernel<true><<<(N + 63) / 64, 64, 0, ctx->stream>>>(P, N, z, nullptr, nullptr, nullptr, nullptr, nullptr, lnL, ln_prior,
                                                                 nullptr);
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

int ile_launch_lnL_z(ile_ctx* ctx, int p, int N, int d, const double* z, const int* perm, double* lnL, double* ln_prior) {
    LnlParams P;
    int rc = ile_fill_params(ctx, p, d, &P);
    if (rc) return rc;
    if (N < 0 || (N > 0 && (!z || !lnL))) return ile_fail(ctx, ILE_EINVAL, "lnL_z: bad argument");
    if (N == 0) return ILE_OK;
    if (ctx->zbox_hint) {                        // a batch drawn inside a box that lies within the prior box needs no box test
        bool inside = true;
        for (int c = 0; c < d; c++) inside = inside && ctx->zbox_lo[c] >= P.lo[c] && ctx->zbox_hi[c] <= P.hi[c];
        P.box_trusted = inside ? 1 : 0;
    }
    if (ctx->variant == 1) return ile_launch_lnL_plain_z(ctx, P, N, z, lnL, ln_prior);
    return ile_launch_lnL_fused(ctx, P, N, z, perm, lnL, ln_prior);
}

extern "C" int ile_lnL_z(ile_ctx* ctx, int p, int N, int d, const double* z, double* lnL, double* ln_prior) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    return ile_launch_lnL_z(ctx, p, N, d, z, nullptr, lnL, ln_prior);
}
