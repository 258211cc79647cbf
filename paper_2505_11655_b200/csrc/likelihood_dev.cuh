// Device functions for steps 1-4 of the hot path: antenna patterns and delays,
// spin-weighted harmonics, prior, the U/V quadratic term.  Used by every lnL kernel.
#pragma once
#include "common.cuh"

struct SampleIn {
    double ra, sd, cd, psi, phi_ref, ch, sh, dist;
    bool valid;
};

// angles: RA, Dec, psi, phi_ref, inclination, distance
__device__ __forceinline__ SampleIn sample_from_angles(double ra, double dec, double psi, double phi_ref, double incl, double dist) {
    SampleIn s;
    s.ra = ra;
    sincos(dec, &s.sd, &s.cd);
    s.psi = psi;
    s.phi_ref = phi_ref;
    sincos(0.5 * incl, &s.sh, &s.ch);
    s.dist = dist;
    s.valid = true;
    return s;
}

// integrator coordinates z = (RA, sin Dec, psi, phi_ref, cos incl[, D]) (G38): only sqrt
__device__ __forceinline__ SampleIn sample_from_z(const LnlParams& P, const double* __restrict__ z, long long N, long long i) {
    SampleIn s;
    double v[6];
    // all coordinate loads first (a check right after each load serialises six memory round trips)
#pragma unroll
    for (int c = 0; c < 6; c++) v[c] = c < P.d ? __ldg(z + (long long)c * N + i) : 1.0;
    bool ok = true;
#pragma unroll
    for (int c = 0; c < 6; c++)
        if (c < P.d) ok = ok & (v[c] >= P.lo[c]) & (v[c] < P.hi[c]);
    s.valid = ok;
    s.ra = v[0];
    s.sd = v[1];
    s.cd = sqrt(fmax((1.0 - v[1]) * (1.0 + v[1]), 0.0));
    s.psi = v[2];
    s.phi_ref = v[3];
    s.ch = sqrt(fmax(0.5 * (1.0 + v[4]), 0.0));
    s.sh = sqrt(fmax(0.5 * (1.0 - v[4]), 0.0));
    s.dist = v[5];
    return s;
}

__device__ __forceinline__ double ln_prior_dev(const LnlParams& P, const SampleIn& s) {
    double lp = P.ln_prior_const;
    if (P.d > 5) lp += log(P.dist_norm * s.dist * s.dist);
    return lp;
}

// Step 1: F_k = F+ - i Fx and tau_k = -x_k.n/c for all detectors.
__device__ __forceinline__ void antenna_dev(const LnlParams& P, const SampleIn& s, double* Fp, double* Fx, double* tau) {
    double sg, cg, sp, cp;
    sincos(P.gmst - s.ra, &sg, &cg);
    sincos(s.psi, &sp, &cp);
    const double sd = s.sd, cd = s.cd;
    double n[3] = {cd * cg, -cd * sg, sd};
    double X[3] = {-cp * sg - sp * cg * sd, -cp * cg + sp * sg * sd, sp * cd};
    double Y[3] = {sp * sg - cp * cg * sd, sp * cg + cp * sg * sd, cp * cd};
#pragma unroll
    for (int k = 0; k < ILE_MAX_K; k++) {
        if (k >= P.K) break;
        double fp = 0.0, fx = 0.0;
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) {
                double Dab = P.D[k][a * 3 + b];
                fp += X[a] * Dab * X[b] - Y[a] * Dab * Y[b];
                fx += X[a] * Dab * Y[b] + Y[a] * Dab * X[b];
            }
        Fp[k] = fp;
        Fx[k] = fx;
        tau[k] = -(P.pos[k][0] * n[0] + P.pos[k][1] * n[1] + P.pos[k][2] * n[2]) / ILE_C_LIGHT;
    }
}

// Step 2 (Eq. 4): -2Y_lm(theta, phi) with cos/sin of theta/2 given.  Yr/Yi: M entries.
template <typename Store>
__device__ __forceinline__ void ylm_dev(const YlmTable* __restrict__ T, double ch, double sh, double phi, Store store) {
    double pc[2 * ILE_MAX_L + 1], ps[2 * ILE_MAX_L + 1];
    const int mp = T->max_pow;
    pc[0] = 1.0;
    ps[0] = 1.0;
    for (int q = 1; q <= mp; q++) {
        pc[q] = pc[q - 1] * ch;
        ps[q] = ps[q - 1] * sh;
    }
    double cm[ILE_MAX_L + 1], sm[ILE_MAX_L + 1];
    const int mm = T->max_abs_m;
    cm[0] = 1.0;
    sm[0] = 0.0;
    for (int q = 1; q <= mm; q++) sincos((double)q * phi, &sm[q], &cm[q]);
    const int M = T->M;
    for (int i = 0; i < M; i++) {
        const YlmMode& Y = T->mode[i];
        double acc = 0.0;
        for (int t = 0; t < Y.nterms; t++) acc += Y.coef[t] * pc[Y.pc[t]] * ps[Y.ps[t]];
        int m = Y.m;
        int am = m < 0 ? -m : m;
        double c = cm[am], s = m < 0 ? -sm[am] : sm[am];
        store(i, acc * c, acc * s);
    }
}

// The same with the power and phase tables in shared memory, scr[q * stride + thread] (they are indexed by the
// mode table at run time: as per-thread arrays they live in local memory, i.e. in L2/DRAM at 2^20 threads).
// scr holds 2 (max_pow + 1) + 2 (max_abs_m + 1) doubles per thread.
template <typename Store>
__device__ __forceinline__ void ylm_dev_smem(const YlmTable* __restrict__ T, double ch, double sh, double phi, double* scr, int stride, Store store) {
    const int mp = T->max_pow, mm = T->max_abs_m;
    double* pc = scr;
    double* ps = pc + (mp + 1) * stride;
    double* cm = ps + (mp + 1) * stride;
    double* sm = cm + (mm + 1) * stride;
    double a = 1.0, b = 1.0;
    pc[0] = 1.0;
    ps[0] = 1.0;
    for (int q = 1; q <= mp; q++) {
        a *= ch;
        b *= sh;
        pc[q * stride] = a;
        ps[q * stride] = b;
    }
    cm[0] = 1.0;
    sm[0] = 0.0;
    for (int q = 1; q <= mm; q++) {
        double sq, cq;
        sincos((double)q * phi, &sq, &cq);
        cm[q * stride] = cq;
        sm[q * stride] = sq;
    }
    const int M = T->M;
    for (int i = 0; i < M; i++) {
        const YlmMode& Y = T->mode[i];
        double acc = 0.0;
        for (int t = 0; t < Y.nterms; t++) acc += Y.coef[t] * pc[Y.pc[t] * stride] * ps[Y.ps[t] * stride];
        const int m = Y.m, am = m < 0 ? -m : m;
        const double c = cm[am * stride], s = m < 0 ? -sm[am * stride] : sm[am * stride];
        store(i, acc * c, acc * s);
    }
}

// Step 4 (Eq. 7, G1-G3): B = 1/4 sum_k [ |F_k|^2 Re(y^H U_k y) + Re(F_k^2 y^T V_k y) ], plain loops.
__device__ __forceinline__ double quadratic_dev(const LnlParams& P, const double* Fp, const double* Fx, const double* Yr, const double* Yi) {
    const int M = P.M;
    double B = 0.0;
    for (int k = 0; k < P.K; k++) {
        const double* U = P.U + (size_t)k * M * M * 2;
        const double* V = P.V + (size_t)k * M * M * 2;
        double uu = 0.0, vr = 0.0, vi = 0.0;
        for (int a = 0; a < M; a++) {
            double tUr = 0.0, tUi = 0.0, tVr = 0.0, tVi = 0.0;   // sum_b U_ab y_b, sum_b V_ab y_b
            for (int b = 0; b < M; b++) {
                double ur = __ldg(U + (a * M + b) * 2), ui = __ldg(U + (a * M + b) * 2 + 1);
                double wr = __ldg(V + (a * M + b) * 2), wi = __ldg(V + (a * M + b) * 2 + 1);
                tUr += ur * Yr[b] - ui * Yi[b];
                tUi += ur * Yi[b] + ui * Yr[b];
                tVr += wr * Yr[b] - wi * Yi[b];
                tVi += wr * Yi[b] + wi * Yr[b];
            }
            uu += Yr[a] * tUr + Yi[a] * tUi;                       // Re(conj(y_a) t)
            vr += Yr[a] * tVr - Yi[a] * tVi;
            vi += Yr[a] * tVi + Yi[a] * tVr;
        }
        double fr = Fp[k], fi = -Fx[k];                            // F = F+ - i Fx
        double f2r = fr * fr - fi * fi, f2i = 2.0 * fr * fi;
        B += (fr * fr + fi * fi) * uu + (f2r * vr - f2i * vi);
    }
    return 0.25 * B;
}

// Distance-marginalised lnT(A, B): bilinear, clamped (G28).
__device__ __forceinline__ double table_lookup(const LnlParams& P, double A, double B) {
    double a = (A - P.A_lo) / (P.A_hi - P.A_lo) * (double)(P.nA - 1);
    double b = (B - P.B_lo) / (P.B_hi - P.B_lo) * (double)(P.nB - 1);
    a = fmin(fmax(a, 0.0), (double)(P.nA - 1));
    b = fmin(fmax(b, 0.0), (double)(P.nB - 1));
    int ia = min((int)floor(a), P.nA - 2), ib = min((int)floor(b), P.nB - 2);
    double fa = a - ia, fb = b - ib;
    const double* T0 = P.lnT + (size_t)ib * P.nA + ia;
    double t0 = (1.0 - fa) * __ldg(T0) + fa * __ldg(T0 + 1);
    double t1 = (1.0 - fa) * __ldg(T0 + P.nA) + fa * __ldg(T0 + P.nA + 1);
    return (1.0 - fb) * t0 + fb * t1;
}
