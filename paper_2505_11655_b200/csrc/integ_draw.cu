// libile: integrator draws and sampling-prior densities.
//   UNIFORM   z = lo + u (hi - lo)
//   AC        inverse-cdf draw from the per-dimension piecewise-constant marginals
//   AV        uniform in the union of active cells (reading G21)
//   GMM       Box-Muller normals through the component's Cholesky factor
//   PORTFOLIO members draw disjoint index ranges; every sample gets the mixture density
//             p_s = sum_a W_a p_{s,a}
// Counter-based generator: Philox4x32-10, counter (sample index, iteration, stream).
#include "integ.cuh"
#include <algorithm>

#define TWO_PI 6.283185307179586

// ---------------------------------------------------------------- member densities
template <int D>
__device__ __forceinline__ double ln_pdf_ac(const IntegDev& I, const SamplerDev& S, const double* zz) {
    // one logarithm of the product of the D marginal densities (each within [1e-30, 1e30]: no overflow for D <= 8)
    double prod = 1.0;
#pragma unroll
    for (int c = 0; c < D; c++) {
        const long long b = bin_index_dev(zz[c], I.lo[c], I.hi[c], S.nb);
        prod *= __ddiv_rn(__dmul_rn(S.pi[c * S.nb + b], (double)S.nb), __dsub_rn(I.hi[c], I.lo[c]));
    }
    return log(prod);
}

template <int D>
__device__ __forceinline__ double ln_pdf_av(const IntegDev& I, const SamplerDev& S, const double* zz) {
    const AvState av = *S.av;
    unsigned long long key = 0, mul = 1;
#pragma unroll
    for (int c = 0; c < D; c++) {
        key += (unsigned long long)bin_index_dev(zz[c], I.lo[c], I.hi[c], av.n) * mul;
        mul *= (unsigned long long)av.n;
    }
    long long lo = 0, hi = av.C;          // first position with keys[pos] >= key
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (S.keys[mid] < key) lo = mid + 1; else hi = mid;
    }
    return (lo < av.C && S.keys[lo] == key) ? av.ln_ps : neg_inf();
}

// Block-shared constants (dynamic shared memory): ln W_a of the members, then one GMM block (integ.cuh, GMS_*) per
// GMM member in member order.
#define DRAW_LNW 0
#define DRAW_GMS ILE_MAX_MEMBERS
__device__ __forceinline__ const double* member_gms(const IntegDev& I, int a, const double* sh) {
    int slot = 0;
    for (int b = 0; b < a; b++) slot += I.mem[b].kind == ILE_KIND_GMM;
    return sh + DRAW_GMS + slot * GMS_DOUBLES;
}

// ln N(z; mu_c, Sigma_c) + ln omega_c for every component; returns the log-sum-exp
// the modelled coordinates of a sample, in the mixture's order (static register indices: gdim is matched, not indexed)
template <int D>
__device__ __forceinline__ void gmm_gather(const IntegDev& I, const double* zz, double* zg) {
#pragma unroll
    for (int r = 0; r < D; r++) {
        zg[r] = 0.0;
#pragma unroll
        for (int c = 0; c < D; c++)
            if (I.gdim[r] == c) zg[r] = zz[c];
    }
}

template <int D>
__device__ __forceinline__ double ln_pdf_gmm(const IntegDev& I, const double* zz, const double* gs) {
    const int d = I.gd;
    const int C = I.n_gmm;
    double zg[D];
    gmm_gather<D>(I, zz, zg);
    bool uok = true;                       // the dimensions the mixture leaves alone: uniform over the box, zero outside
#pragma unroll
    for (int q = 0; q < D; q++)
        if (q < D - d) {
#pragma unroll
            for (int c = 0; c < D; c++)
                if (I.udim[q] == c) uok = uok && (zz[c] >= I.lo[c]) && (zz[c] < I.hi[c]);
        }
    double e[16];
    const double mx = gmm_ln_comps<D>(I, gs, zg, e);
    double sum = 0.0;
    for (int c = 0; c < C; c++) sum += exp(e[c] - mx);
    const double out = mx + log(sum);
    if (d == D) return out;
    return uok ? out - I.ln_uvol : neg_inf();
}

template <int D>
__device__ __forceinline__ double member_ln_pdf(const IntegDev& I, int a, const double* zz, bool inbox, const double* sh) {
    const SamplerDev& S = I.mem[a];
    switch (S.kind) {
        case ILE_KIND_UNIFORM: return inbox ? -log(I.V0) : neg_inf();
        case ILE_KIND_AC: return inbox ? ln_pdf_ac<D>(I, S, zz) : neg_inf();
        case ILE_KIND_AV: return inbox ? ln_pdf_av<D>(I, S, zz) : neg_inf();
        case ILE_KIND_GMM: return ln_pdf_gmm<D>(I, zz, member_gms(I, a, sh));
    }
    return neg_inf();
}

template <int D>
__device__ __forceinline__ double mixture_ln_pdf(const IntegDev& I, const double* zz, const double* sh) {
    bool inbox = true;
#pragma unroll
    for (int c = 0; c < D; c++) inbox = inbox && (zz[c] >= I.lo[c]) && (zz[c] < I.hi[c]);
    if (I.n_members == 1) return member_ln_pdf<D>(I, 0, zz, inbox, sh);
    double e[ILE_MAX_MEMBERS];
    double mx = neg_inf();
    for (int a = 0; a < I.n_members; a++) {
        // members that are not activated yet or contribute silently have weight 0 (ln W = -inf): no term
        const double lw = sh[DRAW_LNW + a];
        e[a] = lw == neg_inf() ? neg_inf() : lw + member_ln_pdf<D>(I, a, zz, inbox, sh);
        mx = fmax(mx, e[a]);
    }
    if (!is_finite_d(mx)) return neg_inf();
    double sum = 0.0;
    for (int a = 0; a < I.n_members; a++) sum += exp(e[a] - mx);
    return mx + log(sum);
}

// ---------------------------------------------------------------- allocation (portfolio, readings G25, G41, G42)
// Activated set at iteration g; when it changes the weights restart uniform over the contributing
// members.  Silent activated members take N / N_active samples each; the contributing ones share the rest,
// N_a = floor(N_c W_a) with the remainder to them in index order.
__global__ void alloc_kernel(IntegDev I, long long N, unsigned int g) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    PortState* P = I.port;
    const int Ns = I.n_members;
    bool changed = false;
    int n_act = 0, n_sil = 0, n_con = 0;
    for (int a = 0; a < Ns; a++) {
        const int act = (unsigned int)I.first_iter[a] <= g ? 1 : 0;
        changed = changed || (act != P->active[a]);
        P->active[a] = act;
        n_act += act;
        n_sil += act && I.silent[a];
        n_con += act && !I.silent[a];
    }
    P->restarted = 0;
    if (changed) {
        for (int a = 0; a < Ns; a++) {
            P->W[a] = (P->active[a] && !I.silent[a]) ? __ddiv_rn(1.0, (double)n_con) : 0.0;
            P->frozen[a] = 0;
        }
        P->restarted = 1;
    }
    const long long each = n_sil ? N / n_act : 0;
    const long long Nc = N - n_sil * each;
    long long tot = 0;
    for (int a = 0; a < Ns; a++) {
        const bool con = P->active[a] && !I.silent[a];
        P->alloc[a] = con ? (long long)floor(__dmul_rn((double)Nc, P->W[a])) : 0;
        tot += P->alloc[a];
    }
    long long rem = Nc - tot;
    int a = 0;
    while (rem > 0) {
        if (P->active[a % Ns] && !I.silent[a % Ns]) {
            P->alloc[a % Ns] += 1;
            rem--;
        }
        a++;
    }
    for (int b = 0; b < Ns; b++)
        if (P->active[b] && I.silent[b]) P->alloc[b] = each;
    long long off = 0;
    for (int b = 0; b < Ns; b++) {
        P->offset[b] = off;
        off += P->alloc[b];
    }
    P->offset[Ns] = off;
    P->n_contrib = (int)Nc;
}

// ---------------------------------------------------------------- draw
// every GMM member's constants and the members' ln W_a, once per block
__device__ __forceinline__ void block_consts(const IntegDev& I, double* sh) {
    if (I.n_members > 1 && threadIdx.x < I.n_members) sh[DRAW_LNW + threadIdx.x] = I.port->W[threadIdx.x] > 0.0 ? log(I.port->W[threadIdx.x]) : neg_inf();
    int slot = 0;
    for (int a = 0; a < I.n_members; a++)
        if (I.mem[a].kind == ILE_KIND_GMM) gmm_load_shared(I, I.mem[a].gmm, sh + DRAW_GMS + (slot++) * GMS_DOUBLES);
    __syncthreads();
}
static size_t draw_smem_bytes(const IntegDev& I) {
    int n = 0;
    for (int a = 0; a < I.n_members; a++) n += I.mem[a].kind == ILE_KIND_GMM;
    return ((size_t)ILE_MAX_MEMBERS + (size_t)n * GMS_DOUBLES) * sizeof(double);
}

template <int D>
__global__ void __launch_bounds__(128, 6) draw_kernel(IntegDev I, int N, unsigned int g, double* __restrict__ z, double* __restrict__ ln_ps) {
    extern __shared__ double draw_sh[];
    block_consts(I, draw_sh);
    // grid-stride: a block builds the shared constants once for all its samples
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    int a = 0;
    while (a + 1 < I.n_members && i >= I.port->offset[a + 1]) a++;
    const SamplerDev& S = I.mem[a];
    constexpr int d = D;
    double zz[D];
    double u0, u1;
    philox_pair(I.seed, (unsigned long long)i, g, 0u, &u0, &u1);
    if (S.kind == ILE_KIND_GMM) {
        const int C = I.n_gmm, gd = I.gd;
        const double* omega = S.gmm;
        const double* mu = omega + C;
        const double* L = mu + C * gd + C * gd * gd;
        int comp = 0;
        double cw = 0.0;
        for (int c = 0; c < C; c++) {     // number of cumulative weights <= u0
            cw = cw + omega[c];
            if (cw <= u0) comp = c + 1;
        }
        if (comp > C - 1) comp = C - 1;
        double nrm[D + 1];
        const int npair = (gd + 1) / 2;
#pragma unroll
        for (int p = 0; p < (D + 1) / 2; p++)
            if (p < npair) {
                double ua, ub;
                philox_pair(I.seed, (unsigned long long)i, g, (unsigned int)(1 + p), &ua, &ub);
                const double r = sqrt(-2.0 * log(1.0 - ua));
                double sn, cs;
                sincos(TWO_PI * ub, &sn, &cs);
                nrm[2 * p] = r * cs;
                nrm[2 * p + 1] = r * sn;
            }
        double zg[D];
#pragma unroll
        for (int r = 0; r < D; r++)
            if (r < gd) {
                double s = mu[comp * gd + r];
#pragma unroll
                for (int k = 0; k <= r; k++) s = s + L[comp * gd * gd + r * gd + k] * nrm[k];
                zg[r] = s;
            }
        // scatter to the modelled dimensions; the others are uniform over the box (streams after the Box-Muller pairs)
#pragma unroll
        for (int c = 0; c < D; c++) zz[c] = 0.0;
#pragma unroll
        for (int r = 0; r < D; r++)
            if (r < gd) {
#pragma unroll
                for (int c = 0; c < D; c++)
                    if (I.gdim[r] == c) zz[c] = zg[r];
            }
        double ua = 0.0, ub = 0.0;
#pragma unroll
        for (int q = 0; q < D; q++)
            if (q < D - gd) {
                if ((q & 1) == 0) philox_pair(I.seed, (unsigned long long)i, g, (unsigned int)(1 + npair + (q >> 1)), &ua, &ub);
                const double u = (q & 1) ? ub : ua;
#pragma unroll
                for (int c = 0; c < D; c++)
                    if (I.udim[q] == c) zz[c] = fmin(__dadd_rn(I.lo[c], __dmul_rn(u, __dsub_rn(I.hi[c], I.lo[c]))), I.below_hi[c]);
            }
    } else {
        unsigned long long key = 0;
        long long n = 1;
        if (S.kind == ILE_KIND_AV) {
            const AvState av = *S.av;
            n = av.n;
            long long cell = (long long)floor(__dmul_rn(u0, (double)av.C));
            if (cell > av.C - 1) cell = av.C - 1;
            key = S.keys[cell];
        }
        // all the uniforms first: the Philox calls are independent chains the scheduler can interleave
        double uc[D + 1];
#pragma unroll
        for (int pq = 0; pq < (D + 1) / 2; pq++) philox_pair(I.seed, (unsigned long long)i, g, (unsigned int)(1 + pq), &uc[2 * pq], &uc[2 * pq + 1]);
#pragma unroll
        for (int c = 0; c < d; c++) {
            const double u = uc[c];
            const double lo = I.lo[c], hi = I.hi[c];
            double zc;
            if (S.kind == ILE_KIND_UNIFORM) {
                zc = __dadd_rn(lo, __dmul_rn(u, __dsub_rn(hi, lo)));
            } else if (S.kind == ILE_KIND_AC) {
                const double* cdf = S.cdf + c * (S.nb + 1);
                const double* pi = S.pi + c * S.nb;
                int b0 = 0, b1 = S.nb;            // last b in [0, nb) with cdf[b] <= u
                while (b1 - b0 > 1) {
                    const int mid = (b0 + b1) >> 1;
                    if (cdf[mid] <= u) b0 = mid; else b1 = mid;
                }
                double r = __ddiv_rn(__dsub_rn(u, cdf[b0]), pi[b0]);
                r = fmin(r, 1.0 - 0x1.0p-53);
                const double delta = __ddiv_rn(__dsub_rn(hi, lo), (double)S.nb);
                zc = __dadd_rn(lo, __dmul_rn(__dadd_rn((double)b0, r), delta));
            } else {                                // AV
                const unsigned long long ic = key % (unsigned long long)n;
                key = key / (unsigned long long)n;
                const double y = __ddiv_rn(__dadd_rn((double)ic, u), (double)n);
                zc = __dadd_rn(lo, __dmul_rn(y, __dsub_rn(hi, lo)));
            }
            zz[c] = fmin(zc, I.below_hi[c]);
        }
    }
#pragma unroll
    for (int c = 0; c < d; c++) z[(long long)c * N + i] = zz[c];
    // a standalone AV draws inside its own cells: p_s is the constant 1 / (v V0)
    ln_ps[i] = (I.n_members == 1 && S.kind == ILE_KIND_AV) ? S.av->ln_ps : mixture_ln_pdf<D>(I, zz, draw_sh);
    }
}

template <int D>
__global__ void __launch_bounds__(128, 6) ln_pdf_kernel(IntegDev I, int N, const double* __restrict__ z, double* __restrict__ ln_ps) {
    extern __shared__ double draw_sh[];
    block_consts(I, draw_sh);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        double zz[D];
#pragma unroll
        for (int c = 0; c < D; c++) zz[c] = z[(long long)c * N + i];
        ln_ps[i] = mixture_ln_pdf<D>(I, zz, draw_sh);
    }
}

int integ_launch_draw(ile_integrator* it, int N, unsigned int g, double* z, double* ln_ps) {
    ile_ctx* ctx = it->ctx;
    alloc_kernel<<<1, 32, 0, ctx->stream>>>(it->I, (long long)N, g);
    ILE_LAUNCH_CHECK(ctx);
    const size_t smem = draw_smem_bytes(it->I);
    int grid = (int)std::min<long long>(((long long)N + 127) / 128, (long long)ctx->sm_count * 32), per_sm = 1;
    switch (it->I.d) {
#define DRAW_CASE(D_)                                                                                                  \
    case D_:                                                                                                           \
        ILE_CUDA(ctx, cudaFuncSetAttribute(draw_kernel<D_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        ILE_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, draw_kernel<D_>, 128, smem));             \
        grid = (int)std::min<long long>(grid, (long long)std::max(1, per_sm) * ctx->sm_count * 2);   /* two full waves */ \
        draw_kernel<D_><<<grid, 128, smem, ctx->stream>>>(it->I, N, g, z, ln_ps);                                      \
        break;
        DRAW_CASE(1) DRAW_CASE(2) DRAW_CASE(3) DRAW_CASE(4) DRAW_CASE(5) DRAW_CASE(6) DRAW_CASE(7) DRAW_CASE(8)
#undef DRAW_CASE
        default: return ile_fail(ctx, ILE_EINVAL, "draw: d = %d", it->I.d);
    }
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}

int integ_launch_ln_pdf(ile_integrator* it, int N, const double* z, double* ln_ps) {
    ile_ctx* ctx = it->ctx;
    const size_t smem = draw_smem_bytes(it->I);
    const int grid = (int)std::min<long long>(((long long)N + 127) / 128, (long long)ctx->sm_count * 32);
    switch (it->I.d) {
#define PDF_CASE(D_)                                                                                                     \
    case D_:                                                                                                             \
        ILE_CUDA(ctx, cudaFuncSetAttribute(ln_pdf_kernel<D_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        ln_pdf_kernel<D_><<<grid, 128, smem, ctx->stream>>>(it->I, N, z, ln_ps);                                         \
        break;
        PDF_CASE(1) PDF_CASE(2) PDF_CASE(3) PDF_CASE(4) PDF_CASE(5) PDF_CASE(6) PDF_CASE(7) PDF_CASE(8)
#undef PDF_CASE
        default: return ile_fail(ctx, ILE_EINVAL, "ln_pdf: d = %d", it->I.d);
    }
    ILE_LAUNCH_CHECK(ctx);
    return ILE_OK;
}
