// libile: integrator handles and the device-resident iteration driver (include/ile.h,
// "integrators").  draw -> lnL -> ln w = lnL + ln p - ln p_s -> reduce (Eq. 8, 9, 16) -> update,
// enqueued back to back on the context's stream with no host round-trip.
#include <stdlib.h>
#include <vector>
#include "integ.cuh"
#include "radix_sort.cuh"

// ---------------------------------------------------------------- host helpers
static void philox_host(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t* out) {
    for (int r = 0; r < 10; r++) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
static double uniform_host(uint64_t seed, uint64_t i, uint32_t g, int e) {
    uint32_t r[4];
    philox_host((uint32_t)i, (uint32_t)(i >> 32), g, (uint32_t)(e / 2), (uint32_t)seed, (uint32_t)(seed >> 32), r);
    const uint64_t w = (e & 1) ? (((uint64_t)r[3] << 32) | r[2]) : (((uint64_t)r[1] << 32) | r[0]);
    return (double)(w >> 11) * 0x1.0p-53;
}
static long long av_n_max_host(int d) {     // largest n with n^d < 2^62
    long long lo = 1, hi = (1ll << 31);
    if (d == 1) return (1ll << 62) - 1;
    while (lo < hi) {
        const long long mid = (lo + hi + 1) / 2;
        unsigned __int128 p = 1;
        bool over = false;
        for (int c = 0; c < d; c++) {
            p *= (unsigned __int128)mid;
            if (p >= ((unsigned __int128)1 << 62)) { over = true; break; }
        }
        if (!over) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// Arena layout: one device allocation behind all the small sampler state, with a second copy of
// its iteration-0 contents so that reset is one device-to-device copy.
struct ArenaPlan {
    size_t port, av[ILE_MAX_MEMBERS], H[ILE_MAX_MEMBERS], pi[ILE_MAX_MEMBERS], cdf[ILE_MAX_MEMBERS], gmm[ILE_MAX_MEMBERS], total;
};
static size_t gmm_doubles(int C, int d) { return (size_t)C + (size_t)C * d + 2 * (size_t)C * d * d; }
static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static ArenaPlan plan_arena(const IntegDev& I) {
    ArenaPlan A;
    memset(&A, 0, sizeof(A));
    size_t off = 0;
    A.port = off; off = align256(off + sizeof(PortState));
    for (int a = 0; a < I.n_members; a++) {
        const int k = I.mem[a].kind;
        if (k == ILE_KIND_AV) { A.av[a] = off; off = align256(off + sizeof(AvState)); }
        if (k == ILE_KIND_AC) {
            const int nb = I.mem[a].nb;
            A.H[a] = off; off = align256(off + (size_t)I.d * nb * 8);
            A.pi[a] = off; off = align256(off + (size_t)I.d * nb * 8);
            A.cdf[a] = off; off = align256(off + (size_t)I.d * (nb + 1) * 8);
        }
        if (k == ILE_KIND_GMM) { A.gmm[a] = off; off = align256(off + gmm_doubles(I.n_gmm, I.gd) * 8); }
    }
    A.total = off;
    return A;
}

static void host_chol(int d, const double* S, double* L) {
    for (int i = 0; i < d * d; i++) L[i] = 0.0;
    for (int i = 0; i < d; i++)
        for (int j = 0; j <= i; j++) {
            double s = S[i * d + j];
            for (int k = 0; k < j; k++) s = s - L[i * d + k] * L[j * d + k];
            L[i * d + j] = (i == j) ? sqrt(s) : s / L[j * d + j];
        }
}

// iteration-0 state: AC uniform marginals; AV one cell; GMM seeded means, wide
// covariances; portfolio equal weights
static void fill_initial(const IntegDev& I, const ArenaPlan& A, unsigned char* h) {
    PortState* P = (PortState*)(h + A.port);
    // iteration 0: the members whose first iteration is 0 are activated; uniform weights over the contributing ones
    int n_con = 0;
    for (int a = 0; a < I.n_members; a++) {
        P->active[a] = I.first_iter[a] <= 0 ? 1 : 0;
        n_con += P->active[a] && !I.silent[a];
    }
    for (int a = 0; a < I.n_members; a++) P->W[a] = (P->active[a] && !I.silent[a]) ? 1.0 / (double)n_con : 0.0;
    for (int a = 0; a < I.n_members; a++) {
        const int k = I.mem[a].kind;
        if (k == ILE_KIND_AV) {
            AvState* av = (AvState*)(h + A.av[a]);
            av->n = 1; av->C = 1; av->N_min = 0;
            av->L_thr = -INFINITY;
            av->v = 1.0;
            av->ln_ps = -log(I.V0);
        }
        if (k == ILE_KIND_AC) {
            double* pi = (double*)(h + A.pi[a]);
            double* cdf = (double*)(h + A.cdf[a]);
            for (int c = 0; c < I.d; c++) {
                double acc = 0.0;
                const int nb = I.mem[a].nb;
                cdf[c * (nb + 1)] = 0.0;
                for (int b = 0; b < nb; b++) {
                    pi[c * nb + b] = 1.0 / (double)nb;
                    acc = acc + pi[c * nb + b];
                    cdf[c * (nb + 1) + b + 1] = acc;
                }
            }
        }
        if (k == ILE_KIND_GMM) {
            const int C = I.n_gmm, d = I.gd;                         // modelled dimensions only
            double* omega = (double*)(h + A.gmm[a]);
            double* mu = omega + C;
            double* Sigma = mu + C * d;
            double* L = Sigma + C * d * d;
            for (int c = 0; c < C; c++) {
                omega[c] = 1.0 / (double)C;
                for (int i = 0; i < d; i++) {
                    const int dim = I.gdim[i];                        // the uniform of that dimension, as with every dimension modelled
                    const double u = uniform_host(I.seed, (uint64_t)c, 0xFFFFFFFFu, dim);
                    mu[c * d + i] = I.lo[dim] + u * (I.hi[dim] - I.lo[dim]);
                    const double hw = 0.5 * (I.hi[dim] - I.lo[dim]);
                    Sigma[c * d * d + i * d + i] = hw * hw;
                }
                host_chol(d, Sigma + c * d * d, L + c * d * d);
            }
        }
    }
}

// ---------------------------------------------------------------- small kernels of the driver
__global__ void lnw_kernel(int N, const double* __restrict__ lnL, const double* __restrict__ ln_prior, const double* __restrict__ ln_ps,
                           double* __restrict__ lnw) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double L = lnL[i];
    lnw[i] = is_finite_d(L) ? (L + ln_prior[i]) - ln_ps[i] : neg_inf();
}

// sampler state at draw time (pre = 1) / after the update (pre = 0) into the result struct
__global__ void annotate_kernel(IntegDev I, ile_result* r, int pre) {
    if (threadIdx.x || blockIdx.x) return;
    int av = -1;
    for (int a = 0; a < I.n_members; a++)
        if (I.mem[a].kind == ILE_KIND_AV && av < 0) av = a;
    if (pre) {
        r->n_cells = 0; r->n_bins = 0; r->N_min = 0; r->ln_volume = 0.0; r->L_thr = 0.0;
        for (int a = 0; a < ILE_MAX_MEMBERS; a++) r->W[a] = (I.kind == ILE_KIND_PORTFOLIO && a < I.n_members) ? I.port->W[a] : 0.0;
        if (av >= 0) {
            const AvState s = *I.mem[av].av;
            r->n_cells = (unsigned long long)s.C;
            r->n_bins = s.n;
            r->ln_volume = -s.ln_ps;
        }
    } else if (av >= 0) {
        const AvState s = *I.mem[av].av;
        r->N_min = (unsigned long long)s.N_min;
        r->L_thr = s.L_thr;
    }
}

__global__ void av_refresh_kernel(IntegDev I, int a) {     // derived fields after set_state
    if (threadIdx.x || blockIdx.x) return;
    AvState* av = I.mem[a].av;
    av->v = __ddiv_rn((double)av->C, pow_d_dev(av->n, I.d));
    av->ln_ps = -log(__dmul_rn(av->v, I.V0));
}

// ---------------------------------------------------------------- options, create, destroy
extern "C" int ile_integrator_opts_default(ile_integrator_opts* o, int kind, int d) {
    if (!o || kind < 0 || kind > ILE_KIND_PORTFOLIO || d < 1 || d > ILE_MAX_D) return ILE_EINVAL;
    memset(o, 0, sizeof(*o));
    o->kind = kind;
    o->d = d;
    const double PI = 3.14159265358979323846;
    const double lo[6] = {0.0, -1.0, 0.0, 0.0, -1.0, 100.0}, hi[6] = {2 * PI, 1.0, PI, 2 * PI, 1.0, 2000.0};
    for (int c = 0; c < d; c++) {
        o->lo[c] = c < 6 ? lo[c] : 0.0;
        o->hi[c] = c < 6 ? hi[c] : 1.0;
    }
    o->seed = 1;
    o->max_batch = 1 << 20;
    o->n_bins = 100;
    o->eps = 0.1;
    o->beta = 1.0;
    o->P_thr = 0.999;
    o->N_min_star = 4096;
    o->n_gmm = 8;
    if (kind == ILE_KIND_PORTFOLIO) {
        o->n_members = 3;
        o->member_kind[0] = ILE_KIND_AC;
        o->member_kind[1] = ILE_KIND_AV;
        o->member_kind[2] = ILE_KIND_GMM;
    }
    return ILE_OK;
}

static void free_integrator(ile_integrator* it) {
    if (!it) return;
    cudaFree(it->z); cudaFree(it->ln_ps); cudaFree(it->lnL); cudaFree(it->lnw); cudaFree(it->ln_prior);
    cudaFree(it->us); cudaFree(it->skey); cudaFree(it->q); cudaFree(it->kbuf0); cudaFree(it->kbuf1);
    cudaFree(it->sel_hist); cudaFree(it->blk_count); cudaFree(it->sort_scratch); cudaFree(it->gmm_part);
    cudaFree(it->port_part); cudaFree(it->res); cudaFree(it->arena);
    for (int a = 0; a < ILE_MAX_MEMBERS; a++) cudaFree(it->I.mem[a].keys);
    free(it);
}

#define IT_ALLOC(ptr, bytes)                                                                  \
    do {                                                                                      \
        if (cudaMalloc((void**)&(ptr), (bytes)) != cudaSuccess) {                             \
            cudaGetLastError();                                                               \
            free_integrator(it);                                                              \
            return ile_fail(ctx, ILE_ENOMEM, "integrator_create: device allocation of %zu bytes failed", (size_t)(bytes)); \
        }                                                                                     \
    } while (0)

extern "C" int ile_integrator_reset(ile_integrator* it);

extern "C" int ile_integrator_create(ile_ctx* ctx, const ile_integrator_opts* o, ile_integrator** out) {
    if (!ctx) return ILE_EINVAL;
    cudaSetDevice(ctx->device);   // every entry runs on the context's device, whatever the caller's current one
    if (!o || !out) return ile_fail(ctx, ILE_EINVAL, "integrator_create: null argument");
    *out = nullptr;
    // max_batch: the fixed-point sums (q <= 2^40 per sample, uint64) cannot overflow up to 2^24 samples with flat weights
    if (o->kind < 0 || o->kind > ILE_KIND_PORTFOLIO || o->d < 1 || o->d > ILE_MAX_D || o->max_batch < 1 || o->max_batch > (1ll << 24))
        return ile_fail(ctx, ILE_EINVAL, "integrator_create: kind, d (1..%d) or max_batch (1..2^24) out of range", ILE_MAX_D);
    for (int c = 0; c < o->d; c++)
        if (!(o->hi[c] > o->lo[c])) return ile_fail(ctx, ILE_EINVAL, "integrator_create: empty box in dimension %d", c);
    int kinds[ILE_MAX_MEMBERS], nbs[ILE_MAX_MEMBERS], Ns = 1;
    kinds[0] = o->kind;
    nbs[0] = o->n_bins;
    if (o->kind == ILE_KIND_PORTFOLIO) {
        Ns = o->n_members;
        if (Ns < 1 || Ns > ILE_MAX_MEMBERS) return ile_fail(ctx, ILE_EINVAL, "integrator_create: n_members in 1..%d", ILE_MAX_MEMBERS);
        for (int a = 0; a < Ns; a++) {
            kinds[a] = o->member_kind[a];
            if (kinds[a] < 0 || kinds[a] > ILE_KIND_GMM) return ile_fail(ctx, ILE_EINVAL, "integrator_create: member %d has kind %d", a, kinds[a]);
            nbs[a] = o->member_n_bins[a] ? o->member_n_bins[a] : o->n_bins;
            if (o->member_first_iter[a] < 0 || (a == 0 && o->member_first_iter[0] != 0))
                return ile_fail(ctx, ILE_EINVAL, "integrator_create: member_first_iter must be >= 0 and 0 for member 0 (PAPER.md:297)");
            if (o->member_silent[a] != 0 && o->member_silent[a] != 1) return ile_fail(ctx, ILE_EINVAL, "integrator_create: member_silent is 0 or 1");
            if (o->member_silent[a] && a == 0) return ile_fail(ctx, ILE_EINVAL, "integrator_create: member 0 contributes to the integral");
            if (a > 0 && o->member_silent[a - 1] && !o->member_silent[a])
                return ile_fail(ctx, ILE_EINVAL, "integrator_create: silent members are listed after the contributing ones");
        }
    }
    bool has_ac = false, has_av = false, has_gmm = false;
    for (int a = 0; a < Ns; a++) {
        has_ac |= kinds[a] == ILE_KIND_AC;
        has_av |= kinds[a] == ILE_KIND_AV;
        has_gmm |= kinds[a] == ILE_KIND_GMM;
    }
    if (has_ac && (!(o->eps >= 0.0 && o->eps <= 1.0) || !(o->beta > 0.0)))
        return ile_fail(ctx, ILE_EINVAL, "integrator_create: AC needs eps in [0,1], beta > 0");
    for (int a = 0; a < Ns; a++)   // the histogram kernel keeps d x n_bins 64-bit counters in shared memory (48 KB without opt-in)
        if (kinds[a] == ILE_KIND_AC && (nbs[a] < 1 || nbs[a] > 4096 || (long long)o->d * nbs[a] > 6144))
            return ile_fail(ctx, ILE_EINVAL, "integrator_create: AC needs n_bins in 1..4096 and d * n_bins <= 6144");
    if (has_av && (!(o->P_thr > 0.0 && o->P_thr <= 1.0) || o->N_min_star < 1))
        return ile_fail(ctx, ILE_EINVAL, "integrator_create: AV needs P_thr in (0,1], N_min_star >= 1");
    if (has_gmm && (o->n_gmm < 1 || o->n_gmm > 16)) return ile_fail(ctx, ILE_EINVAL, "integrator_create: n_gmm in 1..16");
    if (o->gmm_dims_mask >> o->d) return ile_fail(ctx, ILE_EINVAL, "integrator_create: gmm_dims_mask names a dimension >= d");

    ile_integrator* it = (ile_integrator*)calloc(1, sizeof(ile_integrator));
    if (!it) return ile_fail(ctx, ILE_ENOMEM, "integrator_create: out of host memory");
    it->ctx = ctx;
    it->o = *o;
    it->cap = o->max_batch;
    IntegDev& I = it->I;
    I.kind = o->kind; I.d = o->d; I.n_members = Ns; I.nb = has_ac ? o->n_bins : 1; I.n_gmm = has_gmm ? o->n_gmm : 1;
    for (int a = 0; a < Ns; a++) {
        I.mem[a].nb = kinds[a] == ILE_KIND_AC ? nbs[a] : 1;
        I.first_iter[a] = o->kind == ILE_KIND_PORTFOLIO ? o->member_first_iter[a] : 0;
        I.silent[a] = o->kind == ILE_KIND_PORTFOLIO ? o->member_silent[a] : 0;
    }
    I.V0 = 1.0;
    for (int c = 0; c < o->d; c++) {
        I.lo[c] = o->lo[c];
        I.hi[c] = o->hi[c];
        I.below_hi[c] = nextafter(o->hi[c], o->lo[c]);
        I.V0 = I.V0 * (o->hi[c] - o->lo[c]);
    }
    I.seed = o->seed; I.eps = o->eps; I.beta = o->beta; I.P_thr = o->P_thr; I.N_min_star = o->N_min_star;
    {   // the mixture models the dimensions of the mask (0 = all), the others are uniform over the box
        const unsigned mask = o->gmm_dims_mask ? o->gmm_dims_mask : (1u << o->d) - 1u;
        int nu = 0;
        I.gd = 0;
        I.ln_uvol = 0.0;
        for (int c = 0; c < ILE_MAX_D; c++) { I.gdim[c] = -1; I.udim[c] = -1; }
        for (int c = 0; c < o->d; c++) {
            if ((mask >> c) & 1u) I.gdim[I.gd++] = c;
            else {
                I.udim[nu++] = c;
                I.ln_uvol = I.ln_uvol + log(o->hi[c] - o->lo[c]);
            }
        }
    }
    I.n_max = av_n_max_host(o->d);
    for (int a = 0; a < Ns; a++) I.mem[a].kind = kinds[a];

    cudaSetDevice(ctx->device);
    const size_t cap = (size_t)it->cap;
    const ArenaPlan A = plan_arena(I);
    IT_ALLOC(it->arena, 2 * A.total);
    IT_ALLOC(it->z, cap * o->d * 8);
    IT_ALLOC(it->ln_ps, cap * 8);
    IT_ALLOC(it->lnL, cap * 8);
    IT_ALLOC(it->lnw, cap * 8);
    IT_ALLOC(it->ln_prior, cap * 8);
    IT_ALLOC(it->us, sizeof(UpdScratch));
    IT_ALLOC(it->res, sizeof(ile_result));
    if (has_av) {
        IT_ALLOC(it->skey, cap * 8);
        IT_ALLOC(it->q, cap * 8);
        IT_ALLOC(it->kbuf0, cap * 8);
        IT_ALLOC(it->kbuf1, cap * 8);
        IT_ALLOC(it->sel_hist, 2 * 2 * 256 * 8);
        IT_ALLOC(it->blk_count, ((cap + 2047) / 2048 + 1) * 4);
        IT_ALLOC(it->sort_scratch, radix_sort_scratch_bytes((int)cap));
    }
    if (has_gmm) {
        it->gmm_blocks = ctx->sm_count * 4;
        IT_ALLOC(it->gmm_part, (size_t)I.n_gmm * it->gmm_blocks * 48 * 8);
    }
    it->port_blocks = ctx->sm_count;
    IT_ALLOC(it->port_part, (size_t)Ns * it->port_blocks * 3 * 8);
    unsigned char* base = (unsigned char*)it->arena;
    I.port = (PortState*)(base + A.port);
    for (int a = 0; a < Ns; a++) {
        SamplerDev& S = I.mem[a];
        if (S.kind == ILE_KIND_AV) {
            S.av = (AvState*)(base + A.av[a]);
            IT_ALLOC(S.keys, cap * 8);
        }
        if (S.kind == ILE_KIND_AC) {
            S.H = (unsigned long long*)(base + A.H[a]);
            S.pi = (double*)(base + A.pi[a]);
            S.cdf = (double*)(base + A.cdf[a]);
        }
        if (S.kind == ILE_KIND_GMM) S.gmm = (double*)(base + A.gmm[a]);
    }
    std::vector<unsigned char> h(A.total, 0);
    fill_initial(I, A, h.data());
    if (cudaMemcpy(base + A.total, h.data(), A.total, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        free_integrator(it);
        return ile_fail(ctx, ILE_ECUDA, "integrator_create: initial state upload failed");
    }
    int rc = ile_integrator_reset(it);
    if (rc) {
        free_integrator(it);
        return rc;
    }
    *out = it;
    return ILE_OK;
}

extern "C" int ile_integrator_destroy(ile_integrator* it) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    cudaSetDevice(it->ctx->device);
    cudaStreamSynchronize(it->ctx->stream);
    free_integrator(it);
    return ILE_OK;
}

extern "C" int ile_integrator_reset(ile_integrator* it) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    ile_ctx* ctx = it->ctx;
    const ArenaPlan A = plan_arena(it->I);
    unsigned char* base = (unsigned char*)it->arena;
    ILE_CUDA(ctx, cudaMemcpyAsync(base, base + A.total, A.total, cudaMemcpyDeviceToDevice, ctx->stream));
    for (int a = 0; a < it->I.n_members; a++)
        if (it->I.mem[a].kind == ILE_KIND_AV) ILE_CUDA(ctx, cudaMemsetAsync(it->I.mem[a].keys, 0, 8, ctx->stream));
    ILE_CUDA(ctx, cudaMemsetAsync(it->res, 0, sizeof(ile_result), ctx->stream));
    it->drew = false;
    it->last_N = 0;
    return ILE_OK;
}

// ---------------------------------------------------------------- draw / ln_pdf / update
static int check_N(ile_integrator* it, int N, const char* what) {
    if (N < 1 || N > it->cap) return ile_fail(it->ctx, ILE_EINVAL, "%s: N = %d outside 1..max_batch (%lld)", what, N, it->cap);
    return ILE_OK;
}

extern "C" int ile_integrator_draw(ile_integrator* it, int N, uint64_t iter, double* z, double* ln_ps) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    int rc = check_N(it, N, "integrator_draw");
    if (rc) return rc;
    if (!z || !ln_ps) return ile_fail(it->ctx, ILE_EINVAL, "integrator_draw: null output");
    rc = integ_launch_draw(it, N, (unsigned int)iter, z, ln_ps);
    if (rc) return rc;
    it->drew = true;
    it->last_N = N;
    return ILE_OK;
}

extern "C" int ile_integrator_ln_pdf(ile_integrator* it, int N, const double* z, double* ln_ps) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    if (N < 1 || !z || !ln_ps) return ile_fail(it->ctx, ILE_EINVAL, "integrator_ln_pdf: bad argument");
    return integ_launch_ln_pdf(it, N, z, ln_ps);
}

extern "C" int ile_integrator_update(ile_integrator* it, int N, const double* z, const double* lnw, const double* ln_ps) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    int rc = check_N(it, N, "integrator_update");
    if (rc) return rc;
    if (!z || !lnw) return ile_fail(it->ctx, ILE_EINVAL, "integrator_update: null input");
    if (it->I.n_members > 1) {
        if (!ln_ps) return ile_fail(it->ctx, ILE_EINVAL, "integrator_update: a portfolio needs ln_ps");
        if (!it->drew || it->last_N != N)
            return ile_fail(it->ctx, ILE_ESTATE, "integrator_update: a portfolio must have drawn this batch (member allocation)");
    }
    return integ_launch_update(it, N, z, lnw, ln_ps);
}

static int draws_stay_in_box(const IntegDev& I) {
    for (int a = 0; a < I.n_members; a++)
        if (I.mem[a].kind == ILE_KIND_GMM) return 0;
    return 1;
}

// samples of the contributing members in a batch of N at iteration g (alloc_kernel's N_c): silent
// activated members take N / N_active each and sit after the contributing ones
static int contributing_samples(const IntegDev& I, int N, uint64_t g) {
    int n_act = 0, n_sil = 0;
    for (int a = 0; a < I.n_members; a++) {
        const bool act = (uint64_t)I.first_iter[a] <= g;
        n_act += act;
        n_sil += act && I.silent[a];
    }
    return n_sil ? N - n_sil * (N / n_act) : N;
}

// ---------------------------------------------------------------- step / run
static int step_internal(ile_integrator* it, int p, int N, uint64_t iter, ile_result* out_dev) {
    ile_ctx* ctx = it->ctx;
    const IntegDev& I = it->I;
    int rc = integ_launch_draw(it, N, (unsigned int)iter, it->z, it->ln_ps);
    if (rc) return rc;
    it->drew = true;
    it->last_N = N;
    if (draws_stay_in_box(I)) {
        ctx->zbox_hint = 1;
        for (int c = 0; c < I.d; c++) { ctx->zbox_lo[c] = I.lo[c]; ctx->zbox_hi[c] = I.hi[c]; }
    }
    rc = ile_launch_lnL_z(ctx, p, N, I.d, it->z, nullptr, it->lnL, it->ln_prior);
    ctx->zbox_hint = 0;
    if (rc) return rc;
    lnw_kernel<<<(N + 255) / 256, 256, 0, ctx->stream>>>(N, it->lnL, it->ln_prior, it->ln_ps, it->lnw);
    ILE_LAUNCH_CHECK(ctx);
    rc = ile_launch_reduce(ctx, contributing_samples(I, N, iter), it->lnw, it->res, 1);   // silent members' samples stay out of the estimate
    if (rc) return rc;
    annotate_kernel<<<1, 32, 0, ctx->stream>>>(I, it->res, 1);
    ILE_LAUNCH_CHECK(ctx);
    // a standalone AV samples uniformly inside its cells: V_{g+1} = V_g N_min / N
    const double* lp = (I.n_members == 1 && I.mem[0].kind == ILE_KIND_AV) ? nullptr : it->ln_ps;
    it->I.box_trusted = draws_stay_in_box(it->I);          // UNIFORM, AC and AV draws lie in [lo, hi) by construction; Gaussian tails do not
    rc = integ_launch_update(it, N, it->z, it->lnw, lp);
    it->I.box_trusted = 0;
    if (rc) return rc;
    annotate_kernel<<<1, 32, 0, ctx->stream>>>(I, it->res, 0);
    ILE_LAUNCH_CHECK(ctx);
    if (out_dev) ILE_CUDA(ctx, cudaMemcpyAsync(out_dev, it->res, sizeof(ile_result), cudaMemcpyDeviceToDevice, ctx->stream));
    return ILE_OK;
}

// ---------------------------------------------------------------- built-in test integrands
__global__ void __launch_bounds__(256) integrand_kernel(IntegDev I, ile_integrand F, int N, const double* __restrict__ z,
                                                        const double* __restrict__ ln_ps, double* __restrict__ lnf, double* __restrict__ lnw) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int d = I.d;
    double zz[ILE_MAX_D];
    bool inbox = true;
    for (int c = 0; c < d; c++) {
        zz[c] = z[(long long)c * N + i];
        inbox = inbox && (zz[c] >= I.lo[c]) && (zz[c] < I.hi[c]);
    }
    double v = neg_inf();
    if (inbox) {
        if (F.kind == ILE_F_GAUSSIAN_MIX) {
            double e[4], mx = neg_inf();
            for (int c = 0; c < F.n_comp; c++) {
                const double* pc = F.par + c * (ILE_MAX_D + 2);
                double r2 = 0.0;
                for (int k = 0; k < d; k++) r2 = r2 + (zz[k] - pc[k]) * (zz[k] - pc[k]);
                const double sg = pc[ILE_MAX_D];
                e[c] = pc[ILE_MAX_D + 1] - 0.5 * r2 / (sg * sg);
                mx = fmax(mx, e[c]);
            }
            double sum = 0.0;
            for (int c = 0; c < F.n_comp; c++) sum += exp(e[c] - mx);
            v = mx + log(sum);
        } else {
            const double a = F.par[0], b = F.par[1], T = F.par[2];
            double sacc = 0.0;
            for (int k = 0; k + 1 < d; k++) {
                const double t1 = a - zz[k], t2 = zz[k + 1] - zz[k] * zz[k];
                sacc = sacc + t1 * t1 + b * (t2 * t2);
            }
            v = -sacc / T;
        }
    }
    lnf[i] = v;
    lnw[i] = is_finite_d(v) ? v - ln_ps[i] : neg_inf();
}

extern "C" int ile_integrator_step_integrand(ile_integrator* it, const ile_integrand* f, int N, uint64_t iter, ile_result* out_dev) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    ile_ctx* ctx = it->ctx;
    int rc = check_N(it, N, "integrator_step_integrand");
    if (rc) return rc;
    if (!f || f->kind < 0 || f->kind > ILE_F_ROSENBROCK || (f->kind == ILE_F_GAUSSIAN_MIX && (f->n_comp < 1 || f->n_comp > 4)))
        return ile_fail(ctx, ILE_EINVAL, "integrator_step_integrand: unknown integrand or n_comp outside 1..4");
    if (f->kind == ILE_F_ROSENBROCK && (it->I.d < 2 || !(f->par[2] > 0.0)))
        return ile_fail(ctx, ILE_EINVAL, "integrator_step_integrand: Rosenbrock needs d >= 2 and T > 0");
    const IntegDev& I = it->I;
    rc = integ_launch_draw(it, N, (unsigned int)iter, it->z, it->ln_ps);
    if (rc) return rc;
    it->drew = true;
    it->last_N = N;
    integrand_kernel<<<(N + 255) / 256, 256, 0, ctx->stream>>>(I, *f, N, it->z, it->ln_ps, it->lnL, it->lnw);
    ILE_LAUNCH_CHECK(ctx);
    rc = ile_launch_reduce(ctx, contributing_samples(I, N, iter), it->lnw, it->res, 1);
    if (rc) return rc;
    annotate_kernel<<<1, 32, 0, ctx->stream>>>(I, it->res, 1);
    ILE_LAUNCH_CHECK(ctx);
    const double* lp = (I.n_members == 1 && I.mem[0].kind == ILE_KIND_AV) ? nullptr : it->ln_ps;
    it->I.box_trusted = draws_stay_in_box(it->I);          // UNIFORM, AC and AV draws lie in [lo, hi) by construction; Gaussian tails do not
    rc = integ_launch_update(it, N, it->z, it->lnw, lp);
    it->I.box_trusted = 0;
    if (rc) return rc;
    annotate_kernel<<<1, 32, 0, ctx->stream>>>(I, it->res, 0);
    ILE_LAUNCH_CHECK(ctx);
    if (out_dev) ILE_CUDA(ctx, cudaMemcpyAsync(out_dev, it->res, sizeof(ile_result), cudaMemcpyDeviceToDevice, ctx->stream));
    return ILE_OK;
}

extern "C" int ile_integrator_step(ile_integrator* it, int p, int N, uint64_t iter, ile_result* out_dev) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    int rc = check_N(it, N, "integrator_step");
    if (rc) return rc;
    return step_internal(it, p, N, iter, out_dev);
}

extern "C" int ile_integrator_run(ile_integrator* it, int p_first, int p_count, int n_iter, int N, ile_result* out_dev) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    int rc = check_N(it, N, "integrator_run");
    if (rc) return rc;
    if (p_count < 1 || n_iter < 1 || p_first < 0 || !out_dev) return ile_fail(it->ctx, ILE_EINVAL, "integrator_run: bad argument");
    for (int p = 0; p < p_count; p++) {
        rc = ile_integrator_reset(it);
        if (rc) return rc;
        for (int g = 0; g < n_iter; g++) {
            rc = step_internal(it, p_first + p, N, (uint64_t)g, out_dev + (size_t)p * n_iter + g);
            if (rc) return rc;
        }
    }
    return ILE_OK;
}

extern "C" int ile_integrator_last_batch(ile_integrator* it, const double** z, const double** ln_ps, const double** lnL,
                                         const double** lnw) {
    if (!it) return ILE_EINVAL;
    if (z) *z = it->z;
    if (ln_ps) *ln_ps = it->ln_ps;
    if (lnL) *lnL = it->lnL;
    if (lnw) *lnw = it->lnw;
    return ILE_OK;
}

// ---------------------------------------------------------------- state (de)serialisation
static size_t member_blob_bytes(const IntegDev& I, int a, long long C_av) {
    size_t b = 16;   // header: kind, d
    switch (I.mem[a].kind) {
        case ILE_KIND_AC: b += 8 + (size_t)I.d * I.mem[a].nb * 16 + (size_t)I.d * (I.mem[a].nb + 1) * 8; break;
        case ILE_KIND_AV: b += 32 + (size_t)C_av * 8; break;
        case ILE_KIND_GMM: b += 16 + gmm_doubles(I.n_gmm, I.gd) * 8; break;
        default: break;
    }
    return b;
}

extern "C" int ile_integrator_get_state(ile_integrator* it, void* buf, size_t* bytes) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    ile_ctx* ctx = it->ctx;
    if (!bytes) return ile_fail(ctx, ILE_EINVAL, "integrator_get_state: bytes is null");
    const IntegDev& I = it->I;
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    AvState av[ILE_MAX_MEMBERS];
    memset(av, 0, sizeof(av));
    for (int a = 0; a < I.n_members; a++)
        if (I.mem[a].kind == ILE_KIND_AV) ILE_CUDA(ctx, cudaMemcpy(&av[a], I.mem[a].av, sizeof(AvState), cudaMemcpyDeviceToHost));
    size_t need = 0;
    if (I.kind == ILE_KIND_PORTFOLIO) {
        need = 16 + 8 + 4 * 8 * ILE_MAX_MEMBERS;
        for (int a = 0; a < I.n_members; a++) need += 8 + member_blob_bytes(I, a, av[a].C);
    } else {
        need = member_blob_bytes(I, 0, av[0].C);
    }
    if (!buf) {
        *bytes = need;
        return ILE_OK;
    }
    if (*bytes < need) {
        *bytes = need;
        return ile_fail(ctx, ILE_EINVAL, "integrator_get_state: buffer too small (%zu needed)", need);
    }
    *bytes = need;
    unsigned char* w = (unsigned char*)buf;
    auto put_i64 = [&](long long v) { memcpy(w, &v, 8); w += 8; };
    auto put_dev = [&](const void* src, size_t n) -> int {
        if (n && cudaMemcpy(w, src, n, cudaMemcpyDeviceToHost) != cudaSuccess) return 1;
        w += n;
        return 0;
    };
    auto put_member = [&](int a) -> int {
        const SamplerDev& S = I.mem[a];
        put_i64(S.kind);
        put_i64(I.d);
        if (S.kind == ILE_KIND_AC) {
            put_i64(S.nb);
            if (put_dev(S.H, (size_t)I.d * S.nb * 8) || put_dev(S.pi, (size_t)I.d * S.nb * 8) || put_dev(S.cdf, (size_t)I.d * (S.nb + 1) * 8)) return 1;
        } else if (S.kind == ILE_KIND_AV) {
            put_i64(av[a].n); put_i64(av[a].C); put_i64(av[a].N_min);
            memcpy(w, &av[a].L_thr, 8); w += 8;
            if (put_dev(S.keys, (size_t)av[a].C * 8)) return 1;
        } else if (S.kind == ILE_KIND_GMM) {
            put_i64(I.n_gmm);
            put_i64(I.gd);
            if (put_dev(S.gmm, gmm_doubles(I.n_gmm, I.gd) * 8)) return 1;
        }
        return 0;
    };
    int bad = 0;
    if (I.kind == ILE_KIND_PORTFOLIO) {
        PortState P;
        ILE_CUDA(ctx, cudaMemcpy(&P, I.port, sizeof(P), cudaMemcpyDeviceToHost));
        put_i64(ILE_KIND_PORTFOLIO);
        put_i64(I.d);
        put_i64(I.n_members);
        memcpy(w, P.W, 8 * ILE_MAX_MEMBERS); w += 8 * ILE_MAX_MEMBERS;
        for (int a = 0; a < ILE_MAX_MEMBERS; a++) put_i64(P.frozen[a]);
        for (int a = 0; a < ILE_MAX_MEMBERS; a++) put_i64(P.alloc[a]);
        for (int a = 0; a < ILE_MAX_MEMBERS; a++) put_i64(P.active[a]);
        for (int a = 0; a < I.n_members && !bad; a++) {
            put_i64((long long)member_blob_bytes(I, a, av[a].C));
            bad = put_member(a);
        }
    } else {
        bad = put_member(0);
    }
    if (bad) {
        cudaGetLastError();
        return ile_fail(ctx, ILE_ECUDA, "integrator_get_state: device-to-host copy failed");
    }
    return ILE_OK;
}

extern "C" int ile_integrator_set_state(ile_integrator* it, const void* buf, size_t bytes) {
    if (!it) return ILE_EINVAL;
    cudaSetDevice(it->ctx->device);
    ile_ctx* ctx = it->ctx;
    if (!buf) return ile_fail(ctx, ILE_EINVAL, "integrator_set_state: null buffer");
    const IntegDev& I = it->I;
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const unsigned char* r = (const unsigned char*)buf;
    const unsigned char* end = r + bytes;
    bool dry = true;                       // first pass validates the whole blob, second pass writes
    auto get_i64 = [&](long long* v) -> bool {
        if (r + 8 > end) return false;
        memcpy(v, r, 8);
        r += 8;
        return true;
    };
    auto get_dev = [&](void* dst, size_t n) -> bool {
        if (r + n > end) return false;
        if (!dry && n && cudaMemcpy(dst, r, n, cudaMemcpyHostToDevice) != cudaSuccess) return false;
        r += n;
        return true;
    };
    auto get_member = [&](int a) -> bool {
        const SamplerDev& S = I.mem[a];
        long long kind, d;
        if (!get_i64(&kind) || !get_i64(&d) || kind != S.kind || d != I.d) return false;
        if (S.kind == ILE_KIND_AC) {
            long long nb;
            if (!get_i64(&nb) || nb != S.nb) return false;
            return get_dev(S.H, (size_t)I.d * S.nb * 8) && get_dev(S.pi, (size_t)I.d * S.nb * 8) && get_dev(S.cdf, (size_t)I.d * (S.nb + 1) * 8);
        }
        if (S.kind == ILE_KIND_AV) {
            AvState s;
            memset(&s, 0, sizeof(s));
            if (!get_i64(&s.n) || !get_i64(&s.C) || !get_i64(&s.N_min)) return false;
            if (r + 8 > end) return false;
            memcpy(&s.L_thr, r, 8);
            r += 8;
            if (s.n < 1 || s.n > I.n_max || s.C < 1 || s.C > it->cap) return false;
            if (r + (size_t)s.C * 8 > end) return false;
            {   // the draw's binary search and ln p_s assume sorted unique keys below n^d
                unsigned long long lim = 1, prev = 0, k;
                for (int c = 0; c < I.d; c++) lim *= (unsigned long long)s.n;
                for (long long q = 0; q < s.C; q++) {
                    memcpy(&k, r + 8 * q, 8);
                    if (k >= lim || (q > 0 && k <= prev)) return false;
                    prev = k;
                }
            }
            if (!dry && cudaMemcpy(S.av, &s, sizeof(s), cudaMemcpyHostToDevice) != cudaSuccess) return false;
            if (!get_dev(S.keys, (size_t)s.C * 8)) return false;
            if (!dry) {
                av_refresh_kernel<<<1, 32, 0, ctx->stream>>>(I, a);
                ctx->launches++;
            }
            return true;
        }
        if (S.kind == ILE_KIND_GMM) {
            long long C;
            long long gd;
            if (!get_i64(&C) || C != I.n_gmm || !get_i64(&gd) || gd != I.gd) return false;
            if (!get_dev(S.gmm, gmm_doubles(I.n_gmm, I.gd) * 8)) return false;
            if (!dry && integ_gmm_refresh(it, a) != ILE_OK) return false;     // Cholesky factors from the restored Sigma, not from the blob
            return true;
        }
        return true;
    };
    bool ok = true;
  for (int pass = 0; pass < 2 && ok; pass++) {
    dry = pass == 0;
    r = (const unsigned char*)buf;
    if (I.kind == ILE_KIND_PORTFOLIO) {
        long long kind, d, Ns;
        ok = get_i64(&kind) && get_i64(&d) && get_i64(&Ns) && kind == ILE_KIND_PORTFOLIO && d == I.d && Ns == I.n_members;
        PortState P;
        memset(&P, 0, sizeof(P));
        if (ok && r + 8 * ILE_MAX_MEMBERS <= end) {
            memcpy(P.W, r, 8 * ILE_MAX_MEMBERS);
            r += 8 * ILE_MAX_MEMBERS;
        } else ok = false;
        for (int a = 0; a < ILE_MAX_MEMBERS && ok; a++) { long long v; ok = get_i64(&v); P.frozen[a] = (int)v; }
        for (int a = 0; a < ILE_MAX_MEMBERS && ok; a++) { long long v; ok = get_i64(&v) && v >= 0 && v <= it->cap; P.alloc[a] = v; }
        for (int a = 0; a < ILE_MAX_MEMBERS && ok; a++) { long long v; ok = get_i64(&v) && (v == 0 || v == 1); P.active[a] = (int)v; }
        if (ok) {
            long long off = 0;
            for (int a = 0; a < I.n_members; a++) { P.offset[a] = off; off += P.alloc[a]; }
            P.offset[I.n_members] = off;
            ok = off <= it->cap;
            // the allocation belongs to a batch of that size: an update needs a draw first unless it is the resident one
            if (!dry && off != it->last_N) it->drew = false;
            ok = dry || cudaMemcpy(I.port, &P, sizeof(P), cudaMemcpyHostToDevice) == cudaSuccess;
        }
        for (int a = 0; a < I.n_members && ok; a++) {
            long long nb;
            ok = get_i64(&nb) && get_member(a);
        }
    } else {
        ok = get_member(0);
    }
    if (ok && r != end) ok = false;        // trailing bytes: not a blob of this integrator
  }
    if (!ok) {
        cudaGetLastError();
        return ile_fail(ctx, ILE_EINVAL, "integrator_set_state: blob does not match this integrator (kind, d, sizes) or is truncated");
    }
    ILE_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return ILE_OK;
}
