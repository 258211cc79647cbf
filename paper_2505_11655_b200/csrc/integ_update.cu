// libile: integrator training steps, all device-resident.
//   AC         per-dimension fixed-point weighted histograms -> marginals
//   AV         threshold for enclosed probability P_thr by radix select on (ln f desc, index asc),
//              N_min, V_{g+1}, Delta V, n_bins (Eq. 13), sorted unique cell keys
//   GMM        one weighted EM step (reading G26)
//   PORTFOLIO  per-member n_ESS -> W, floor 0.05/N_s, freeze below 5 %
// Every decision (N_min, n_bins, frozen members, "nothing to train on") is taken on the device;
// the kernels that follow read it from UpdScratch, so an iteration needs no host round-trip.
#include "integ.cuh"
#include <algorithm>
#include "radix_sort.cuh"

enum { MASK_BOX = 1, MASK_LNPS = 2 };

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
        v = w > v ? w : v;
    }
    return v;
}
__device__ __forceinline__ unsigned long long warp_min_u64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
        v = w < v ? w : v;
    }
    return v;
}

// ---------------------------------------------------------------- common: init, masked max
__global__ void upd_init_kernel(UpdScratch* us, const int* skip, unsigned long long* zero_ptr, int zero_count, unsigned long long* sel_hist) {
    const bool dead = skip && *skip;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        memset(us, 0, sizeof(UpdScratch));
        us->mn_ord = ~0ull;
        us->abort = dead ? 1 : 0;
    }
    if (dead) return;
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < zero_count; q += gridDim.x * blockDim.x) zero_ptr[q] = 0ull;
    if (sel_hist)
        for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < 2 * 2 * 256; q += gridDim.x * blockDim.x) sel_hist[q] = 0ull;
}

__global__ void __launch_bounds__(256) mask_max_kernel(IntegDev I, int N, const double* __restrict__ z, const double* __restrict__ lnw,
                                                       const double* __restrict__ ln_ps, int mode, UpdScratch* us) {
    if (us->abort) return;
    unsigned long long mx = 0ull, mn = ~0ull, cnt = 0ull;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const double w = lnw[i];
        bool ok = is_finite_d(w);
        if (ok && (mode & MASK_BOX)) ok = in_box_dev(I, z, N, i);
        double lp = 0.0;
        if (ok && (mode & MASK_LNPS)) {
            lp = ln_ps[i];
            ok = is_finite_d(lp);
        }
        if (ok) {
            const unsigned long long o = ord_from_double(w);
            mx = o > mx ? o : mx;
            if (mode & MASK_LNPS) {
                const unsigned long long p = ord_from_double(lp);
                mn = p < mn ? p : mn;
            }
            cnt++;
        }
    }
    mx = warp_max_u64(mx);
    mn = warp_min_u64(mn);
    cnt = warp_sum_u64(cnt);
    if ((threadIdx.x & 31) == 0 && cnt) {
        atomicMax(&us->m_ord, mx);
        atomicMin(&us->mn_ord, mn);
        atomicAdd(&us->n_valid, cnt);
    }
}

// ---------------------------------------------------------------- AC
__global__ void __launch_bounds__(256) ac_hist_kernel(IntegDev I, int a, int N, const double* __restrict__ z, const double* __restrict__ lnw,
                                                      const UpdScratch* __restrict__ us) {
    if (us->abort || us->n_valid == 0) return;
    extern __shared__ unsigned long long sh_h[];
    const int nb = I.mem[a].nb, tot = I.d * nb;
    for (int q = threadIdx.x; q < tot; q += blockDim.x) sh_h[q] = 0ull;
    __syncthreads();
    const double m = double_from_ord(us->m_ord);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const double w = lnw[i];
        if (!is_finite_d(w) || !in_box_dev(I, z, N, i)) continue;
        const unsigned long long q = qfix_dev(__dmul_rn(I.beta, __dsub_rn(w, m)));
        if (!q) continue;
        for (int c = 0; c < I.d; c++) {
            const long long b = bin_index_dev(z[(long long)c * N + i], I.lo[c], I.hi[c], nb);
            atomicAdd(&sh_h[c * nb + (int)b], q);
        }
    }
    __syncthreads();
    unsigned long long* H = I.mem[a].H;
    for (int q = threadIdx.x; q < tot; q += blockDim.x)
        if (sh_h[q]) atomicAdd(&H[q], sh_h[q]);
}

// pi_c[b] = (1 - eps) H_c[b] / sum H_c + eps / n_b; cdf = left-to-right running sum.  One block per dimension: the
// integer total and the bins' divisions in parallel, the running sum by one thread in bin order (the oracle's order)
__global__ void __launch_bounds__(256) ac_finish_kernel(IntegDev I, int a, const UpdScratch* __restrict__ us) {
    if (us->abort) return;
    const int c = blockIdx.x, t = threadIdx.x;
    const int nb = I.mem[a].nb;
    const unsigned long long* H = I.mem[a].H + c * nb;
    double* pi = I.mem[a].pi + c * nb;
    double* cdf = I.mem[a].cdf + c * (nb + 1);
    __shared__ unsigned long long part[8];
    __shared__ unsigned long long tot_sh;
    unsigned long long s = 0;
    for (int b = t; b < nb; b += blockDim.x) s += H[b];
    s = warp_sum_u64(s);
    if ((t & 31) == 0) part[t >> 5] = s;
    __syncthreads();
    if (t == 0) {
        unsigned long long tot = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) tot += part[w];
        tot_sh = tot;
    }
    __syncthreads();
    const unsigned long long tot = tot_sh;
    if (tot == 0) return;                         // keep the old marginal
    for (int b = t; b < nb; b += blockDim.x) {
        const double frac = __ddiv_rn(__ull2double_rn(H[b]), __ull2double_rn(tot));
        pi[b] = __dadd_rn(__dmul_rn(__dsub_rn(1.0, I.eps), frac), __ddiv_rn(I.eps, (double)nb));
    }
    __syncthreads();
    if (t == 0) {
        double acc = 0.0;
        cdf[0] = 0.0;
        for (int b = 0; b < nb; b++) {
            acc = __dadd_rn(acc, pi[b]);
            cdf[b + 1] = acc;
        }
    }
}

// ---------------------------------------------------------------- AV
// ordered key (ascending = ln f descending), fixed-point weight q, total weight
__global__ void __launch_bounds__(256) av_prepare_kernel(IntegDev I, int N, const double* __restrict__ z, const double* __restrict__ lnw,
                                                         const double* __restrict__ ln_ps, UpdScratch* us, unsigned long long* __restrict__ skey,
                                                         unsigned long long* __restrict__ qv) {
    if (us->abort || us->n_valid == 0) return;
    const double m = double_from_ord(us->m_ord);
    unsigned long long tot = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const double w = lnw[i];
        bool ok = is_finite_d(w) && in_box_dev(I, z, N, i);
        double lp = 0.0;
        if (ok && ln_ps) {
            lp = ln_ps[i];
            ok = is_finite_d(lp);
        }
        unsigned long long k = ~0ull, q = 0ull;
        if (ok) {
            double lnf = __dadd_rn(w, lp);
            if (lnf == 0.0) lnf = 0.0;            // -0 and +0 are one value in the ordering
            k = ~ord_from_double(lnf);
            q = qfix_dev(__dsub_rn(w, m));
        }
        skey[i] = k;
        qv[i] = q;
        tot += q;
    }
    tot = warp_sum_u64(tot);
    if ((threadIdx.x & 31) == 0 && tot) atomicAdd(&us->total_q, tot);
}

__global__ void av_sel_init_kernel(IntegDev I, UpdScratch* us) {
    if (threadIdx.x || blockIdx.x) return;
    if (us->abort) return;
    if (us->n_valid == 0 || us->total_q == 0) {
        us->abort = 1;
        return;
    }
    const double Td = ceil(__dmul_rn(I.P_thr, __ull2double_rn(us->total_q)));
    const unsigned long long T = (unsigned long long)Td;
    us->path[0].target = T;
    us->path[0].fail = T > us->total_q ? 1 : 0;
    unsigned long long want = (unsigned long long)I.N_min_star;
    if (want > us->n_valid) want = us->n_valid;
    if (want < 1) want = 1;
    us->path[1].target = want;
}

__device__ __forceinline__ bool sel_match(const SelPath& P, unsigned long long k, unsigned int idx) {
    const int nd = P.ndig;
    if (nd == 0) return true;
    if (nd <= 8) {
        const int sh = 64 - 8 * nd;
        return (k >> sh) == (P.prefix_key >> sh);
    }
    if (k != P.prefix_key) return false;
    const int sh = 32 - 8 * (nd - 8);
    return sh >= 32 ? true : (idx >> sh) == (P.prefix_idx >> sh);
}
__device__ __forceinline__ int sel_digit(int nd, unsigned long long k, unsigned int idx) {
    return nd < 8 ? (int)((k >> (56 - 8 * nd)) & 0xffull) : (int)((idx >> (24 - 8 * (nd - 8))) & 0xffu);
}

// Fix the next digit of each live path and clear the histogram for the next pass: one block of 256 threads, thread b = bin b.
// The digit is the first bin at which the running metric reaches the target; the running sums are exact integers, so the
// block scan gives what a bin-by-bin walk gives.
__device__ void sel_pick_block(UpdScratch* us, unsigned long long* hist) {
    __shared__ unsigned long long wtot[2][8];
    __shared__ int dg_sh;
    const int b = threadIdx.x, lane = b & 31, wp = b >> 5;
    for (int p = 0; p < 2; p++) {
        SelPath P = us->path[p];
        if (P.done || P.fail) continue;                      // the same for every thread
        const unsigned long long cnt = __ldcg(hist + (p * 2 + 0) * 256 + b), met = __ldcg(hist + (p * 2 + 1) * 256 + b);
        unsigned long long sm = met, sc = cnt;                // inclusive sums over the warp's bins
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long tm = __shfl_up_sync(0xffffffffu, sm, o), tc = __shfl_up_sync(0xffffffffu, sc, o);
            if (lane >= o) { sm += tm; sc += tc; }
        }
        if (lane == 31) { wtot[0][wp] = sm; wtot[1][wp] = sc; }
        if (b == 0) dg_sh = 256;
        __syncthreads();
        unsigned long long om = P.cum_metric, oc = P.cum_count;
        for (int w2 = 0; w2 < wp; w2++) { om += wtot[0][w2]; oc += wtot[1][w2]; }
        if (om + sm >= P.target) atomicMin(&dg_sh, b);
        __syncthreads();
        const int dg = dg_sh;
        if (dg == 256) {
            if (b == 0) { P.fail = 1; us->path[p] = P; }
        } else if (b == dg) {
            P.cum_metric = om + sm - met;
            P.cum_count = oc + sc - cnt;
            if (P.ndig < 8) P.prefix_key |= (unsigned long long)dg << (56 - 8 * P.ndig);
            else P.prefix_idx |= (unsigned int)dg << (24 - 8 * (P.ndig - 8));
            P.ndig++;
            if (cnt == 1 || P.ndig == AV_SEL_PASSES) P.done = 1;
            us->path[p] = P;
        }
        __syncthreads();
    }
    for (int q = b; q < 1024; q += 256) hist[q] = 0ull;
}

// histogram of the next digit among the elements matching each path's prefix
// hist layout: [path][0 = count, 1 = metric][256]
__global__ void __launch_bounds__(256) av_sel_hist_kernel(int N, const unsigned long long* __restrict__ skey,
                                                          const unsigned long long* __restrict__ qv, UpdScratch* us,
                                                          unsigned long long* hist) {
    if (us->abort) return;
    __shared__ unsigned long long sh[2][2][256];
    __shared__ SelPath P[2];
    if (threadIdx.x < 2) P[threadIdx.x] = us->path[threadIdx.x];
    for (int q = threadIdx.x; q < 1024; q += blockDim.x) (&sh[0][0][0])[q] = 0ull;
    __syncthreads();
    const bool live0 = !P[0].done && !P[0].fail, live1 = !P[1].done;
    if (!live0 && !live1) return;
    const int lane = threadIdx.x & 31;
    const long long Npad = ((long long)N + 31) & ~31ll;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < Npad; i += (long long)gridDim.x * blockDim.x) {
        const bool act = i < N;
        const unsigned long long k = act ? skey[i] : ~0ull;
        const unsigned long long q = act ? qv[i] : 0ull;
#pragma unroll
        for (int p = 0; p < 2; p++) {
            if (!(p == 0 ? live0 : live1)) continue;
            const bool mt = act && sel_match(P[p], k, (unsigned int)i);
            const int dg = mt ? sel_digit(P[p].ndig, k, (unsigned int)i) : 256;
            const unsigned mask = __match_any_sync(0xffffffffu, dg);
            if (mask == 0xffffffffu) {            // whole warp in one bucket: one atomic each
                if (dg == 256) continue;
                const unsigned long long qs = p == 0 ? warp_sum_u64(q) : 32ull;
                if (lane == 0) {
                    atomicAdd(&sh[p][0][dg], 32ull);
                    atomicAdd(&sh[p][1][dg], qs);
                }
            } else if (mt) {
                if (lane == __ffs(mask) - 1) atomicAdd(&sh[p][0][dg], (unsigned long long)__popc(mask));
                if (p == 0) { if (q) atomicAdd(&sh[p][1][dg], q); }
                else if (lane == __ffs(mask) - 1) atomicAdd(&sh[p][1][dg], (unsigned long long)__popc(mask));
            }
        }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < 1024; q += blockDim.x) {
        const unsigned long long v = (&sh[0][0][0])[q];
        if (v) atomicAdd(&hist[q], v);
    }
    // the last block to get here sees every block's sums and fixes the digit (no second launch per pass)
    __shared__ bool last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = atomicAdd(&us->ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!last) return;
    __threadfence();
    sel_pick_block(us, hist);
    if (threadIdx.x == 0) us->ticket = 0u;
}

__device__ __forceinline__ bool av_kept(const UpdScratch& U, const SelPath& P, unsigned long long k, unsigned int idx) {
    if (k == ~0ull) return false;
    if (U.use_path == 2) return true;
    const int nd = P.ndig;
    if (nd <= 8) {
        const int sh = 64 - 8 * nd;
        return (k >> sh) <= (P.prefix_key >> sh);
    }
    if (k != P.prefix_key) return k < P.prefix_key;
    const int sh = 32 - 8 * (nd - 8);
    return (idx >> sh) <= (P.prefix_idx >> sh);
}

// N_P, N_min = min(n_valid, max(N_P, N_min*)), and which threshold realises it
__global__ void av_decide_kernel(IntegDev I, int N, UpdScratch* us) {
    if (threadIdx.x || blockIdx.x) return;
    if (us->abort) return;
    const SelPath A = us->path[0], B = us->path[1];
    const unsigned long long n_valid = us->n_valid;
    const unsigned long long N_P = (A.fail || !A.done) ? (unsigned long long)N + 1ull : A.cum_count + 1ull;
    unsigned long long want = N_P > (unsigned long long)I.N_min_star ? N_P : (unsigned long long)I.N_min_star;
    const unsigned long long N_min = want < n_valid ? want : n_valid;
    int use;
    if (N_min == n_valid) use = 2;                         // keep every valid sample
    else if (N_min == N_P) use = 0;
    else use = 1;                                          // N_min = N_min* (B's target)
    (void)B;
    us->use_path = use;
    us->N_min = (long long)N_min;
}

// over the kept samples: count, fixed-point sum of 1/p_s (portfolio member), last kept ln f
__global__ void __launch_bounds__(256) av_stats_kernel(int N, const double* __restrict__ ln_ps, UpdScratch* us,
                                                       const unsigned long long* __restrict__ skey) {
    if (us->abort) return;
    __shared__ UpdScratch U;
    if (threadIdx.x == 0) U = *us;
    __syncthreads();
    const SelPath P = U.path[U.use_path < 2 ? U.use_path : 0];
    const double mn = double_from_ord(U.mn_ord);
    unsigned long long R = 0, mk = 0, cnt = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long k = skey[i];
        if (!av_kept(U, P, k, (unsigned int)i)) continue;
        cnt++;
        mk = k > mk ? k : mk;
        if (ln_ps) R += qfix_dev(__dsub_rn(mn, ln_ps[i]));
    }
    R = warp_sum_u64(R);
    cnt = warp_sum_u64(cnt);
    mk = warp_max_u64(mk);
    if ((threadIdx.x & 31) == 0 && cnt) {
        atomicAdd(&us->R, R);
        atomicAdd((unsigned long long*)&us->n_kept, cnt);
        atomicMax(&us->max_skey, mk);
    }
}

// V_{g+1} = V_g N_min / N (or its importance estimate), Delta V = V_{g+1} / sqrt(N_min),
// n_{g+1} = largest n with n^d <= 1 / Delta V (Eq. 13, reading G20)
__global__ void av_nnew_kernel(IntegDev I, int a, int N, UpdScratch* us, int has_lnps) {
    if (threadIdx.x || blockIdx.x) return;
    if (us->abort) return;
    const AvState av = *I.mem[a].av;
    const double Nm = (double)us->N_min;
    double v_new;
    if (!has_lnps) {
        v_new = __ddiv_rn(__dmul_rn(av.v, Nm), (double)N);
    } else {
        const double mn = double_from_ord(us->mn_ord);
        v_new = __ddiv_rn(__dmul_rn(__dmul_rn(__ull2double_rn(us->R), 0x1.0p-40), exp(-mn)), __dmul_rn((double)N, I.V0));
    }
    const double dv = __ddiv_rn(v_new, sqrt(Nm));
    const double inv = __ddiv_rn(1.0, dv);
    long long lo_n = 1, hi_n = I.n_max;
    while (lo_n < hi_n) {
        const long long mid = (lo_n + hi_n + 1) / 2;
        if (pow_d_dev(mid, I.d) <= inv) lo_n = mid; else hi_n = mid - 1;
    }
    unsigned long long top = 1;
    for (int c = 0; c < I.d; c++) top *= (unsigned long long)lo_n;
    top -= 1;                                               // largest key
    int bits = 0;
    while (top) { bits++; top >>= 1; }
    us->v_new = v_new;
    us->n_new = lo_n;
    us->n_bits = bits;
    us->n_kept = 0;                                         // reused as the compaction cursor
}

__global__ void __launch_bounds__(256) av_compact_kernel(IntegDev I, int N, const double* __restrict__ z, UpdScratch* us,
                                                         const unsigned long long* __restrict__ skey, unsigned long long* __restrict__ out) {
    if (us->abort) return;
    __shared__ UpdScratch U;
    if (threadIdx.x == 0) U = *us;
    __syncthreads();
    const SelPath P = U.path[U.use_path < 2 ? U.use_path : 0];
    const int lane = threadIdx.x & 31;
    const long long Npad = ((long long)N + 31) & ~31ll;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < Npad; i += (long long)gridDim.x * blockDim.x) {
        const bool keep = i < N && av_kept(U, P, skey[i], (unsigned int)i);
        const unsigned mask = __ballot_sync(0xffffffffu, keep);
        if (!mask) continue;
        long long base = 0;
        if (lane == __ffs(mask) - 1) base = (long long)atomicAdd((unsigned long long*)&us->n_kept, (unsigned long long)__popc(mask));
        base = __shfl_sync(0xffffffffu, base, __ffs(mask) - 1);
        if (keep) out[base + __popc(mask & ((1u << lane) - 1u))] = av_key_dev(I, z, N, i, U.n_new);
    }
}

// sorted keys -> unique keys (three kernels: heads per block, scan, write)
#define UQ_TILE 2048
__global__ void __launch_bounds__(256) uniq_count_kernel(const unsigned long long* __restrict__ k, const UpdScratch* __restrict__ us,
                                                         unsigned int* __restrict__ blk) {
    if (us->abort) return;
    const long long n = us->n_kept;
    const long long base = (long long)blockIdx.x * UQ_TILE;
    if (base >= n) return;
    unsigned int c = 0;
    for (int r = 0; r < UQ_TILE / 256; r++) {
        const long long i = base + r * 256 + threadIdx.x;
        if (i < n && (i == 0 || k[i] != k[i - 1])) c++;
    }
    __shared__ unsigned int sh;
    if (threadIdx.x == 0) sh = 0;
    __syncthreads();
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(&sh, c);
    __syncthreads();
    if (threadIdx.x == 0) blk[blockIdx.x] = sh;
}
__global__ void __launch_bounds__(1024) uniq_scan_kernel(UpdScratch* us, unsigned int* __restrict__ blk) {
    if (us->abort) return;
    const long long n = us->n_kept;
    const int nblocks = (int)((n + UQ_TILE - 1) / UQ_TILE);
    __shared__ unsigned int part[1024];
    const int t = threadIdx.x;
    const int per = (nblocks + 1023) / 1024;
    const int b0 = min(t * per, nblocks), b1 = min(b0 + per, nblocks);
    unsigned int s = 0;
    for (int b = b0; b < b1; b++) s += blk[b];
    part[t] = s;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
        unsigned int add = t >= o ? part[t - o] : 0;
        __syncthreads();
        part[t] += add;
        __syncthreads();
    }
    unsigned int run = part[t] - s;
    for (int b = b0; b < b1; b++) {
        unsigned int c = blk[b];
        blk[b] = run;
        run += c;
    }
    if (t == 1023) us->n_heads = (long long)part[1023];
}
__global__ void __launch_bounds__(256) uniq_write_kernel(const unsigned long long* __restrict__ k, const UpdScratch* __restrict__ us,
                                                         const unsigned int* __restrict__ blk, unsigned long long* __restrict__ out) {
    if (us->abort) return;
    const long long n = us->n_kept;
    const long long base = (long long)blockIdx.x * UQ_TILE;
    if (base >= n) return;
    // thread t owns UQ_TILE/256 consecutive keys so that ranks follow the sorted order
    const int PER = UQ_TILE / 256;
    const long long i0 = base + (long long)threadIdx.x * PER;
    unsigned int c = 0;
    for (int r = 0; r < PER; r++) {
        const long long i = i0 + r;
        if (i < n && (i == 0 || k[i] != k[i - 1])) c++;
    }
    __shared__ unsigned int sc[256];
    sc[threadIdx.x] = c;
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {
        unsigned int add = threadIdx.x >= o ? sc[threadIdx.x - o] : 0;
        __syncthreads();
        sc[threadIdx.x] += add;
        __syncthreads();
    }
    unsigned int pos = blk[blockIdx.x] + sc[threadIdx.x] - c;
    for (int r = 0; r < PER; r++) {
        const long long i = i0 + r;
        if (i < n && (i == 0 || k[i] != k[i - 1])) out[pos++] = k[i];
    }
}

__global__ void av_commit_kernel(IntegDev I, int a, UpdScratch* us) {
    if (threadIdx.x || blockIdx.x) return;
    if (us->abort) return;
    AvState* av = I.mem[a].av;
    av->n = us->n_new;
    av->C = us->n_heads;
    av->N_min = us->N_min;
    av->L_thr = double_from_ord(~us->max_skey);
    av->v = __ddiv_rn((double)av->C, pow_d_dev(av->n, I.d));
    av->ln_ps = -log(__dmul_rn(av->v, I.V0));
}

// ---------------------------------------------------------------- GMM (one weighted EM step)
#define GMM_NACC 36                                         // 1 + d + d(d+1)/2 at d = 7; d = 8 needs 45
#define GMM_NACC_MAX 48
// One weighted EM step's sums in one pass (E step + M-step moments).  Per round of 256 samples: thread t evaluates the
// mixture at its sample and leaves the responsibilities x importance weight R[t][c] (0 outside the box or for a
// non-finite weight) and the modelled coordinates Z[t][.] in shared memory; then thread (slice, component c, moment q)
// adds its slice of the round to its moment about the component's old mean: q = 0: sum R, 1 + r: sum R dz_r,
// 1 + D + r (r + 1) / 2 + s: sum R dz_r dz_s (layout by the total dimension D; entries past gd stay 0).  Column D of Z is
// the constant 1 with mean 0, so every moment is sum R (Z[ia] - mu[ia]) (Z[ib] - mu[ib]) for an index pair (ia, ib).
#define GMM_SLOTS 3                                          // moment slots per thread: 16 components x 45 moments / 256
template <int D>
__global__ void __launch_bounds__(256) gmm_em_kernel(IntegDev I, int a, int N, const double* __restrict__ z, const double* __restrict__ lnw,
                                                     const UpdScratch* __restrict__ us, double* __restrict__ part) {
    if (us->abort || us->n_valid == 0) return;
    constexpr int NACC = 1 + D + D * (D + 1) / 2, ZP = D + 1 + ((D + 1) & 1 ? 0 : 1);      // odd row strides: no bank conflicts
    constexpr int CP = 17;                   // row stride of R (16 components)
    const int d = I.gd, C = I.n_gmm, t = threadIdx.x;
    const double* g = I.mem[a].gmm;
    extern __shared__ double em_sh[];
    double* gs = em_sh;                      // the member's constants
    double* R = gs + GMS_DOUBLES;            // [256][CP]
    double* Z = R + 256 * CP;                // [256][ZP]
    double* mu_s = Z + 256 * ZP;             // [C][D + 1]
    gmm_load_shared(I, g, gs);
    for (int q = t; q < C * (D + 1); q += 256) {
        const int c = q / (D + 1), r = q - c * (D + 1);
        mu_s[q] = r < d ? g[C + c * d + r] : 0.0;
    }
    // the moments this thread accumulates
    const int NP = C * NACC, SL = NP >= 256 ? 1 : 256 / NP;
    int sc[GMM_SLOTS], sia[GMM_SLOTS], sib[GMM_SLOTS], sl[GMM_SLOTS];
    bool used[GMM_SLOTS];
    double acc[GMM_SLOTS];
#pragma unroll
    for (int k = 0; k < GMM_SLOTS; k++) {
        const int item = t + 256 * k;
        acc[k] = 0.0;
        sc[k] = sia[k] = sib[k] = sl[k] = 0;
        used[k] = item < NP * SL;
        if (used[k]) {
            const int pair = item % NP;
            sl[k] = item / NP;
            const int c = pair / NACC, q = pair - c * NACC;
            int ia = D, ib = D;
            if (q >= 1 && q <= D) ia = q - 1;
            else if (q > D) {
                int r = 0;
                while (1 + D + (r + 1) * (r + 2) / 2 <= q) r++;
                ia = r;
                ib = q - (1 + D + r * (r + 1) / 2);
            }
            sc[k] = c; sia[k] = ia; sib[k] = ib;
        }
    }
    __syncthreads();
    const double m = double_from_ord(us->m_ord);
    __shared__ int wcnt[8];
    const int lane = t & 31, wid = t >> 5;
    for (long long base = (long long)blockIdx.x * 256; base < N; base += (long long)gridDim.x * 256) {
        const long long i = base + t;
        // samples whose weight exp(ln w - max) underflows to 0 (most of a batch, PAPER.md:107 weights are peaked) add
        // exactly nothing to any sum: they skip the mixture evaluation and are left out of the round's list
        double wt = 0.0;
        if (i < N) {
            const double w = lnw[i];
            if (is_finite_d(w) && in_box_dev(I, z, N, i)) wt = exp(w - m);
        }
        const bool ok = wt > 0.0;
        const unsigned bal = __ballot_sync(0xffffffffu, ok);
        if (lane == 0) wcnt[wid] = __popc(bal);
        __syncthreads();
        int pos = __popc(bal & ((1u << lane) - 1u)), nround = 0;
#pragma unroll
        for (int q = 0; q < 8; q++) {
            pos += q < wid ? wcnt[q] : 0;
            nround += wcnt[q];
        }
        if (ok) {
            double zz[D], e[16];
#pragma unroll
            for (int c = 0; c < D; c++) zz[c] = c < d ? z[(long long)I.gdim[c] * N + i] : 0.0;
            const double mx = gmm_ln_comps<D>(I, gs, zz, e);
            double sum = 0.0;
            for (int c = 0; c < C; c++) {
                e[c] = exp(e[c] - mx);
                sum += e[c];
            }
            wt = wt / sum;
            for (int c = 0; c < C; c++) R[pos * CP + c] = e[c] * wt;
#pragma unroll
            for (int c = 0; c < D; c++) Z[pos * ZP + c] = zz[c];
            Z[pos * ZP + D] = 1.0;
        }
        __syncthreads();
        const int per = (nround + SL - 1) / SL;
#pragma unroll
        for (int k = 0; k < GMM_SLOTS; k++) {
            if (!used[k]) continue;
            const int b0 = min(nround, sl[k] * per), b1 = min(nround, b0 + per);
            if (b1 <= b0) continue;
            const double ma = mu_s[sc[k] * (D + 1) + sia[k]], mb = mu_s[sc[k] * (D + 1) + sib[k]];
            const double* pr = R + b0 * CP + sc[k];
            const double* pa = Z + b0 * ZP + sia[k];
            const double* pb = Z + b0 * ZP + sib[k];
            double v = acc[k];
            int n = b1 - b0;
            for (; n >= 4; n -= 4) {
#pragma unroll
                for (int u = 0; u < 4; u++) v = fma(pr[u * CP], (pa[u * ZP] - ma) * (pb[u * ZP] - mb), v);
                pr += 4 * CP;
                pa += 4 * ZP;
                pb += 4 * ZP;
            }
            for (; n > 0; n--) {
                v = fma(pr[0], (pa[0] - ma) * (pb[0] - mb), v);
                pr += CP;
                pa += ZP;
                pb += ZP;
            }
            acc[k] = v;
        }
        __syncthreads();
    }
    // slices of a moment meet in shared memory; one partial per (component, block, moment)
    double* red = R;
#pragma unroll
    for (int k = 0; k < GMM_SLOTS; k++)
        if (t + 256 * k < NP * SL) red[t + 256 * k] = acc[k];
    __syncthreads();
    for (int pair = t; pair < NP; pair += 256) {
        double v = 0.0;
        for (int q = 0; q < SL; q++) v += red[q * NP + pair];
        const int c = pair / NACC, q = pair - c * NACC;
        part[((size_t)c * gridDim.x + blockIdx.x) * GMM_NACC_MAX + q] = v;
    }
}

__device__ void gmm_chol_dev(int d, const double* S, double* L) {
    for (int i = 0; i < d * d; i++) L[i] = 0.0;
    for (int i = 0; i < d; i++)
        for (int j = 0; j <= i; j++) {
            double s = S[i * d + j];
            for (int k = 0; k < j; k++) s = s - L[i * d + k] * L[j * d + k];
            L[i * d + j] = (i == j) ? sqrt(s) : s / L[j * d + j];
        }
}

__global__ void gmm_finish_kernel(IntegDev I, int a, const UpdScratch* __restrict__ us, const double* __restrict__ part, int blocks) {
    if (us->abort || us->n_valid == 0) return;
    const int d = I.gd, dt = I.d, C = I.n_gmm, c = threadIdx.x;
    const int nacc = 1 + dt + dt * (dt + 1) / 2;             // the moments kernel lays its accumulators out by the total dimension
    double* g = I.mem[a].gmm;
    double* omega = g;
    double* mu = omega + C;
    double* Sigma = mu + C * d;
    double* L = Sigma + C * d * d;
    __shared__ double s0s[16];
    __shared__ double tot_sh[16][GMM_NACC_MAX];
    // thread (component, accumulator) sums its column of the per-block partials in block order
    for (int e = threadIdx.x; e < C * nacc; e += blockDim.x) {
        const int cc = e / nacc, q = e - cc * nacc;
        double v = 0.0;
        for (int b = 0; b < blocks; b++) v += part[((size_t)cc * blocks + b) * GMM_NACC_MAX + q];
        tot_sh[cc][q] = v;
    }
    __syncthreads();
    double acc[GMM_NACC_MAX];
    if (c < C) {
        for (int q = 0; q < nacc; q++) acc[q] = tot_sh[c][q];
        s0s[c] = acc[0];
    }
    __syncthreads();
    double tot = 0.0;
    for (int q = 0; q < C; q++) tot += s0s[q];
    if (!(tot > 0.0) || c >= C) return;
    if (acc[0] > 1.0e-300) {
        double mean[ILE_MAX_D];
        for (int r = 0; r < d; r++) mean[r] = acc[1 + r] / acc[0];
        for (int r = 0; r < d; r++)
            for (int s = 0; s <= r; s++) {
                double v = acc[1 + dt + r * (r + 1) / 2 + s] / acc[0] - mean[r] * mean[s];
                if (r == s) {
                    const double rg = I.hi[I.gdim[r]] - I.lo[I.gdim[r]];
                    v = v + 1.0e-6 * (rg * rg);
                }
                Sigma[c * d * d + r * d + s] = v;
                Sigma[c * d * d + s * d + r] = v;
            }
        for (int r = 0; r < d; r++) mu[c * d + r] = mu[c * d + r] + mean[r];
    }
    omega[c] = acc[0] / tot;
    gmm_chol_dev(d, Sigma + c * d * d, L + c * d * d);
}

__global__ void gmm_chol_kernel(IntegDev I, int a) {
    const int d = I.gd, C = I.n_gmm, c = threadIdx.x;
    if (c >= C) return;
    double* Sigma = I.mem[a].gmm + C + C * d;
    gmm_chol_dev(d, Sigma + c * d * d, Sigma + C * d * d + c * d * d);
}

// ---------------------------------------------------------------- PORTFOLIO weights
__global__ void __launch_bounds__(256) port_ness_kernel(IntegDev I, const double* __restrict__ lnw, double* __restrict__ part) {
    const int a = blockIdx.y;
    const long long off = I.port->offset[a], cnt = (I.port->active[a] && !I.silent[a]) ? I.port->alloc[a] : 0;   // n_ESS of contributing members only
    double m = neg_inf(), s1 = 0.0, s2 = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < cnt; i += (long long)gridDim.x * blockDim.x) {
        const double v = lnw[off + i];
        if (!is_finite_d(v)) continue;
        if (v > m) {
            const double e = exp(m - v);
            s1 = s1 * e + 1.0;
            s2 = s2 * e * e + 1.0;
            m = v;
        } else {
            const double e = exp(v - m);
            s1 += e;
            s2 += e * e;
        }
    }
    __shared__ double sm[8], sa[8], sb[8];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const double wm = warp_max(m);
    const double sc = (m == neg_inf()) ? 0.0 : exp(m - wm);
    s1 = warp_sum(s1 * sc);
    s2 = warp_sum(s2 * sc * sc);
    if (lane == 0) { sm[w] = wm; sa[w] = s1; sb[w] = s2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double bm = neg_inf();
        for (int q = 0; q < 8; q++) bm = fmax(bm, sm[q]);
        double t1 = 0.0, t2 = 0.0;
        for (int q = 0; q < 8; q++)
            if (sm[q] != neg_inf()) {
                const double e = exp(sm[q] - bm);
                t1 += sa[q] * e;
                t2 += sb[q] * e * e;
            }
        double* o = part + ((size_t)a * gridDim.x + blockIdx.x) * 3;
        o[0] = bm; o[1] = t1; o[2] = t2;
    }
}

__global__ void port_weights_kernel(IntegDev I, const double* __restrict__ part, int blocks) {
    // one warp: the lanes share the per-block partials of a member, lane 0 then sets the weights
    PortState* P = I.port;
    const int Ns = I.n_members, lane = threadIdx.x;
    double ness[ILE_MAX_MEMBERS], tot = 0.0;
    for (int a = 0; a < Ns; a++) {
        double bm = neg_inf();
        for (int b = lane; b < blocks; b += 32) bm = fmax(bm, part[((size_t)a * blocks + b) * 3]);
        bm = warp_max(bm);
        double t1 = 0.0, t2 = 0.0;
        for (int b = lane; b < blocks; b += 32) {
            const double* o = part + ((size_t)a * blocks + b) * 3;
            if (o[0] == neg_inf()) continue;
            const double e = exp(o[0] - bm);
            t1 += o[1] * e;
            t2 += o[2] * e * e;
        }
        t1 = warp_sum(t1);
        t2 = warp_sum(t2);
        ness[a] = (bm == neg_inf() || !(t2 > 0.0)) ? 0.0 : t1 * t1 / t2;
        tot += ness[a];
    }
    if (lane) return;
    // members that are not activated are never trained; silent ones always are
    int n_con = 0;
    for (int a = 0; a < Ns; a++) {
        const bool con = P->active[a] && !I.silent[a];
        n_con += con;
        if (!P->active[a]) P->frozen[a] = 1;
        else if (!con) P->frozen[a] = 0;
    }
    if (!(tot > 0.0)) {
        P->restarted = 0;
        return;
    }
    double W[ILE_MAX_MEMBERS], ws = 0.0;
    for (int a = 0; a < Ns; a++) {
        const bool con = P->active[a] && !I.silent[a];
        if (!con) {
            W[a] = 0.0;
            continue;
        }
        const double raw = ness[a] / tot;
        // the batch after a restart was drawn with uniform weights (none below 5 %): nobody is frozen on it
        P->frozen[a] = (raw < 0.05 && !P->restarted) ? 1 : 0;
        W[a] = fmax(raw, 0.05 / (double)n_con);
        ws += W[a];
    }
    for (int a = 0; a < Ns; a++) P->W[a] = W[a] / ws;
    P->restarted = 0;
}

// ---------------------------------------------------------------- host: update dispatch
static int member_update(ile_integrator* it, int a, int N, const double* z, const double* lnw, const double* ln_ps, const int* skip) {
    ile_ctx* ctx = it->ctx;
    const IntegDev& I = it->I;
    const SamplerDev& S = I.mem[a];
    cudaStream_t st = ctx->stream;
    const int grid = ctx->sm_count * 8;
    switch (S.kind) {
        case ILE_KIND_UNIFORM:
            return ILE_OK;
        case ILE_KIND_AC: {
            upd_init_kernel<<<8, 256, 0, st>>>(it->us, skip, S.H, I.d * S.nb, nullptr);
            ILE_LAUNCH_CHECK(ctx);
            mask_max_kernel<<<grid, 256, 0, st>>>(I, N, z, lnw, nullptr, 0, it->us);
            ILE_LAUNCH_CHECK(ctx);
            ac_hist_kernel<<<grid, 256, (size_t)I.d * S.nb * 8, st>>>(I, a, N, z, lnw, it->us);
            ILE_LAUNCH_CHECK(ctx);
            ac_finish_kernel<<<I.d, 256, 0, st>>>(I, a, it->us);
            ILE_LAUNCH_CHECK(ctx);
            return ILE_OK;
        }
        case ILE_KIND_AV: {
            upd_init_kernel<<<8, 256, 0, st>>>(it->us, skip, nullptr, 0, it->sel_hist);
            ILE_LAUNCH_CHECK(ctx);
            mask_max_kernel<<<grid, 256, 0, st>>>(I, N, z, lnw, ln_ps, MASK_BOX | (ln_ps ? MASK_LNPS : 0), it->us);
            ILE_LAUNCH_CHECK(ctx);
            av_prepare_kernel<<<grid, 256, 0, st>>>(I, N, z, lnw, ln_ps, it->us, it->skey, it->q);
            ILE_LAUNCH_CHECK(ctx);
            av_sel_init_kernel<<<1, 32, 0, st>>>(I, it->us);
            ILE_LAUNCH_CHECK(ctx);
            for (int p = 0; p < AV_SEL_PASSES; p++) {
                av_sel_hist_kernel<<<grid, 256, 0, st>>>(N, it->skey, it->q, it->us, it->sel_hist);
                ILE_LAUNCH_CHECK(ctx);
            }
            av_decide_kernel<<<1, 32, 0, st>>>(I, N, it->us);
            ILE_LAUNCH_CHECK(ctx);
            av_stats_kernel<<<grid, 256, 0, st>>>(N, ln_ps, it->us, it->skey);
            ILE_LAUNCH_CHECK(ctx);
            av_nnew_kernel<<<1, 32, 0, st>>>(I, a, N, it->us, ln_ps ? 1 : 0);
            ILE_LAUNCH_CHECK(ctx);
            av_compact_kernel<<<grid, 256, 0, st>>>(I, N, z, it->us, it->skey, it->kbuf0);
            ILE_LAUNCH_CHECK(ctx);
            // the sort reads its element count and key width from the device (no host round-trip);
            // after an abort n_kept = 0, so it moves nothing
            int rc = radix_sort_device(ctx, (int)it->cap, &it->us->n_kept, &it->us->n_bits, (uint64_t*)it->kbuf0, nullptr, (uint64_t*)it->kbuf1, nullptr,
                                       it->sort_scratch, 8);
            if (rc) return rc;
            const int ub = (int)((it->cap + UQ_TILE - 1) / UQ_TILE);
            uniq_count_kernel<<<ub, 256, 0, st>>>(it->kbuf0, it->us, it->blk_count);
            ILE_LAUNCH_CHECK(ctx);
            uniq_scan_kernel<<<1, 1024, 0, st>>>(it->us, it->blk_count);
            ILE_LAUNCH_CHECK(ctx);
            uniq_write_kernel<<<ub, 256, 0, st>>>(it->kbuf0, it->us, it->blk_count, S.keys);
            ILE_LAUNCH_CHECK(ctx);
            av_commit_kernel<<<1, 32, 0, st>>>(I, a, it->us);
            ILE_LAUNCH_CHECK(ctx);
            return ILE_OK;
        }
        case ILE_KIND_GMM: {
            upd_init_kernel<<<8, 256, 0, st>>>(it->us, skip, nullptr, 0, nullptr);
            ILE_LAUNCH_CHECK(ctx);
            mask_max_kernel<<<grid, 256, 0, st>>>(I, N, z, lnw, nullptr, MASK_BOX, it->us);
            ILE_LAUNCH_CHECK(ctx);
            const size_t em_smem = ((size_t)GMS_DOUBLES + 256 * (17 + 10) + (size_t)I.n_gmm * 9 + 16) * sizeof(double);
            int per_sm = 1, em_blocks = it->gmm_blocks;
            switch (I.d) {
#define GMM_CASE(D)                                                                                                        \
    case D:                                                                                                                \
        ILE_CUDA(ctx, cudaFuncSetAttribute(gmm_em_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)em_smem)); \
        ILE_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gmm_em_kernel<D>, 256, em_smem));             \
        em_blocks = std::max(1, std::min(it->gmm_blocks, per_sm * ctx->sm_count));        /* one full wave, grid-stride */ \
        gmm_em_kernel<D><<<em_blocks, 256, em_smem, st>>>(I, a, N, z, lnw, it->us, it->gmm_part);                          \
        break;
                GMM_CASE(1) GMM_CASE(2) GMM_CASE(3) GMM_CASE(4) GMM_CASE(5) GMM_CASE(6) GMM_CASE(7) GMM_CASE(8)
#undef GMM_CASE
            }
            ILE_LAUNCH_CHECK(ctx);
            gmm_finish_kernel<<<1, 256, 0, st>>>(I, a, it->us, it->gmm_part, em_blocks);
            ILE_LAUNCH_CHECK(ctx);
            return ILE_OK;
        }
    }
    return ile_fail(ctx, ILE_EINVAL, "update: unknown member kind %d", S.kind);
}

int integ_gmm_refresh(ile_integrator* it, int a) {
    gmm_chol_kernel<<<1, 32, 0, it->ctx->stream>>>(it->I, a);
    ILE_LAUNCH_CHECK(it->ctx);
    return ILE_OK;
}

int integ_launch_update(ile_integrator* it, int N, const double* z, const double* lnw, const double* ln_ps) {
    ile_ctx* ctx = it->ctx;
    const IntegDev& I = it->I;
    if (I.n_members == 1) return member_update(it, 0, N, z, lnw, I.kind == ILE_KIND_PORTFOLIO ? nullptr : ln_ps, nullptr);
    // weights from the per-member n_ESS of the last batch; then every member that
    // is not frozen trains on all samples with the overall weights
    dim3 g(it->port_blocks, I.n_members);
    port_ness_kernel<<<g, 256, 0, ctx->stream>>>(I, lnw, it->port_part);
    ILE_LAUNCH_CHECK(ctx);
    port_weights_kernel<<<1, 32, 0, ctx->stream>>>(I, it->port_part, it->port_blocks);
    ILE_LAUNCH_CHECK(ctx);
    for (int a = 0; a < I.n_members; a++) {
        int rc = member_update(it, a, N, z, lnw, ln_ps, &I.port->frozen[a]);
        if (rc) return rc;
    }
    return ILE_OK;
}
