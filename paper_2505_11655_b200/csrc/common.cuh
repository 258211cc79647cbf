// Internal declarations shared by the translation units of libile (CUDA, sm_100a only).
// Nothing here is shared with oracle/ (the CPU oracle is independent numpy code).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <math.h>
#include "../../include/ile.h"

#define ILE_C_LIGHT 299792458.0
#define ILE_MAX_L 8
#define ILE_YLM_MAX_TERMS 12
#define ILE_TIMING_SLOTS 256
#define ILE_QT_ROW 48            // doubles per stored bin in the tiled Q layout (24 complex modes)

// ---------------------------------------------------------------- Ylm term table (device global)
// -2Y_lm(theta, phi) = e^{i m phi} * sum_t coef[t] * cos(theta/2)^pc[t] * sin(theta/2)^ps[t]
struct YlmMode {
    int m;
    int nterms;
    int pc[ILE_YLM_MAX_TERMS];
    int ps[ILE_YLM_MAX_TERMS];
    double coef[ILE_YLM_MAX_TERMS];
};
struct YlmTable {
    int M;
    int max_abs_m;
    int max_pow;
    int pad;
    YlmMode mode[ILE_MAX_M];
};

// ---------------------------------------------------------------- kernel parameter block (by value)
struct LnlParams {
    int K, M, N_Q, N_t, stride, interp, d, use_table;
    int box_trusted;              // 1: every sample of the batch lies in the prior box (the integrator drew it inside a box within it): no test
    int N_Qpad;                   // bins allocated per (p,k) in the tiled layout
    double fs, t_Q0, t_lo, dt, D_ref, gmst;
    double D[ILE_MAX_K][9];
    double pos[ILE_MAX_K][3];
    double lo[6], hi[6];          // prior box in z
    double ln_prior_const;        // -ln(2pi) - ln2 - ln(pi) - ln(2pi) - ln2
    double dist_norm;             // 3 / (D_max^3 - D_min^3)
    double ln_Nt;                 // ln N_t (time-marginalisation normaliser)
    // distance table
    int nA, nB;
    double A_lo, A_hi, B_lo, B_hi;
    const double* lnT;
    const double* lnT4;           // cells of the table, see ile_ctx
    // per intrinsic point data (already offset to point p)
    const double* Qc;             // [K][M][N_Q][2]
    const double* Qf;             // [K][N_Qpad/2][6][2][8] fragment-major: one 128-byte line per (bin pair, k-step pair)
    const double* U;              // [K][M][M][2]
    const double* V;              // [K][M][M][2]
    const YlmTable* ylm;
    // upper-triangle pair list (a <= b) and the matching packed matrices, Eq. 17-18:
    // UVp[pair][k] = w (Re U_ab, Im U_ab, Re V_ab, Im V_ab), w = 1 on the diagonal and 2 off it
    const int2* pairs;
    int n_pairs;
    const double* UVp;
    // signed 8-bit digits of Q for the tcgen05 contraction (lnl_split.cu): image of point p, groups of 8 bins per
    // detector, biased exponent of max |Q_k| (the integer scale is 2^(45 - (qeb - 1023)))
    const unsigned char* Qs;
    int NG8;
    int qeb[ILE_MAX_K];
    // step 4 in the tcgen05 kernel: the thread group (0..3) of a sample that walks row a of the upper triangle.  Groups
    // 0..K-1 also cut one detector's coefficients into digits, so they get fewer pairs (ile_fill_params balances the two)
    unsigned char tri_group[24];
};

struct ile_ctx {
    int device;
    cudaStream_t stream;
    char err[512];
    bool have_net, have_modes, have_quv, have_grid, have_prior;
    int K, M, P, N_Q, N_Qpad, quv_K, quv_M;
    double D[ILE_MAX_K][9], pos[ILE_MAX_K][3], gmst, max_delay;
    int ell[ILE_MAX_M], m[ILE_MAX_M];
    YlmTable h_ylm;
    YlmTable* d_ylm;
    double fs, t_Q0, D_ref;
    double *d_Qc, *d_Qf, *d_U, *d_V, *d_UVp;
    unsigned char* d_Qs;          // Q digits for the tcgen05 contraction, [P][K][NG8][2432 bytes]
    int* d_qeb;                   // [P][K] biased exponent of max |Q|
    unsigned int* d_qhi;          // scratch of the same size
    int* h_qeb;                   // host copy of d_qeb
    int2* d_pairs;
    int n_pairs;
    double t_lo, dt;
    int N_t, interp, stride;
    double D_min, D_max;
    int nA, nB;
    double A_lo, A_hi, B_lo, B_hi;
    double* d_lnT;
    double* d_lnT4;               // the same table as cells: [nB-1][nA-1][4] = (T[b][a], T[b][a+1], T[b+1][a], T[b+1][a+1]): one 32-byte read per bilinear lookup
    int variant;
    int ylm_max_pow, ylm_max_abs_m;   // sizes of the harmonics' power and phase tables (shared-memory scratch of the prep kernel)
    void* pc_buf;                 // scratch of ile_precompute_quv (grow-only, freed at destroy)
    size_t pc_bytes;
    int pc_W_nf;                 // N_f of the twiddle table held in pc_buf (0: none)
    int qf_valid;                 // d_Qf matches d_Qc
    int zbox_hint;                // set by the integrator around its own lnL call: the batch lies in [zbox_lo, zbox_hi)
    double zbox_lo[8], zbox_hi[8];
    int lnl_split;                // 1 (default): tcgen05 integer-digit fused kernel (lnl_split.cu) where the shape allows
    int sky_sort;                 // 1 (default): order samples by delay cell before the fused kernel
    int sm_count;
    // scratch
    void* d_scratch;
    size_t scratch_bytes;
    uint64_t launches;            // kernels launched so far (for bench's gpu_launches)
    // optional device timing of the fused lnL kernel (ile_kernel_timing): event pairs on the stream
    int timing_on;
    cudaEvent_t* tev;             // [2 * ILE_TIMING_SLOTS]
    int tev_used;
    double t_ms_total;
    uint64_t t_count;
};

int ile_fail(ile_ctx* ctx, int code, const char* fmt, ...);
int ile_scratch(ile_ctx* ctx, size_t bytes, void** out);
int ile_fill_params(ile_ctx* ctx, int p, int d, LnlParams* P);
int ile_launch_lnL_z(ile_ctx* ctx, int p, int N, int d, const double* z, const int* perm, double* lnL,
                     double* ln_prior);
int ile_launch_reduce(ile_ctx* ctx, int N, const double* lnw, ile_result* out_dev, int accumulate);
uint64_t ile_launch_count(ile_ctx* ctx);
// tcgen05 path (lnl_split.cu)
struct SpTile;
size_t ile_split_qs_bytes(int P, int K, int N_Q);
int ile_split_ng8(int N_Q);
int ile_split_build_q(ile_ctx* ctx, int P, int K, int M, int N_Q, const double* d_Qc, unsigned char* d_Qs, int* d_qeb, unsigned int* d_qhi);
bool ile_split_supported(const LnlParams& P);
int ile_split_cell_bits(int n_min, int n_max);
int ile_split_max_tiles(int N, int cell_bits, int K);
size_t ile_split_tile_bytes(int max_tiles);
int ile_launch_split_keys(ile_ctx* ctx, const LnlParams& P, int N, const double* z, int n_min, int cell_bits, unsigned long long* key,
                          unsigned int* val, double* rec, long long* n_dev, int* bits_dev, int* ntiles_dev);
size_t ile_split_rec_bytes(int N);
int ile_launch_split(ile_ctx* ctx, const LnlParams& P, int N, int n_min, int cell_bits, const unsigned long long* key, const double* rec,
                     const int* perm, double* lnL, double* ln_prior, int* tstart, SpTile* tiles, int* ntiles_dev);
int ile_timing_begin(ile_ctx* ctx);            // returns a slot (or -1 when timing is off)
void ile_timing_end(ile_ctx* ctx, int slot);
int ile_timing_drain(ile_ctx* ctx);

#define ILE_CUDA(ctx, call)                                                                   \
    do {                                                                                      \
        cudaError_t e__ = (call);                                                             \
        if (e__ != cudaSuccess)                                                               \
            return ile_fail((ctx), ILE_ECUDA, "%s failed: %s (%s:%d)", #call,                 \
                            cudaGetErrorString(e__), __FILE__, __LINE__);                     \
    } while (0)
#define ILE_LAUNCH_CHECK(ctx)                                                                 \
    do {                                                                                      \
        (ctx)->launches++;                                                                    \
        cudaError_t e__ = cudaGetLastError();                                                 \
        if (e__ != cudaSuccess)                                                               \
            return ile_fail((ctx), ILE_ECUDA, "kernel launch failed: %s (%s:%d)",             \
                            cudaGetErrorString(e__), __FILE__, __LINE__);                     \
    } while (0)

// ---------------------------------------------------------------- device helpers
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double neg_inf() { return __longlong_as_double(0xfff0000000000000LL); }
__device__ __forceinline__ double pos_inf() { return __longlong_as_double(0x7ff0000000000000LL); }
int ile_load_quv_impl(ile_ctx* ctx, int P, int N_Q, double fs, double t_Q0, const double* Q, const double* U, const double* V, double D_ref,
                      int src_is_device, bool trusted);
int ile_quv_alloc(ile_ctx* ctx, int P, int N_Q);
int ile_ensure_qf(ile_ctx* ctx);
