// rw_internal.h -- private declarations shared by the translation units of librw.so.
// Nothing here is visible through the C ABI (include/rw.h), and nothing under oracle/
// includes it.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/rw.h"

namespace rw {

// ---- basis / coefficient layout -----------------------------------------
// dsigma of Eq. (4) is quadratic in (g~L, g~R) per flavour and Eq. (8) is linear in mu_nu^2, so
//   S_theta(T_i) = sum_b c_b(theta) * Basis_b(T_i),   b = 0..9
//   b = 3a+0: g~L_a^2   b = 3a+1: g~R_a^2   b = 3a+2: g~L_a g~R_a   (a = e, mu, tau)   b = 9: mu_nu^2
// Row 10 carries coefficient 1 and holds N_mc in dead bins (S_SM = 0 => w := 1); row 11 is padding.
constexpr int kNumBasis = 10;
constexpr int kCoefStride = 12;   // doubles per point in coef[P][12] and rows per period in What[D][12][n_T]
constexpr int kNumTerms = 11;     // rows of What that are ever non-zero

// ---- DMMA contraction tile geometry (rw_fold_gemm.cu) ------------------------------------------
constexpr int kBM = 128;          // points per CTA tile
constexpr int kBN = 128;          // reconstructed bins per CTA tile
constexpr int kBK = 16;           // recoil bins per pipeline stage
constexpr int kStages = 6;
constexpr int kGemmConsumerWarps = 8;
constexpr int kGemmThreads = kGemmConsumerWarps * 32;

// ---- streaming fold geometry (rw_fold_stream.cu) -----------------------------------------------
constexpr int kStreamThreads = 256;
constexpr int kStreamCols = 2 * kStreamThreads;   // columns per CTA strip (one double2 per thread)
constexpr int kStreamMaxPB = 16;                  // points folded per pass over R

// ---- streaming DMMA fold geometry (rw_fold_ridge.cu) -------------------------------------------
constexpr int kRidgeCols = 256;                   // columns per strip (8 warps x 32)
constexpr int kRidgeMaxP = 64;                    // points per launch (tile heights 8, 16, 24, ... 64)
constexpr int kRidgePlanSMs = 148;                // B200: the stream-K grid is one wave of these SMs' slots

struct Consts {
    double sin2w, m_e, G_F, alpha;
    double C0;        // 2 G_F^2 m_e / pi        (Eq. 4 prefactor)
    double Cmm;       // pi alpha^2 / m_e^2      (Eq. 8 prefactor)
    double gL[3], gR[3];   // Eq. (2)-(3)
};

// Which parameter a column of param[P][k] holds (include/rw.h RW_EPS_EE_L ... RW_MU_NU); -1 = unused.
struct Kinds { int k; int kind[RW_N_KINDS]; };

struct Layout {           // byte offsets into the workspace (all 256-byte aligned)
    size_t E, fw, P3, T, Tmax_invE, N_mc, bkg, counts, R_copy;
    size_t basis, S_sm, What, sat_const, flag, G, ident, stream_cnt, strip_part, comp8, rate;
    size_t param_stage, coef, A_packed, partial, mu_part, out_stage, mu_stage, mu_tile, mu_prof;
    size_t B8, f_col8, e_row8, tau8, blk_hl8, blk_cm8, tau8b, comp8p;
    size_t gcol8, cert_part, bound_stage, fb_idx, coef_fb, rate_fb, out_fb;
    size_t pee_perm, pee_j0, pee_TmaxS, pee_fS, pee_rho, pee_Y;
    bool pee_scan;        // the sorted-grid suffix-sum tables of rw_eval_pee exist (3 (n_E + 1) doubles fit in shared memory)
    int KP512;            // n_T rounded up to 512 bins (staging chunk of k_slice_A)
    size_t total;
    int ldR;              // row pitch of the workspace copy of R (doubles)
    int KPAD;             // n_T rounded up to kBK
    int64_t A_pitch;      // doubles between consecutive 8-point row blocks of A_packed (>= 8 KPAD)
    int64_t MC;           // points per GEMM chunk (multiple of kBM)
    int n_tiles_n;        // ceil(n_rec / kBN)
    int stream_strips;    // ceil(n_rec / kStreamCols)
    int stream_splits;    // row splits of the streaming fold
    int ridge_strips;     // ceil(n_rec / kRidgeCols)
    int ridge_max_p;      // largest tile height of k_fold_ridge the slot scratch was sized for (16, 32 or 64)
    size_t ridge_cnt, ridge_part, ridge_slots, ridge_frag;
    bool sliced;          // RW_CREATE_SLICED: the INT8 slices of R are in the workspace
    int ns8;              // 8-bit balanced slices per operand: 8 when n_T <= 2048, else 7 (rw_api.cu plan())
    int KT8, NT8;         // k-blocks of 32 recoil bins; 64-column units = 2 x (128-column tiles) (rw_fold_i8.cu)
    int64_t prof_rows;    // points per pass of rw_eval_profile (rows of the mu scratch)
    int64_t pee_rows;     // points per pass of rw_eval_pee (rows of n_T weights the same scratch holds)
    int mu_tile_items;    // capacity of the split-K scratch in (tile, k-range) work items
    int ldG;              // row pitch of the prefolded templates G[D][12][ldG] (n_rec rounded up to even)
    int64_t max_batch;
    bool copy_R;
};

}  // namespace rw

struct rw_ctx {
    int n_E, n_T, n_rec, D;
    int n_comp;               // signal components (>= 1)
    double f_tau;             // tau share of 1 - P_e when no explicit P_mu / P_tau tables were given
    bool have_mu_tau;         // explicit P_mu / P_tau tables (then rw_eval_pee cannot split a per-point P_e)
    uint8_t *comp8;           // [n_T] component of every recoil bin (device); all zero when n_comp == 1
    double *rate;             // [max_batch][4] per-point rate scales of the components (k_coef)
    rw::Consts cst;
    rw::Layout lay;
    char *ws;                 // device workspace base
    // device tables
    double *E, *fw, *P3, *T, *Tmax_invE, *N_mc, *bkg, *counts;
    const double *R;          // [D][n_T][ldR]
    int ldR;
    size_t R_period_stride;   // doubles between periods
    double *basis, *S_sm, *What, *sat_const;
    int *stream_cnt;          // last-CTA-done tickets of the streaming fold: [D * strips] + 1, self-resetting
    int *ridge_cnt;           // tickets of k_fold_ridge: 2 x [D * ridge_strips] + 1
    double *ridge_part;       // [2 kRidgePlanSMs][64] Poisson sums per CTA of k_fold_ridge
    double *ridge_slots;      // [3 G][tile height][256] parked partial tiles of k_fold_ridge
    double *ridge_frag;       // N' as DMMA fragments for its tile heights 32 and 64 (k_ridge_frag)
    double *strip_part;       // [D * strips][16] Poisson sums per column strip
    double *G, *ident;        // prefolded templates [D][12][ldG]; identity coefficients [16][12] used to fold them
    int *flag;
    // per-call scratch
    double *param_stage, *coef, *A_packed, *partial, *mu_part, *out_stage, *mu_stage;
    uint8_t *B8;              // [D][NT8 / 2][KT8][ns8 slices][4 KB] INT8 slices of R (RW_CREATE_SLICED)
    int *f_col8, *e_row8;     // column exponents [D][n_rec]; row exponents of the current chunk [MC]
    int *tau8;                // [D][n_T] per-bin rescaling exponents (2^tau ~ N_mc)
    double *blk_hl8;          // [D][2: hi, lo][11][KT8] block-wise max / min of W^_b 2^-tau (row-exponent bound)
    int *blk_cm8;             // [KT8] components present in each 32-bin block
    int8_t *tau8b;            // [D][KP512] tau as bytes, zero-padded (cp.async staging of k_slice_A)
    uint8_t *comp8p;          // [KP512] comp8, zero-padded
    int *pee_perm, *pee_j0;   // flux grid sorted by T_max; first sorted entry that passes the cut, per recoil bin
    double *pee_TmaxS, *pee_fS, *pee_rho, *pee_Y;   // sorted T_max; f E^-n [n_comp][3][n_E]; rho [n_comp][2][n_E]; totals [n_comp][9][n_E + 1]
    double *gcol8;            // [D][2: full, fast][n_rec] certificate constants g_k of the sliced contraction
    double *cert_part;        // [D][NT8][MC] certified relative error per (half tile, point)
    double *bound_stage;      // [max_batch] certified bound per point of a slice (strict mode without a caller array)
    int *fb_idx;              // [MC] + 1: uncertified points of a chunk (ascending), then their count
    double *coef_fb, *rate_fb, *out_fb;   // [MC][12], [MC][4], [MC]: their coefficient rows / recomputed values
    double *mu_prof;          // rw_eval_profile scratch: mu[prof_rows][D][n_rec]
    double *mu_tile;          // split-K scratch: [mu_tile_items][<=128][128] parked accumulators
    CUtensorMap *tmapR;       // host array [D]
    CUtensorMap tmapA[4];     // N' maps for tile heights 16, 32, 64, 128
    int num_sms;
    int64_t launches;
    int64_t strict_fallbacks; // points recomputed by the DMMA path in strict sliced calls so far
    // measurement hooks (rw_profile_begin/end)
    cudaEvent_t *prof_ev;     // pairs: [2q] before, [2q+1] after fold launch q
    int prof_cap, prof_n;     // pairs allocated / recorded
    bool profiling;
    char err[512];
};

namespace rw {

// error helpers -----------------------------------------------------------------------------------
int fail(rw_ctx *ctx, int status, const char *fmt, ...);
#define RW_CUDA(ctx, call)                                                                   \
    do {                                                                                     \
        cudaError_t e__ = (call);                                                            \
        if (e__ != cudaSuccess)                                                              \
            return rw::fail((ctx), RW_ERR_CUDA, "%s failed: %s (%s:%d)", #call,              \
                            cudaGetErrorString(e__), __FILE__, __LINE__);                    \
    } while (0)

// kernels' host launchers (each returns a cudaError_t from the launch) ---------------------------
cudaError_t launch_setup(rw_ctx *ctx, cudaStream_t s);                       // rw_setup.cu
cudaError_t launch_sat_const(rw_ctx *ctx, cudaStream_t s);                   // rw_setup.cu
cudaError_t launch_validate_counts(rw_ctx *ctx, const double *counts_dev, cudaStream_t s);   // rw_setup.cu
cudaError_t launch_comp8(rw_ctx *ctx, const int32_t *comp_dev, cudaStream_t s);   // rw_setup.cu
cudaError_t launch_validate_device(rw_ctx *ctx, const double *R_src, int ld_src,
                                   size_t period_stride_src, cudaStream_t s); // rw_setup.cu
cudaError_t launch_flavour(rw_ctx *ctx, int have_mu_tau, double f_tau, cudaStream_t s);  // rw_setup.cu
cudaError_t launch_coef(rw_ctx *ctx, const double *param, int64_t P, int k, const int *kinds,
                        cudaStream_t s);                                     // rw_coef.cu
cudaError_t launch_gen_A(rw_ctx *ctx, int d, int64_t p0, int64_t Pc, cudaStream_t s);   // rw_coef.cu
cudaError_t launch_fold_gemm(rw_ctx *ctx, int d, int64_t Pc, double *out_mu, int64_t mu_p0,
                             cudaStream_t s);                                // rw_fold_gemm.cu
// One launch: fold + Poisson terms + final sum for Pb <= 16 points given by coefficients `coef`, raw parameters
// `param` (+ kinds; step a1 then runs inside the kernel) or caller weights `wts`.  out == NULL: fold only (prefold).
cudaError_t launch_fold_stream(rw_ctx *ctx, const double *coef, const double *param, const Kinds *kd,
                               const double *wts, int Pb, double *out, bool full_eq18, double *out_mu,
                               cudaStream_t s, const double *rate_rows = nullptr);   // rw_fold_stream.cu
// The same contract for Pb <= 64 points on the streaming DMMA kernel (rw_fold_ridge.cu); out must not be NULL.
cudaError_t launch_fold_ridge(rw_ctx *ctx, const double *coef, const double *param, const Kinds *kd,
                              const double *wts, int Pb, double *out, bool full_eq18, double *out_mu,
                              cudaStream_t s);                               // rw_fold_ridge.cu
// Grid (CTAs) of k_fold_ridge for tile height 8 << mb_log2 and the number of row blocks per strip.  Host arithmetic only.
int ridge_grid(int n_T, int n_rec, int D, int mb_log2, int num_sms, int *nblk_out);         // rw_fold_ridge.cu
cudaError_t launch_gen_A_weights(rw_ctx *ctx, int d, const double *w, int64_t Pc, cudaStream_t s);  // rw_coef.cu
cudaError_t launch_prefold(rw_ctx *ctx, cudaStream_t s);                     // rw_collapsed.cu
cudaError_t launch_profile(rw_ctx *ctx, const double *mu_rows, int64_t rows, double s0, double sigma,
                           bool full_eq18, double *out, double *out_scale, cudaStream_t s);   // rw_profile.cu
int profile_setup(rw_ctx *ctx);                                              // rw_profile.cu
cudaError_t launch_weights_pee(rw_ctx *ctx, const double *P_e_pts, int64_t Pq, double *w, cudaStream_t s);  // rw_pee.cu
cudaError_t launch_coef_grad(rw_ctx *ctx, const double *param, int64_t P, int k, const int *kinds,
                             cudaStream_t s, bool split = false);            // rw_grad.cu
cudaError_t launch_grad(rw_ctx *ctx, const double *rows, int64_t P, int k, bool full_eq18, double *out,
                        double *grad, cudaStream_t s, bool split = false);   // rw_grad.cu
int pee_setup(rw_ctx *ctx, cudaStream_t s);                                  // rw_pee.cu
int i8_setup(rw_ctx *ctx, cudaStream_t s);                                   // rw_fold_i8.cu
cudaError_t launch_fold_i8(rw_ctx *ctx, int d, int64_t p0, int64_t Pc, double *out_mu, cudaStream_t s,
                           const double *w = nullptr, bool fast = false, bool certify = false);    // rw_fold_i8.cu
cudaError_t launch_reduce_max(rw_ctx *ctx, int n_parts, int64_t part_stride, int64_t Pc, double *bound,
                              cudaStream_t s);                               // rw_fold_stream.cu
cudaError_t launch_collect_uncertified(rw_ctx *ctx, const double *bound, int64_t Ps, double tol, bool gather, cudaStream_t s);   // rw_fold_stream.cu
cudaError_t launch_scatter_fallback(rw_ctx *ctx, int n, double *out, double *bound, cudaStream_t s);               // rw_fold_stream.cu
cudaError_t launch_collapsed(rw_ctx *ctx, int64_t p0, int64_t Pc, double *out_mu,
                             cudaStream_t s);                                // rw_collapsed.cu
cudaError_t launch_reduce(rw_ctx *ctx, int n_parts, int64_t part_stride, int64_t Pc, double *out,
                          bool full_eq18, cudaStream_t s);                   // rw_fold_stream.cu
int make_tensor_maps(rw_ctx *ctx);                                           // rw_fold_gemm.cu
int ridge_setup(rw_ctx *ctx);                                                // rw_fold_ridge.cu
int gemm_rows_per_warp_block(int64_t Pc);                                    // rw_fold_gemm.cu
int gemm_tail_split(int tail, int num_sms, int k_iters, int max_items);      // rw_fold_gemm.cu

// Brackets one fold-kernel launch with CUDA events while profiling is on (rw_api.cu).
struct ProfScope {
    rw_ctx *ctx; cudaStream_t s; bool on;
    ProfScope(rw_ctx *c, cudaStream_t st) : ctx(c), s(st), on(c->profiling && c->prof_n < c->prof_cap)
    {
        if (on) cudaEventRecord(ctx->prof_ev[2 * ctx->prof_n], s);
    }
    ~ProfScope()
    {
        if (on) { cudaEventRecord(ctx->prof_ev[2 * ctx->prof_n + 1], s); ctx->prof_n++; }
    }
};

// Step a1 for one point: g~ = g + eps (Eq. 6), then the monomials the cross section is polynomial
// in: g~L^2, g~R^2, g~L g~R per flavour (Eq. 4/7) and mu_nu^2 (Eq. 8-9).
// c[10] = 1 multiplies the dead-bin row of W^, c[11] = 0 is padding.
// r[c] = rate scale of signal component c (rate_k of Eq. 17; 1 when not scanned).
__device__ __forceinline__ void coef_from_param(const double *__restrict__ prow, const Kinds &kd, const Consts &cst,
                                                double *c /*[12]*/, double *r /*[4]*/)
{
#pragma unroll
    for (int q = 0; q < RW_MAX_COMPONENTS; ++q) r[q] = 1.0;
    for (int a = 0; a < kd.k; ++a) {
#pragma unroll
        for (int q = 0; q < RW_MAX_COMPONENTS; ++q)
            if (kd.kind[a] == RW_RATE_0 + q) r[q] = prow[a];
    }
    double th[RW_RATE_0];
#pragma unroll
    for (int q = 0; q < RW_RATE_0; ++q) th[q] = 0.0;
    for (int a = 0; a < kd.k; ++a) {
        const double v = prow[a];
#pragma unroll
        for (int q = 0; q < RW_RATE_0; ++q)
            if (kd.kind[a] == q) th[q] = v;
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double gl = cst.gL[a] + th[2 * a], gr = cst.gR[a] + th[2 * a + 1];
        c[3 * a + 0] = gl * gl;
        c[3 * a + 1] = gr * gr;
        c[3 * a + 2] = gl * gr;
    }
    c[9] = th[RW_MU_NU] * th[RW_MU_NU];
    c[10] = 1.0;
    c[11] = 0.0;
}

// Poisson term of Eq. (18) relative to its saturated value: mu - n + n ln(n/mu) (x2 applied later).
__device__ __forceinline__ double poisson_term(double mu, double n)
{
    if (n > 0.0) {
        if (mu > 0.0) {
            double d = mu - n;
            return d - n * log1p(d / n);
        }
        return (mu == mu) ? __longlong_as_double(0x7ff0000000000000LL) : mu;   // +inf, NaN stays NaN
    }
    return mu;
}

// Poisson term with the reciprocal count precomputed (inv = 1/n for n > 0, else 0): no division per bin.
// mu == 0 < n must give +inf (n * fl(1/n) is not always exactly 1, so log1p would see -1 + ulp), NaN stays NaN.
__device__ __forceinline__ double poisson_term_inv(double mu, double n, double inv)
{
    const double d = mu - n;
    double t = d - n * log1p(d * inv);
    if (!(mu > 0.0) && n > 0.0) t = (mu == mu) ? __longlong_as_double(0x7ff0000000000000LL) : mu;
    return t;
}

// Sum of four Poisson terms with the reciprocal counts precomputed (inv = 1/n for n > 0, 0 for n == 0):
//   d = mu - n,  term = d - n log1p(d inv)      (n == 0: term = mu;  mu == 0 < n: +inf;  NaN stays NaN)
// Deliberately NOT inlined: the contraction's epilogue evaluates 64 terms per thread, and 64 inlined copies of
// log1p were 11k instructions that missed the instruction cache (4 % of the kernel at N_T = 16384, 14 % at
// 4096).  One copy per kernel, four independent chains per call.
static __device__ __noinline__ double poisson_sum4(double m0, double m1, double m2, double m3,
                                                   double n0, double n1, double n2, double n3,
                                                   double i0, double i1, double i2, double i3)
{
    const double t0 = poisson_term_inv(m0, n0, i0), t1 = poisson_term_inv(m1, n1, i1);
    const double t2 = poisson_term_inv(m2, n2, i2), t3 = poisson_term_inv(m3, n3, i3);
    return (t0 + t1) + (t2 + t3);
}

}  // namespace rw
