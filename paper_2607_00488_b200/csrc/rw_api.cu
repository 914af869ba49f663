// rw_api.cu -- the C ABI of include/rw.h: validation, workspace planning, table placement and
// the stream-ordered launch sequence of one rw_eval_batch.  No arithmetic of the method lives
// here; every step of the path runs in the kernels of rw_setup/rw_coef/rw_fold_*.cu.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "rw_internal.h"

namespace rw {

static thread_local char g_create_err[512] = "";

int fail(rw_ctx *ctx, int status, const char *fmt, ...)
{
    char *dst = ctx ? ctx->err : g_create_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    if (ctx) memcpy(g_create_err, ctx->err, 512);
    return status;
}

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

constexpr int kPlanSMs = 148;            // B200; only used to size the streaming-fold row split
constexpr int64_t kMaxChunkRows = 32768;             // points per contraction chunk
constexpr int64_t kMaxChunkBytes = (int64_t)4 << 30;  // ... and A_packed <= 4 GiB: 180 GB of HBM make large
                                                      // chunks cheap, and the last wave of a launch is <0.5%

static int plan(const rw_inputs *in, int64_t max_batch, Layout *L)
{
    if (!in || !L) return RW_ERR_INVALID;
    if (in->n_E <= 0 || in->n_T <= 0 || in->n_rec <= 0 || in->n_periods <= 0 || max_batch <= 0)
        return RW_ERR_INVALID;
    if (in->mem_kind != RW_MEM_HOST && in->mem_kind != RW_MEM_DEVICE) return RW_ERR_INVALID;
    const size_t n_E = in->n_E, n_T = in->n_T, n_rec = in->n_rec, D = in->n_periods;
    if (in->n_comp < 0 || in->n_comp > RW_MAX_COMPONENTS) return RW_ERR_INVALID;
    const size_t n_comp = in->n_comp > 1 ? in->n_comp : 1;
    memset(L, 0, sizeof(*L));
    L->max_batch = max_batch;
    L->copy_R = (in->mem_kind == RW_MEM_HOST) || (n_rec & 1);
    L->ldR = L->copy_R ? (int)((n_rec + 1) & ~(size_t)1) : (int)n_rec;
    L->KPAD = (int)((n_T + 31) / 32 * 32);      // k-stages of 16 (DMMA) and 32 (INT8 slices) both divide it
    L->A_pitch = (int64_t)L->KPAD * 8;
    L->sliced = (in->create_flags & (RW_CREATE_SLICED | RW_CREATE_FP32)) != 0;     // RW_FP32 runs on the same slices
    L->KT8 = (int)((n_T + 31) / 32);
    // 8 slices (63 bits) are exact in int32 up to n_T = 8192; they are used where the contraction is too short for
    // the tensor pipe to matter.  Beyond, 7 slices (55 bits, 28 instead of 36 products): measured 5e-15 .. 1.2e-13 of mu
    // on configs 3-5 against the 1e-12 bar.
    L->ns8 = (n_T <= 2048) ? 8 : 7;
    L->NT8 = 2 * (int)((n_rec + 127) / 128);     // 64-column units (one epilogue warp set each); tiles are 128 wide
    int64_t cap = kMaxChunkBytes / (L->A_pitch) / kBM * kBM;
    if (cap < kBM) cap = kBM;
    if (cap > kMaxChunkRows) cap = kMaxChunkRows;
    int64_t mc = (max_batch + kBM - 1) / kBM * kBM;
    L->MC = mc < cap ? mc : cap;
    L->n_tiles_n = (int)((n_rec + kBN - 1) / kBN);
    L->stream_strips = (int)((n_rec + kStreamCols - 1) / kStreamCols);
    int splits = (int)((kPlanSMs * 4 + L->stream_strips * D - 1) / (L->stream_strips * D));
    int max_splits = (int)((n_T + 63) / 64);
    if (splits > max_splits) splits = max_splits;
    if (splits < 1) splits = 1;
    L->stream_splits = splits;
    L->ridge_strips = (int)((n_rec + kRidgeCols - 1) / kRidgeCols);
    L->ridge_max_p = max_batch <= 16 ? 16 : max_batch <= 32 ? 32 : kRidgeMaxP;
    size_t ridge_slot_bytes = 0;         // 3 parked partial tiles per CTA, largest variant
    for (int v = 0; (8 << v) <= L->ridge_max_p; ++v) {
        const size_t b = (size_t)3 * ridge_grid((int)n_T, (int)n_rec, (int)D, v, kRidgePlanSMs, nullptr) * (8u << v) * kRidgeCols * 8;
        if (b > ridge_slot_bytes) ridge_slot_bytes = b;
    }
    const size_t nstrip2 = (n_rec + 255) / 256;
    const size_t mu_ld = (n_rec + 1) & ~(size_t)1;

    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align256(off + bytes); return o; };
    L->E = take(n_E * 8);
    L->fw = take(n_comp * n_E * 8);
    L->P3 = take(n_comp * 3 * n_E * 8);
    L->comp8 = take(n_T);
    L->rate = take((size_t)max_batch * RW_MAX_COMPONENTS * 8);
    L->T = take(n_T * 8);
    L->Tmax_invE = take(3 * n_E * 8);
    L->N_mc = take(D * n_T * 8);
    L->bkg = take(D * n_rec * 8);
    L->counts = take(D * n_rec * 8);
    L->R_copy = take(L->copy_R ? D * n_T * (size_t)L->ldR * 8 : 0);
    L->basis = take(kNumBasis * n_T * 8);
    L->S_sm = take(n_T * 8);
    L->What = take(D * kCoefStride * n_T * 8);
    L->sat_const = take(8);
    L->flag = take(4);
    L->ldG = (int)mu_ld;
    L->G = take(D * n_comp * kCoefStride * mu_ld * 8);              // templates [D][n_comp][12][ldG]
    L->stream_cnt = take((D * (size_t)L->stream_strips + 1) * 4);
    L->strip_part = take(D * (size_t)L->stream_strips * kStreamMaxPB * 8);
    L->ident = take(kStreamMaxPB * (kCoefStride + RW_MAX_COMPONENTS) * 8);     // unit coefficient rows + one rate row set
    L->param_stage = take((size_t)max_batch * RW_N_KINDS * 8);
    L->coef = take((size_t)max_batch * kCoefStride * 8);
    L->A_packed = take((size_t)(L->MC / 8) * L->A_pitch * 8);
    size_t part_gemm = D * (size_t)(L->sliced ? L->NT8 : L->n_tiles_n) * L->MC, part_stream = D * nstrip2 * kStreamMaxPB;
    L->partial = take((part_gemm > part_stream ? part_gemm : part_stream) * 8);
    L->mu_part = take(D * (size_t)(max_splits < splits ? max_splits : splits) * kStreamMaxPB * mu_ld * 8);
    L->ridge_slots = take(ridge_slot_bytes);
    L->ridge_cnt = take((2 * D * (size_t)L->ridge_strips + 1) * 4);
    L->ridge_part = take((size_t)2 * kRidgePlanSMs * kRidgeMaxP * 8);
    // N' in fragment order for the ridge kernel's tile heights 32 and 64: [D][n_T / 8 + 8 blocks][points / 8][32] x 16 B
    L->ridge_frag = take(L->ridge_max_p >= 32 ? D * ((n_T + 7) / 8 + 8) * (size_t)(L->ridge_max_p / 8) * 512 : 0);
    L->out_stage = take((size_t)max_batch * 8);
    {   // split-K scratch: at most 8 work items per SM, and never more than 16 k-ranges of every 16-point tile
        int64_t items = (int64_t)L->n_tiles_n * ((L->MC + 15) / 16) * 16;
        if (items > 8 * kPlanSMs) items = 8 * kPlanSMs;
        L->mu_tile_items = (int)items;
        L->mu_tile = take((size_t)items * kBM * kBN * 8);
    }
    {   // rw_eval_profile scratch: mu of one pass, about 256 MB (at least 128 points, at most max_batch); rw_eval_pee
        // keeps the weights w[pee_rows][n_T] of a pass in the same scratch, so it also holds min(max_batch, those
        // rows) rows of n_T doubles (a context made for single evaluations, max_batch = 1, can still call it)
        int64_t rows = ((int64_t)256 << 20) / (int64_t)(D * n_rec * 8);
        if (rows < 128) rows = 128;
        if (rows > max_batch) rows = max_batch;
        L->prof_rows = rows;
        size_t doubles = (size_t)rows * D * n_rec;
        if (doubles < (size_t)rows * n_T) doubles = (size_t)rows * n_T;
        int64_t pr = (int64_t)(doubles / n_T);
        L->pee_rows = pr < max_batch ? pr : max_batch;
        L->mu_prof = take(doubles * 8);
    }
    L->B8 = take(L->sliced ? D * (size_t)L->NT8 * L->KT8 * 16384 : 0);
    L->f_col8 = take(L->sliced ? D * n_rec * 4 : 0);
    L->e_row8 = take(L->sliced ? (size_t)L->MC * 4 : 0);
    L->tau8 = take(L->sliced ? D * n_T * 4 : 0);
    L->blk_hl8 = take(L->sliced ? D * 2 * (size_t)kNumTerms * L->KT8 * 8 : 0);
    L->blk_cm8 = take(L->sliced ? (size_t)L->KT8 * 4 : 0);
    L->KP512 = (int)((n_T + 511) / 512 * 512);
    L->tau8b = take(L->sliced ? D * (size_t)L->KP512 : 0);
    L->comp8p = take(L->sliced ? (size_t)L->KP512 : 0);
    L->pee_scan = 3 * (n_E + 1) * 8 <= (size_t)200 << 10;
    L->pee_perm = take(L->pee_scan ? n_E * 4 : 0);
    L->pee_j0 = take(L->pee_scan ? n_T * 4 : 0);
    L->pee_TmaxS = take(L->pee_scan ? n_E * 8 : 0);
    L->pee_fS = take(L->pee_scan ? n_comp * 3 * n_E * 8 : 0);
    L->pee_rho = take(L->pee_scan ? n_comp * 2 * n_E * 8 : 0);
    L->pee_Y = take(L->pee_scan ? n_comp * 9 * (n_E + 1) * 8 : 0);
    L->gcol8 = take(L->sliced ? D * 2 * n_rec * 8 : 0);
    L->cert_part = take(L->sliced ? D * (size_t)L->NT8 * L->MC * 8 : 0);
    L->bound_stage = take(L->sliced ? (size_t)max_batch * 8 : 0);
    L->fb_idx = take(L->sliced ? ((size_t)L->MC + 1) * 4 : 0);
    L->coef_fb = take(L->sliced ? (size_t)L->MC * kCoefStride * 8 : 0);
    L->rate_fb = take(L->sliced ? (size_t)L->MC * RW_MAX_COMPONENTS * 8 : 0);
    L->out_fb = take(L->sliced ? (size_t)L->MC * 8 : 0);
    L->total = off;
    return RW_OK;
}

static bool host_bad_nonneg(const double *x, size_t n)
{
    for (size_t q = 0; q < n; ++q)
        if (!(x[q] >= 0.0) || isinf(x[q])) return true;
    return false;
}
static bool host_bad_pos(const double *x, size_t n)
{
    for (size_t q = 0; q < n; ++q)
        if (!(x[q] > 0.0) || isinf(x[q])) return true;
    return false;
}
static bool host_bad_prob(const double *x, size_t n)
{
    for (size_t q = 0; q < n; ++q)
        if (!(x[q] >= 0.0 && x[q] <= 1.0)) return true;
    return false;
}

static const char *flag_message(int f)
{
    if (f & 1) return "E_MeV must be finite and > 0";
    if (f & 2) return "flux_w must be finite and >= 0";
    if (f & 4) return "P_e/P_mu/P_tau must lie in [0,1]";
    if (f & 8) return "T_MeV must be finite and > 0 (PAPER.md:108)";
    if (f & 16) return "N_mc must be finite and >= 0";
    if (f & 32) return "bkg must be finite and >= 0";
    if (f & 64) return "counts must be finite and >= 0";
    if (f & 128) return "R must be finite and >= 0";
    if (f & 256) return "comp_of_T must lie in [0, n_comp)";
    return "invalid input";
}

// RW_MODE_AUTO (measured on B200, config-4 size): one point -> the one-launch HBM-streaming kernel; 2..64 points ->
// the streaming DMMA kernel (R read once at HBM speed, contraction on the FP64 tensor cores; one launch up to 16
// points, N' from k_ridge_frag above: 64 points 0.536 ms against 0.574 ms for the tiled contraction); beyond -> the
// tiled DMMA contraction (tile height 128, split-K).  The opt-in contractions (prec != 0) replace the last two.
constexpr int kAutoRidgeMax = 64;
constexpr int kAutoTailRows = 96;        // left-over points of a batch (P mod 128) that go to the ridge kernel in RW_MODE_AUTO
constexpr int64_t kAutoTailMax = 16384;  // ... for batches up to this size (beyond, one more row of tiles is < 1 %)
static bool auto_stream(const rw_ctx *, int64_t P, int prec) { return prec == 0 ? P <= 1 : P <= 4; }
static bool use_stream(const rw_ctx *ctx, uint32_t mode, int64_t P, int prec)
{
    return mode == RW_MODE_STREAM || (mode == RW_MODE_AUTO && auto_stream(ctx, P, prec));
}
static bool use_ridge(const rw_ctx *ctx, uint32_t mode, int64_t P, int prec)
{
    return mode == RW_MODE_RIDGE || (mode == RW_MODE_AUTO && prec == 0 && !auto_stream(ctx, P, prec) && P <= kAutoRidgeMax);
}

// Points of the next call of the streaming DMMA kernel when `rem` are left.  Its time follows the tile height (a
// multiple of 8 points) but never drops below one pass over R (config 4: 0.18 / 0.22 / 0.27 / 0.34 / 0.40 / 0.47 /
// 0.53 ms for <= 16 / 24 / 32 / 40 / 48 / 56 / 64 points), so when two calls are left they share the points evenly
// instead of 64 + rest: 65 points = 40 + 25 (0.34 + 0.27 ms) rather than 64 + 1 (0.53 + 0.18 ms).
static int ridge_group(int64_t rem, int max_p)
{
    if (rem <= max_p) return (int)rem;
    if (rem > 2 * (int64_t)max_p) return max_p;
    const int half = (int)(((rem + 1) / 2 + 7) / 8 * 8);
    return half < max_p ? half : max_p;
}

// RW_MODE_AUTO, FP64, beyond 64 points: the number of left-over points (P mod 128, at most 96) that go through the
// streaming DMMA kernel instead of a partly filled row of tiles, or 0.  The tiled contraction works in rows of 128
// points and a partly filled last row costs as much as a full one (config-4 size: 1.07 ms per row; 192 points 2.02 ms,
// 65 points 1.07 ms); the ridge kernel does <= 16 / 32 / 64 points in 0.18 / 0.27 / 0.53 ms there (192 points 1.60 ms,
// 65 points 0.71 ms).  Scans of "a few hundred" points are the paper's own use.
// Where it pays (measured, never a loss from 1000 x 500 to 16384 x 8192): responses large enough that a row of tiles is
// a sizeable part of a wave of the machine (n_T n_rec >= 4e7 per period: config-4 class), and any batch of <= 256 points
// unless the response is so small that the call is bound by its launches (n_T n_rec D < 4e6: config 2 and below).
static int64_t auto_tail(const rw_ctx *ctx, uint32_t mode, int64_t P, int prec)
{
    const Layout &L = ctx->lay;
    if (mode != RW_MODE_AUTO || prec != 0 || P <= kAutoRidgeMax || L.ridge_max_p < kRidgeMaxP) return 0;
    const double cells = (double)ctx->n_T * (double)ctx->n_rec;
    const bool pays = (P <= kAutoTailMax && cells >= 4e7) || (P <= 256 && cells * ctx->D >= 4e6);
    const int64_t rem = P % kBM;
    return (pays && rem <= kAutoTailRows) ? rem : 0;
}

// Options of the sliced contraction (prec 2 / 3): tol > 0 = strict (RW_SLICED_STRICT, RW_FP32): a point whose certified
// relative error exceeds tol is recomputed by the FP64 DMMA path; bound = device array [Ps] that receives the certified
// bound of every point (0 for points that went through an FP64 path), or NULL.
struct SlicedOpt { double tol = 0.0; double *bound = nullptr; };

// Steps a2-a4 for the Ps <= max_batch points whose coefficients are in ctx->coef: -2lnL -> dout[Ps], and mu ->
// out_mu[Ps][D][n_rec] when asked.
// prec: 0 = FP64 DMMA, 2 = INT8 slices (RW_SLICED), 3 = their top four (RW_SLICED_FAST, RW_FP32); only the contraction
// regime differs
static int fold_slice(rw_ctx *ctx, int64_t Ps, uint32_t mode, bool full, double *dout, double *out_mu, cudaStream_t s,
                      int prec = 0, const SlicedOpt &opt = SlicedOpt())
{
    const Layout &L = ctx->lay;
    const int D = ctx->D, n_rec = ctx->n_rec;
    const bool stream_mode = use_stream(ctx, mode, Ps, prec);
    const bool contraction = mode != RW_MODE_COLLAPSED && !stream_mode && !use_ridge(ctx, mode, Ps, prec);
    if (opt.bound && !(contraction && prec >= 2))                  // every other regime is an FP64 path
        RW_CUDA(ctx, cudaMemsetAsync(opt.bound, 0, (size_t)Ps * 8, s));
    if (const int64_t rem = contraction ? auto_tail(ctx, mode, Ps, prec) : 0) {
        const int64_t main = Ps - rem;
        if (main > 0) {
            const int rc = fold_slice(ctx, main, RW_MODE_GEMM, full, dout, out_mu, s, 0, opt);
            if (rc != RW_OK) return rc;
        }
        for (int64_t g0 = main, step = 0; g0 < Ps; g0 += step) {
            const int Pb = ridge_group(Ps - g0, L.ridge_max_p);
            step = Pb;
            double *mu = out_mu ? out_mu + (size_t)g0 * D * n_rec : nullptr;
            RW_CUDA(ctx, launch_fold_ridge(ctx, ctx->coef + g0 * kCoefStride, nullptr, nullptr, nullptr, Pb,
                                           dout + g0, full, mu, s));
        }
        return RW_OK;
    }
    if (mode == RW_MODE_COLLAPSED) {
        const int nstrip = (n_rec + 511) / 512;
        for (int64_t c0 = 0; c0 < Ps; c0 += L.MC) {
            const int64_t Pc = (Ps - c0 < L.MC) ? Ps - c0 : L.MC;
            double *mu = out_mu ? out_mu + (size_t)c0 * D * n_rec : nullptr;
            RW_CUDA(ctx, launch_collapsed(ctx, c0, Pc, mu, s));
            RW_CUDA(ctx, launch_reduce(ctx, D * nstrip, L.MC, Pc, dout + c0, full, s));
        }
    } else if (stream_mode) {
        for (int64_t g0 = 0; g0 < Ps; g0 += kStreamMaxPB) {
            const int Pb = (int)((Ps - g0 < kStreamMaxPB) ? Ps - g0 : kStreamMaxPB);
            double *mu = out_mu ? out_mu + (size_t)g0 * D * n_rec : nullptr;
            RW_CUDA(ctx, launch_fold_stream(ctx, ctx->coef + g0 * kCoefStride, nullptr, nullptr, nullptr, Pb,
                                            dout + g0, full, mu, s));
        }
    } else if (!contraction) {
        for (int64_t g0 = 0, step = 0; g0 < Ps; g0 += step) {
            const int Pb = ridge_group(Ps - g0, L.ridge_max_p);
            step = Pb;
            double *mu = out_mu ? out_mu + (size_t)g0 * D * n_rec : nullptr;
            RW_CUDA(ctx, launch_fold_ridge(ctx, ctx->coef + g0 * kCoefStride, nullptr, nullptr, nullptr, Pb,
                                           dout + g0, full, mu, s));
        }
    } else {
        const bool certify = prec >= 2 && (opt.tol > 0.0 || opt.bound);
        for (int64_t c0 = 0; c0 < Ps; c0 += L.MC) {
            const int64_t Pc = (Ps - c0 < L.MC) ? Ps - c0 : L.MC;
            double *mu = out_mu ? out_mu + (size_t)c0 * D * n_rec : nullptr;
            for (int d = 0; d < D; ++d) {
                if (prec >= 2) {
                    RW_CUDA(ctx, launch_fold_i8(ctx, d, c0, Pc, mu, s, nullptr, prec == 3, certify));
                } else {
                    RW_CUDA(ctx, launch_gen_A(ctx, d, c0, Pc, s));
                    RW_CUDA(ctx, launch_fold_gemm(ctx, d, Pc, mu, 0, s));
                }
            }
            RW_CUDA(ctx, launch_reduce(ctx, D * (prec >= 2 ? L.NT8 : L.n_tiles_n), L.MC, Pc, dout + c0, full, s));
            if (!certify) continue;
            double *bnd = opt.bound ? opt.bound + c0 : ctx->bound_stage + c0;
            RW_CUDA(ctx, launch_reduce_max(ctx, D * L.NT8, L.MC, Pc, bnd, s));
            if (!(opt.tol > 0.0)) continue;
            // ---- strict: how many points of this chunk are not certified?  (the one place the library reads a number
            // back: the stream is synchronised once per chunk, so a strict call cannot be captured in a CUDA graph)
            double *coef_all = ctx->coef, *rate_all = ctx->rate;
            ctx->coef = coef_all + c0 * kCoefStride; ctx->rate = rate_all + c0 * RW_MAX_COMPONENTS;
            cudaError_t e = launch_collect_uncertified(ctx, bnd, Pc, opt.tol, true, s);
            ctx->coef = coef_all; ctx->rate = rate_all;
            RW_CUDA(ctx, e);
            int n_bad = 0;
            RW_CUDA(ctx, cudaMemcpyAsync(&n_bad, ctx->fb_idx + L.MC, 4, cudaMemcpyDeviceToHost, s));
            RW_CUDA(ctx, cudaStreamSynchronize(s));
            ctx->strict_fallbacks += n_bad;
            if (n_bad == 0) continue;
            if (mu) {            // mu rows cannot be scattered: the whole chunk goes through the DMMA path again
                ctx->coef = coef_all + c0 * kCoefStride; ctx->rate = rate_all + c0 * RW_MAX_COMPONENTS;
                int rc = fold_slice(ctx, Pc, RW_MODE_GEMM, full, dout + c0, mu, s, 0);
                ctx->coef = coef_all; ctx->rate = rate_all;
                if (rc != RW_OK) return rc;
                if (opt.bound) RW_CUDA(ctx, cudaMemsetAsync(opt.bound + c0, 0, (size_t)Pc * 8, s));
            } else {             // only the uncertified points, from their gathered coefficient rows
                ctx->coef = ctx->coef_fb; ctx->rate = ctx->rate_fb;
                int rc = fold_slice(ctx, n_bad, RW_MODE_AUTO, full, ctx->out_fb, nullptr, s, 0);
                ctx->coef = coef_all; ctx->rate = rate_all;
                if (rc != RW_OK) return rc;
                RW_CUDA(ctx, launch_scatter_fallback(ctx, n_bad, dout + c0, opt.bound ? opt.bound + c0 : nullptr, s));
            }
        }
    }
    return RW_OK;
}

// Contraction regime asked for by the flags: 0 = FP64 DMMA, 2 = RW_SLICED, 3 = RW_SLICED_FAST / RW_FP32; *tol > 0 when
// the call is strict (RW_SLICED_STRICT; RW_FP32 always is: its contract is a relative error, not a scale bound).
static int pick_prec(rw_ctx *ctx, const char *fn, uint32_t flags, bool fp32_ok, int *prec, double *tol)
{
    const bool fp32 = flags & RW_FP32, fast = (flags & RW_SLICED_FAST) || fp32, sliced = (flags & RW_SLICED) || fast;
    if ((flags & RW_SLICED) && fast)
        return fail(ctx, RW_ERR_INVALID, "%s: RW_SLICED, RW_SLICED_FAST and RW_FP32 exclude each other", fn);
    if (fp32 && (flags & RW_SLICED_FAST))
        return fail(ctx, RW_ERR_INVALID, "%s: RW_SLICED, RW_SLICED_FAST and RW_FP32 exclude each other", fn);
    if (fp32 && !fp32_ok) return fail(ctx, RW_ERR_UNSUPPORTED, "%s: RW_FP32 is not supported here", fn);
    if ((flags & RW_SLICED_STRICT) && !sliced)
        return fail(ctx, RW_ERR_INVALID, "%s: RW_SLICED_STRICT goes with RW_SLICED or RW_SLICED_FAST", fn);
    if (sliced && !ctx->lay.sliced)
        return fail(ctx, RW_ERR_UNSUPPORTED, "%s: RW_SLICED / RW_SLICED_FAST / RW_FP32 need a context created with "
                                             "RW_CREATE_SLICED (or RW_CREATE_FP32)", fn);
    *prec = fast ? 3 : (sliced ? 2 : 0);
    *tol = (fp32 || (flags & RW_SLICED_STRICT)) ? (fast ? 1e-5 : 1e-12) : 0.0;
    return RW_OK;
}

static int check_kinds(rw_ctx *ctx, const char *fn, int32_t k, const int32_t *param_kind, int *kinds)
{
    for (int a = 0; a < k; ++a) {
        kinds[a] = param_kind[a];
        if (kinds[a] < 0 || kinds[a] >= RW_RATE_0 + ctx->n_comp)
            return fail(ctx, RW_ERR_INVALID, "%s: param_kind[%d] = %d out of range", fn, a, kinds[a]);
        for (int b = 0; b < a; ++b)
            if (kinds[b] == kinds[a]) return fail(ctx, RW_ERR_INVALID, "%s: duplicate param_kind %d", fn, kinds[a]);
    }
    return RW_OK;
}

}  // namespace rw

using namespace rw;

extern "C" {

int rw_workspace_bytes(const rw_inputs *in, int64_t max_batch, size_t *bytes)
{
    Layout L;
    int rc = plan(in, max_batch, &L);
    if (rc != RW_OK) return fail(nullptr, rc, "rw_workspace_bytes: invalid sizes/mem_kind/max_batch");
    if (!bytes) return fail(nullptr, RW_ERR_INVALID, "rw_workspace_bytes: bytes is NULL");
    *bytes = L.total;
    return RW_OK;
}

int rw_create(const rw_inputs *in, int64_t max_batch, void *dev_workspace, size_t workspace_bytes,
              void *cuda_stream, rw_ctx **out)
{
    if (!out) return fail(nullptr, RW_ERR_INVALID, "rw_create: out is NULL");
    *out = nullptr;
    Layout L;
    int rc = plan(in, max_batch, &L);
    if (rc != RW_OK) return fail(nullptr, rc, "rw_create: invalid sizes/mem_kind/max_batch");
    if (!in->E_MeV || !in->flux_w || !in->P_e || !in->T_MeV || !in->N_mc || !in->R || !in->bkg || !in->counts)
        return fail(nullptr, RW_ERR_INVALID, "rw_create: a required input array is NULL");
    if ((in->P_mu == nullptr) != (in->P_tau == nullptr))
        return fail(nullptr, RW_ERR_INVALID, "rw_create: P_mu and P_tau must both be given or both be NULL");
    const bool have_mt = in->P_mu != nullptr;
    const size_t n_comp = in->n_comp > 1 ? in->n_comp : 1;
    if (n_comp > 1 && !in->comp_of_T)
        return fail(nullptr, RW_ERR_INVALID, "rw_create: comp_of_T is NULL with n_comp = %d", in->n_comp);
    double f_tau = in->f_tau;
    if (!have_mt && !(f_tau >= 0.0 && f_tau <= 1.0))
        return fail(nullptr, RW_ERR_INVALID, "rw_create: f_tau must lie in [0,1]");
    if (!dev_workspace || ((uintptr_t)dev_workspace & 255) || workspace_bytes < L.total)
        return fail(nullptr, RW_ERR_WORKSPACE, "rw_create: workspace NULL, not 256-byte aligned, or smaller than %zu bytes",
                    L.total);
    const rw_constants &k = in->consts;
    double vals[4] = {k.sin2_theta_w, k.m_e_MeV, k.G_F_MeV2, k.alpha_em};
    for (double v : vals)
        if (!(v >= 0.0) || isinf(v)) return fail(nullptr, RW_ERR_INVALID, "rw_create: constants must be finite and >= 0");

    int dev = 0, major = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return fail(nullptr, RW_ERR_CUDA, "rw_create: no usable CUDA device: %s", cudaGetErrorString(cudaGetLastError()));
    if (major != 10) return fail(nullptr, RW_ERR_UNSUPPORTED, "rw_create: built for sm_100a, device is sm_%d", major * 10);

    const size_t n_E = in->n_E, n_T = in->n_T, n_rec = in->n_rec, D = in->n_periods;
    const bool host = in->mem_kind == RW_MEM_HOST;
    if (host) {
        int f = 0;
        if (host_bad_pos(in->E_MeV, n_E)) f |= 1;
        if (host_bad_nonneg(in->flux_w, n_comp * n_E)) f |= 2;
        if (host_bad_prob(in->P_e, n_comp * n_E) ||
            (have_mt && (host_bad_prob(in->P_mu, n_comp * n_E) || host_bad_prob(in->P_tau, n_comp * n_E)))) f |= 4;
        if (n_comp > 1)
            for (size_t i = 0; i < n_T; ++i)
                if (in->comp_of_T[i] < 0 || in->comp_of_T[i] >= (int32_t)n_comp) f |= 256;
        if (host_bad_pos(in->T_MeV, n_T)) f |= 8;
        if (host_bad_nonneg(in->N_mc, D * n_T)) f |= 16;
        if (host_bad_nonneg(in->bkg, D * n_rec)) f |= 32;
        if (host_bad_nonneg(in->counts, D * n_rec)) f |= 64;
        if (host_bad_nonneg(in->R, D * n_T * n_rec)) f |= 128;
        if (f) return fail(nullptr, RW_ERR_INVALID, "rw_create: %s", flag_message(f));
    } else if (!L.copy_R && ((uintptr_t)in->R & 15)) {
        return fail(nullptr, RW_ERR_INVALID, "rw_create: a borrowed device R must be 16-byte aligned");
    }

    rw_ctx *ctx = (rw_ctx *)calloc(1, sizeof(rw_ctx));
    if (!ctx) return fail(nullptr, RW_ERR_NOMEM, "rw_create: out of host memory");
    ctx->tmapR = (CUtensorMap *)calloc(D, sizeof(CUtensorMap));
    if (!ctx->tmapR) { free(ctx); return fail(nullptr, RW_ERR_NOMEM, "rw_create: out of host memory"); }
    ctx->n_E = in->n_E; ctx->n_T = in->n_T; ctx->n_rec = in->n_rec; ctx->D = in->n_periods;
    ctx->n_comp = (int)n_comp;
    ctx->f_tau = f_tau; ctx->have_mu_tau = have_mt;
    ctx->lay = L;
    ctx->num_sms = sms;
    ctx->ws = (char *)dev_workspace;
    Consts &c = ctx->cst;
    c.sin2w = k.sin2_theta_w > 0 ? k.sin2_theta_w : 0.23121;
    c.m_e = k.m_e_MeV > 0 ? k.m_e_MeV : 0.51099895;
    c.G_F = k.G_F_MeV2 > 0 ? k.G_F_MeV2 : 1.1663788e-11;
    c.alpha = k.alpha_em > 0 ? k.alpha_em : 1.0 / 137.035999084;
    const double pi = 3.14159265358979323846;
    c.C0 = 2.0 * c.G_F * c.G_F * c.m_e / pi;                 // Eq. (4) prefactor
    c.Cmm = pi * c.alpha * c.alpha / (c.m_e * c.m_e);        // Eq. (8) prefactor
    c.gL[0] = 0.5 + c.sin2w;  c.gR[0] = c.sin2w;              // Eq. (2)
    c.gL[1] = -0.5 + c.sin2w; c.gR[1] = c.sin2w;              // Eq. (3)
    c.gL[2] = -0.5 + c.sin2w; c.gR[2] = c.sin2w;

    char *ws = ctx->ws;
    ctx->E = (double *)(ws + L.E);          ctx->fw = (double *)(ws + L.fw);
    ctx->P3 = (double *)(ws + L.P3);        ctx->T = (double *)(ws + L.T);
    ctx->comp8 = (uint8_t *)(ws + L.comp8);       // all zero with a single component
    ctx->rate = (double *)(ws + L.rate);
    ctx->Tmax_invE = (double *)(ws + L.Tmax_invE);
    ctx->N_mc = (double *)(ws + L.N_mc);    ctx->bkg = (double *)(ws + L.bkg);
    ctx->counts = (double *)(ws + L.counts);
    ctx->basis = (double *)(ws + L.basis);  ctx->S_sm = (double *)(ws + L.S_sm);
    ctx->What = (double *)(ws + L.What);    ctx->sat_const = (double *)(ws + L.sat_const);
    ctx->flag = (int *)(ws + L.flag);
    ctx->G = (double *)(ws + L.G);          ctx->ident = (double *)(ws + L.ident);
    ctx->stream_cnt = (int *)(ws + L.stream_cnt);
    ctx->strip_part = (double *)(ws + L.strip_part);
    ctx->ridge_cnt = (int *)(ws + L.ridge_cnt);
    ctx->ridge_part = (double *)(ws + L.ridge_part);
    ctx->ridge_frag = (double *)(ws + L.ridge_frag);
    ctx->ridge_slots = (double *)(ws + L.ridge_slots);
    ctx->param_stage = (double *)(ws + L.param_stage);
    ctx->coef = (double *)(ws + L.coef);    ctx->A_packed = (double *)(ws + L.A_packed);
    ctx->partial = (double *)(ws + L.partial);
    ctx->mu_part = (double *)(ws + L.mu_part);
    ctx->out_stage = (double *)(ws + L.out_stage);
    ctx->mu_tile = (double *)(ws + L.mu_tile);
    ctx->mu_prof = (double *)(ws + L.mu_prof);
    ctx->pee_perm = (int *)(ws + L.pee_perm);      ctx->pee_j0 = (int *)(ws + L.pee_j0);
    ctx->pee_TmaxS = (double *)(ws + L.pee_TmaxS); ctx->pee_fS = (double *)(ws + L.pee_fS);
    ctx->pee_rho = (double *)(ws + L.pee_rho);     ctx->pee_Y = (double *)(ws + L.pee_Y);
    ctx->gcol8 = (double *)(ws + L.gcol8);
    ctx->cert_part = (double *)(ws + L.cert_part);
    ctx->bound_stage = (double *)(ws + L.bound_stage);
    ctx->fb_idx = (int *)(ws + L.fb_idx);
    ctx->coef_fb = (double *)(ws + L.coef_fb);
    ctx->rate_fb = (double *)(ws + L.rate_fb);
    ctx->out_fb = (double *)(ws + L.out_fb);
    ctx->B8 = (uint8_t *)(ws + L.B8);
    ctx->f_col8 = (int *)(ws + L.f_col8);
    ctx->e_row8 = (int *)(ws + L.e_row8);
    ctx->tau8 = (int *)(ws + L.tau8);
    ctx->blk_hl8 = (double *)(ws + L.blk_hl8);
    ctx->blk_cm8 = (int *)(ws + L.blk_cm8);
    ctx->tau8b = (int8_t *)(ws + L.tau8b);
    ctx->comp8p = (uint8_t *)(ws + L.comp8p);
    ctx->ldR = L.ldR;
    ctx->R_period_stride = n_T * (size_t)L.ldR;
    ctx->R = L.copy_R ? (const double *)(ws + L.R_copy) : in->R;

    cudaStream_t s = (cudaStream_t)cuda_stream;
    const cudaMemcpyKind kind = host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
#define RW_TRY(call)                                                                            \
    do {                                                                                        \
        cudaError_t e__ = (call);                                                               \
        if (e__ != cudaSuccess) {                                                               \
            fail(nullptr, RW_ERR_CUDA, "rw_create: %s failed: %s", #call, cudaGetErrorString(e__)); \
            free(comp_host); free(ctx->tmapR); free(ctx);                                       \
            return RW_ERR_CUDA;                                                                 \
        }                                                                                       \
    } while (0)
    uint8_t *comp_host = nullptr;                              // host staging of comp_of_T, freed after the sync
    RW_TRY(cudaMemcpyAsync(ctx->E, in->E_MeV, n_E * 8, kind, s));
    RW_TRY(cudaMemcpyAsync(ctx->fw, in->flux_w, n_comp * n_E * 8, kind, s));
    for (size_t q = 0; q < n_comp; ++q) {                      // [n_comp][n_E] tables -> P3[n_comp][3][n_E]
        RW_TRY(cudaMemcpyAsync(ctx->P3 + q * 3 * n_E, in->P_e + q * n_E, n_E * 8, kind, s));
        if (have_mt) {
            RW_TRY(cudaMemcpyAsync(ctx->P3 + q * 3 * n_E + n_E, in->P_mu + q * n_E, n_E * 8, kind, s));
            RW_TRY(cudaMemcpyAsync(ctx->P3 + q * 3 * n_E + 2 * n_E, in->P_tau + q * n_E, n_E * 8, kind, s));
        }
    }
    if (n_comp == 1) RW_TRY(cudaMemsetAsync(ctx->comp8, 0, n_T, s));
    if (n_comp > 1) {
        RW_TRY(cudaMemsetAsync(ctx->flag, 0, 4, s));
        if (host) {
            comp_host = (uint8_t *)malloc(n_T);
            if (!comp_host) { free(ctx->tmapR); free(ctx); return fail(nullptr, RW_ERR_NOMEM, "rw_create: out of host memory"); }
            for (size_t i = 0; i < n_T; ++i) comp_host[i] = (uint8_t)in->comp_of_T[i];
            RW_TRY(cudaMemcpyAsync(ctx->comp8, comp_host, n_T, cudaMemcpyHostToDevice, s));
        }
    }
    RW_TRY(cudaMemcpyAsync(ctx->T, in->T_MeV, n_T * 8, kind, s));
    RW_TRY(cudaMemcpyAsync(ctx->N_mc, in->N_mc, D * n_T * 8, kind, s));
    RW_TRY(cudaMemcpyAsync(ctx->bkg, in->bkg, D * n_rec * 8, kind, s));
    RW_TRY(cudaMemcpyAsync(ctx->counts, in->counts, D * n_rec * 8, kind, s));
    if (L.copy_R) {
        if ((size_t)L.ldR != n_rec) RW_TRY(cudaMemsetAsync(ws + L.R_copy, 0, D * n_T * (size_t)L.ldR * 8, s));
        RW_TRY(cudaMemcpy2DAsync(ws + L.R_copy, (size_t)L.ldR * 8, in->R, n_rec * 8, n_rec * 8, D * n_T, kind, s));
    }
    RW_TRY(cudaMemsetAsync(ctx->flag, 0, 4, s));
    if (n_comp > 1 && !host) RW_TRY(launch_comp8(ctx, in->comp_of_T, s));
    RW_TRY(cudaMemsetAsync(ctx->stream_cnt, 0, (D * (size_t)L.stream_strips + 1) * 4, s));
    RW_TRY(cudaMemsetAsync(ctx->ridge_cnt, 0, (2 * D * (size_t)L.ridge_strips + 1) * 4, s));
    RW_TRY(launch_flavour(ctx, have_mt ? 1 : 0, f_tau, s));
    if (!host) RW_TRY(launch_validate_device(ctx, ctx->R, ctx->ldR, ctx->R_period_stride, s));
    RW_TRY(launch_setup(ctx, s));
    RW_TRY(launch_sat_const(ctx, s));
    RW_TRY(launch_prefold(ctx, s));
    int flag = 0;
    RW_TRY(cudaMemcpyAsync(&flag, ctx->flag, 4, cudaMemcpyDeviceToHost, s));
    RW_TRY(cudaStreamSynchronize(s));
    free(comp_host);
#undef RW_TRY
    if (flag) {
        fail(nullptr, RW_ERR_INVALID, "rw_create: %s", flag_message(flag));
        free(ctx->tmapR); free(ctx);
        return RW_ERR_INVALID;
    }
    rc = make_tensor_maps(ctx);
    if (rc == RW_OK) rc = ridge_setup(ctx);
    if (rc == RW_OK) rc = profile_setup(ctx);
    if (rc == RW_OK) {
        rc = pee_setup(ctx, s);
        if (rc == RW_OK && cudaStreamSynchronize(s) != cudaSuccess)
            rc = fail(nullptr, RW_ERR_CUDA, "rw_create: per-point P_ee tables failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    if (rc == RW_OK && L.sliced) {
        rc = i8_setup(ctx, s);
        if (rc == RW_OK && cudaStreamSynchronize(s) != cudaSuccess)
            rc = fail(nullptr, RW_ERR_CUDA, "rw_create: slicing R failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    if (rc != RW_OK) { free(ctx->tmapR); free(ctx); return rc; }
    ctx->err[0] = 0;
    *out = ctx;
    return RW_OK;
}

int rw_set_counts(rw_ctx *ctx, const double *counts, int32_t mem_kind, void *cuda_stream)
{
    if (!ctx) return fail(nullptr, RW_ERR_INVALID, "rw_set_counts: ctx is NULL");
    if (!counts || (mem_kind != RW_MEM_HOST && mem_kind != RW_MEM_DEVICE))
        return fail(ctx, RW_ERR_INVALID, "rw_set_counts: counts NULL or bad mem_kind");
    const size_t n = (size_t)ctx->D * ctx->n_rec;
    if (mem_kind == RW_MEM_HOST && host_bad_nonneg(counts, n))
        return fail(ctx, RW_ERR_INVALID, "rw_set_counts: counts must be finite and >= 0");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (mem_kind == RW_MEM_DEVICE) {
        // validate the caller's array BEFORE the context changes: a rejected call leaves counts and the saturated
        // constant as they were
        int flag = 0;
        RW_CUDA(ctx, cudaMemsetAsync(ctx->flag, 0, 4, s));
        RW_CUDA(ctx, launch_validate_counts(ctx, counts, s));
        RW_CUDA(ctx, cudaMemcpyAsync(&flag, ctx->flag, 4, cudaMemcpyDeviceToHost, s));
        RW_CUDA(ctx, cudaStreamSynchronize(s));
        if (flag) return fail(ctx, RW_ERR_INVALID, "rw_set_counts: counts must be finite and >= 0");
    }
    RW_CUDA(ctx, cudaMemsetAsync(ctx->flag, 0, 4, s));
    RW_CUDA(ctx, cudaMemcpyAsync(ctx->counts, counts, n * 8,
                                 mem_kind == RW_MEM_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, s));
    RW_CUDA(ctx, launch_sat_const(ctx, s));
    RW_CUDA(ctx, cudaStreamSynchronize(s));
    return RW_OK;
}

static int eval_batch_impl(const char *fn, rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                           double *out_m2lnL, double *out_mu, double *out_bound, uint32_t flags, void *cuda_stream)
{
    if (!ctx) return fail(nullptr, RW_ERR_INVALID, "%s: ctx is NULL", fn);
    if (P < 0 || k < 0 || k > RW_N_KINDS) return fail(ctx, RW_ERR_INVALID, "%s: P < 0 or k outside [0,11]", fn);
    if (P == 0) return RW_OK;
    if (!out_m2lnL || (k > 0 && (!param || !param_kind)))
        return fail(ctx, RW_ERR_INVALID, "%s: param, param_kind or out_m2lnL is NULL", fn);
    int kinds[RW_N_KINDS];
    { int rc = check_kinds(ctx, fn, k, param_kind, kinds); if (rc != RW_OK) return rc; }
    const uint32_t mode = flags & RW_MODE_MASK;
    const bool param_host = flags & RW_PARAM_HOST, out_host = flags & RW_OUT_HOST, full = flags & RW_FULL_EQ18;
    int prec = 0;
    double tol = 0.0;
    { int rc = pick_prec(ctx, fn, flags, true, &prec, &tol); if (rc != RW_OK) return rc; }
    if (mode > RW_MODE_RIDGE) return fail(ctx, RW_ERR_INVALID, "%s: unknown mode in flags", fn);

    cudaStream_t s = (cudaStream_t)cuda_stream;
    const Layout &L = ctx->lay;
    const int D = ctx->D, n_rec = ctx->n_rec;
    // mu for a host caller is staged through the scratch of rw_eval_profile (prof_rows points of D n_rec doubles),
    // slice by slice, and copied D2H on the stream like -2lnL
    const bool mu_host = out_host && out_mu;
    const int64_t slice = (mu_host && L.prof_rows < L.max_batch) ? L.prof_rows : L.max_batch;
    for (int64_t s0 = 0; s0 < P; s0 += slice) {
        const int64_t Ps = (P - s0 < slice) ? P - s0 : slice;
        double *dmu = !out_mu ? nullptr : mu_host ? ctx->mu_prof : out_mu + (size_t)s0 * D * n_rec;
        const double *dparam = nullptr;
        if (k > 0) {
            dparam = param + s0 * k;
            if (param_host) {
                RW_CUDA(ctx, cudaMemcpyAsync(ctx->param_stage, dparam, (size_t)Ps * k * 8, cudaMemcpyHostToDevice, s));
                dparam = ctx->param_stage;
            }
        }
        double *dout = out_host ? ctx->out_stage : out_m2lnL + s0;
        const bool stream_mode = use_stream(ctx, mode, Ps, prec);
        if (stream_mode || use_ridge(ctx, mode, Ps, prec)) {
            if (out_bound) RW_CUDA(ctx, cudaMemsetAsync(out_bound + s0, 0, (size_t)Ps * 8, s));       // FP64 paths
            // up to 64 points: ONE launch per group does a1-a4 (coefficients computed in the kernel) -- the
            // HBM-streaming kernel (groups of 16) or the streaming DMMA kernel (groups of 64)
            Kinds kd;
            kd.k = k;
            for (int a = 0; a < RW_N_KINDS; ++a) kd.kind[a] = (a < k) ? kinds[a] : -1;
            for (int64_t g0 = 0, step = 0; g0 < Ps; g0 += step) {
                const int Pb = stream_mode ? (int)((Ps - g0 < kStreamMaxPB) ? Ps - g0 : kStreamMaxPB)
                                           : ridge_group(Ps - g0, L.ridge_max_p);
                step = Pb;
                double *mu = dmu ? dmu + (size_t)g0 * D * n_rec : nullptr;
                const double *cf = nullptr, *pr = (k > 0) ? dparam + g0 * k : nullptr;
                if (k == 0) {
                    RW_CUDA(ctx, launch_coef(ctx, nullptr, Pb, 0, kinds, s));
                    cf = ctx->coef;
                }
                if (stream_mode)
                    RW_CUDA(ctx, launch_fold_stream(ctx, cf, pr, k > 0 ? &kd : nullptr, nullptr, Pb, dout + g0, full, mu, s));
                else
                    RW_CUDA(ctx, launch_fold_ridge(ctx, cf, pr, k > 0 ? &kd : nullptr, nullptr, Pb, dout + g0, full, mu, s));
            }
        } else {
        RW_CUDA(ctx, launch_coef(ctx, dparam, Ps, k, kinds, s));
        SlicedOpt opt;
        opt.tol = tol; opt.bound = out_bound ? out_bound + s0 : nullptr;
        { int rc = fold_slice(ctx, Ps, mode, full, dout, dmu, s, prec, opt); if (rc != RW_OK) return rc; }
        }
        if (out_host)
            RW_CUDA(ctx, cudaMemcpyAsync(out_m2lnL + s0, ctx->out_stage, (size_t)Ps * 8, cudaMemcpyDeviceToHost, s));
        if (mu_host)
            RW_CUDA(ctx, cudaMemcpyAsync(out_mu + (size_t)s0 * D * n_rec, ctx->mu_prof, (size_t)Ps * D * n_rec * 8,
                                         cudaMemcpyDeviceToHost, s));
    }
    return RW_OK;
}

int rw_eval_batch(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                  double *out_m2lnL, double *out_mu, uint32_t flags, void *cuda_stream)
{
    return eval_batch_impl("rw_eval_batch", ctx, param, P, k, param_kind, out_m2lnL, out_mu, nullptr, flags, cuda_stream);
}

int rw_eval_certified(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                      double *out_m2lnL, double *out_bound, uint32_t flags, void *cuda_stream)
{
    if (!ctx) return fail(nullptr, RW_ERR_INVALID, "rw_eval_certified: ctx is NULL");
    if (!out_bound && P > 0) return fail(ctx, RW_ERR_INVALID, "rw_eval_certified: out_bound is NULL");
    if (flags & (RW_PARAM_HOST | RW_OUT_HOST))
        return fail(ctx, RW_ERR_UNSUPPORTED, "rw_eval_certified: host buffers are not supported");
    if (!(flags & (RW_SLICED | RW_SLICED_FAST | RW_FP32)))
        return fail(ctx, RW_ERR_INVALID, "rw_eval_certified: needs RW_SLICED, RW_SLICED_FAST or RW_FP32 (the FP64 paths "
                                         "have no input-dependent bound)");
    return eval_batch_impl("rw_eval_certified", ctx, param, P, k, param_kind, out_m2lnL, nullptr, out_bound, flags, cuda_stream);
}

int64_t rw_strict_fallback_count(const rw_ctx *ctx) { return ctx ? ctx->strict_fallbacks : 0; }

int rw_eval_profile(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                    double s0, double sigma, double *out_m2lnL, double *out_scale, uint32_t flags,
                    void *cuda_stream)
{
    if (!ctx) return fail(nullptr, RW_ERR_INVALID, "rw_eval_profile: ctx is NULL");
    if (P < 0 || k < 0 || k > RW_N_KINDS) return fail(ctx, RW_ERR_INVALID, "rw_eval_profile: P < 0 or k outside [0,11]");
    if (P == 0) return RW_OK;
    if (!out_m2lnL || (k > 0 && (!param || !param_kind)))
        return fail(ctx, RW_ERR_INVALID, "rw_eval_profile: param, param_kind or out_m2lnL is NULL");
    if (flags & (RW_PARAM_HOST | RW_OUT_HOST))
        return fail(ctx, RW_ERR_UNSUPPORTED, "rw_eval_profile: host buffers are not supported");
    if (!(s0 == s0) || !(sigma == sigma) || isinf(s0) || (sigma > 0.0 && s0 < 0.0))
        return fail(ctx, RW_ERR_INVALID, "rw_eval_profile: s0 must be finite (and >= 0 with a pull), sigma not NaN");
    int kinds[RW_N_KINDS];
    { int rc = check_kinds(ctx, "rw_eval_profile", k, param_kind, kinds); if (rc != RW_OK) return rc; }
    const uint32_t mode = flags & RW_MODE_MASK;
    const bool full = flags & RW_FULL_EQ18;
    int prec = 0;
    SlicedOpt opt;
    { int rc = pick_prec(ctx, "rw_eval_profile", flags, true, &prec, &opt.tol); if (rc != RW_OK) return rc; }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const Layout &L = ctx->lay;
    // passes of <= prof_rows points: fold with mu written to the scratch, then one CTA per point profiles s
    for (int64_t q0 = 0; q0 < P; q0 += L.prof_rows) {
        const int64_t Pq = (P - q0 < L.prof_rows) ? P - q0 : L.prof_rows;
        RW_CUDA(ctx, launch_coef(ctx, k > 0 ? param + q0 * k : nullptr, Pq, k, kinds, s));
        int rc = fold_slice(ctx, Pq, mode, false, ctx->out_stage, ctx->mu_prof, s, prec, opt);
        if (rc != RW_OK) return rc;
        RW_CUDA(ctx, launch_profile(ctx, ctx->mu_prof, Pq, s0, sigma, full, out_m2lnL + q0,
                                    out_scale ? out_scale + q0 : nullptr, s));
    }
    return RW_OK;
}

int rw_eval_grad(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                 double *out_m2lnL, double *out_grad, uint32_t flags, void *cuda_stream)
{
    if (!ctx) return fail(nullptr, RW_ERR_INVALID, "rw_eval_grad: ctx is NULL");
    if (P < 0 || k < 1 || k > RW_N_KINDS) return fail(ctx, RW_ERR_INVALID, "rw_eval_grad: P < 0 or k outside [1,11]");
    if (P == 0) return RW_OK;
    if (!out_m2lnL || !out_grad || !param || !param_kind)
        return fail(ctx, RW_ERR_INVALID, "rw_eval_grad: param, param_kind, out_m2lnL or out_grad is NULL");
    if (flags & (RW_PARAM_HOST | RW_OUT_HOST | RW_FP32 | RW_SLICED_STRICT))
        return fail(ctx, RW_ERR_UNSUPPORTED, "rw_eval_grad: host buffers, RW_FP32 and RW_SLICED_STRICT are not supported "
                                             "(a derivative row has no certificate: it is a difference of two folds)");
    int kinds[RW_N_KINDS];
    { int rc = check_kinds(ctx, "rw_eval_grad", k, param_kind, kinds); if (rc != RW_OK) return rc; }
    const uint32_t mode = flags & RW_MODE_MASK;
    int prec = 0;
    double tol = 0.0;
    { int rc = pick_prec(ctx, "rw_eval_grad", flags, false, &prec, &tol); if (rc != RW_OK) return rc; }
    const bool full = flags & RW_FULL_EQ18;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const Layout &L = ctx->lay;
    // a point is 1 + k rows of the ordinary fold (value row + one derivative row per parameter); where the rows go
    // through the sliced contraction every derivative row goes as its positive and its negative part: 1 + 2 k rows
    const int max_rows_per_point = 1 + ((prec >= 2 && mode != RW_MODE_COLLAPSED) ? 2 : 1) * k;
    const int64_t per_pass = L.prof_rows / max_rows_per_point;
    if (per_pass < 1)
        return fail(ctx, RW_ERR_WORKSPACE, "rw_eval_grad: max_batch (%lld) is smaller than %d rows per point",
                    (long long)L.max_batch, max_rows_per_point);
    for (int64_t q0 = 0; q0 < P; q0 += per_pass) {
        const int64_t Pq = (P - q0 < per_pass) ? P - q0 : per_pass;
        // a pass small enough for the streaming kernels is folded in FP64 by fold_slice whatever the flags: no split
        const int64_t plain_rows = Pq * (1 + k);
        const bool split = max_rows_per_point > 1 + k && !use_stream(ctx, mode, plain_rows, prec) &&
                           !use_ridge(ctx, mode, plain_rows, prec);
        const int64_t rows = split ? Pq * max_rows_per_point : plain_rows;
        RW_CUDA(ctx, launch_coef_grad(ctx, param + q0 * k, Pq, k, kinds, s, split));
        int rc = fold_slice(ctx, rows, mode, false, ctx->out_stage, ctx->mu_prof, s, split ? prec : 0);
        if (rc != RW_OK) return rc;
        RW_CUDA(ctx, launch_grad(ctx, ctx->mu_prof, Pq, k, full, out_m2lnL + q0, out_grad + q0 * k, s, split));
    }
    return RW_OK;
}

// Dense fold + likelihood for P rows of caller-visible weights w[P][n_T] (device).
static int weights_rows(rw_ctx *ctx, const double *w, int64_t P, uint32_t mode, bool full, double *out, double *out_mu,
                        cudaStream_t s, int prec, double tol = 0.0)
{
    const Layout &L = ctx->lay;
    const int D = ctx->D, n_rec = ctx->n_rec;
    const size_t n_T = ctx->n_T;
    if (use_stream(ctx, mode, P, prec)) {
        for (int64_t g0 = 0; g0 < P; g0 += kStreamMaxPB) {
            const int Pb = (int)((P - g0 < kStreamMaxPB) ? P - g0 : kStreamMaxPB);
            double *mu = out_mu ? out_mu + (size_t)g0 * D * n_rec : nullptr;
            RW_CUDA(ctx, launch_fold_stream(ctx, nullptr, nullptr, nullptr, w + (size_t)g0 * n_T, Pb, out + g0, full, mu, s));
        }
    } else if (use_ridge(ctx, mode, P, prec)) {
        for (int64_t g0 = 0, step = 0; g0 < P; g0 += step) {
            const int Pb = ridge_group(P - g0, L.ridge_max_p);
            step = Pb;
            double *mu = out_mu ? out_mu + (size_t)g0 * D * n_rec : nullptr;
            RW_CUDA(ctx, launch_fold_ridge(ctx, nullptr, nullptr, nullptr, w + (size_t)g0 * n_T, Pb, out + g0, full, mu, s));
        }
    } else if (const int64_t rem = auto_tail(ctx, mode, P, prec)) {     // full rows of tiles, then the left-over points
        const int64_t main = P - rem;
        if (main > 0) {
            const int rc = weights_rows(ctx, w, main, RW_MODE_GEMM, full, out, out_mu, s, prec, tol);
            if (rc != RW_OK) return rc;
        }
        for (int64_t g0 = main, step = 0; g0 < P; g0 += step) {
            const int Pb = ridge_group(P - g0, L.ridge_max_p);
            step = Pb;
            double *mu = out_mu ? out_mu + (size_t)g0 * D * n_rec : nullptr;
            RW_CUDA(ctx, launch_fold_ridge(ctx, nullptr, nullptr, nullptr, w + (size_t)g0 * n_T, Pb, out + g0, full, mu, s));
        }
    } else {
        for (int64_t c0 = 0; c0 < P; c0 += L.MC) {
            const int64_t Pc = (P - c0 < L.MC) ? P - c0 : L.MC;
            double *mu = out_mu ? out_mu + (size_t)c0 * D * n_rec : nullptr;
            for (int d = 0; d < D; ++d) {
                if (prec >= 2) {
                    RW_CUDA(ctx, launch_fold_i8(ctx, d, 0, Pc, mu, s, w + (size_t)c0 * n_T, prec == 3, tol > 0.0));
                } else {
                    RW_CUDA(ctx, launch_gen_A_weights(ctx, d, w + (size_t)c0 * n_T, Pc, s));
                    RW_CUDA(ctx, launch_fold_gemm(ctx, d, Pc, mu, 0, s));
                }
            }
            RW_CUDA(ctx, launch_reduce(ctx, D * (prec >= 2 ? L.NT8 : L.n_tiles_n), L.MC, Pc, out + c0, full, s));
            if (prec >= 2 && tol > 0.0) {
                // strict: arbitrary weights have no coefficient rows to gather, so a chunk with ANY uncertified point
                // goes through the DMMA path again as a whole (one stream synchronisation per chunk)
                RW_CUDA(ctx, launch_reduce_max(ctx, D * L.NT8, L.MC, Pc, ctx->out_fb, s));
                RW_CUDA(ctx, launch_collect_uncertified(ctx, ctx->out_fb, Pc, tol, false, s));
                int n_bad = 0;
                RW_CUDA(ctx, cudaMemcpyAsync(&n_bad, ctx->fb_idx + L.MC, 4, cudaMemcpyDeviceToHost, s));
                RW_CUDA(ctx, cudaStreamSynchronize(s));
                ctx->strict_fallbacks += n_bad;
                if (n_bad > 0) {
                    for (int d = 0; d < D; ++d) {
                        RW_CUDA(ctx, launch_gen_A_weights(ctx, d, w + (size_t)c0 * n_T, Pc, s));
                        RW_CUDA(ctx, launch_fold_gemm(ctx, d, Pc, mu, 0, s));
                    }
                    RW_CUDA(ctx, launch_reduce(ctx, D * L.n_tiles_n, L.MC, Pc, out + c0, full, s));
                }
            }
        }
    }
    return RW_OK;
}

int rw_eval_weights(rw_ctx *ctx, const double *w, int64_t P, double *out_m2lnL, double *out_mu,
                    uint32_t flags, void *cuda_stream)
{
    if (!ctx) return fail(nullptr, RW_ERR_INVALID, "rw_eval_weights: ctx is NULL");
    if (P < 0) return fail(ctx, RW_ERR_INVALID, "rw_eval_weights: P < 0");
    if (P == 0) return RW_OK;
    if (!w || !out_m2lnL) return fail(ctx, RW_ERR_INVALID, "rw_eval_weights: w or out_m2lnL is NULL");
    const uint32_t mode = flags & RW_MODE_MASK;
    if (mode == RW_MODE_COLLAPSED || (flags & (RW_PARAM_HOST | RW_OUT_HOST | RW_FP32)))
        return fail(ctx, RW_ERR_UNSUPPORTED, "rw_eval_weights: collapsed mode, RW_FP32 and host buffers are not supported "
                                             "(arbitrary weights are not low-rank; w is a device array)");
    int prec = 0;
    double tol = 0.0;
    { int rc = pick_prec(ctx, "rw_eval_weights", flags, false, &prec, &tol); if (rc != RW_OK) return rc; }
    return weights_rows(ctx, w, P, mode, flags & RW_FULL_EQ18, out_m2lnL, out_mu, (cudaStream_t)cuda_stream, prec, tol);
}

int rw_eval_pee(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                const double *P_e_pts, double *out_m2lnL, double *out_mu, uint32_t flags, void *cuda_stream)
{
    if (!ctx) return fail(nullptr, RW_ERR_INVALID, "rw_eval_pee: ctx is NULL");
    if (P < 0 || k < 0 || k > RW_RATE_0) return fail(ctx, RW_ERR_INVALID, "rw_eval_pee: P < 0 or k outside [0,7]");
    if (P == 0) return RW_OK;
    if (!out_m2lnL || !P_e_pts || (k > 0 && (!param || !param_kind)))
        return fail(ctx, RW_ERR_INVALID, "rw_eval_pee: param, param_kind, P_e_pts or out_m2lnL is NULL");
    const uint32_t mode = flags & RW_MODE_MASK;
    if (mode == RW_MODE_COLLAPSED || (flags & (RW_PARAM_HOST | RW_OUT_HOST | RW_FP32)))
        return fail(ctx, RW_ERR_UNSUPPORTED, "rw_eval_pee: collapsed mode, RW_FP32 and host buffers are not supported");
    if ((ctx->n_comp > 1 || ctx->have_mu_tau) && !ctx->lay.pee_scan)
        return fail(ctx, RW_ERR_UNSUPPORTED, "rw_eval_pee: several components / explicit P_mu, P_tau need the sorted-grid "
                                             "path, i.e. a flux grid of at most ~8500 entries (n_E = %d)", ctx->n_E);
    int kinds[RW_N_KINDS], prec = 0;
    double tol = 0.0;
    { int rc = check_kinds(ctx, "rw_eval_pee", k, param_kind, kinds); if (rc != RW_OK) return rc; }
    { int rc = pick_prec(ctx, "rw_eval_pee", flags, false, &prec, &tol); if (rc != RW_OK) return rc; }
    for (int a = 0; a < k; ++a)
        if (kinds[a] >= RW_RATE_0) return fail(ctx, RW_ERR_INVALID, "rw_eval_pee: rate kinds are not accepted");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const Layout &L = ctx->lay;
    // passes sized by the mu scratch, which holds the weights w[Pq][n_T] here (plan(): at least one row)
    const int64_t per_pass = L.pee_rows;
    for (int64_t q0 = 0; q0 < P; q0 += per_pass) {
        const int64_t Pq = (P - q0 < per_pass) ? P - q0 : per_pass;
        RW_CUDA(ctx, launch_coef(ctx, k > 0 ? param + q0 * k : nullptr, Pq, k, kinds, s));
        RW_CUDA(ctx, launch_weights_pee(ctx, P_e_pts + (size_t)q0 * ctx->n_comp * ctx->n_E, Pq, ctx->mu_prof, s));
        int rc = weights_rows(ctx, ctx->mu_prof, Pq, mode, flags & RW_FULL_EQ18, out_m2lnL + q0,
                              out_mu ? out_mu + (size_t)q0 * ctx->D * ctx->n_rec : nullptr, s, prec, tol);
        if (rc != RW_OK) return rc;
    }
    return RW_OK;
}

int rw_get_table(const rw_ctx *ctx, int32_t which, const double **dev_ptr, int64_t *n_elems)
{
    if (!ctx || !dev_ptr || !n_elems) return RW_ERR_INVALID;
    switch (which) {
    case RW_TABLE_S_SM: *dev_ptr = ctx->S_sm; *n_elems = ctx->n_T; return RW_OK;
    case RW_TABLE_BASIS: *dev_ptr = ctx->basis; *n_elems = (int64_t)kNumBasis * ctx->n_T; return RW_OK;
    case RW_TABLE_WHAT: *dev_ptr = ctx->What; *n_elems = (int64_t)ctx->D * kCoefStride * ctx->n_T; return RW_OK;
    case RW_TABLE_G: *dev_ptr = ctx->G; *n_elems = (int64_t)ctx->D * ctx->n_comp * kCoefStride * ctx->lay.ldG; return RW_OK;
    default: return RW_ERR_INVALID;
    }
}

int64_t rw_launch_count(const rw_ctx *ctx) { return ctx ? ctx->launches : 0; }

int rw_profile_begin(rw_ctx *ctx)
{
    if (!ctx) return RW_ERR_INVALID;
    if (!ctx->prof_ev) {
        const int cap = 32768;
        ctx->prof_ev = (cudaEvent_t *)calloc(2 * cap, sizeof(cudaEvent_t));
        if (!ctx->prof_ev) return fail(ctx, RW_ERR_NOMEM, "rw_profile_begin: out of host memory");
        for (int q = 0; q < 2 * cap; ++q) RW_CUDA(ctx, cudaEventCreate(&ctx->prof_ev[q]));
        ctx->prof_cap = cap;
    }
    ctx->prof_n = 0;
    ctx->profiling = true;
    return RW_OK;
}

int rw_profile_end(rw_ctx *ctx, double *fold_ms_total, int64_t *fold_launches)
{
    if (!ctx || !fold_ms_total || !fold_launches) return RW_ERR_INVALID;
    ctx->profiling = false;
    double total = 0.0;
    for (int q = 0; q < ctx->prof_n; ++q) {
        float ms = 0.f;
        RW_CUDA(ctx, cudaEventSynchronize(ctx->prof_ev[2 * q + 1]));
        RW_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->prof_ev[2 * q], ctx->prof_ev[2 * q + 1]));
        total += ms;
    }
    *fold_ms_total = total;
    *fold_launches = ctx->prof_n;
    return RW_OK;
}

int rw_destroy(rw_ctx *ctx)
{
    if (!ctx) return RW_OK;
    if (ctx->prof_ev) {
        for (int q = 0; q < 2 * ctx->prof_cap; ++q) cudaEventDestroy(ctx->prof_ev[q]);
        free(ctx->prof_ev);
    }
    free(ctx->tmapR);
    free(ctx);
    return RW_OK;
}

const char *rw_strerror(int status)
{
    switch (status) {
    case RW_OK: return "ok";
    case RW_ERR_INVALID: return "invalid argument or input table";
    case RW_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case RW_ERR_CUDA: return "CUDA call failed";
    case RW_ERR_UNSUPPORTED: return "unsupported device or option";
    case RW_ERR_NOMEM: return "out of host memory";
    default: return "unknown status";
    }
}

const char *rw_last_error(const rw_ctx *ctx) { return ctx ? ctx->err : g_create_err; }

}  // extern "C"
