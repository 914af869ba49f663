// rw_fold_stream.cu -- the whole path for a handful of points (Pb <= 16 per launch) in ONE kernel:
// HBM-streaming fold with the coefficient step in front and the likelihood reduction behind it.
//
// With few points the fold mu[p][k] = sum_i N'[p][i] R[i][k] + bkg[k] (Eq. 11) reads
// every byte of R once and does 2P flop per 8 bytes: it is bound by HBM bandwidth, not arithmetic.
// R is row-major with the reconstructed index fastest, so a thread owns two adjacent columns
// (one 16-byte load per row), a CTA owns a 512-column strip, and the recoil rows are split over
// gridDim.y so that the grid fills all SMs several times over.
//   a1  the CTA computes the coefficients of its points from the raw parameters (Eq. 6)
//   a2  N'[p][i] (Eq. 14 / Eq. 1) is formed on the fly from the 11-term pre-scaled basis into shared memory
//   a3  each CTA folds its row range; the partial sums of a strip go to mu_part
//   a4  the LAST CTA of a strip to finish (ticket counter) adds the row ranges in a fixed order, adds the
//       background and reduces the Poisson terms of Eq. (18) of its 512 columns; the LAST strip
//       to finish adds the strips and periods in a fixed order and writes -2lnL.  Results do not depend on
//       which CTA is last: only who does the (fixed-order) sums changes.  The counters reset themselves.
// A single evaluation -- the call a minimiser makes -- is therefore one launch.
#include "rw_internal.h"

namespace rw {

constexpr int kRC = 64;   // recoil rows staged per iteration

struct StreamArgs {
    const double *R; size_t R_period_stride; int ldR, n_T, n_rec, D;
    const double *coef;       // [Pb][12], or NULL
    const double *param;      // [Pb][k] raw parameters (coefficients computed here), or NULL
    const double *wts;        // [Pb][n_T] caller weights (rw_eval_weights), or NULL
    const double *rate;       // [Pb][4] rate scales matching `coef` (ignored with `param`: computed here), or NULL
    const uint8_t *comp8;     // [n_T] component of every recoil bin, or NULL (one component)
    const double *What, *N_mc, *bkg, *counts, *sat_const;
    int Pb, rows_per_split, n_splits, mu_ld;
    double *mu_part;          // [D][n_splits][PB][mu_ld]
    double *strip_part;       // [D * strips][16]
    int *cnt;                 // [D * strips] strip tickets, then one global ticket
    double *out;              // [Pb] -2lnL, or NULL: fold only
    double *out_mu;           // NULL or [Pb][D][n_rec]
};

template <int PB>
__global__ void __launch_bounds__(kStreamThreads)
k_fold_stream(const StreamArgs A, const Kinds kd, const Consts cst)
{
    __shared__ __align__(16) double sN[2][kRC][PB];
    __shared__ double sC[PB][kCoefStride];
    __shared__ double sRate[PB][RW_MAX_COMPONENTS];
    __shared__ double red[kStreamThreads / 32][PB];
    __shared__ int s_last;
    const int d = blockIdx.z, split = blockIdx.y, strip = blockIdx.x;
    const int n_T = A.n_T, n_rec = A.n_rec, Pb = A.Pb;
    const int col = strip * kStreamCols + 2 * threadIdx.x;
    const int i0 = split * A.rows_per_split;
    const int i1 = min(n_T, i0 + A.rows_per_split);
    const double *Rd = A.R + (size_t)d * A.R_period_stride;
    const double *Wd = A.What + (size_t)d * kCoefStride * n_T;
    const double *wts = A.wts;

    if (!wts) {
        if (A.param) {
            if (threadIdx.x < PB) {
                double c[kCoefStride], r[RW_MAX_COMPONENTS];
                if (threadIdx.x < Pb) {
                    coef_from_param(A.param + (size_t)threadIdx.x * kd.k, kd, cst, c, r);
                } else {
#pragma unroll
                    for (int b = 0; b < kCoefStride; ++b) c[b] = 0.0;
#pragma unroll
                    for (int q = 0; q < RW_MAX_COMPONENTS; ++q) r[q] = 1.0;
                }
#pragma unroll
                for (int b = 0; b < kCoefStride; ++b) sC[threadIdx.x][b] = c[b];
#pragma unroll
                for (int q = 0; q < RW_MAX_COMPONENTS; ++q) sRate[threadIdx.x][q] = r[q];
            }
        } else {
            for (int q = threadIdx.x; q < PB * kCoefStride; q += kStreamThreads) {
                int p = q / kCoefStride, b = q - p * kCoefStride;
                sC[p][b] = (p < Pb) ? A.coef[(size_t)p * kCoefStride + b] : 0.0;
            }
            for (int q = threadIdx.x; q < PB * RW_MAX_COMPONENTS; q += kStreamThreads) {
                int p = q / RW_MAX_COMPONENTS, cq = q - p * RW_MAX_COMPONENTS;
                sRate[p][cq] = (p < Pb && A.rate) ? A.rate[(size_t)p * RW_MAX_COMPONENTS + cq] : 1.0;
            }
        }
    }
    double acc[PB][2];
#pragma unroll
    for (int p = 0; p < PB; ++p) acc[p][0] = acc[p][1] = 0.0;
    const bool col_ok = col < n_rec;

    // N' of a 64-row chunk: N' = sum_b c_b W^_b (Eq. 14 folded into the pre-scaled basis) or w N_mc (Eq. 1 with
    // caller-supplied weights).  Double-buffered: chunk ic + 64 is staged after chunk ic has been streamed, so one
    // barrier per chunk and the warps that finish streaming early stage while the others still load R.
    auto stage = [&](int ic, int buf) {
        for (int q = threadIdx.x; q < kRC * PB; q += kStreamThreads) {
            const int p = q / kRC, row = q - p * kRC;     // consecutive threads -> consecutive bins
            const int i = ic + row;
            double v = 0.0;
            if (i < i1) {
                if (wts) {
                    if (p < Pb) v = wts[(size_t)p * n_T + i] * A.N_mc[(size_t)d * n_T + i];
                } else {
#pragma unroll
                    for (int b = 0; b < kNumTerms; ++b) v = fma(sC[p][b], Wd[(size_t)b * n_T + i], v);
                    if (A.comp8) v *= sRate[p][A.comp8[i]];        // rate_k of Eq. (17)
                }
            }
            sN[buf][row][p] = v;
        }
    };
    __syncthreads();                                               // sC, sRate
    if (i0 < i1) stage(i0, 0);
    int buf = 0;
    for (int ic = i0; ic < i1; ic += kRC, buf ^= 1) {
        __syncthreads();                                           // sN[buf] staged; sN[buf ^ 1] no longer read
        if (col_ok) {
            const double *Rp = Rd + (size_t)ic * A.ldR + col;
            const int nrows = min(kRC, i1 - ic);
#pragma unroll 1
            for (int r0 = 0; r0 < nrows; r0 += 8) {
                double2 rv[8];
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    rv[u] = (r0 + u < nrows)
                                ? __ldg(reinterpret_cast<const double2 *>(Rp + (size_t)(r0 + u) * A.ldR))
                                : make_double2(0.0, 0.0);
#pragma unroll
                for (int u = 0; u < 8; ++u) {
#pragma unroll
                    for (int p = 0; p < PB; ++p) {
                        const double n = sN[buf][r0 + u][p];
                        acc[p][0] = fma(n, rv[u].x, acc[p][0]);
                        acc[p][1] = fma(n, rv[u].y, acc[p][1]);
                    }
                }
            }
        }
        if (ic + kRC < i1) stage(ic + kRC, buf ^ 1);
    }
    const int n_splits = A.n_splits, mu_ld = A.mu_ld;
    if (col_ok) {
#pragma unroll
        for (int p = 0; p < PB; ++p) {
            double *dst = A.mu_part + (((size_t)d * n_splits + split) * PB + p) * mu_ld + col;
            __stcg(reinterpret_cast<double2 *>(dst), make_double2(acc[p][0], acc[p][1]));
        }
    }
    if (!A.out) return;                      // fold only (template prefold)

    // ---------------------------------------------------------------- last CTA of this strip: a4 for 512 columns
    const int n_strips = gridDim.x, sid = d * n_strips + strip;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(A.cnt + sid, 1) == n_splits - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double bk0 = 0.0, bk1 = 0.0, cn0 = 0.0, cn1 = 0.0;
    const bool ok1 = col + 1 < n_rec;
    if (col_ok) { bk0 = A.bkg[(size_t)d * n_rec + col]; cn0 = A.counts[(size_t)d * n_rec + col]; }
    if (ok1) { bk1 = A.bkg[(size_t)d * n_rec + col + 1]; cn1 = A.counts[(size_t)d * n_rec + col + 1]; }
    double m0[PB], m1[PB];
#pragma unroll
    for (int p = 0; p < PB; ++p) m0[p] = m1[p] = 0.0;
    if (col_ok) {
        // row ranges in a fixed order, kBatch of them (16 loads) in flight: left to the compiler the loop ran ~4 loads
        // deep, ten dependent round trips to L2 for the 37 row ranges of a config-4 strip (~10 us of a 0.17 ms call)
        constexpr int kBatch = (PB >= 16) ? 1 : 16 / PB;
        for (int s0 = 0; s0 < n_splits; s0 += kBatch) {
            double2 v[kBatch][PB];
#pragma unroll
            for (int u = 0; u < kBatch; ++u) {
                const int s = min(s0 + u, n_splits - 1);
#pragma unroll
                for (int p = 0; p < PB; ++p)
                    v[u][p] = __ldcg(reinterpret_cast<const double2 *>(
                        A.mu_part + (((size_t)d * n_splits + s) * PB + p) * mu_ld + col));
            }
#pragma unroll
            for (int u = 0; u < kBatch; ++u)
                if (s0 + u < n_splits) {
#pragma unroll
                    for (int p = 0; p < PB; ++p) { m0[p] += v[u][p].x; m1[p] += v[u][p].y; }
                }
        }
    }
#pragma unroll
    for (int p = 0; p < PB; ++p) {
        double t = 0.0;
        if (col_ok && p < Pb) {
            const double a0 = m0[p] + bk0, a1 = m1[p] + bk1;
            if (A.out_mu) {
                double *dst = A.out_mu + ((size_t)p * A.D + d) * n_rec + col;
                dst[0] = a0;
                if (ok1) dst[1] = a1;
            }
            t = poisson_term(a0, cn0) + (ok1 ? poisson_term(a1, cn1) : 0.0);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) red[warp][p] = t;
    }
    __syncthreads();
    if (threadIdx.x < PB) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kStreamThreads / 32; ++w) v += red[w][threadIdx.x];
        __stcg(A.strip_part + (size_t)sid * kStreamMaxPB + threadIdx.x, v);
    }

    // ---------------------------------------------------------------- last strip: sum strips and periods, write
    const int n_sid = n_strips * A.D;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(A.cnt + n_sid, 1) == n_sid - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    {   // warp w adds the strips w, w + 8, ... of point `lane`, then the eight warps in order: fixed order, one round trip
        double v = 0.0;
        if (lane < Pb)
            for (int q = warp; q < n_sid; q += kStreamThreads / 32) v += __ldcg(A.strip_part + (size_t)q * kStreamMaxPB + lane);
        if (lane < PB) red[warp][lane] = v;
    }
    __syncthreads();
    if (threadIdx.x < Pb) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kStreamThreads / 32; ++w) v += red[w][threadIdx.x];
        v *= 2.0;
        if (A.sat_const) v += A.sat_const[0];
        A.out[threadIdx.x] = v;
    }
    for (int q = threadIdx.x; q <= n_sid; q += kStreamThreads) A.cnt[q] = 0;     // ready for the next launch
}

template <int PB>
static void launch_stream_t(const StreamArgs &A, const Kinds &kd, const Consts &cst, dim3 grid, cudaStream_t s)
{
    k_fold_stream<PB><<<grid, kStreamThreads, 0, s>>>(A, kd, cst);
}

cudaError_t launch_fold_stream(rw_ctx *ctx, const double *coef, const double *param, const Kinds *kd,
                               const double *wts, int Pb, double *out, bool full_eq18, double *out_mu,
                               cudaStream_t s, const double *rate_rows)
{
    // `coef` is ctx->coef + 12 g0 for the group starting at point g0 (or the identity of the prefold, which is
    // never run with several components): its rates are ctx->rate + 4 g0
    const double *rate = rate_rows;
    if (!rate && coef && ctx->comp8 && coef >= ctx->coef && coef < ctx->coef + (size_t)ctx->lay.max_batch * kCoefStride)
        rate = ctx->rate + (coef - ctx->coef) / kCoefStride * RW_MAX_COMPONENTS;
    const Layout &L = ctx->lay;
    StreamArgs A;
    A.R = ctx->R; A.R_period_stride = ctx->R_period_stride; A.ldR = ctx->ldR;
    A.n_T = ctx->n_T; A.n_rec = ctx->n_rec; A.D = ctx->D;
    A.coef = coef; A.param = param; A.wts = wts;
    A.rate = rate; A.comp8 = ctx->comp8;
    A.What = ctx->What; A.N_mc = ctx->N_mc; A.bkg = ctx->bkg; A.counts = ctx->counts;
    A.sat_const = full_eq18 ? ctx->sat_const : nullptr;
    A.Pb = Pb;
    A.rows_per_split = ((ctx->n_T + L.stream_splits - 1) / L.stream_splits + kRC - 1) / kRC * kRC;
    A.n_splits = (ctx->n_T + A.rows_per_split - 1) / A.rows_per_split;
    A.mu_ld = (ctx->n_rec + 1) & ~1;
    A.mu_part = ctx->mu_part; A.strip_part = ctx->strip_part; A.cnt = ctx->stream_cnt;
    A.out = out; A.out_mu = out_mu;
    Kinds none;
    none.k = 0;
    for (int a = 0; a < RW_N_KINDS; ++a) none.kind[a] = -1;
    const Kinds &k = kd ? *kd : none;
    dim3 grid(L.stream_strips, A.n_splits, ctx->D);
    {
        ProfScope prof(ctx, s);
        if (!out) launch_stream_t<16>(A, k, ctx->cst, grid, s);           // prefold: PB = 16 layout of mu_part
        else if (Pb <= 1) launch_stream_t<1>(A, k, ctx->cst, grid, s);
        else if (Pb <= 2) launch_stream_t<2>(A, k, ctx->cst, grid, s);
        else if (Pb <= 4) launch_stream_t<4>(A, k, ctx->cst, grid, s);
        else if (Pb <= 8) launch_stream_t<8>(A, k, ctx->cst, grid, s);
        else launch_stream_t<16>(A, k, ctx->cst, grid, s);
    }
    ctx->launches++;
    return cudaGetLastError();
}

// out[p] = 2 * sum_parts partial[part][p] (+ saturated constant for the literal Eq. 18), fixed order.
__global__ void k_reduce(const double *__restrict__ partial, int n_parts, int64_t part_stride, int64_t Pc,
                         const double *__restrict__ sat_const, double *__restrict__ out)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= Pc) return;
    double v = 0.0;
    for (int q = 0; q < n_parts; ++q) v += partial[(size_t)q * part_stride + p];
    v *= 2.0;
    if (sat_const) v += sat_const[0];
    out[p] = v;
}

// bound[p] = max over parts of cert[part][p]: the certified relative error of the sliced contraction per point.
__global__ void k_reduce_max(const double *__restrict__ cert, int n_parts, int64_t part_stride, int64_t Pc,
                             double *__restrict__ bound)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= Pc) return;
    double v = 0.0;
    for (int q = 0; q < n_parts; ++q) v = fmax(v, cert[(size_t)q * part_stride + p]);
    bound[p] = v;
}

cudaError_t launch_reduce_max(rw_ctx *ctx, int n_parts, int64_t part_stride, int64_t Pc, double *bound, cudaStream_t s)
{
    k_reduce_max<<<(unsigned)((Pc + 255) / 256), 256, 0, s>>>(ctx->cert_part, n_parts, part_stride, Pc, bound);
    ctx->launches++;
    return cudaGetLastError();
}

// Strict mode: the points of a slice whose certified bound exceeds `tol` (NaN bounds included) -> compact list.
// idx[0 .. *count) ascending (one thread block scans in order, so the list -- and with it the fallback -- is
// deterministic); their coefficient and rate rows are gathered next to it.
__global__ void __launch_bounds__(1024)
k_collect_uncertified(const double *__restrict__ bound, int64_t Ps, double tol, const double *__restrict__ coef,
                      const double *__restrict__ rate, int *__restrict__ idx, int *__restrict__ count,
                      double *__restrict__ coef_fb, double *__restrict__ rate_fb)
{
    __shared__ int s_warp[32], s_base;
    if (threadIdx.x == 0) s_base = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int64_t p0 = 0; p0 < Ps; p0 += 1024) {
        const int64_t p = p0 + threadIdx.x;
        const bool bad = p < Ps && !(bound[p] <= tol);
        const unsigned m = __ballot_sync(0xffffffffu, bad);
        if (lane == 0) s_warp[warp] = __popc(m);
        __syncthreads();
        int off = s_base;
        for (int w = 0; w < warp; ++w) off += s_warp[w];
        if (bad) {
            const int q = off + __popc(m & ((1u << lane) - 1));
            idx[q] = (int)p;
            if (coef) {
#pragma unroll
            for (int b = 0; b < kCoefStride; ++b) coef_fb[(size_t)q * kCoefStride + b] = coef[(size_t)p * kCoefStride + b];
#pragma unroll
            for (int c = 0; c < RW_MAX_COMPONENTS; ++c) rate_fb[(size_t)q * RW_MAX_COMPONENTS + c] = rate[(size_t)p * RW_MAX_COMPONENTS + c];
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) { int t = 0; for (int w = 0; w < 32; ++w) t += s_warp[w]; s_base += t; }
        __syncthreads();
    }
    if (threadIdx.x == 0) *count = s_base;
}

// out[idx[q]] = out_fb[q], bound[idx[q]] = 0 (recomputed in FP64 by the DMMA path)
__global__ void k_scatter_fallback(const int *__restrict__ idx, int n, const double *__restrict__ out_fb,
                                   double *__restrict__ out, double *__restrict__ bound)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    out[idx[q]] = out_fb[q];
    if (bound) bound[idx[q]] = 0.0;
}

cudaError_t launch_collect_uncertified(rw_ctx *ctx, const double *bound, int64_t Ps, double tol, bool gather, cudaStream_t s)
{
    k_collect_uncertified<<<1, 1024, 0, s>>>(bound, Ps, tol, gather ? ctx->coef : nullptr, ctx->rate, ctx->fb_idx, ctx->fb_idx + ctx->lay.MC,
                                             ctx->coef_fb, ctx->rate_fb);
    ctx->launches++;
    return cudaGetLastError();
}

cudaError_t launch_scatter_fallback(rw_ctx *ctx, int n, double *out, double *bound, cudaStream_t s)
{
    k_scatter_fallback<<<(n + 255) / 256, 256, 0, s>>>(ctx->fb_idx, n, ctx->out_fb, out, bound);
    ctx->launches++;
    return cudaGetLastError();
}

cudaError_t launch_reduce(rw_ctx *ctx, int n_parts, int64_t part_stride, int64_t Pc, double *out,
                          bool full_eq18, cudaStream_t s)
{
    k_reduce<<<(unsigned)((Pc + 255) / 256), 256, 0, s>>>(ctx->partial, n_parts, part_stride, Pc,
                                                          full_eq18 ? ctx->sat_const : nullptr, out);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
