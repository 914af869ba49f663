// rw_fold_stream.cu -- steps a3 + a4 for small batches (P <= 16 per pass): HBM-streaming fold.
//
// With few points the fold mu[p][k] = sum_i N'[p][i] R[i][k] + bkg[k] (Eq. 11) reads
// every byte of R once and does 2P flop per 8 bytes: it is bound by HBM bandwidth, not arithmetic.
// R is row-major with the reconstructed index fastest, so a thread owns two adjacent columns
// (one 16-byte load per row), a CTA owns a 512-column strip, and the recoil rows are split over
// gridDim.y so that the grid fills all SMs several times over.  N'[p][i] (Eq. 14 / Eq. 1) is
// formed on the fly from the 11-term pre-scaled basis and staged in shared memory.
// The row-split partial sums are combined in a fixed order by k_stream_deviance, which adds the
// background and reduces the Poisson terms of Eq. (18) per point: warp shuffles,
// then one shared-memory pass per CTA; k_reduce finishes over strips and periods.
#include "rw_internal.h"

namespace rw {

constexpr int kRC = 64;   // recoil rows staged per iteration

template <int PB>
__global__ void __launch_bounds__(kStreamThreads)
k_fold_stream(const double *__restrict__ R, size_t R_period_stride, int ldR, int n_T, int n_rec,
              const double *__restrict__ coef, int Pb, const double *__restrict__ What,
              const double *__restrict__ wts /*NULL, or caller weights [Pb][n_T] (rw_eval_weights)*/,
              const double *__restrict__ N_mc /*[D][n_T], used with wts*/,
              int rows_per_split, int n_splits, int mu_ld, double *__restrict__ mu_part)
{
    __shared__ __align__(16) double sN[kRC][PB];
    __shared__ double sC[PB][kNumTerms];
    const int d = blockIdx.z;
    const int split = blockIdx.y;
    const int col = blockIdx.x * kStreamCols + 2 * threadIdx.x;
    const int i0 = split * rows_per_split;
    const int i1 = min(n_T, i0 + rows_per_split);
    const double *Rd = R + (size_t)d * R_period_stride;
    const double *Wd = What + (size_t)d * kCoefStride * n_T;

    if (!wts)
        for (int q = threadIdx.x; q < PB * kNumTerms; q += kStreamThreads) {
            int p = q / kNumTerms, b = q - p * kNumTerms;
            sC[p][b] = (p < Pb) ? coef[(size_t)p * kCoefStride + b] : 0.0;
        }
    double acc[PB][2];
#pragma unroll
    for (int p = 0; p < PB; ++p) acc[p][0] = acc[p][1] = 0.0;
    const bool col_ok = col < n_rec;

    for (int ic = i0; ic < i1; ic += kRC) {
        __syncthreads();
        for (int q = threadIdx.x; q < kRC * PB; q += kStreamThreads) {
            const int p = q / kRC, row = q - p * kRC;     // consecutive threads -> consecutive bins
            const int i = ic + row;
            double v = 0.0;
            if (i < i1) {
                if (wts) {          // N' = w N_mc (Eq. 1 with caller-supplied weights)
                    if (p < Pb) v = wts[(size_t)p * n_T + i] * N_mc[(size_t)d * n_T + i];
                } else {            // N' = sum_b c_b W^_b (Eq. 14 folded into the pre-scaled basis)
#pragma unroll
                    for (int b = 0; b < kNumTerms; ++b) v = fma(sC[p][b], Wd[(size_t)b * n_T + i], v);
                }
            }
            sN[row][p] = v;
        }
        __syncthreads();
        if (col_ok) {
            const double *Rp = Rd + (size_t)ic * ldR + col;
            const int nrows = min(kRC, i1 - ic);
#pragma unroll 1
            for (int r0 = 0; r0 < nrows; r0 += 8) {
                double2 rv[8];
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    rv[u] = (r0 + u < nrows)
                                ? __ldg(reinterpret_cast<const double2 *>(Rp + (size_t)(r0 + u) * ldR))
                                : make_double2(0.0, 0.0);
#pragma unroll
                for (int u = 0; u < 8; ++u) {
#pragma unroll
                    for (int p = 0; p < PB; ++p) {
                        const double n = sN[r0 + u][p];
                        acc[p][0] = fma(n, rv[u].x, acc[p][0]);
                        acc[p][1] = fma(n, rv[u].y, acc[p][1]);
                    }
                }
            }
        }
    }
    if (col_ok) {
#pragma unroll
        for (int p = 0; p < PB; ++p) {
            double *dst = mu_part + (((size_t)d * n_splits + split) * PB + p) * mu_ld + col;
            *reinterpret_cast<double2 *>(dst) = make_double2(acc[p][0], acc[p][1]);
        }
    }
}

// mu = sum_split partial + bkg; Poisson term; per-CTA reduction -> partial[(d*nstrip + strip)][p].
__global__ void __launch_bounds__(256)
k_stream_deviance(const double *__restrict__ mu_part, int n_splits, int PB, int mu_ld, int n_rec,
                  const double *__restrict__ bkg, const double *__restrict__ counts, int D,
                  double *__restrict__ out_mu /*[P][D][n_rec] rows of this group, or NULL*/,
                  double *__restrict__ partial /*[D*nstrip][kStreamMaxPB]*/)
{
    const int p = blockIdx.y, d = blockIdx.z;
    const int col = blockIdx.x * 256 + threadIdx.x;
    double term = 0.0;
    if (col < n_rec) {
        double mu = 0.0;
        for (int s = 0; s < n_splits; ++s)
            mu += mu_part[(((size_t)d * n_splits + s) * PB + p) * mu_ld + col];
        mu += bkg[(size_t)d * n_rec + col];
        if (out_mu) out_mu[((size_t)p * D + d) * n_rec + col] = mu;
        term = poisson_term(mu, counts[(size_t)d * n_rec + col]);
    }
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) term += __shfl_down_sync(0xffffffffu, term, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = term;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) v += red[w];
        partial[((size_t)d * gridDim.x + blockIdx.x) * kStreamMaxPB + p] = v;
    }
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

template <int PB>
static void launch_stream_t(rw_ctx *ctx, const double *coef, const double *wts, int Pb, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    const int rows_per_split = ((ctx->n_T + L.stream_splits - 1) / L.stream_splits + kRC - 1) / kRC * kRC;
    const int n_splits = (ctx->n_T + rows_per_split - 1) / rows_per_split;
    dim3 grid(L.stream_strips, n_splits, ctx->D);
    const int mu_ld = (ctx->n_rec + 1) & ~1;
    k_fold_stream<PB><<<grid, kStreamThreads, 0, s>>>(
        ctx->R, ctx->R_period_stride, ctx->ldR, ctx->n_T, ctx->n_rec, coef, Pb,
        ctx->What, wts, ctx->N_mc, rows_per_split, n_splits, mu_ld, ctx->mu_part);
}

// Pb > 0: fold Pb points (coefficients `coef`, or caller weights `wts`) and reduce the Poisson terms.
// Pb < 0: fold -Pb coefficient vectors only (the template prefold of rw_collapsed.cu; partials stay in mu_part
//         laid out for PB = 16).
cudaError_t launch_fold_stream(rw_ctx *ctx, const double *coef, const double *wts, int Pb, double *out_mu,
                               cudaStream_t s)
{
    const Layout &L = ctx->lay;
    if (Pb < 0) {
        launch_stream_t<16>(ctx, coef, nullptr, -Pb, s);
        ctx->launches++;
        return cudaGetLastError();
    }
    int PB;
    {
        ProfScope prof(ctx, s);
        if (Pb <= 1) { PB = 1; launch_stream_t<1>(ctx, coef, wts, Pb, s); }
        else if (Pb <= 2) { PB = 2; launch_stream_t<2>(ctx, coef, wts, Pb, s); }
        else if (Pb <= 4) { PB = 4; launch_stream_t<4>(ctx, coef, wts, Pb, s); }
        else if (Pb <= 8) { PB = 8; launch_stream_t<8>(ctx, coef, wts, Pb, s); }
        else { PB = 16; launch_stream_t<16>(ctx, coef, wts, Pb, s); }
    }
    const int rows_per_split = ((ctx->n_T + L.stream_splits - 1) / L.stream_splits + kRC - 1) / kRC * kRC;
    const int n_splits = (ctx->n_T + rows_per_split - 1) / rows_per_split;
    const int mu_ld = (ctx->n_rec + 1) & ~1;
    const int nstrip2 = (ctx->n_rec + 255) / 256;
    dim3 grid2(nstrip2, Pb, ctx->D);
    k_stream_deviance<<<grid2, 256, 0, s>>>(ctx->mu_part, n_splits, PB, mu_ld, ctx->n_rec, ctx->bkg,
                                            ctx->counts, ctx->D, out_mu, ctx->partial);
    ctx->launches += 2;
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
