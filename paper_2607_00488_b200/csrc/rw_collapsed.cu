// rw_collapsed.cu -- opt-in RW_MODE_COLLAPSED: rank-K prefolded templates.
//
// Eq. (4) is quadratic in the couplings, Eq. (8) linear in mu_nu^2, and the
// fold of Eq. (11) is linear in the recoil spectrum, so
//     mu[p][d][k] - bkg[d][k] = sum_{b<11} c_b(theta_p) G[d][b][k],   G[d][b][k] = sum_i W^[d][b][i] R[d][i][k]
// holds exactly.  rw_create folds the 11 templates once (k_fold_stream with identity coefficients: the
// templates are "points" whose coefficient vectors are unit vectors), and a point then costs
// 2*11*n_rec*D flop plus the Poisson terms of Eq. (18) instead of 2*n_T*n_rec*D.
// This path is bound by plain FP64 ALU work (the log1p of every bin), not by HBM or the tensor pipe;
// bench.py reports it on its own line and never mixes it into the dense-fold figure.
#include "rw_internal.h"

namespace rw {

constexpr int kColThreads = 256;
constexpr int kColCols = 2 * kColThreads;   // reconstructed bins per CTA strip, two per thread
constexpr int kColPB = 64;                  // points per CTA

// G[d][b][k] = sum over row splits of the streaming fold's partial sums (fixed order).
__global__ void k_sum_splits(const double *__restrict__ mu_part, int n_splits, int PB, int mu_ld, int n_rec,
                             int ldG, int n_comp, int q, double *__restrict__ G /*[D][n_comp][12][ldG]*/)
{
    const int b = blockIdx.y, d = blockIdx.z;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= ldG) return;
    double v = 0.0;
    if (col < n_rec && b < kNumTerms)
        for (int s = 0; s < n_splits; ++s) v += mu_part[(((size_t)d * n_splits + s) * PB + b) * mu_ld + col];
    G[(((size_t)d * n_comp + q) * kCoefStride + b) * ldG + col] = v;
}

// ident[16][12] unit coefficient rows, then rate[16][4]: every row the unit vector of component `comp` (a template of
// component q is the fold of W^_b masked to the bins of q: rate_q = 1, the others 0)
__global__ void k_identity(double *__restrict__ ident, int comp)
{
    const int q = threadIdx.x;
    if (q < kStreamMaxPB * kCoefStride) ident[q] = (q / kCoefStride == q % kCoefStride) ? 1.0 : 0.0;
    if (q < kStreamMaxPB * RW_MAX_COMPONENTS)
        ident[kStreamMaxPB * kCoefStride + q] = (q % RW_MAX_COMPONENTS == comp) ? 1.0 : 0.0;
}

// One CTA: kColPB points x one 512-column strip of one period.  The 11 template values of the thread's two
// columns stay in registers; per point: 11-term dot product, + bkg, Poisson term, warp-shuffle sum, then one
// shared-memory pass over the 8 warps.  partial[(d * nstrip + strip)][p] feeds k_reduce (fixed order).
// Several components (Eq. 17): mu - bkg = sum_q rate_q sum_b c_b G[d][q][b][k]; the templates are read through L1
// (11 n_comp x 512 columns x 8 bytes per strip) instead of living in registers.
__global__ void __launch_bounds__(kColThreads)
k_collapsed_multi(const double *__restrict__ G, int ldG, int n_rec, int D, int n_comp, const double *__restrict__ coef,
                  const double *__restrict__ rate, int64_t Pc, const double *__restrict__ bkg,
                  const double *__restrict__ counts, double *__restrict__ partial, int64_t part_stride,
                  double *__restrict__ out_mu)
{
    __shared__ double sC[kColPB][kCoefStride];
    __shared__ double sR[kColPB][RW_MAX_COMPONENTS];
    __shared__ double red[kColThreads / 32][kColPB];
    const int d = blockIdx.z;
    const int64_t p0 = (int64_t)blockIdx.y * kColPB;
    const int np = (int)min((int64_t)kColPB, Pc - p0);
    const int col = blockIdx.x * kColCols + 2 * threadIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int q = threadIdx.x; q < kColPB * kCoefStride; q += kColThreads) {
        const int p = q / kCoefStride, b = q - p * kCoefStride;
        sC[p][b] = (p < np) ? coef[(p0 + p) * kCoefStride + b] : 0.0;
    }
    for (int q = threadIdx.x; q < kColPB * RW_MAX_COMPONENTS; q += kColThreads) {
        const int p = q / RW_MAX_COMPONENTS, c = q - p * RW_MAX_COMPONENTS;
        sR[p][c] = (p < np) ? rate[(p0 + p) * RW_MAX_COMPONENTS + c] : 0.0;
    }
    const bool ok0 = col < n_rec, ok1 = col + 1 < n_rec;
    const double bk0 = ok0 ? bkg[(size_t)d * n_rec + col] : 0.0, bk1 = ok1 ? bkg[(size_t)d * n_rec + col + 1] : 0.0;
    const double cn0 = ok0 ? counts[(size_t)d * n_rec + col] : 0.0, cn1 = ok1 ? counts[(size_t)d * n_rec + col + 1] : 0.0;
    const double ci0 = cn0 > 0.0 ? 1.0 / cn0 : 0.0, ci1 = cn1 > 0.0 ? 1.0 / cn1 : 0.0;
    __syncthreads();
    for (int p = 0; p < np; ++p) {
        double m0 = bk0, m1 = bk1;
        for (int q = 0; q < n_comp; ++q) {
            const double *Gq = G + ((size_t)d * n_comp + q) * kCoefStride * ldG + col;
            double a0 = 0.0, a1 = 0.0;
#pragma unroll
            for (int b = 0; b < kNumTerms; ++b) {
                const double2 v = ok0 ? __ldg(reinterpret_cast<const double2 *>(Gq + (size_t)b * ldG)) : make_double2(0.0, 0.0);
                a0 = fma(sC[p][b], v.x, a0);
                a1 = fma(sC[p][b], v.y, a1);
            }
            m0 = fma(sR[p][q], a0, m0);
            m1 = fma(sR[p][q], a1, m1);
        }
        if (out_mu) {
            double *dst = out_mu + ((size_t)(p0 + p) * D + d) * n_rec + col;
            if (ok0) dst[0] = m0;
            if (ok1) dst[1] = m1;
        }
        double t = poisson_term_inv(m0, cn0, ci0) + poisson_term_inv(m1, cn1, ci1);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) red[warp][p] = t;
    }
    __syncthreads();
    if (threadIdx.x < np) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kColThreads / 32; ++w) v += red[w][threadIdx.x];
        partial[((size_t)d * gridDim.x + blockIdx.x) * part_stride + p0 + threadIdx.x] = v;
    }
}

// (three CTAs per SM: 80 registers and 48 bytes of spills beat 91 registers and two CTAs by 9 % -- the kernel is bound
// by the FP64 pipe behind the dependent chain of its log1p, profiles/r02_alu_kernels.md)
__global__ void __launch_bounds__(kColThreads, 3)
k_collapsed(const double *__restrict__ G, int ldG, int n_rec, int D, const double *__restrict__ coef,
            const double *__restrict__ rate /*[.][4]: rate[.][0] scales the single component*/, int64_t Pc, const double *__restrict__ bkg, const double *__restrict__ counts,
            double *__restrict__ partial, int64_t part_stride, double *__restrict__ out_mu)
{
    __shared__ double sC[kColPB][kCoefStride];
    __shared__ double red[kColThreads / 32][kColPB];
    const int d = blockIdx.z;
    const int64_t p0 = (int64_t)blockIdx.y * kColPB;
    const int np = (int)min((int64_t)kColPB, Pc - p0);
    const int col = blockIdx.x * kColCols + 2 * threadIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    for (int q = threadIdx.x; q < kColPB * kCoefStride; q += kColThreads) {
        const int p = q / kCoefStride, b = q - p * kCoefStride;
        // slot 11 of the coefficient row is padding: it carries the point's rate scale here
        sC[p][b] = (p < np) ? (b == kCoefStride - 1 ? rate[(p0 + p) * RW_MAX_COMPONENTS] : coef[(p0 + p) * kCoefStride + b]) : 0.0;
    }
    double g[kNumTerms][2], bk[2], cn[2], ci[2];
    const bool ok0 = col < n_rec, ok1 = col + 1 < n_rec;
    {
        const double *Gd = G + (size_t)d * kCoefStride * ldG;
#pragma unroll
        for (int b = 0; b < kNumTerms; ++b) {
            // ldG is even and col is even: one 16-byte load; columns >= n_rec hold zeros
            const double2 v = ok0 ? *reinterpret_cast<const double2 *>(Gd + (size_t)b * ldG + col)
                                  : make_double2(0.0, 0.0);
            g[b][0] = v.x; g[b][1] = v.y;
        }
        bk[0] = ok0 ? bkg[(size_t)d * n_rec + col] : 0.0;
        bk[1] = ok1 ? bkg[(size_t)d * n_rec + col + 1] : 0.0;
        cn[0] = ok0 ? counts[(size_t)d * n_rec + col] : 0.0;
        cn[1] = ok1 ? counts[(size_t)d * n_rec + col + 1] : 0.0;
        ci[0] = cn[0] > 0.0 ? 1.0 / cn[0] : 0.0;
        ci[1] = cn[1] > 0.0 ? 1.0 / cn[1] : 0.0;
    }
    __syncthreads();
    // two points per trip: four independent log1p chains per thread keep the FP64 pipe fed at 16 warps per SM
    for (int p = 0; p < np; p += 2) {
        double m[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
        for (int b = 0; b < kNumTerms; ++b) {
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const double c = sC[p + u][b];            // rows >= np hold zeros
                m[u][0] = fma(c, g[b][0], m[u][0]);
                m[u][1] = fma(c, g[b][1], m[u][1]);
            }
        }
        double t[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const double rt = sC[p + u][kCoefStride - 1];             // rate_k of Eq. (17), 1 when not scanned
            const double m0 = fma(rt, m[u][0], bk[0]), m1 = fma(rt, m[u][1], bk[1]);
            if (out_mu && p + u < np) {
                double *dst = out_mu + ((size_t)(p0 + p + u) * D + d) * n_rec + col;
                if (ok0) dst[0] = m0;
                if (ok1) dst[1] = m1;
            }
            // columns >= n_rec carry template 0, bkg 0, n 0: their term is exactly 0
            t[u] = poisson_term_inv(m0, cn[0], ci[0]) + poisson_term_inv(m1, cn[1], ci[1]);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            t[0] += __shfl_xor_sync(0xffffffffu, t[0], o);
            t[1] += __shfl_xor_sync(0xffffffffu, t[1], o);
        }
        if (lane == 0) { red[warp][p] = t[0]; red[warp][p + 1] = t[1]; }
    }
    __syncthreads();
    if (threadIdx.x < np) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kColThreads / 32; ++w) v += red[w][threadIdx.x];
        partial[((size_t)d * gridDim.x + blockIdx.x) * part_stride + p0 + threadIdx.x] = v;
    }
}

cudaError_t launch_prefold(rw_ctx *ctx, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    const int rows_per_split = ((ctx->n_T + L.stream_splits - 1) / L.stream_splits + 63) / 64 * 64;
    const int n_splits = (ctx->n_T + rows_per_split - 1) / rows_per_split;
    const int mu_ld = (ctx->n_rec + 1) & ~1;
    for (int q = 0; q < ctx->n_comp; ++q) {
        k_identity<<<1, 256, 0, s>>>(ctx->ident, q);
        ctx->launches++;
        // the 11 templates of component q are folded as 11 "points" with unit coefficient vectors and the unit rate
        // vector of q (no deviance pass)
        cudaError_t e = launch_fold_stream(ctx, ctx->ident, nullptr, nullptr, nullptr, kNumTerms, nullptr, false, nullptr, s,
                                           ctx->ident + kStreamMaxPB * kCoefStride);
        if (e != cudaSuccess) return e;
        dim3 grid((L.ldG + 255) / 256, kCoefStride, ctx->D);
        k_sum_splits<<<grid, 256, 0, s>>>(ctx->mu_part, n_splits, kStreamMaxPB, mu_ld, ctx->n_rec, L.ldG, ctx->n_comp, q, ctx->G);
        ctx->launches++;
    }
    return cudaGetLastError();
}

cudaError_t launch_collapsed(rw_ctx *ctx, int64_t p0, int64_t Pc, double *out_mu, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    const int nstrip = (ctx->n_rec + kColCols - 1) / kColCols;
    dim3 grid(nstrip, (unsigned)((Pc + kColPB - 1) / kColPB), ctx->D);
    ProfScope prof(ctx, s);
    if (ctx->n_comp > 1)
        k_collapsed_multi<<<grid, kColThreads, 0, s>>>(ctx->G, L.ldG, ctx->n_rec, ctx->D, ctx->n_comp, ctx->coef + p0 * kCoefStride,
                                                       ctx->rate + p0 * RW_MAX_COMPONENTS, Pc, ctx->bkg, ctx->counts,
                                                       ctx->partial, L.MC, out_mu);
    else
    k_collapsed<<<grid, kColThreads, 0, s>>>(ctx->G, L.ldG, ctx->n_rec, ctx->D, ctx->coef + p0 * kCoefStride,
                                             ctx->rate + p0 * RW_MAX_COMPONENTS, Pc,
                                             ctx->bkg, ctx->counts, ctx->partial, L.MC, out_mu);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
