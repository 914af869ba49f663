// rw_coef.cu -- steps a1 + a2: per-point coefficients and the reweighted MC spectrum.
//
//   k_coef    param[P][k] -> coef[P][12]:  g~ = g + eps (Eq. 6), then the monomials the
//             cross section is polynomial in: g~L^2, g~R^2, g~L g~R per flavour (Eq. 4/7,
//             PAPER.md:65,83) and mu_nu^2 (Eq. 8-9)
//   k_gen_A   N'[p][i] = w_i(theta_p) N_mc[i] = sum_b coef[p][b] W^[b][i]  (Eq. 14 and the
//             diag(r) E_true of Eq. 1), written in the 8x8-blocked layout the
//             DMMA contraction reads (rw_fold_gemm.cu).  Materialised once per (chunk, period):
//             regenerating it per output tile would redo these flops n_rec/128 times.
#include "rw_internal.h"

namespace rw {

__global__ void k_coef(const double *__restrict__ param, int64_t P, Kinds kd, Consts cst,
                       double *__restrict__ coef, double *__restrict__ rate)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= P) return;
    double c[kCoefStride], r[RW_MAX_COMPONENTS];
    coef_from_param(param + p * kd.k, kd, cst, c, r);
#pragma unroll
    for (int b = 0; b < kCoefStride; ++b) coef[p * kCoefStride + b] = c[b];
#pragma unroll
    for (int q = 0; q < RW_MAX_COMPONENTS; ++q) rate[p * RW_MAX_COMPONENTS + q] = r[q];
}

constexpr int kGenThreads = 256;   // 32 row-blocks of 8 points
constexpr int kGenKT = 128;        // recoil bins staged per CTA

// A_packed[mb][kb][r][2 c + e] = N'[p0 + 8 mb + r][8 kb + c + 4 e] (the DMMA A fragment of k-step e is the
// even/odd half of one 16-byte load); rows >= Pc and bins >= n_T are zero.
__global__ void __launch_bounds__(kGenThreads)
k_gen_A(const double *__restrict__ coef, int64_t p0, int64_t Pc, int64_t rows_pad,
        const double *__restrict__ What /*[12][n_T] of this period*/, int n_T, int KPAD, int64_t A_pitch,
        const double *__restrict__ rate /*[P][4]*/, const uint8_t *__restrict__ comp8 /*[n_T] or NULL*/,
        double *__restrict__ A)
{
    __shared__ __align__(16) double sW[kNumTerms][kGenKT];
    __shared__ uint8_t sComp[kGenKT];
    if (comp8)
        for (int q = threadIdx.x; q < kGenKT; q += kGenThreads) {
            const int i = blockIdx.y * kGenKT + q;
            sComp[q] = (i < n_T) ? comp8[i] : 0;
        }
    const int k0 = blockIdx.y * kGenKT;
    for (int q = threadIdx.x; q < kNumTerms * kGenKT; q += kGenThreads) {
        int b = q / kGenKT, kk = q - b * kGenKT;
        int i = k0 + kk;
        sW[b][kk] = (i < n_T) ? What[(size_t)b * n_T + i] : 0.0;
    }
    __syncthreads();
    const int r = threadIdx.x & 7;
    const int64_t mb = blockIdx.x * (int64_t)(kGenThreads / 8) + (threadIdx.x >> 3);
    const int64_t row = mb * 8 + r;
    if (row >= rows_pad) return;
    double c[kNumTerms];
    const bool valid = row < Pc;
#pragma unroll
    for (int b = 0; b < kNumTerms; ++b) c[b] = valid ? coef[(p0 + row) * kCoefStride + b] : 0.0;
    double rt[RW_MAX_COMPONENTS];
#pragma unroll
    for (int q = 0; q < RW_MAX_COMPONENTS; ++q) rt[q] = (valid && comp8) ? rate[(p0 + row) * RW_MAX_COMPONENTS + q] : 1.0;
    const int nkb = min(kGenKT, KPAD - k0) / 8;
    for (int kb = 0; kb < nkb; ++kb) {
        double v[8];
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) v[kk] = 0.0;
#pragma unroll
        for (int b = 0; b < kNumTerms; ++b) {
            const double2 *w2 = reinterpret_cast<const double2 *>(&sW[b][kb * 8]);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                double2 w = w2[h];
                v[2 * h] = fma(c[b], w.x, v[2 * h]);
                v[2 * h + 1] = fma(c[b], w.y, v[2 * h + 1]);
            }
        }
        if (comp8) {            // rate_k of Eq. (17): scale every bin by its component's rate
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
                const int cq = sComp[kb * 8 + kk];
                v[kk] *= (cq == 0) ? rt[0] : (cq == 1) ? rt[1] : (cq == 2) ? rt[2] : rt[3];
            }
        }
        double2 *dst = reinterpret_cast<double2 *>(A + (mb * A_pitch + (size_t)(k0 / 8 + kb) * 64 + r * 8));
#pragma unroll
        for (int h = 0; h < 4; ++h) dst[h] = make_double2(v[h], v[h + 4]);   // bins k and k+4 interleaved
    }
}

// Caller-supplied weights (rw_eval_weights): A_packed[mb][kb][r][2 c + e] = (w N_mc)[8 mb + r][8 kb + c + 4 e]
// (Eq. 1: diag(r) E_true).  A CTA transposes a 64-point x 64-bin tile through shared
// memory: rows of w are read 512 contiguous bytes per warp, the 8x8 blocks are written 512 contiguous bytes each.
constexpr int kGwRows = 64, kGwCols = 64;
__global__ void __launch_bounds__(256)
k_gen_A_weights(const double *__restrict__ w /*[Pc][n_T]*/, int64_t Pc, int64_t rows_pad,
                const double *__restrict__ N_mc /*[n_T] of this period*/, int n_T, int KPAD, int64_t A_pitch,
                double *__restrict__ A)
{
    __shared__ double tile[kGwRows][kGwCols + 1];
    const int64_t row0 = (int64_t)blockIdx.x * kGwRows;
    const int k0 = blockIdx.y * kGwCols;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int rr = warp; rr < kGwRows; rr += 8) {
        const int64_t row = row0 + rr;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int i = k0 + lane + 32 * h;
            double v = 0.0;
            if (row < Pc && i < n_T) v = w[(size_t)row * n_T + i] * N_mc[i];
            tile[rr][lane + 32 * h] = v;
        }
    }
    __syncthreads();
    // 8 x 8 blocks of this tile; warp `warp` writes the blocks of row block mb = warp
    const int64_t mb = row0 / 8 + warp;
    if (mb * 8 >= rows_pad) return;
    for (int kb = 0; kb < kGwCols / 8; ++kb) {
        if (k0 + kb * 8 >= KPAD) break;
        double *dst = A + (mb * A_pitch + (size_t)(k0 / 8 + kb) * 64);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int e = lane + 32 * h;               // element of the block: r = e / 8, position 2 c + e' = e % 8
            dst[e] = tile[warp * 8 + (e >> 3)][kb * 8 + ((e & 7) >> 1) + 4 * (e & 1)];
        }
    }
}

cudaError_t launch_gen_A_weights(rw_ctx *ctx, int d, const double *w, int64_t Pc, cudaStream_t s)
{
    const int64_t rows_pad = (Pc + kBM - 1) / kBM * kBM;
    dim3 grid((unsigned)((rows_pad + kGwRows - 1) / kGwRows), (unsigned)((ctx->lay.KPAD + kGwCols - 1) / kGwCols));
    k_gen_A_weights<<<grid, 256, 0, s>>>(w, Pc, rows_pad, ctx->N_mc + (size_t)d * ctx->n_T, ctx->n_T,
                                         ctx->lay.KPAD, ctx->lay.A_pitch, ctx->A_packed);
    ctx->launches++;
    return cudaGetLastError();
}

cudaError_t launch_coef(rw_ctx *ctx, const double *param, int64_t P, int k, const int *kinds,
                        cudaStream_t s)
{
    Kinds kd;
    kd.k = k;
    for (int a = 0; a < RW_N_KINDS; ++a) kd.kind[a] = (a < k) ? kinds[a] : -1;
    k_coef<<<(unsigned)((P + 127) / 128), 128, 0, s>>>(param, P, kd, ctx->cst, ctx->coef, ctx->rate);
    ctx->launches++;
    return cudaGetLastError();
}

cudaError_t launch_gen_A(rw_ctx *ctx, int d, int64_t p0, int64_t Pc, cudaStream_t s)
{
    const int64_t rows_pad = (Pc + kBM - 1) / kBM * kBM;
    dim3 grid((unsigned)((rows_pad + kGenThreads - 1) / kGenThreads),
              (unsigned)((ctx->lay.KPAD + kGenKT - 1) / kGenKT));
    k_gen_A<<<grid, kGenThreads, 0, s>>>(ctx->coef, p0, Pc, rows_pad,
                                         ctx->What + (size_t)d * kCoefStride * ctx->n_T, ctx->n_T,
                                         ctx->lay.KPAD, ctx->lay.A_pitch, ctx->rate, ctx->comp8, ctx->A_packed);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
