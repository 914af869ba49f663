// rw_grad.cu -- analytic gradient of -2lnL with respect to the scanned parameters (rest of SURVEY.md section 8 f-2:
// "analytic gradient for minimisers"; the paper minimises Eq. 18 with MIGRAD).
//
// Everything on the path is linear in the coefficient vector c(theta) and in the rates, so the derivative of the
// prediction is the SAME fold applied to derivative coefficients:
//     dmu/dtheta_m = fold( rate_c(i) * sum_b (dc_b/dtheta_m) W^_b[i] )            (Eq. 11 is linear)
//     dc/d eps^L_a : d(gL^2) = 2 gL, d(gL gR) = gR;   dc/d eps^R_a : d(gR^2) = 2 gR, d(gL gR) = gL   (Eq. 4/6)
//     dc/d mu_nu   : d(mu_nu^2) = 2 mu_nu                                                          (Eq. 8)
//     d/d rate_c   : the component's own content (coefficients c, rate vector = unit vector e_c)    (Eq. 17)
//     d(-2lnL)/dtheta_m = sum_j 2 (1 - n_j/mu_j) dmu_j/dtheta_m                     (Eq. 18; n_j = 0: 2 dmu_j)
// A point therefore becomes 1 + k rows of the ordinary batched fold (k_coef_grad writes their coefficient and
// rate rows), mu of all rows goes to the scratch, and k_grad (one CTA per point) contracts them.
// Under RW_SLICED / RW_SLICED_FAST the rows must be non-negative (fixed point): a derivative row, which changes sign
// along the recoil bins, is folded as TWO rows -- its positive part max(v, 0) with coefficients dc and its negative
// part max(-v, 0) with coefficients -dc (slot 11 of the coefficient row = 1 tells k_slice_A to clamp instead of
// rejecting the row) -- and k_grad takes their difference: 1 + 2 k rows per point.
#include "rw_internal.h"

namespace rw {

template <bool SPLIT>
__global__ void k_coef_grad(const double *__restrict__ param, int64_t P, Kinds kd, Consts cst,
                            double *__restrict__ coef /*[(1+k) P][12]*/, double *__restrict__ rate /*[(1+k) P][4]*/)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= P) return;
    const double *prow = param + p * kd.k;
    double c[kCoefStride], r[RW_MAX_COMPONENTS];
    coef_from_param(prow, kd, cst, c, r);
    const int64_t row0 = p * (1 + (SPLIT ? 2 : 1) * kd.k);
#pragma unroll
    for (int b = 0; b < kCoefStride; ++b) coef[row0 * kCoefStride + b] = c[b];
#pragma unroll
    for (int q = 0; q < RW_MAX_COMPONENTS; ++q) rate[row0 * RW_MAX_COMPONENTS + q] = r[q];
    // couplings at this point (Eq. 6): needed for the derivative monomials
    double th[RW_RATE_0];
#pragma unroll
    for (int q = 0; q < RW_RATE_0; ++q) th[q] = 0.0;
    for (int a = 0; a < kd.k; ++a)
#pragma unroll
        for (int q = 0; q < RW_RATE_0; ++q)
            if (kd.kind[a] == q) th[q] = prow[a];
    for (int a = 0; a < kd.k; ++a) {
        const int kind = kd.kind[a];
        double dc[kCoefStride], dr[RW_MAX_COMPONENTS];
#pragma unroll
        for (int b = 0; b < kCoefStride; ++b) dc[b] = 0.0;
#pragma unroll
        for (int q = 0; q < RW_MAX_COMPONENTS; ++q) dr[q] = r[q];
        if (kind >= RW_RATE_0) {                       // rate of one component: its own content
#pragma unroll
            for (int b = 0; b < kCoefStride; ++b) dc[b] = c[b];
#pragma unroll
            for (int q = 0; q < RW_MAX_COMPONENTS; ++q) dr[q] = (q == kind - RW_RATE_0) ? 1.0 : 0.0;
        } else if (kind == RW_MU_NU) {
            dc[9] = 2.0 * th[RW_MU_NU];
        } else {
            const int fl = kind >> 1;
            const double gl = cst.gL[fl] + th[2 * fl], gr = cst.gR[fl] + th[2 * fl + 1];
            if ((kind & 1) == 0) { dc[3 * fl] = 2.0 * gl; dc[3 * fl + 2] = gr; }
            else                 { dc[3 * fl + 1] = 2.0 * gr; dc[3 * fl + 2] = gl; }
        }
        if (!SPLIT) {
            const int64_t row = row0 + 1 + a;
#pragma unroll
            for (int b = 0; b < kCoefStride; ++b) coef[row * kCoefStride + b] = dc[b];
#pragma unroll
            for (int q = 0; q < RW_MAX_COMPONENTS; ++q) rate[row * RW_MAX_COMPONENTS + q] = dr[q];
        } else {
            const int64_t row = row0 + 1 + 2 * a;            // positive part, then negative part
#pragma unroll
            for (int b = 0; b < kCoefStride - 1; ++b) {
                coef[row * kCoefStride + b] = dc[b];
                coef[(row + 1) * kCoefStride + b] = -dc[b];
            }
            coef[row * kCoefStride + kCoefStride - 1] = 1.0;  // clamp marker (W^ row 11 is zero: no contribution)
            coef[(row + 1) * kCoefStride + kCoefStride - 1] = 1.0;
#pragma unroll
            for (int q = 0; q < RW_MAX_COMPONENTS; ++q) {
                rate[row * RW_MAX_COMPONENTS + q] = dr[q];
                rate[(row + 1) * RW_MAX_COMPONENTS + q] = dr[q];
            }
        }
    }
}

constexpr int kGradThreads = 256;

// One CTA per point.  rows[(1+k)][nb]: mu of the point, then (dmu/dtheta_m + bkg) for every parameter; SPLIT:
// rows[(1+2k)][nb] with (positive part + bkg, negative part + bkg) per parameter.
template <bool SPLIT>
__global__ void __launch_bounds__(kGradThreads)
k_grad(const double *__restrict__ rows, int nb, int k, const double *__restrict__ bkg,
       const double *__restrict__ counts, const double *__restrict__ sat_const, double *__restrict__ out,
       double *__restrict__ grad)
{
    __shared__ double red[kGradThreads / 32][1 + RW_N_KINDS];
    const double *mu_row = rows + (size_t)blockIdx.x * (1 + (SPLIT ? 2 : 1) * k) * nb;
    double acc[1 + RW_N_KINDS];
#pragma unroll
    for (int m = 0; m <= RW_N_KINDS; ++m) acc[m] = 0.0;
    for (int j = threadIdx.x; j < nb; j += kGradThreads) {
        const double mu = mu_row[j], n = counts[j], b = bkg[j];
        acc[0] += poisson_term(mu, n);
        const double g = (n > 0.0) ? 1.0 - n / mu : 1.0;          // d term / d mu
#pragma unroll
        for (int m = 0; m < RW_N_KINDS; ++m)
            if (m < k) {
                const double dmu = SPLIT ? mu_row[(size_t)(1 + 2 * m) * nb + j] - mu_row[(size_t)(2 + 2 * m) * nb + j]
                                         : mu_row[(size_t)(1 + m) * nb + j] - b;
                acc[1 + m] = fma(g, dmu, acc[1 + m]);
            }
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int m = 0; m <= RW_N_KINDS; ++m) {
        double v = acc[m];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][m] = v;
    }
    __syncthreads();
    if (threadIdx.x <= k) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kGradThreads / 32; ++w) v += red[w][threadIdx.x];
        v *= 2.0;
        if (threadIdx.x == 0) out[blockIdx.x] = sat_const ? v + sat_const[0] : v;
        else grad[(size_t)blockIdx.x * k + threadIdx.x - 1] = v;
    }
}

cudaError_t launch_coef_grad(rw_ctx *ctx, const double *param, int64_t P, int k, const int *kinds, cudaStream_t s,
                             bool split)
{
    Kinds kd;
    kd.k = k;
    for (int a = 0; a < RW_N_KINDS; ++a) kd.kind[a] = (a < k) ? kinds[a] : -1;
    if (split) k_coef_grad<true><<<(unsigned)((P + 127) / 128), 128, 0, s>>>(param, P, kd, ctx->cst, ctx->coef, ctx->rate);
    else k_coef_grad<false><<<(unsigned)((P + 127) / 128), 128, 0, s>>>(param, P, kd, ctx->cst, ctx->coef, ctx->rate);
    ctx->launches++;
    return cudaGetLastError();
}

cudaError_t launch_grad(rw_ctx *ctx, const double *rows, int64_t P, int k, bool full_eq18, double *out, double *grad,
                        cudaStream_t s, bool split)
{
    if (split) k_grad<true><<<(unsigned)P, kGradThreads, 0, s>>>(rows, ctx->D * ctx->n_rec, k, ctx->bkg, ctx->counts,
                                                                 full_eq18 ? ctx->sat_const : nullptr, out, grad);
    else k_grad<false><<<(unsigned)P, kGradThreads, 0, s>>>(rows, ctx->D * ctx->n_rec, k, ctx->bkg, ctx->counts,
                                               full_eq18 ? ctx->sat_const : nullptr, out, grad);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
