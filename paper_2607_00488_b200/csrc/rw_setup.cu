// rw_setup.cu -- step a0 (once per rw_create): theta-independent tables.
//
//   Basis_b(T_i), b = 0..9   the recoil spectrum of Eq. (12) split by its polynomial
//                            dependence on the couplings: Eq. (4) is quadratic in
//                            (gL, gR) per flavour, Eq. (8) linear in mu_nu^2
//   S_SM(T_i)                Eq. (12) at theta = 0  -- the fixed denominator of Eq. (14)
//   W^_d[b][i]               Basis_b[i] * N_mc[d][i] / S_SM[i]: weights x MC spectrum (Eq. 14, Eq. 1)
//                            reduced to an 11-term dot product per (point, recoil bin)
//   sat_const                sum 2[lnGamma(n+1) - n ln n + n]: Eq. (18) minus the deviance
//
// The paper recomputes the (E_nu x T) grid on every likelihood call; here it is
// done once, because nothing on that grid depends on theta except through 10 coefficients.
#include "rw_internal.h"

namespace rw {

// Per flux-grid entry: kinematic limit T_max = 2E^2/(m_e+2E) (north_star; reading R2:
// binary64, one expression, round-to-nearest, no contraction), 1/E and m_e/E^2.
__global__ void k_energy_tables(int n_E, const double *__restrict__ E, double m_e,
                                double *__restrict__ out /*[3][n_E]*/)
{
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_E) return;
    double e = E[j];
    double num = __dmul_rn(__dmul_rn(2.0, e), e);
    double den = __dadd_rn(m_e, __dmul_rn(2.0, e));
    out[j] = __ddiv_rn(num, den);
    double inv = 1.0 / e;
    out[n_E + j] = inv;
    out[2 * n_E + j] = m_e * inv * inv;
}

// Flavour probabilities: row 0 = P_e; rows 1,2 = P_mu, P_tau or the f_tau split of 1 - P_e (R3).
// Layout P3[n_comp][3][n_E]; blockIdx.y = component.
__global__ void k_flavour(int n_E, double *__restrict__ P3, int have_mu_tau, double f_tau)
{
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_E || have_mu_tau) return;
    double *Pc = P3 + (size_t)blockIdx.y * 3 * n_E;
    double pe = Pc[j];
    Pc[n_E + j] = (1.0 - pe) * (1.0 - f_tau);
    Pc[2 * n_E + j] = (1.0 - pe) * f_tau;
}

constexpr int kBasisThreads = 128;

// One CTA per recoil bin: ten sums over the flux grid, fixed-order tree reduction (deterministic).
__global__ void __launch_bounds__(kBasisThreads)
k_basis(int n_E, const double *__restrict__ fw, const double *__restrict__ P3,
        const double *__restrict__ etab, int n_T, const double *__restrict__ T, double C0, double Cmm,
        const uint8_t *__restrict__ comp8 /*NULL: one component*/, double *__restrict__ basis /*[10][n_T]*/)
{
    const int i = blockIdx.x;
    if (comp8) {                  // the bin's own component: its flux table and flavour probabilities (Eq. 17)
        fw += (size_t)comp8[i] * n_E;
        P3 += (size_t)comp8[i] * 3 * n_E;
    }
    const double Ti = T[i];
    const double invT = 1.0 / Ti;
    const double *Tmax = etab, *invE = etab + n_E, *meE2 = etab + 2 * n_E;
    double acc[kNumBasis];
#pragma unroll
    for (int b = 0; b < kNumBasis; ++b) acc[b] = 0.0;
    for (int j = threadIdx.x; j < n_E; j += kBasisThreads) {
        if (!(Ti <= Tmax[j])) continue;              // kinematic cut, inclusive
        const double f = fw[j];
        const double u = 1.0 - Ti * invE[j];
        const double u2 = u * u;
        const double v = Ti * meE2[j];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double pa = f * P3[a * n_E + j];
            acc[3 * a + 0] += pa;                    // gL^2 term
            acc[3 * a + 1] += pa * u2;               // gR^2 (1 - T/E)^2 term
            acc[3 * a + 2] += pa * v;                // gL gR m_e T / E^2 term (sign applied below)
        }
        acc[9] += f * (invT - invE[j]);              // (1/T - 1/E), flavour independent
    }
    __shared__ double red[kBasisThreads / 32][kNumBasis];
#pragma unroll
    for (int b = 0; b < kNumBasis; ++b) {
        double v = acc[b];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5][b] = v;
    }
    __syncthreads();
    if (threadIdx.x < kNumBasis) {
        const int b = threadIdx.x;
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kBasisThreads / 32; ++w) v += red[w][b];
        double scale = (b == 9) ? Cmm : ((b % 3 == 2) ? -C0 : C0);
        basis[(size_t)b * n_T + i] = scale * v;
    }
}

struct Coef0 { double c[kNumBasis]; };

// S_SM and the pre-scaled basis W^ (per period).  Dead bins (S_SM == 0): w := 1 (reading R9), so
// N' = N_mc there for every theta -- row 10, whose coefficient is the constant 1.
__global__ void k_finalize(int n_T, int D, const double *__restrict__ basis, Coef0 c0,
                           const double *__restrict__ N_mc, double *__restrict__ S_sm,
                           double *__restrict__ What /*[D][12][n_T]*/)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_T) return;
    double bas[kNumBasis];
    double S = 0.0;
#pragma unroll
    for (int b = 0; b < kNumBasis; ++b) {
        bas[b] = basis[(size_t)b * n_T + i];
        S += c0.c[b] * bas[b];
    }
    S_sm[i] = S;
    const bool live = S > 0.0;
    for (int d = 0; d < D; ++d) {
        const double N = N_mc[(size_t)d * n_T + i];
        const double q = live ? N / S : 0.0;
        double *W = What + (size_t)d * kCoefStride * n_T + i;
#pragma unroll
        for (int b = 0; b < kNumBasis; ++b) W[(size_t)b * n_T] = bas[b] * q;
        W[(size_t)10 * n_T] = live ? 0.0 : N;
        W[(size_t)11 * n_T] = 0.0;
    }
}

// Saturated-likelihood constant of Eq. (18): 2 sum_k [lnGamma(n+1) - n ln n + n]  (n = 0 => 0).
__global__ void k_sat_const(int64_t n, const double *__restrict__ counts, double *__restrict__ out)
{
    __shared__ double red[32];
    double acc = 0.0;
    for (int64_t q = threadIdx.x; q < n; q += blockDim.x) {
        double c = counts[q];
        if (c > 0.0) acc += lgamma(c + 1.0) - c * log(c) + c;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += red[w];
        out[0] = 2.0 * v;
    }
}

// Device-side validation (RW_MEM_DEVICE inputs): sets bits in *flag, read once by rw_create.
enum { F_E = 1, F_FW = 2, F_P = 4, F_T = 8, F_NMC = 16, F_BKG = 32, F_CNT = 64, F_R = 128 };

__device__ __forceinline__ bool bad_nonneg(double x) { return !(x >= 0.0) || isinf(x); }

__global__ void k_validate_small(int n_E, int n_comp, const double *E, const double *fw, const double *P3, int n_T,
                                 const double *T, int64_t nN, const double *N_mc, int64_t nB,
                                 const double *bkg, const double *counts, int *flag)
{
    int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int f = 0;
    if (t < n_E && (!(E[t] > 0.0) || isinf(E[t]))) f |= F_E;
    if (t < (int64_t)n_comp * n_E && bad_nonneg(fw[t])) f |= F_FW;
    if (t < (int64_t)n_comp * 3 * n_E) {
        double p = P3[t];
        if (!(p >= 0.0 && p <= 1.0)) f |= F_P;
    }
    if (t < n_T && (!(T[t] > 0.0) || isinf(T[t]))) f |= F_T;
    if (t < nN && bad_nonneg(N_mc[t])) f |= F_NMC;
    if (t < nB) {
        if (bad_nonneg(bkg[t])) f |= F_BKG;
        if (bad_nonneg(counts[t])) f |= F_CNT;
    }
    if (f) atomicOr(flag, f);
}

__global__ void k_validate_R(const double *__restrict__ R, int64_t rows, int n_rec, int ld,
                             int *flag)
{
    int64_t total = rows * n_rec;
    int f = 0;
    for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < total;
         q += (int64_t)gridDim.x * blockDim.x) {
        int64_t r = q / n_rec;
        int c = (int)(q - r * n_rec);
        if (bad_nonneg(R[r * ld + c])) f = F_R;
    }
    if (f) atomicOr(flag, f);
}

__global__ void k_validate_counts(int64_t n, const double *counts, int *flag)
{
    int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t < n && bad_nonneg(counts[t])) atomicOr(flag, F_CNT);
}

cudaError_t launch_validate_device(rw_ctx *ctx, const double *R_src, int ld_src,
                                   size_t period_stride_src, cudaStream_t s)
{
    int64_t nN = (int64_t)ctx->D * ctx->n_T, nB = (int64_t)ctx->D * ctx->n_rec;
    int64_t m = (int64_t)ctx->n_comp * 3 * ctx->n_E;
    if (ctx->n_T > m) m = ctx->n_T;
    if (nN > m) m = nN;
    if (nB > m) m = nB;
    k_validate_small<<<(unsigned)((m + 255) / 256), 256, 0, s>>>(
        ctx->n_E, ctx->n_comp, ctx->E, ctx->fw, ctx->P3, ctx->n_T, ctx->T, nN, ctx->N_mc, nB, ctx->bkg, ctx->counts,
        ctx->flag);
    ctx->launches++;
    for (int d = 0; d < ctx->D; ++d) {
        k_validate_R<<<ctx->num_sms * 8, 256, 0, s>>>(R_src + d * period_stride_src, ctx->n_T,
                                                      ctx->n_rec, ld_src, ctx->flag);
        ctx->launches++;
    }
    return cudaGetLastError();
}

// comp_of_T (int32, device) -> comp8, flagging indices outside [0, n_comp)
__global__ void k_comp8(int n_T, int n_comp, const int32_t *__restrict__ comp, uint8_t *__restrict__ comp8, int *flag)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_T) return;
    const int c = comp[i];
    if (c < 0 || c >= n_comp) { atomicOr(flag, 256); comp8[i] = 0; }
    else comp8[i] = (uint8_t)c;
}

cudaError_t launch_comp8(rw_ctx *ctx, const int32_t *comp_dev, cudaStream_t s)
{
    k_comp8<<<(ctx->n_T + 255) / 256, 256, 0, s>>>(ctx->n_T, ctx->n_comp, comp_dev, ctx->comp8, ctx->flag);
    ctx->launches++;
    return cudaGetLastError();
}

// Sets F_CNT in ctx->flag when a device array of D * n_rec counts holds a negative or non-finite value.
cudaError_t launch_validate_counts(rw_ctx *ctx, const double *counts_dev, cudaStream_t s)
{
    int64_t nB = (int64_t)ctx->D * ctx->n_rec;
    k_validate_counts<<<(unsigned)((nB + 255) / 256), 256, 0, s>>>(nB, counts_dev, ctx->flag);
    ctx->launches++;
    return cudaGetLastError();
}

cudaError_t launch_sat_const(rw_ctx *ctx, cudaStream_t s)
{
    int64_t nB = (int64_t)ctx->D * ctx->n_rec;
    k_validate_counts<<<(unsigned)((nB + 255) / 256), 256, 0, s>>>(nB, ctx->counts, ctx->flag);
    k_sat_const<<<1, 1024, 0, s>>>(nB, ctx->counts, ctx->sat_const);
    ctx->launches += 2;
    return cudaGetLastError();
}

cudaError_t launch_setup(rw_ctx *ctx, cudaStream_t s)
{
    const int n_E = ctx->n_E, n_T = ctx->n_T;
    k_energy_tables<<<(n_E + 255) / 256, 256, 0, s>>>(n_E, ctx->E, ctx->cst.m_e, ctx->Tmax_invE);
    k_basis<<<n_T, kBasisThreads, 0, s>>>(n_E, ctx->fw, ctx->P3, ctx->Tmax_invE, n_T, ctx->T,
                                          ctx->cst.C0, ctx->cst.Cmm, ctx->comp8, ctx->basis);
    Coef0 c0;
    for (int a = 0; a < 3; ++a) {
        c0.c[3 * a + 0] = ctx->cst.gL[a] * ctx->cst.gL[a];
        c0.c[3 * a + 1] = ctx->cst.gR[a] * ctx->cst.gR[a];
        c0.c[3 * a + 2] = ctx->cst.gL[a] * ctx->cst.gR[a];
    }
    c0.c[9] = 0.0;
    k_finalize<<<(n_T + 127) / 128, 128, 0, s>>>(n_T, ctx->D, ctx->basis, c0, ctx->N_mc, ctx->S_sm,
                                                 ctx->What);
    ctx->launches += 3;
    return cudaGetLastError();
}

cudaError_t launch_flavour(rw_ctx *ctx, int have_mu_tau, double f_tau, cudaStream_t s)
{
    k_flavour<<<dim3((ctx->n_E + 255) / 256, ctx->n_comp), 256, 0, s>>>(ctx->n_E, ctx->P3, have_mu_tau, f_tau);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
