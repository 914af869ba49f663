// rw_pee.cu -- step a1 in its general form: the recoil spectrum with a survival-probability table per point
// (the "physics update" of PAPER.md:220: oscillation probabilities and cross sections on the discretised grid,
// combined with the fluxes into f_T(T_l; eps), Eq. 12).  With P_ee varying per point the weights
//     w[p][i] = S_theta(T_i; P_e_pts[p]) / S_SM(T_i; nominal P_e)              (Eq. 14; reading R16)
// are no longer a rank-11 function of the point, so they are computed on the (E_nu x T) grid per point and fed to
// the dense fold of rw_eval_weights.  The couplings still enter through the monomials of Eq. (4)/(8): per
// (point, bin) seven sums over the flux grid are enough --
//     nu_e:      sum f P_e {1, (1 - T/E)^2, m_e T/E^2}        nu_mu,tau: the same with (1 - P_e)
//     mu_nu:     sum f (1/T - 1/E)
// all under the kinematic cut T <= 2E^2/(m_e + 2E) (tabulated once per E entry, reading R2).
#include "rw_internal.h"

namespace rw {

constexpr int kPeeThreads = 128;     // recoil bins per CTA
constexpr int kPeeChunk = 128;       // flux-grid entries staged per iteration

__global__ void __launch_bounds__(kPeeThreads)
k_weights_pee(int n_E, const double *__restrict__ etab /*[3][n_E]: T_max, 1/E, m_e/E^2*/,
              const double *__restrict__ fw, const double *__restrict__ P_e_pts /*[P][n_E]*/, double f_tau,
              int n_T, const double *__restrict__ T, const double *__restrict__ S_sm,
              const double *__restrict__ coef /*[P][12]*/, double C0, double Cmm, double *__restrict__ w /*[P][n_T]*/)
{
    __shared__ double sTmax[kPeeChunk], sInvE[kPeeChunk], sMeE2[kPeeChunk], sFw[kPeeChunk], sPe[kPeeChunk];
    const int64_t p = blockIdx.y;
    const int i = blockIdx.x * kPeeThreads + threadIdx.x;
    const bool ok = i < n_T;
    const double Ti = ok ? T[i] : 1.0;
    const double invT = 1.0 / Ti;
    const double *Pp = P_e_pts + p * n_E;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, b0 = 0.0, b1 = 0.0, b2 = 0.0, dm = 0.0;
    for (int j0 = 0; j0 < n_E; j0 += kPeeChunk) {
        __syncthreads();
        {
            const int j = j0 + threadIdx.x;
            const bool in = j < n_E;
            sTmax[threadIdx.x] = in ? etab[j] : -1.0;              // T_i <= -1 never holds: padded entries drop out
            sInvE[threadIdx.x] = in ? etab[n_E + j] : 0.0;
            sMeE2[threadIdx.x] = in ? etab[2 * n_E + j] : 0.0;
            sFw[threadIdx.x] = in ? fw[j] : 0.0;
            sPe[threadIdx.x] = in ? Pp[j] : 0.0;
        }
        __syncthreads();
#pragma unroll 4
        for (int jj = 0; jj < kPeeChunk; ++jj) {
            if (!(Ti <= sTmax[jj])) continue;                      // kinematic cut, inclusive
            const double f = sFw[jj], pe = sPe[jj];
            const double u = 1.0 - Ti * sInvE[jj], u2 = u * u, v = Ti * sMeE2[jj];
            const double fe = f * pe, fo = f * (1.0 - pe);
            a0 += fe; a1 = fma(fe, u2, a1); a2 = fma(fe, v, a2);
            b0 += fo; b1 = fma(fo, u2, b1); b2 = fma(fo, v, b2);
            dm = fma(f, invT - sInvE[jj], dm);
        }
    }
    if (!ok) return;
    const double *c = coef + p * kCoefStride;
    const double g = 1.0 - f_tau;
    const double cL = g * c[3] + f_tau * c[6], cR = g * c[4] + f_tau * c[7], cLR = g * c[5] + f_tau * c[8];
    const double S = C0 * ((c[0] * a0 + c[1] * a1 - c[2] * a2) + (cL * b0 + cR * b1 - cLR * b2)) + Cmm * c[9] * dm;
    const double S0 = S_sm[i];
    w[p * n_T + i] = (S0 > 0.0) ? S / S0 : 1.0;                    // dead bins keep w = 1 (reading R9)
}

cudaError_t launch_weights_pee(rw_ctx *ctx, const double *P_e_pts, int64_t Pq, double *w, cudaStream_t s)
{
    dim3 grid((ctx->n_T + kPeeThreads - 1) / kPeeThreads, (unsigned)Pq);
    k_weights_pee<<<grid, kPeeThreads, 0, s>>>(ctx->n_E, ctx->Tmax_invE, ctx->fw, P_e_pts, ctx->f_tau, ctx->n_T, ctx->T,
                                               ctx->S_sm, ctx->coef, ctx->cst.C0, ctx->cst.Cmm, w);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
