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
constexpr int kPeeMaxPts = 8;        // points per CTA: the cut and the kinematic factors of a (E, T) pair serve all of them

// Thread = one recoil bin, kPeePts points.  Per (E_j, T_i) pair the cut, f, f (1 - T/E)^2 and f m_e T/E^2 are
// computed once; each point then costs six FMAs with its (P_e, 1 - P_e) pair read as one broadcast 16-byte load.
template <int kPeePts>
__global__ void __launch_bounds__(kPeeThreads)
k_weights_pee(int n_E, const double *__restrict__ etab /*[3][n_E]: T_max, 1/E, m_e/E^2*/,
              const double *__restrict__ fw, const double *__restrict__ P_e_pts /*[P][n_E]*/, int64_t P, double f_tau,
              int n_T, const double *__restrict__ T, const double *__restrict__ S_sm,
              const double *__restrict__ coef /*[P][12]*/, double C0, double Cmm, double *__restrict__ w /*[P][n_T]*/)
{
    __shared__ double sTmax[kPeeChunk], sInvE[kPeeChunk], sMeE2[kPeeChunk], sFw[kPeeChunk];
    __shared__ __align__(16) double2 sPe[kPeeChunk][kPeePts];      // (P_e, 1 - P_e) of the CTA's points
    const int64_t p0 = (int64_t)blockIdx.y * kPeePts;
    const int i = blockIdx.x * kPeeThreads + threadIdx.x;
    const bool ok = i < n_T;
    const double Ti = ok ? T[i] : 1.0;
    const double invT = 1.0 / Ti;
    double a0[kPeePts], a1[kPeePts], a2[kPeePts], b0[kPeePts], b1[kPeePts], b2[kPeePts], dm = 0.0;
#pragma unroll
    for (int q = 0; q < kPeePts; ++q) a0[q] = a1[q] = a2[q] = b0[q] = b1[q] = b2[q] = 0.0;
    for (int j0 = 0; j0 < n_E; j0 += kPeeChunk) {
        __syncthreads();
        {
            const int j = j0 + threadIdx.x;
            const bool in = j < n_E;
            sTmax[threadIdx.x] = in ? etab[j] : -1.0;              // T_i <= -1 never holds: padded entries drop out
            sInvE[threadIdx.x] = in ? etab[n_E + j] : 0.0;
            sMeE2[threadIdx.x] = in ? etab[2 * n_E + j] : 0.0;
            sFw[threadIdx.x] = in ? fw[j] : 0.0;
        }
        for (int q = threadIdx.x; q < kPeeChunk * kPeePts; q += kPeeThreads) {
            const int pt = q / kPeeChunk, jj = q - pt * kPeeChunk;     // consecutive threads -> consecutive E entries
            const bool in = j0 + jj < n_E && p0 + pt < P;
            const double pe = in ? P_e_pts[(p0 + pt) * n_E + j0 + jj] : 0.0;
            sPe[jj][pt] = make_double2(pe, in ? 1.0 - pe : 0.0);
        }
        __syncthreads();
#pragma unroll 2
        for (int jj = 0; jj < kPeeChunk; ++jj) {
            if (!(Ti <= sTmax[jj])) continue;                      // kinematic cut, inclusive
            const double f = sFw[jj];
            const double u = 1.0 - Ti * sInvE[jj], k1 = f * (u * u), k2 = f * (Ti * sMeE2[jj]);
            dm = fma(f, invT - sInvE[jj], dm);
#pragma unroll
            for (int q = 0; q < kPeePts; ++q) {
                const double2 pp = sPe[jj][q];
                a0[q] = fma(f, pp.x, a0[q]); a1[q] = fma(k1, pp.x, a1[q]); a2[q] = fma(k2, pp.x, a2[q]);
                b0[q] = fma(f, pp.y, b0[q]); b1[q] = fma(k1, pp.y, b1[q]); b2[q] = fma(k2, pp.y, b2[q]);
            }
        }
    }
    if (!ok) return;
    const double S0 = S_sm[i];
    const double g = 1.0 - f_tau;
#pragma unroll
    for (int q = 0; q < kPeePts; ++q) {
        const int64_t p = p0 + q;
        if (p >= P) break;
        const double *c = coef + p * kCoefStride;
        const double cL = g * c[3] + f_tau * c[6], cR = g * c[4] + f_tau * c[7], cLR = g * c[5] + f_tau * c[8];
        const double S = C0 * ((c[0] * a0[q] + c[1] * a1[q] - c[2] * a2[q]) + (cL * b0[q] + cR * b1[q] - cLR * b2[q])) +
                         Cmm * c[9] * dm;
        w[p * n_T + i] = (S0 > 0.0) ? S / S0 : 1.0;                // dead bins keep w = 1 (reading R9)
    }
}

// A handful of points (a minimiser's single evaluation): one WARP per recoil bin, the lanes stride over the flux
// grid and a fixed-order shuffle tree combines their sums, so the 4096-entry loop of a bin is 128 steps deep
// instead of 4096.
template <int PTS>
__global__ void __launch_bounds__(128)
k_weights_pee_warp(int n_E, const double *__restrict__ etab, const double *__restrict__ fw,
                   const double *__restrict__ P_e_pts, int64_t P, double f_tau, int n_T, const double *__restrict__ T,
                   const double *__restrict__ S_sm, const double *__restrict__ coef, double C0, double Cmm,
                   double *__restrict__ w)
{
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int64_t p0 = (int64_t)blockIdx.y * PTS;
    if (i >= n_T) return;
    const double Ti = T[i], invT = 1.0 / Ti;
    double a0[PTS], a1[PTS], a2[PTS], b0[PTS], b1[PTS], b2[PTS], dm = 0.0;
#pragma unroll
    for (int q = 0; q < PTS; ++q) a0[q] = a1[q] = a2[q] = b0[q] = b1[q] = b2[q] = 0.0;
    for (int j = lane; j < n_E; j += 32) {
        if (!(Ti <= etab[j])) continue;                            // kinematic cut, inclusive
        const double f = fw[j], invE = etab[n_E + j];
        const double u = 1.0 - Ti * invE, k1 = f * (u * u), k2 = f * (Ti * etab[2 * n_E + j]);
        dm = fma(f, invT - invE, dm);
#pragma unroll
        for (int q = 0; q < PTS; ++q) {
            const double pe = (p0 + q < P) ? P_e_pts[(p0 + q) * n_E + j] : 0.0, po = 1.0 - pe;
            a0[q] = fma(f, pe, a0[q]); a1[q] = fma(k1, pe, a1[q]); a2[q] = fma(k2, pe, a2[q]);
            b0[q] = fma(f, po, b0[q]); b1[q] = fma(k1, po, b1[q]); b2[q] = fma(k2, po, b2[q]);
        }
    }
    auto wsum = [](double v) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        return v;
    };
    dm = wsum(dm);
    const double S0 = S_sm[i];
    const double g = 1.0 - f_tau;
#pragma unroll
    for (int q = 0; q < PTS; ++q) {
        const double A0 = wsum(a0[q]), A1 = wsum(a1[q]), A2 = wsum(a2[q]);
        const double B0 = wsum(b0[q]), B1 = wsum(b1[q]), B2 = wsum(b2[q]);
        const int64_t p = p0 + q;
        if (p >= P || lane != 0) continue;
        const double *c = coef + p * kCoefStride;
        const double cL = g * c[3] + f_tau * c[6], cR = g * c[4] + f_tau * c[7], cLR = g * c[5] + f_tau * c[8];
        const double S = C0 * ((c[0] * A0 + c[1] * A1 - c[2] * A2) + (cL * B0 + cR * B1 - cLR * B2)) + Cmm * c[9] * dm;
        w[p * n_T + i] = (S0 > 0.0) ? S / S0 : 1.0;
    }
}

cudaError_t launch_weights_pee(rw_ctx *ctx, const double *P_e_pts, int64_t Pq, double *w, cudaStream_t s)
{
    if (Pq <= 4) {      // measured on B200 (config 4): 1 point 0.45 -> 0.33 ms per rw_eval_pee; at 16 points the blocked kernel wins
        const int pts = (int)Pq;
        dim3 grid((ctx->n_T + 3) / 4, (unsigned)((Pq + pts - 1) / pts));
#define RW_PEE_LAUNCH(N)                                                                                               \
    k_weights_pee_warp<N><<<grid, 128, 0, s>>>(ctx->n_E, ctx->Tmax_invE, ctx->fw, P_e_pts, Pq, ctx->f_tau, ctx->n_T,     \
                                               ctx->T, ctx->S_sm, ctx->coef, ctx->cst.C0, ctx->cst.Cmm, w)
        if (pts == 4) RW_PEE_LAUNCH(4);
        else if (pts == 3) RW_PEE_LAUNCH(3);
        else if (pts == 2) RW_PEE_LAUNCH(2);
        else RW_PEE_LAUNCH(1);
#undef RW_PEE_LAUNCH
    } else {
        dim3 grid((ctx->n_T + kPeeThreads - 1) / kPeeThreads, (unsigned)((Pq + kPeeMaxPts - 1) / kPeeMaxPts));
        k_weights_pee<kPeeMaxPts><<<grid, kPeeThreads, 0, s>>>(ctx->n_E, ctx->Tmax_invE, ctx->fw, P_e_pts, Pq, ctx->f_tau,
                                                              ctx->n_T, ctx->T, ctx->S_sm, ctx->coef, ctx->cst.C0,
                                                              ctx->cst.Cmm, w);
    }
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
