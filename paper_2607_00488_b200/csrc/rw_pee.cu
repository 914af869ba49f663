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

// ------------------------------------------------------------------------------------------------------------------
// The same weights in O(n_E + n_T) per point instead of O(n_E n_T).  T_max(E) = 2E^2/(m_e + 2E) grows with E, so with
// the flux grid SORTED by T_max the cut T_i <= T_max(E_j) is a threshold: the entries j >= j0(i) of the sorted grid.
// And the three kinematic factors are polynomials in T_i with coefficients E_j^-n,
//     1,   (1 - T/E)^2 = 1 - 2 T E^-1 + T^2 E^-2,   m_e T E^-2,
// so all six flavour sums of a bin are combinations of the three SUFFIX SUMS
//     X_n[p][j] = sum_{l >= j} f_l omega_l P_e^p[l] E_l^-n,   n = 0, 1, 2
// read at j0(i); the nu_mu / nu_tau sums are (point-independent suffix sums Y_n of f omega E^-n) - X_n with
// omega = rho_mu, rho_tau the share of 1 - P_e each flavour takes (f_tau split, or the nominal tables' ratio,
// reading R17).  One CTA per point: suffix scans in shared memory, then every bin of the scanned component.
// (1 - T/E)^2 is evaluated as x0 - T (2 x1 - T x2): its cancellation error is relative to x0, i.e. to the g~L^2 term
// that comes with it -- below 1e-15 of the spectrum unless g~L of a flavour is tuned to zero.
constexpr int kScanThreads = 1024;

__global__ void k_pee_rank(int n_E, const double *__restrict__ Tmax, int *__restrict__ perm)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_E) return;
    const double t = Tmax[j];
    int rank = 0;
    for (int l = 0; l < n_E; ++l) {
        const double u = Tmax[l];
        rank += (u < t) || (u == t && l < j);
    }
    perm[rank] = j;
}

// sorted copies: fS[q][n][j] = f_q E^-n, rho[q][w][j] = share of 1 - P_e that goes to nu_mu (w = 0) / nu_tau (w = 1)
__global__ void k_pee_tables(int n_E, int n_comp, const int *__restrict__ perm, const double *__restrict__ etab,
                             const double *__restrict__ fw, const double *__restrict__ P3, int have_mu_tau, double f_tau,
                             double *__restrict__ TmaxS, double *__restrict__ fS, double *__restrict__ rho)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y;
    if (j >= n_E) return;
    const int o = perm[j];
    const double invE = etab[n_E + o], f = fw[(size_t)q * n_E + o];
    if (q == 0) TmaxS[j] = etab[o];
    fS[((size_t)q * 3 + 0) * n_E + j] = f;
    fS[((size_t)q * 3 + 1) * n_E + j] = f * invE;
    fS[((size_t)q * 3 + 2) * n_E + j] = f * invE * invE;
    double rm = 1.0 - f_tau, rt = f_tau;
    if (have_mu_tau) {
        const double pm = P3[((size_t)q * 3 + 1) * n_E + o], pt = P3[((size_t)q * 3 + 2) * n_E + o];
        if (pm + pt > 0.0) { rm = pm / (pm + pt); rt = pt / (pm + pt); }
    }
    rho[((size_t)q * 2 + 0) * n_E + j] = rm;
    rho[((size_t)q * 2 + 1) * n_E + j] = rt;
}

// Y[q][w][n][j] = sum_{l >= j} f_q omega_w E^-n (w = 0: omega = 1), compensated, one thread per array; Y[..][n_E] = 0
__global__ void k_pee_totals(int n_E, int n_comp, const double *__restrict__ fS, const double *__restrict__ rho,
                             double *__restrict__ Y)
{
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n_comp * 9) return;
    const int q = a / 9, w = (a % 9) / 3, n = a % 3;
    const double *f = fS + ((size_t)q * 3 + n) * n_E;
    const double *r = (w == 0) ? nullptr : rho + ((size_t)q * 2 + (w - 1)) * n_E;
    double *y = Y + (size_t)a * (n_E + 1);
    double sum = 0.0, comp = 0.0;
    y[n_E] = 0.0;
    for (int j = n_E - 1; j >= 0; --j) {
        const double v = (r ? f[j] * r[j] : f[j]) - comp;
        const double t = sum + v;
        comp = (t - sum) - v;
        sum = t;
        y[j] = sum;
    }
}

__global__ void k_pee_j0(int n_T, const double *__restrict__ T, int n_E, const double *__restrict__ TmaxS, int *__restrict__ j0)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_T) return;
    const double t = T[i];
    int lo = 0, hi = n_E;                       // first sorted entry with T_i <= T_max (the cut, inclusive)
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (t <= TmaxS[mid]) hi = mid; else lo = mid + 1;
    }
    j0[i] = lo;
}

struct PeeScanArgs {
    int n_E, n_T, n_comp, have_mu_tau, tables_per_point;     // tables_per_point: P_e_pts is [P][n_comp][n_E] (else [P][n_E])
    double f_tau, C0, m_e;
    const int *perm, *j0;
    const uint8_t *comp8;
    const double *fS, *rho, *Y, *T, *S_sm, *basis9, *coef, *P_e_pts;
    double *w;
};

// Suffix sums of three arrays held in shared memory, in place: x[n][j] <- sum_{l >= j} x[n][l]; x[n][n_E] = 0.
__device__ __forceinline__ void pee_suffix_scan3(double *x, int n_E, int pitch, double *s_tot /*[3][32]*/)
{
    const int L = (n_E + kScanThreads - 1) / kScanThreads;
    const int j1 = min(n_E, (int)(threadIdx.x + 1) * L), jb = min(n_E, (int)threadIdx.x * L);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double tot[3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        double acc = 0.0;
        for (int j = j1 - 1; j >= jb; --j) { acc += x[n * pitch + j]; x[n * pitch + j] = acc; }
        tot[n] = acc;
    }
    // exclusive suffix scan of the segment totals: what lies behind this thread's segment
    double off[3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        double v = tot[n];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double u = __shfl_down_sync(0xffffffffu, v, o);
            if (lane + o < 32) v += u;
        }
        if (lane == 0) s_tot[n * 32 + warp] = v;        // warp total (inclusive suffix at lane 0)
        off[n] = v - tot[n];                            // behind this lane, inside the warp
    }
    __syncthreads();
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        double behind = 0.0;
        for (int wq = kScanThreads / 32 - 1; wq > warp; --wq) behind += s_tot[n * 32 + wq];
        off[n] += behind;
        for (int j = jb; j < j1; ++j) x[n * pitch + j] += off[n];
        if (threadIdx.x == 0) x[n * pitch + n_E] = 0.0;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kScanThreads)
k_pee_scan(const PeeScanArgs A)
{
    extern __shared__ __align__(16) double pee_smem[];
    const int n_E = A.n_E, pitch = n_E + 1;
    double *x = pee_smem;                                  // [3][n_E + 1]
    __shared__ double s_tot[3 * 32];
    const int64_t p = blockIdx.x;
    double c[kNumBasis];
#pragma unroll
    for (int b = 0; b < kNumBasis; ++b) c[b] = A.coef[p * kCoefStride + b];
    const int n_w = A.have_mu_tau ? 3 : 1;                 // f_tau split: rho is constant, one scan serves all flavours
    const double g = 1.0 - A.f_tau;
    for (int q = 0; q < A.n_comp; ++q) {
        const double *Pp = A.P_e_pts + (A.tables_per_point ? ((size_t)p * A.n_comp + q) * n_E : (size_t)p * n_E);
        for (int wq = 0; wq < n_w; ++wq) {
            __syncthreads();                               // the previous pass has read x
            for (int j = threadIdx.x; j < n_E; j += kScanThreads) {
                double pe = Pp[A.perm[j]];
                if (wq > 0) pe *= A.rho[((size_t)q * 2 + (wq - 1)) * n_E + j];
#pragma unroll
                for (int n = 0; n < 3; ++n) x[n * pitch + j] = A.fS[((size_t)q * 3 + n) * n_E + j] * pe;
            }
            __syncthreads();
            pee_suffix_scan3(x, n_E, pitch, s_tot);
            const double *Y1 = A.Y + ((size_t)q * 9 + 0) * pitch;                  // omega = 1
            const double *Yw = A.Y + ((size_t)q * 9 + 3 * wq) * pitch;             // omega of this pass
            for (int i = threadIdx.x; i < A.n_T; i += kScanThreads) {
                if (A.comp8[i] != q) continue;
                const int j = A.j0[i];
                const double Ti = A.T[i];
                const double x0 = x[j], x1 = x[pitch + j], x2 = x[2 * pitch + j];
                double S;
                if (wq == 0) {
                    // nu_e: sums weighted by P_e
                    const double a0 = x0, a1 = x0 - Ti * (2.0 * x1 - Ti * x2), a2 = A.m_e * Ti * x2;
                    S = c[0] * a0 + c[1] * a1 - c[2] * a2;
                    if (!A.have_mu_tau) {                  // nu_mu, nu_tau share the sums weighted by 1 - P_e
                        const double y0 = Y1[j] - x0, y1 = Y1[pitch + j] - x1, y2 = Y1[2 * pitch + j] - x2;
                        const double b0 = y0, b1 = y0 - Ti * (2.0 * y1 - Ti * y2), b2 = A.m_e * Ti * y2;
                        const double cL = g * c[3] + A.f_tau * c[6], cR = g * c[4] + A.f_tau * c[7],
                                     cLR = g * c[5] + A.f_tau * c[8];
                        S += cL * b0 + cR * b1 - cLR * b2;
                    }
                    S = A.C0 * S + c[9] * A.basis9[i];       // + magnetic-moment term (Eq. 8; no flavour factor)
                } else {
                    // nu_mu (wq = 1) / nu_tau (wq = 2): rho (1 - P_e) = Y^rho - X^rho
                    const double y0 = Yw[j] - x0, y1 = Yw[pitch + j] - x1, y2 = Yw[2 * pitch + j] - x2;
                    const double b0 = y0, b1 = y0 - Ti * (2.0 * y1 - Ti * y2), b2 = A.m_e * Ti * y2;
                    S = A.w[p * A.n_T + i] + A.C0 * (c[3 * wq] * b0 + c[3 * wq + 1] * b1 - c[3 * wq + 2] * b2);
                }
                if (wq == n_w - 1) {
                    const double S0 = A.S_sm[i];
                    S = (S0 > 0.0) ? S / S0 : 1.0;           // dead bins keep w = 1 (reading R9)
                }
                A.w[p * A.n_T + i] = S;
            }
        }
    }
}

int pee_setup(rw_ctx *ctx, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    if (!L.pee_scan) return RW_OK;
    const int n_E = ctx->n_E, n_T = ctx->n_T, nc = ctx->n_comp;
    k_pee_rank<<<(n_E + 127) / 128, 128, 0, s>>>(n_E, ctx->Tmax_invE, ctx->pee_perm);
    k_pee_tables<<<dim3((n_E + 127) / 128, nc), 128, 0, s>>>(n_E, nc, ctx->pee_perm, ctx->Tmax_invE, ctx->fw, ctx->P3,
                                                              ctx->have_mu_tau ? 1 : 0, ctx->f_tau, ctx->pee_TmaxS,
                                                              ctx->pee_fS, ctx->pee_rho);
    k_pee_totals<<<(nc * 9 + 31) / 32, 32, 0, s>>>(n_E, nc, ctx->pee_fS, ctx->pee_rho, ctx->pee_Y);
    k_pee_j0<<<(n_T + 127) / 128, 128, 0, s>>>(n_T, ctx->T, n_E, ctx->pee_TmaxS, ctx->pee_j0);
    ctx->launches += 4;
    if (cudaGetLastError() != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "per-point P_ee tables failed at launch");
    // The attribute belongs to the function on this device, not to the context: always raise it to the cap plan() admits
    // (L.pee_scan), so that a later context with a smaller flux grid cannot lower it under a live context's launches.
    cudaError_t e = cudaFuncSetAttribute(k_pee_scan, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 << 10);
    if (e != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "cudaFuncSetAttribute(k_pee_scan): %s", cudaGetErrorString(e));
    return RW_OK;
}

cudaError_t launch_weights_pee(rw_ctx *ctx, const double *P_e_pts, int64_t Pq, double *w, cudaStream_t s)
{
    if (ctx->lay.pee_scan) {        // sorted-grid suffix sums: O(n_E + n_T) per point
        PeeScanArgs A;
        A.n_E = ctx->n_E; A.n_T = ctx->n_T; A.n_comp = ctx->n_comp; A.have_mu_tau = ctx->have_mu_tau ? 1 : 0;
        A.tables_per_point = ctx->n_comp > 1;
        A.f_tau = ctx->f_tau; A.C0 = ctx->cst.C0; A.m_e = ctx->cst.m_e;
        A.perm = ctx->pee_perm; A.j0 = ctx->pee_j0; A.comp8 = ctx->comp8;
        A.fS = ctx->pee_fS; A.rho = ctx->pee_rho; A.Y = ctx->pee_Y; A.T = ctx->T; A.S_sm = ctx->S_sm;
        A.basis9 = ctx->basis + (size_t)9 * ctx->n_T; A.coef = ctx->coef; A.P_e_pts = P_e_pts; A.w = w;
        k_pee_scan<<<(unsigned)Pq, kScanThreads, 3 * (ctx->n_E + 1) * 8, s>>>(A);
        ctx->launches++;
        return cudaGetLastError();
    }
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
