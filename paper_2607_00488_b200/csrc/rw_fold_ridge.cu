// rw_fold_ridge.cu -- the whole path for 5..64 points in ONE kernel: the regime around the ridge of the
// roofline (P* = 4 F / BW ~ 23 points on B200), where the fold
//   mu[p][k] = sum_i N'[p][i] R[i][k] + bkg[k]                                  (Eq. 11)
// has to read every byte of R exactly once at HBM speed AND do 2 P flop per 8 bytes, more than scalar DFMA
// can issue next to the loads.  Design:
//   * decomposition of k_fold_stream: a CTA owns a 256-column strip x a range of recoil rows (grid =
//     strips x row ranges x periods, one wave of one or two CTAs per SM), so R streams from HBM exactly once;
//   * a producer warp keeps a ring of 4-6 stages of 8 or 16 rows in flight (up to 200 KB per SM -- registers
//     cannot hold that much, a first version with the loads going straight into the fragments stayed at 5.4 TB/s):
//     one plain bulk copy (cp.async.bulk, mbarrier completion) per row, 2 KB long requests, exactly the strip's
//     bytes; the rows land at a pitch of 2080 bytes (= 32 mod 128), which makes the fragment loads below
//     conflict free without a swizzle;
//   * the arithmetic of k_fold_gemm: mma.sync.m8n8k4.f64 (DMMA.8x8x4).  Eight consumer warps own 32 columns
//     each and all points of the tile; lane (r = lane / 4, c = lane % 4) reads the 16 bytes
//     R[i + c][col + 2 r .. + 1] -- one B fragment for the even and one for the odd columns of a 16-column group;
//   * N' of 64 recoil rows x 8 MB points (steps a1 + a2: coefficients from the raw parameters, Eq. 6, PAPER.md:79;
//     N' = sum_b c_b W^_b, Eq. 14 / Eq. 1) is formed on the fly into shared memory, double
//     buffered, pitch 68 doubles so that the A-fragment loads are conflict free;
//   * a4 as in k_fold_stream: the partial tile of a row range is parked; the LAST CTA of a strip (ticket) adds
//     the ranges in a fixed order, adds bkg and reduces the Poisson terms of Eq. (18); the last
//     strip adds strips and periods in a fixed order and writes -2lnL.  One launch per call, deterministic.
#include <type_traits>

#include "rw_internal.h"

namespace rw {

constexpr int kRgWarps = 8;                           // consumer (DMMA) warps
constexpr int kRgConsumers = kRgWarps * 32;
constexpr int kRgThreads = kRgConsumers + 32;         // + the producer warp (tile heights 8, 16, 32)
constexpr int kRgThreads64 = kRgConsumers + 128;      // tile height 64: a producer warpgroup, so that setmaxnreg can
                                                      // move its registers to the consumers (128 accumulators each)
constexpr int kRgWarpCols = 32;                       // two 16-column groups per warp
constexpr int kRgCols = kRgWarps * kRgWarpCols;       // 256 columns per CTA strip
constexpr int kRgKC = 64;                             // recoil rows of N' staged per chunk
constexpr int kRgPitch = kRgKC + 4;                   // = 4 (mod 16) doubles: the A-fragment rows land in distinct banks
constexpr int kRgRowBytes = kRgCols * 8 + 32;         // ring pitch 2080 B = 32 (mod 128): rows c = 0..3 -> 4 bank groups
static_assert(kRgCols == kRidgeCols && kRgKC == kRidgeRowQuantum * 4, "plan() in rw_api.cu assumes this geometry");

struct RidgeArgs {
    const double *R; size_t R_period_stride; int ldR, n_T, n_rec, D;
    const double *coef;       // [Pb][12], or NULL
    const double *param;      // [Pb][k] raw parameters (coefficients computed here), or NULL
    const double *wts;        // [Pb][n_T] caller weights, or NULL
    const double *rate;       // [Pb][4] rate scales matching `coef`, or NULL
    const uint8_t *comp8;     // [n_T] component of every recoil bin
    const double *What, *N_mc, *bkg, *counts, *sat_const;
    int Pb, rows_per_split, n_splits, mu_ld;
    double *mu_part;          // [D][n_splits][8 MB][mu_ld]
    double *strip_part;       // [D * strips][64]
    int *cnt;                 // [D * strips] strip tickets, then one global ticket
    double *out;              // [Pb]
    double *out_mu;           // NULL or [Pb][D][n_rec]
};

__device__ __forceinline__ void rg_dmma(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ uint32_t rg_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void rg_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void rg_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void rg_mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void rg_mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// one row of the strip, global -> shared, completion counted on `bar`; R is read once: evict-first in L2, so that
// the parked partial tiles and W^ stay resident
__device__ __forceinline__ void rg_bulk_row(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}

template <int MB> struct RidgeCfg {
    static constexpr int PP = 8 * MB;                                  // points of the tile
    static constexpr int RS = (MB <= 2) ? 8 : 16;                      // recoil rows per ring stage
    static constexpr int NS = (MB == 1) ? 6 : (MB == 8) ? 4 : 5;       // ring stages
    static constexpr int MinCtas = (MB <= 2) ? 2 : 1;
    static constexpr int Threads = (MB == 8) ? kRgThreads64 : kRgThreads;
    static constexpr int StageBytes = RS * kRgRowBytes;
    static constexpr int RingBytes = NS * StageBytes;
    static constexpr int SmemDoubles = 2 * PP * kRgPitch + PP * kCoefStride + PP * RW_MAX_COMPONENTS + kRgWarps * PP;
    static constexpr int Smem = RingBytes + SmemDoubles * 8 + 2 * NS * 8;           // + barriers
};

template <int MB>
__global__ void __launch_bounds__(RidgeCfg<MB>::Threads, RidgeCfg<MB>::MinCtas)
k_fold_ridge(const RidgeArgs A, const Kinds kd, const Consts cst)
{
    using Cfg = RidgeCfg<MB>;
    constexpr int PP = Cfg::PP, RS = Cfg::RS, NS = Cfg::NS, kThreads = Cfg::Threads;
    // 128-byte aligned so that the bank analysis of the ring pitch holds; indexed directly (a re-aligned pointer
    // would lose its address space and turn the fragment loads into generic LD)
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t ring = rg_smem_u32(smem);
    double *sN = reinterpret_cast<double *>(smem + Cfg::RingBytes);     // [2][PP][kRgPitch]
    double *sC = sN + 2 * PP * kRgPitch;                               // [PP][12]
    double *sRate = sC + PP * kCoefStride;                             // [PP][4]
    double *red = sRate + PP * RW_MAX_COMPONENTS;                      // [8 warps][PP]
    const uint32_t full_bar = rg_smem_u32(red + kRgWarps * PP);
    const uint32_t empty_bar = full_bar + NS * 8;
    __shared__ int s_last;

    const int d = blockIdx.z, split = blockIdx.y, strip = blockIdx.x;
    const int n_T = A.n_T, n_rec = A.n_rec, Pb = A.Pb;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r = lane >> 2, c = lane & 3;
    const int i0 = split * A.rows_per_split;
    const int i1 = min(n_T, i0 + A.rows_per_split);
    const int nrows = i1 - i0;
    const int n_iters = (nrows + RS - 1) / RS;                         // ring stage-iterations of this CTA
    const double *Rd = A.R + (size_t)d * A.R_period_stride;
    const double *Wd = A.What + (size_t)d * kCoefStride * n_T;
    const double *wts = A.wts;
    const int cols_avail = min(kRgCols, A.ldR - strip * kRgCols);      // even; the pad column of a copied R is zero

    if (threadIdx.x == 0) {
        for (int s = 0; s < NS; ++s) {
            rg_mbar_init(full_bar + 8 * s, 1);
            rg_mbar_init(empty_bar + 8 * s, kRgWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // ragged strip or row range: the ring is also read where no copy ever lands (times N' = 0), so it must hold
    // finite numbers there
    if (cols_avail < kRgCols || (nrows % RS) != 0) {
        for (int q = threadIdx.x; q < Cfg::RingBytes / 16; q += kThreads)
            reinterpret_cast<double2 *>(smem)[q] = make_double2(0.0, 0.0);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }

    // ---------------------------------------------------------------- a1: coefficients of the tile's points
    if (!wts) {
        if (A.param) {
            if (threadIdx.x < PP) {
                double cc[kCoefStride], rr[RW_MAX_COMPONENTS];
                if (threadIdx.x < Pb) {
                    coef_from_param(A.param + (size_t)threadIdx.x * kd.k, kd, cst, cc, rr);
                } else {
#pragma unroll
                    for (int b = 0; b < kCoefStride; ++b) cc[b] = 0.0;
#pragma unroll
                    for (int q = 0; q < RW_MAX_COMPONENTS; ++q) rr[q] = 1.0;
                }
#pragma unroll
                for (int b = 0; b < kCoefStride; ++b) sC[threadIdx.x * kCoefStride + b] = cc[b];
#pragma unroll
                for (int q = 0; q < RW_MAX_COMPONENTS; ++q) sRate[threadIdx.x * RW_MAX_COMPONENTS + q] = rr[q];
            }
        } else {
            for (int q = threadIdx.x; q < PP * kCoefStride; q += kThreads) {
                const int p = q / kCoefStride;
                sC[q] = (p < Pb) ? A.coef[q] : 0.0;
            }
            for (int q = threadIdx.x; q < PP * RW_MAX_COMPONENTS; q += kThreads) {
                const int p = q / RW_MAX_COMPONENTS;
                sRate[q] = (p < Pb && A.rate) ? A.rate[q] : 1.0;
            }
        }
    }
    __syncthreads();                                                // barriers, zeroed ring, sC, sRate

    if (warp >= kRgWarps) {
        // ------------------------------------------------------------ producer warp: lane l copies row l of a stage
        if constexpr (MB == 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == kRgWarps) {                                      // (the other warps of that group idle)
            uint64_t policy;
            asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
            const uint32_t row_bytes = (uint32_t)cols_avail * 8;
            const double *src = Rd + (size_t)(i0 + lane) * A.ldR + (size_t)strip * kRgCols;
            int stage = 0;
            uint32_t phase = 0;
            for (int q = 0; q < n_iters; ++q) {
                rg_mbar_wait(empty_bar + 8 * stage, phase ^ 1);
                const int rows = min(RS, nrows - q * RS);
                const uint32_t fb = full_bar + 8 * stage;
                if (lane == 0) rg_mbar_expect_tx(fb, (uint32_t)rows * row_bytes);
                __syncwarp();
                if (lane < rows)
                    rg_bulk_row(ring + stage * Cfg::StageBytes + lane * kRgRowBytes, src + (size_t)q * RS * A.ldR, row_bytes, fb,
                                policy);
                if (++stage == NS) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        if constexpr (MB == 8) asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
        // ------------------------------------------------------------ a2: N' of a 64-row chunk -> sN[buf][p][row]
        // thread = (row, quarter of the points): the 11 basis values of its row are loaded once for all its points
        auto stage_n = [&](int ic, int buf) {
            const int row = threadIdx.x & (kRgKC - 1), pq = threadIdx.x >> 6;
            const int i = ic + row;
            const bool ok = i < i1;
            double *dst = sN + (size_t)buf * PP * kRgPitch + row;
            if (wts) {
                const double nm = ok ? A.N_mc[(size_t)d * n_T + i] : 0.0;
#pragma unroll
                for (int j = 0; j < PP / 4; ++j) {
                    const int p = pq + 4 * j;
                    dst[p * kRgPitch] = (ok && p < Pb) ? wts[(size_t)p * n_T + i] * nm : 0.0;
                }
            } else {
                double w[kNumTerms];
#pragma unroll
                for (int b = 0; b < kNumTerms; ++b) w[b] = ok ? __ldg(Wd + (size_t)b * n_T + i) : 0.0;
                const int cq = ok ? A.comp8[i] : 0;
#pragma unroll
                for (int j = 0; j < PP / 4; ++j) {
                    const int p = pq + 4 * j;
                    double v = 0.0;
#pragma unroll
                    for (int b = 0; b < kNumTerms; ++b) v = fma(sC[p * kCoefStride + b], w[b], v);
                    dst[p * kRgPitch] = v * sRate[p * RW_MAX_COMPONENTS + cq];     // rate_k of Eq. (17); 1 when not scanned
                }
            }
        };

        // ------------------------------------------------------------ a3: DMMA over the ring
        double acc[MB][2][2][2];
#pragma unroll
        for (int mb = 0; mb < MB; ++mb)
#pragma unroll
            for (int g = 0; g < 2; ++g)
#pragma unroll
                for (int nb = 0; nb < 2; ++nb) acc[mb][g][nb][0] = acc[mb][g][nb][1] = 0.0;
        // B fragments: row 4 ks + c of the stage, columns 32 warp + 16 g + 2 r + {0, 1}
        const uint32_t b_off = (uint32_t)c * kRgRowBytes + (uint32_t)(kRgWarpCols * warp + 2 * r) * 8;
        if (nrows > 0) stage_n(i0, 0);
        int stage = 0, buf = 0, q = 0;
        uint32_t phase = 0;
        for (int ch = 0; ch * kRgKC < nrows; ++ch, buf ^= 1) {
            asm volatile("bar.sync 1, %0;" ::"n"(kRgConsumers) : "memory");   // sN[buf] staged; sN[buf ^ 1] no longer read
            const double *sA = sN + (size_t)buf * PP * kRgPitch + r * kRgPitch + c;
#pragma unroll
            for (int sq = 0; sq < kRgKC / RS; ++sq) {
                if (q < n_iters) {
                    rg_mbar_wait(full_bar + 8 * stage, phase);
                    const uint32_t st = ring + stage * Cfg::StageBytes + b_off;
#pragma unroll
                    for (int ks = 0; ks < RS / 4; ++ks) {
                        double a[MB];
                        double2 b[2];
#pragma unroll
                        for (int g = 0; g < 2; ++g)
                            asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(b[g].x), "=d"(b[g].y)
                                         : "r"(st + (uint32_t)ks * (4 * kRgRowBytes) + (uint32_t)g * 128));
#pragma unroll
                        for (int mb = 0; mb < MB; ++mb) a[mb] = sA[mb * 8 * kRgPitch + sq * RS + 4 * ks];
#pragma unroll
                        for (int mb = 0; mb < MB; ++mb)
#pragma unroll
                            for (int g = 0; g < 2; ++g) {
                                rg_dmma(acc[mb][g][0][0], acc[mb][g][0][1], a[mb], b[g].x);
                                rg_dmma(acc[mb][g][1][0], acc[mb][g][1][1], a[mb], b[g].y);
                            }
                    }
                    __syncwarp();
                    if (lane == 0) rg_mbar_arrive(empty_bar + 8 * stage);
                    if (++stage == NS) { stage = 0; phase ^= 1; }
                    ++q;
                }
            }
            if ((ch + 1) * kRgKC < nrows) stage_n(i0 + (ch + 1) * kRgKC, buf ^ 1);
        }

        // ------------------------------------------------------------ park the partial tile of this row range
        // column 4 c + 2 e + nb of a 16-column group holds acc[.][.][nb][e]
        const int colw = strip * kRgCols + warp * kRgWarpCols;
#pragma unroll
        for (int mb = 0; mb < MB; ++mb)
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                const int col = colw + 16 * g + 4 * c;
                double *dst = A.mu_part + (((size_t)d * A.n_splits + split) * PP + 8 * mb + r) * A.mu_ld + col;
                if (col < n_rec)
                    __stcg(reinterpret_cast<double2 *>(dst), make_double2(acc[mb][g][0][0], acc[mb][g][1][0]));
                if (col + 2 < n_rec)
                    __stcg(reinterpret_cast<double2 *>(dst + 2), make_double2(acc[mb][g][0][1], acc[mb][g][1][1]));
            }
    }

    // ---------------------------------------------------------------- last CTA of this strip: a4 for 256 columns
    const int n_splits = A.n_splits, mu_ld = A.mu_ld;
    const int n_strips = gridDim.x, sid = d * n_strips + strip;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(A.cnt + sid, 1) == n_splits - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (warp < kRgWarps) {
        const int col = strip * kRgCols + threadIdx.x;
        const bool col_ok = col < n_rec;
        double bk = 0.0, cn = 0.0;
        if (col_ok) { bk = A.bkg[(size_t)d * n_rec + col]; cn = A.counts[(size_t)d * n_rec + col]; }
#pragma unroll 1
        for (int pb = 0; pb < MB; ++pb) {
            double m[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) m[q] = 0.0;
            if (col_ok) {
                const double *src = A.mu_part + ((size_t)d * n_splits * PP + 8 * pb) * mu_ld + col;
                for (int s = 0; s < n_splits; ++s) {      // row ranges in a fixed order; the 8 loads of a step overlap
#pragma unroll
                    for (int q = 0; q < 8; ++q) m[q] += __ldcg(src + ((size_t)s * PP + q) * mu_ld);
                }
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int p = 8 * pb + q;
                double t = 0.0;
                if (col_ok && p < Pb) {
                    const double a = m[q] + bk;
                    if (A.out_mu) A.out_mu[((size_t)p * A.D + d) * n_rec + col] = a;
                    t = poisson_term(a, cn);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                if (lane == 0) red[warp * PP + p] = t;
            }
        }
    }
    __syncthreads();
    if (threadIdx.x < PP) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kRgWarps; ++w) v += red[w * PP + threadIdx.x];
        __stcg(A.strip_part + (size_t)sid * kRidgeMaxP + threadIdx.x, v);
    }

    // ---------------------------------------------------------------- last strip: sum strips and periods, write
    const int n_sid = n_strips * A.D;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(A.cnt + n_sid, 1) == n_sid - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x < Pb) {
        double v = 0.0;
        for (int q = 0; q < n_sid; ++q) v += __ldcg(A.strip_part + (size_t)q * kRidgeMaxP + threadIdx.x);
        v *= 2.0;
        if (A.sat_const) v += A.sat_const[0];
        A.out[threadIdx.x] = v;
    }
    for (int q = threadIdx.x; q <= n_sid; q += kThreads) A.cnt[q] = 0;       // ready for the next launch
}

template <int MB>
static cudaError_t launch_ridge_t(const RidgeArgs &A, const Kinds &kd, const Consts &cst, dim3 grid, cudaStream_t s)
{
    static bool attr_set = false;          // per instantiation; the attribute is per device function
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(k_fold_ridge<MB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             RidgeCfg<MB>::Smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    k_fold_ridge<MB><<<grid, RidgeCfg<MB>::Threads, RidgeCfg<MB>::Smem, s>>>(A, kd, cst);
    return cudaSuccess;
}

int ridge_plan(int n_T, int n_rec, int D, int mb_log2, int num_sms, int *rows_per_split)
{
    const int strips = (n_rec + kRgCols - 1) / kRgCols;
    const int slots = num_sms * ((mb_log2 <= 1) ? 2 : 1);           // resident CTAs (RidgeCfg::MinCtas)
    const int max_splits = n_T / kRgKC > 1 ? n_T / kRgKC : 1;       // at least one 64-row chunk per CTA
    int best = 1;
    double best_eff = 0.0;
    for (int S = 1; S <= max_splits; ++S) {
        const int64_t ctas = (int64_t)strips * D * S;
        if (ctas > 2 * (int64_t)slots && S > 1) break;              // at most two waves: partial tiles cost traffic
        const double eff = (double)ctas / (double)((ctas + slots - 1) / slots * slots);
        if (eff > best_eff + 0.01) { best_eff = eff; best = S; }
    }
    int rows = (n_T + best - 1) / best;
    rows = (rows + kRidgeRowQuantum - 1) / kRidgeRowQuantum * kRidgeRowQuantum;
    *rows_per_split = rows;
    return (n_T + rows - 1) / rows;
}

cudaError_t launch_fold_ridge(rw_ctx *ctx, const double *coef, const double *param, const Kinds *kd,
                              const double *wts, int Pb, double *out, bool full_eq18, double *out_mu,
                              cudaStream_t s)
{
    // `coef` is ctx->coef + 12 g0 for the group starting at point g0: its rates are ctx->rate + 4 g0
    const double *rate = nullptr;
    if (coef && coef >= ctx->coef && coef < ctx->coef + (size_t)ctx->lay.max_batch * kCoefStride)
        rate = ctx->rate + (coef - ctx->coef) / kCoefStride * RW_MAX_COMPONENTS;
    const Layout &L = ctx->lay;
    RidgeArgs A;
    A.R = ctx->R; A.R_period_stride = ctx->R_period_stride; A.ldR = ctx->ldR;
    A.n_T = ctx->n_T; A.n_rec = ctx->n_rec; A.D = ctx->D;
    A.coef = coef; A.param = param; A.wts = wts;
    A.rate = rate; A.comp8 = ctx->comp8;
    A.What = ctx->What; A.N_mc = ctx->N_mc; A.bkg = ctx->bkg; A.counts = ctx->counts;
    A.sat_const = full_eq18 ? ctx->sat_const : nullptr;
    A.Pb = Pb;
    const int mbl = Pb <= 8 ? 0 : Pb <= 16 ? 1 : Pb <= 32 ? 2 : 3;     // tile height 8 << mbl
    A.rows_per_split = L.ridge_rows[mbl];
    A.n_splits = (ctx->n_T + A.rows_per_split - 1) / A.rows_per_split;
    A.mu_ld = (ctx->n_rec + 1) & ~1;
    A.mu_part = ctx->mu_part; A.strip_part = ctx->ridge_part; A.cnt = ctx->ridge_cnt;
    A.out = out; A.out_mu = out_mu;
    Kinds none;
    none.k = 0;
    for (int a = 0; a < RW_N_KINDS; ++a) none.kind[a] = -1;
    const Kinds &k = kd ? *kd : none;
    dim3 grid(L.ridge_strips, A.n_splits, ctx->D);
    cudaError_t e;
    {
        ProfScope prof(ctx, s);
        if (mbl == 0) e = launch_ridge_t<1>(A, k, ctx->cst, grid, s);
        else if (mbl == 1) e = launch_ridge_t<2>(A, k, ctx->cst, grid, s);
        else if (mbl == 2) e = launch_ridge_t<4>(A, k, ctx->cst, grid, s);
        else e = launch_ridge_t<8>(A, k, ctx->cst, grid, s);
    }
    if (e != cudaSuccess) return e;
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
