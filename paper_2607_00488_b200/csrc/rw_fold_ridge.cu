// rw_fold_ridge.cu -- the whole path for 2..64 points in ONE kernel: the regime around the ridge of the
// roofline (P* = 4 F / BW ~ 23 points on B200), where the fold
//   mu[p][k] = sum_i N'[p][i] R[i][k] + bkg[k]                                  (Eq. 11)
// has to read every byte of R exactly once at HBM speed AND do 2 P flop per 8 bytes, more than scalar DFMA
// can issue next to the loads.  Design:
//   * stream-K decomposition: the work is the sequence of (period, 256-column strip, block of RS recoil rows)
//     units, strip-major; CTA j of G takes the units [j U / G, (j + 1) U / G) -- one wave, every SM streams the
//     same number of bytes whatever the shape.  A span that crosses a strip boundary is cut into segments; a strip
//     shared by several CTAs is finished by whichever of them arrives last (ticket), adding the parked partial tiles
//     in CTA order, so the result does not depend on the arrival order;
//   * a producer warp keeps a ring of 4-6 stages of RS rows in flight (up to 200 KB per SM -- registers cannot
//     hold that much: a first version with the loads going straight into the fragments stayed at 5.4 TB/s): one plain
//     bulk copy (cp.async.bulk, mbarrier completion, L2 evict-first) per row, 2 KB requests, exactly the strip's
//     bytes; the rows land at a pitch of 2064 bytes (= 16 mod 64: the rows 2 c + j a quarter-warp reads fall in four
//     different 32-byte bank groups), which makes the fragment loads conflict free without a swizzle;
//   * the arithmetic of k_fold_gemm: mma.sync.m8n8k4.f64 (DMMA.8x8x4).  Eight consumer warps own 32 columns each
//     and all points of the tile; lane (r = lane / 4, c = lane % 4) reads the 16 bytes R[i + 2 c + j][col + 2 r .. + 1]
//     -- one B fragment for the even and one for the odd columns of a 16-column group;
//   * N' of the next 64 recoil rows x 8 MB points (steps a1 + a2: coefficients from the raw parameters, Eq. 6,
//     PAPER.md:79; N' = sum_b c_b W^_b, Eq. 14 / Eq. 1) is itself a [8 MB x 12] x [12 x 8] DMMA per
//     8 rows -- consumer warp w forms the 8-row block w of the next chunk (operands prefetched a chunk ahead) -- whose
//     C fragment (point r, rows 2 c and 2 c + 1) IS the A fragment of the fold's two k-steps when k-step j takes the
//     rows {2 c + j}: the lanes store and reload their own 16 bytes (double-buffered, lane-linear: no bank conflicts,
//     no transposition).  3 MB DMMAs per warp and chunk instead of 22 MB DFMAs per thread: with scalar staging the
//     tensor pipe was 75 % busy at 64 points, and separate scalar stager warps could not keep up at all;
//   * tile heights 32 and 64 (17..64 points) take N' ready-made instead: k_ridge_frag writes it once per call in the
//     fragment layout and one more warp copies it chunk by chunk (one bulk copy) into the two buffers -- formed in the
//     consumer warps, the dependent chain load -> 3 DMMA -> store and its bar.sync cost 10 % of the kernel there, and
//     stager warps (DMMA or scalar) only queue behind the consumers: on B200 DFMA and DMMA share one pipe;
//   * at 64 points setmaxnreg moves the registers of the producer warpgroup to the consumers (128 accumulators);
//   * a4: the finishing CTA of a strip adds bkg and reduces the Poisson terms of Eq. (18) of its 256
//     columns; the last strip adds strips and periods in a fixed order and writes -2lnL.  One launch per call.
#include "rw_internal.h"

namespace rw {

constexpr int kRgWarps = 8;                           // consumer (DMMA) warps: two warpgroups
constexpr int kRgConsumers = kRgWarps * 32;
constexpr int kRgThreads = kRgConsumers + 32;         // + the producer warp (tile heights 8, 16, 32)
constexpr int kRgThreads64 = kRgConsumers + 128;      // tile height 64: a producer warpgroup for setmaxnreg (3 warps idle)
constexpr int kRgWarpCols = 32;                       // two 16-column groups per warp
constexpr int kRgCols = kRgWarps * kRgWarpCols;       // 256 columns per strip
constexpr int kRgKC = 64;                             // recoil rows of N' per chunk: one 8-row block per consumer warp
constexpr int kRgNB = 2;                              // N' buffers
constexpr int kRgRowBytes = kRgCols * 8 + 16;         // ring pitch 2064 B = 16 (mod 64): rows 2 c + j -> 4 bank groups
static_assert(kRgCols == kRidgeCols, "plan() in rw_api.cu assumes this strip width");

struct RidgeArgs {
    const double *R; size_t R_period_stride; int ldR, n_T, n_rec, D;
    const double *coef;       // [Pb][12], or NULL
    const double *param;      // [Pb][k] raw parameters (coefficients computed here), or NULL
    const double *wts;        // [Pb][n_T] caller weights, or NULL
    const double *rate;       // [Pb][4] rate scales matching `coef`, or NULL
    const uint8_t *comp8;     // [n_T] component of every recoil bin
    const double *What, *N_mc, *bkg, *counts, *sat_const;
    int Pb, n_strips, nblk;   // strips per period; blocks of RS rows per strip
    int zero_ring;            // ragged strip or row tail: the ring is read where no copy lands
    int zero;                 // 0, opaque to the compiler (release of a ring stage at 16 points)
    double *frag;             // tile heights 32, 64: N' as DMMA fragments [D][nblk8][MB][32 lanes] x 16 B (k_ridge_frag)
    int nblk8;                // 8-row blocks per period in `frag` (n_T / 8 rounded up, + 8 zero blocks)
    double *slots;            // [3 G][8 MB][256] parked partial tiles
    double *strip_part;       // [G][64] Poisson sums of everything a CTA finished
    int *cnt;                 // [D * strips] "parked" tickets, [D * strips] "left" tickets, one global ticket
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
__device__ __forceinline__ void rg_bar_consumers() { asm volatile("bar.sync 1, %0;" ::"n"(kRgConsumers) : "memory"); }

template <int MB> struct RidgeCfg {
    static constexpr int PP = 8 * MB;                                  // points of the tile
    // Tile heights 24 .. 64 (MB >= 3) read N' ready-made (k_ridge_frag writes it once per call instead of once per column
    // strip in every CTA; in the consumer warps the chain load W^ -> 3 DMMA -> store and the bar.sync behind it idled the
    // tensor pipe for 10 % of the kernel there): one more warp copies it chunk by chunk into the two N' buffers.
    // Every multiple of 8 points has its own instantiation: above 16 points the kernel is bound by the DMMA pipe, so its
    // time follows the tile height, not the number of points (33 points in a 64-row tile ran at 0.46 of the bound).
    static constexpr bool Prefab = (MB >= 3);
    static constexpr bool Big = (MB >= 7);                             // 112 / 128 accumulator registers: setmaxnreg
    static constexpr int RS = Prefab ? 16 : 8;                         // recoil rows per ring stage (= per work unit)
    static constexpr int NS = (MB == 1) ? 6 : Big ? 4 : 5;             // ring stages
    static constexpr int MinCtas = Prefab ? 1 : 2;
    // How a ring stage is handed back safely (see the consumer loop): one iteration late (free, but one stage less in
    // flight), or at once through a register dependence on its fragment loads (16 points: five 16 KB stages per CTA
    // are too few to give one away -- 0.199 ms against 0.214 ms on config 4)
    static constexpr bool LateRelease = (MB != 2);
    static constexpr int Threads = Big ? kRgThreads64 : Prefab ? kRgThreads + 32 : kRgThreads;
    // tile heights 56, 64: setmaxnreg redistributes the registers the CTA was LAUNCHED with (384 x 168): 256 ConsumerRegs +
    // 128 HelperRegs must not exceed that pool, or the consumers wait for ever
    static constexpr int ConsumerRegs = 224, HelperRegs = 40;
    static_assert(kRgConsumers * ConsumerRegs + 128 * HelperRegs <= kRgThreads64 * 168, "setmaxnreg pool");
    static constexpr int StageBytes = RS * kRgRowBytes;
    static constexpr int RingBytes = NS * StageBytes;
    static constexpr int NBytes = kRgNB * (kRgKC / 8) * MB * 512;      // N' fragments: [buffer][8-row block][mb][lane] x 16 B
    static constexpr int SmemDoubles = PP * kCoefStride + PP * RW_MAX_COMPONENTS + kRgWarps * PP;
    static constexpr int Smem = RingBytes + NBytes + SmemDoubles * 8 + 2 * NS * 8 + 2 * kRgNB * 8;
};

// Work split shared by the three roles.  Units u = tile * nblk + block; CTA j owns [u0(j), u0(j + 1)).
struct RidgeSplit {
    long long U;
    int G, nblk;
    __device__ __forceinline__ long long u0(int j) const { return (long long)j * U / G; }
    __device__ __forceinline__ int cta_of(long long u) const { return (int)(((u + 1) * G - 1) / U); }
    // slot of CTA j's partial tile of `tile`: 3 j + {0: the tile its span starts in, 2: the tile it ends in, 1: a
    // whole tile in between (private, reused)}.  Four 64-bit divisions: never inside a loop over contributors.
    __device__ __forceinline__ int slot_of(int j, int tile) const
    {
        const long long a = u0(j), b = u0(j + 1) - 1;
        if (tile == (int)(a / nblk)) return 3 * j;
        if (tile == (int)(b / nblk)) return 3 * j + 2;
        return 3 * j + 1;
    }
};

template <int MB>
__global__ void __launch_bounds__(RidgeCfg<MB>::Threads, RidgeCfg<MB>::MinCtas)
k_fold_ridge(const RidgeArgs A, const Kinds kd, const Consts cst)
{
    using Cfg = RidgeCfg<MB>;
    constexpr int PP = Cfg::PP, RS = Cfg::RS, NS = Cfg::NS;
    // 128-byte aligned so that the bank analysis of the ring pitch holds; indexed directly (a re-aligned pointer
    // would lose its address space and turn the fragment loads into generic LD)
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t ring = rg_smem_u32(smem);
    const uint32_t sN = ring + Cfg::RingBytes;                         // [2 buffers][8 blocks][MB][32 lanes] double2
    double *sC = reinterpret_cast<double *>(smem + Cfg::RingBytes + Cfg::NBytes);   // [PP][12]
    double *sRate = sC + PP * kCoefStride;                             // [PP][4]
    double *red = sRate + PP * RW_MAX_COMPONENTS;                      // [8 warps][PP]
    const uint32_t full_bar = rg_smem_u32(red + kRgWarps * PP);        // ring: NS full, NS empty
    const uint32_t empty_bar = full_bar + NS * 8;
    const uint32_t nfull_bar = empty_bar + NS * 8;                     // the two N' buffers (tile heights 32, 64)
    const uint32_t nempty_bar = nfull_bar + kRgNB * 8;
    __shared__ int s_flag;
    __shared__ int s_slot[2 * kRidgePlanSMs + 8];                       // slots of the contributors of the tile being finished

    const int n_T = A.n_T, n_rec = A.n_rec, Pb = A.Pb;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_tiles = A.D * A.n_strips;
    RidgeSplit sp;
    sp.nblk = A.nblk; sp.U = (long long)n_tiles * A.nblk; sp.G = gridDim.x;
    const long long ua = sp.u0(blockIdx.x), ub = sp.u0(blockIdx.x + 1);
    const int tile_a = (int)(ua / sp.nblk), tile_b = (int)((ub - 1) / sp.nblk);   // first and last tile of this CTA's span

    if (threadIdx.x == 0) {
        for (int s = 0; s < NS; ++s) {
            rg_mbar_init(full_bar + 8 * s, 1);
            rg_mbar_init(empty_bar + 8 * s, kRgWarps);
        }
        for (int s = 0; s < kRgNB; ++s) {
            rg_mbar_init(nfull_bar + 8 * s, 1);
            rg_mbar_init(nempty_bar + 8 * s, kRgWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (A.zero_ring) {               // the ring is also read where no copy ever lands (times N' = 0): finite numbers
        for (int q = threadIdx.x; q < Cfg::RingBytes / 16; q += Cfg::Threads)
            reinterpret_cast<double2 *>(smem)[q] = make_double2(0.0, 0.0);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (warp >= kRgWarps) {
        if constexpr (Cfg::Big) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(Cfg::HelperRegs));
        if (warp == kRgWarps) {
            // ------------------------------------------------------------ producer: lane l copies row l of a stage
            uint64_t policy;
            asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
            int stage = 0;
            uint32_t phase = 0;
            for (long long u = ua; u < ub;) {
                const int tile = (int)(u / sp.nblk), b0 = (int)(u - (long long)tile * sp.nblk);
                const int nb = (int)min((long long)(sp.nblk - b0), ub - u);
                const int d = tile / A.n_strips, strip = tile - d * A.n_strips;
                const int row0 = b0 * RS, nrows = min(n_T, (b0 + nb) * RS) - row0;
                const uint32_t row_bytes = (uint32_t)min(kRgCols, A.ldR - strip * kRgCols) * 8;   // even; a copied R is zero-padded
                const double *src = A.R + (size_t)d * A.R_period_stride + (size_t)(row0 + lane) * A.ldR + (size_t)strip * kRgCols;
                for (int q = 0; q < nb; ++q) {
                    rg_mbar_wait(empty_bar + 8 * stage, phase ^ 1);
                    const int rows = min(RS, nrows - q * RS);
                    const uint32_t fb = full_bar + 8 * stage;
                    if (lane == 0) rg_mbar_expect_tx(fb, (uint32_t)rows * row_bytes);
                    __syncwarp();
                    if (lane < rows)
                        rg_bulk_row(ring + stage * Cfg::StageBytes + lane * kRgRowBytes, src + (size_t)q * RS * A.ldR,
                                    row_bytes, fb, policy);
                    if (++stage == NS) { stage = 0; phase ^= 1; }
                }
                u += nb;
            }
        } else if (Cfg::Prefab && warp == kRgWarps + 1 && lane == 0) {
            // ------------------------------------------------------------ N' loader: chunk n -> buffer n & 1
            uint64_t policy;
            asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(policy));    // read by every strip
            uint32_t n = 0;
            for (long long u = ua; u < ub;) {
                const int tile = (int)(u / sp.nblk), b0 = (int)(u - (long long)tile * sp.nblk);
                const int nb = (int)min((long long)(sp.nblk - b0), ub - u);
                const int d = tile / A.n_strips;
                const int row0 = b0 * RS, row1 = min(n_T, (b0 + nb) * RS);
                u += nb;
                for (int ic = row0; ic < row1; ic += kRgKC, ++n) {
                    const uint32_t buf = n & 1;
                    rg_mbar_wait(nempty_bar + 8 * buf, ((n >> 1) & 1) ^ 1);     // the consumers are done with chunk n - 2
                    constexpr uint32_t bytes = (kRgKC / 8) * MB * 512;
                    rg_mbar_expect_tx(nfull_bar + 8 * buf, bytes);
                    rg_bulk_row(sN + buf * bytes, A.frag + ((size_t)d * A.nblk8 + ic / 8) * (MB * 64), bytes,
                                nfull_bar + 8 * buf, policy);
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumers
    if constexpr (Cfg::Big) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(Cfg::ConsumerRegs));
    // ---------------------------------------------------------------- a1: coefficients of the tile's points
    const double *wts = A.wts;
    if (!wts && !Cfg::Prefab) {
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
            for (int q = threadIdx.x; q < PP * kCoefStride; q += kRgConsumers) sC[q] = (q / kCoefStride < Pb) ? A.coef[q] : 0.0;
            for (int q = threadIdx.x; q < PP * RW_MAX_COMPONENTS; q += kRgConsumers)
                sRate[q] = (q / RW_MAX_COMPONENTS < Pb && A.rate) ? A.rate[q] : 1.0;
        }
    }
    rg_bar_consumers();                              // (the producer is already streaming R)
    const int r = lane >> 2, c = lane & 3;
    // B fragments: rows 2 c + j of an 8-row block, columns 32 warp + 16 g + 2 r + {0, 1}
    const uint32_t b_off = (uint32_t)(2 * c) * kRgRowBytes + (uint32_t)(kRgWarpCols * warp + 2 * r) * 8;
    // ---------------------------------------------------------------- a4, shared out among the contributors of a tile
    // Once every contributor [jf, jl] of `tile` has parked its partial tile, contributor ci = j - jf finishes the points
    // [ci PPc, (ci + 1) PPc) of it for all 256 columns: sums the parked partials in CTA order (the result does not
    // depend on who arrives when), adds bkg, reduces the Poisson terms of Eq. (18).  One round trip to L2 per CTA instead
    // of one per contributor in a single finishing CTA (which cost 7 / 15 / 21 us of a 0.18 / 0.19 / 0.32 ms call at
    // 4 / 16 / 32 points).  Thread t keeps the running sum of point t over everything this CTA finishes.
    double my_part = 0.0;
    auto finish_slice = [&](const int tile, const int jf, const int jl) {
        const int d = tile / A.n_strips, strip = tile - d * A.n_strips;
        const int ncon = jl - jf + 1, ci = blockIdx.x - jf;
        const int PPc = (Pb + ncon - 1) / ncon;
        const int p_lo = ci * PPc, p_hi = min(Pb, p_lo + PPc);
        if (p_lo >= p_hi) return;                                       // (uniform) more contributors than points
        const int col = strip * kRgCols + threadIdx.x;
        const bool col_ok = col < n_rec;
        double bk = 0.0, cn = 0.0;
        if (col_ok) { bk = A.bkg[(size_t)d * n_rec + col]; cn = A.counts[(size_t)d * n_rec + col]; }
#pragma unroll 1
        for (int p0 = p_lo; p0 < p_hi; p0 += 4) {
            double m[4] = {0.0, 0.0, 0.0, 0.0};
            for (int j0 = 0; j0 < ncon; j0 += 8) {                      // 4 points x 8 contributors = 32 loads in flight
                double v[8][4];
#pragma unroll
                for (int jj = 0; jj < 8; ++jj) {
                    const double *src = A.slots + (size_t)s_slot[min(j0 + jj, ncon - 1)] * (PP * kRgCols) + threadIdx.x;
#pragma unroll
                    for (int e = 0; e < 4; ++e) v[jj][e] = __ldcg(src + (size_t)min(p0 + e, p_hi - 1) * kRgCols);
                }
#pragma unroll
                for (int jj = 0; jj < 8; ++jj)
                    if (j0 + jj < ncon) {
#pragma unroll
                        for (int e = 0; e < 4; ++e) m[e] += v[jj][e];
                    }
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int p = p0 + e;
                double t = 0.0;
                if (col_ok && p < p_hi) {
                    const double a = m[e] + bk;
                    if (A.out_mu) A.out_mu[((size_t)p * A.D + d) * n_rec + col] = a;
                    t = poisson_term(a, cn);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                if (lane == 0 && p < p_hi) red[warp * PP + p] = t;
            }
        }
        rg_bar_consumers();
        if ((int)threadIdx.x >= p_lo && (int)threadIdx.x < p_hi) {
#pragma unroll
            for (int w = 0; w < kRgWarps; ++w) my_part += red[w * PP + threadIdx.x];
        }
        rg_bar_consumers();                                             // red is rewritten by the next tile
    };
    // a shared tile: wait until all its contributors have parked (they are co-resident: one wave, cooperative launch),
    // finish this CTA's share, and let the last one to leave reset the two tickets for the next launch
    auto finish_shared = [&](const int tile) {
        const int jf = sp.cta_of((long long)tile * sp.nblk), jl = sp.cta_of((long long)(tile + 1) * sp.nblk - 1);
        const int ncon = jl - jf + 1;
        for (int t = threadIdx.x; t < ncon; t += kRgConsumers) s_slot[t] = sp.slot_of(jf + t, tile);   // four 64-bit divisions each
        if (threadIdx.x == 0) {
            const volatile int *tk = A.cnt + tile;
            while (*tk < ncon) __nanosleep(64);
        }
        rg_bar_consumers();
        __threadfence();
        finish_slice(tile, jf, jl);
        if (threadIdx.x == 0 && atomicAdd(A.cnt + n_tiles + tile, 1) == ncon - 1) {
            A.cnt[tile] = 0;                                            // everyone is past the wait above
            A.cnt[n_tiles + tile] = 0;
        }
    };
    uint32_t chunk_n = 0;             // chunks folded so far (tile heights 32, 64: N' buffer chunk_n & 1, phase (chunk_n >> 1) & 1)
    int nrelease = -1;                // N' buffer of the previous chunk, not yet handed back to the loader
    int pending = 0;                  // shared tiles this CTA arrived at last: bit 0 the first of its span, bit 1 the last
    int stage = 0, release = -1;      // `release`: the stage consumed in the previous iteration, not yet handed back
    uint32_t phase = 0;
    for (long long u = ua; u < ub;) {
        const int tile = (int)(u / sp.nblk), b0 = (int)(u - (long long)tile * sp.nblk);
        const int nb = (int)min((long long)(sp.nblk - b0), ub - u);
        const int d = tile / A.n_strips;
        const int row0 = b0 * RS, row1 = min(n_T, (b0 + nb) * RS);
        u += nb;

        // ------------------------------------------------------------ a2: this warp's 8-row block of a 64-row chunk
        // Lane (r, c): the B fragment of the staging product is W^[4 ks + c][i + r], the A fragment c[8 mb + r][4 ks + c],
        // and the C fragment N'[8 mb + r][i + 2 c], N'[8 mb + r][i + 2 c + 1] is what the same lane of every warp loads
        // back as the A fragment of the fold.  fetch() runs a chunk ahead of form().
        const double *Wd = A.What + (size_t)d * kCoefStride * n_T;
        double bw[3];
        int cq0 = 0, cq1 = 0;
        auto fetch = [&](int ic) {
            const int i0 = ic + 8 * warp, ia = i0 + 2 * c;
#pragma unroll
            for (int ks = 0; ks < 3; ++ks) {
                const int b = 4 * ks + c;
                bw[ks] = (!wts && b < kNumTerms && i0 + r < row1) ? __ldg(Wd + (size_t)b * n_T + i0 + r) : 0.0;
            }
            cq0 = (ia < row1) ? A.comp8[ia] : 0;
            cq1 = (ia + 1 < row1) ? A.comp8[ia + 1] : 0;
        };
        auto form = [&](int ic, int buf) {
            const int ia = ic + 8 * warp + 2 * c;
            const uint32_t dst = sN + (uint32_t)((buf * (kRgKC / 8) + warp) * MB) * 512 + lane * 16;
            if (wts) {
                const double n0 = (ia < row1) ? A.N_mc[(size_t)d * n_T + ia] : 0.0;
                const double n1 = (ia + 1 < row1) ? A.N_mc[(size_t)d * n_T + ia + 1] : 0.0;
#pragma unroll
                for (int mb = 0; mb < MB; ++mb) {
                    const int p = 8 * mb + r;
                    const double v0 = (p < Pb && ia < row1) ? wts[(size_t)p * n_T + ia] * n0 : 0.0;
                    const double v1 = (p < Pb && ia + 1 < row1) ? wts[(size_t)p * n_T + ia + 1] * n1 : 0.0;
                    asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(dst + mb * 512), "d"(v0), "d"(v1) : "memory");
                }
            } else {
#pragma unroll
                for (int mb = 0; mb < MB; ++mb) {
                    const int p = 8 * mb + r;
                    double v0 = 0.0, v1 = 0.0;
#pragma unroll
                    for (int ks = 0; ks < 3; ++ks) rg_dmma(v0, v1, sC[p * kCoefStride + 4 * ks + c], bw[ks]);
                    v0 *= sRate[p * RW_MAX_COMPONENTS + cq0];     // rate_k of Eq. (17); 1 when not scanned
                    v1 *= sRate[p * RW_MAX_COMPONENTS + cq1];
                    asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(dst + mb * 512), "d"(v0), "d"(v1) : "memory");
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
                for (int e = 0; e < 2; ++e) acc[mb][g][e][0] = acc[mb][g][e][1] = 0.0;
        if constexpr (!Cfg::Prefab) {
            fetch(row0);
            form(row0, 0);
        }
        int q = 0, nbuf = 0;
        for (int ic = row0; ic < row1; ic += kRgKC, nbuf ^= 1) {
            const bool more = ic + kRgKC < row1;
            if constexpr (Cfg::Prefab) {
                nbuf = (int)(chunk_n & 1);
                rg_mbar_wait(nfull_bar + 8 * nbuf, (chunk_n >> 1) & 1);        // N' of this chunk has landed
            } else {
                rg_bar_consumers();                  // N'[nbuf] formed by all warps; N'[nbuf ^ 1] no longer read
                if (more) fetch(ic + kRgKC);
            }
            const uint32_t sA = sN + (uint32_t)(nbuf * (kRgKC / 8) * MB) * 512 + lane * 16;
#pragma unroll
            for (int sq = 0; sq < kRgKC / RS; ++sq) {
                if (q < nb) {
                    rg_mbar_wait(full_bar + 8 * stage, phase);
                    if constexpr (Cfg::Prefab) {
                        // the N' buffer of the previous chunk goes back to the loader only now: every DMMA that read it
                        // has been issued, so its fragment loads have returned (the hazard described at the ring release)
                        if (nrelease >= 0) {
                            if (lane == 0) rg_mbar_arrive(nempty_bar + 8 * nrelease);
                            nrelease = -1;
                        }
                    }
                    const uint32_t st = ring + stage * Cfg::StageBytes + b_off;
                    uint32_t dep = 0;
#pragma unroll
                    for (int hb = 0; hb < RS / 8; ++hb) {              // 8-row blocks of this stage
                        double2 a[MB];
#pragma unroll
                        for (int mb = 0; mb < MB; ++mb)
                            asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(a[mb].x), "=d"(a[mb].y)
                                         : "r"(sA + (uint32_t)((sq * (RS / 8) + hb) * MB + mb) * 512));
#pragma unroll
                        for (int j = 0; j < 2; ++j) {                  // k-step j: rows 2 c + j of the block
                            double2 b[2];
#pragma unroll
                            for (int g = 0; g < 2; ++g)
                                asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(b[g].x), "=d"(b[g].y)
                                             : "r"(st + (uint32_t)(8 * hb + j) * kRgRowBytes + (uint32_t)g * 128));
                            if constexpr (!Cfg::LateRelease)
                                dep |= (uint32_t)__double2hiint(b[0].x) | (uint32_t)__double2hiint(b[1].x);
#pragma unroll
                            for (int mb = 0; mb < MB; ++mb) {
                                const double av = j ? a[mb].y : a[mb].x;
#pragma unroll
                                for (int g = 0; g < 2; ++g) {
                                    rg_dmma(acc[mb][g][0][0], acc[mb][g][0][1], av, b[g].x);
                                    rg_dmma(acc[mb][g][1][0], acc[mb][g][1][1], av, b[g].y);
                                }
                            }
                        }
                    }
                    // A stage may be handed back only when every fragment load of it has RETURNED.  Released right behind
                    // the loop, ptxas issues the arrive directly after the last LDS, and the producer's next copy into the
                    // stage has been seen to overtake that load (two CTAs per SM, 16 points: 32-byte pieces of a later row
                    // in one fragment, -2lnL off by 1e-8 .. 1e-3 relative in every other run).  Either the arrive comes one
                    // iteration late, behind the next stage's barrier wait (every DMMA reading the stage has been issued
                    // by then), or its address depends on the loaded registers (& 0 the compiler cannot see; a warp-wide
                    // LDS completes as one instruction, so lane 0's registers stand for the warp).
                    __syncwarp();
                    if constexpr (Cfg::LateRelease) {
                        if (lane == 0 && release >= 0) rg_mbar_arrive(empty_bar + 8 * release);
                        release = stage;
                    } else {
                        if (lane == 0) rg_mbar_arrive(empty_bar + 8 * stage + (dep & (uint32_t)A.zero));
                    }
                    if (++stage == NS) { stage = 0; phase ^= 1; }
                    ++q;
                }
            }
            if constexpr (Cfg::Prefab) {
                __syncwarp();
                nrelease = nbuf;
                ++chunk_n;
            } else {
                if (more) form(ic + kRgKC, nbuf ^ 1);
            }
        }

        // ------------------------------------------------------------ park the partial tile of this segment
        // column 4 c + 2 e + nb of a 16-column group holds acc[.][.][nb][e]; tile-local layout [8 MB][256]
        {
            const int my_slot = 3 * blockIdx.x + (tile == tile_a ? 0 : tile == tile_b ? 2 : 1);     // = sp.slot_of(blockIdx.x, tile)
            double *slot = A.slots + (size_t)my_slot * (PP * kRgCols);
#pragma unroll
            for (int mb = 0; mb < MB; ++mb)
#pragma unroll
                for (int g = 0; g < 2; ++g) {
                    double *dst = slot + (8 * mb + r) * kRgCols + warp * kRgWarpCols + 16 * g + 4 * c;
                    __stcg(reinterpret_cast<double2 *>(dst), make_double2(acc[mb][g][0][0], acc[mb][g][1][0]));
                    __stcg(reinterpret_cast<double2 *>(dst + 2), make_double2(acc[mb][g][0][1], acc[mb][g][1][1]));
                }
        }
        // ------------------------------------------------------------ a4
        // A tile shared with other CTAs is finished by all of them together -- but not now: a CTA that still has a
        // segment to stream would stall its ring; the partial tile waits in its slot until this CTA has streamed
        // everything.  A tile this CTA owns alone is finished at once (its slot 3 j + 1 is reused by the next one).
        const int jf = sp.cta_of((long long)tile * sp.nblk), jl = sp.cta_of((long long)(tile + 1) * sp.nblk - 1);
        __threadfence();
        rg_bar_consumers();
        if (jl > jf) {
            if (threadIdx.x == 0) atomicAdd(A.cnt + tile, 1);          // parked
            pending |= (tile == tile_a) ? 1 : 2;                       // a shared tile is the first or the last of the span
        } else {
            if (threadIdx.x == 0) s_slot[0] = 3 * blockIdx.x + (tile == tile_a ? 0 : tile == tile_b ? 2 : 1);
            rg_bar_consumers();
            finish_slice(tile, jf, jl);
        }
    }
    if (pending & 1) finish_shared(tile_a);
    if (pending & 2) finish_shared(tile_b);

    // ---------------------------------------------------------------- the last CTA adds the CTAs' sums and writes -2lnL
    if (threadIdx.x < PP) __stcg(A.strip_part + (size_t)blockIdx.x * kRidgeMaxP + threadIdx.x, my_part);
    __threadfence();
    rg_bar_consumers();
    if (threadIdx.x == 0) s_flag = atomicAdd(A.cnt + 2 * n_tiles, 1);
    rg_bar_consumers();
    if (s_flag != (int)gridDim.x - 1) return;
    __threadfence();
    // warp w adds the CTAs w, w + 8, ... for point `lane` (+ 32), eight loads in flight, then the eight warps in order
#pragma unroll
    for (int h = 0; h < (PP + 31) / 32; ++h) {
        const int p = 32 * h + lane;
        double v = 0.0;
        if (p < Pb) {
            for (int j0 = warp; j0 < (int)gridDim.x; j0 += 8 * kRgWarps) {
                double x[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int j = j0 + u * kRgWarps;
                    x[u] = (j < (int)gridDim.x) ? __ldcg(A.strip_part + (size_t)j * kRidgeMaxP + p) : 0.0;
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) v += x[u];
            }
        }
        if (p < PP) red[warp * PP + p] = v;
    }
    rg_bar_consumers();
    if (threadIdx.x < Pb) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < kRgWarps; ++w) v += red[w * PP + threadIdx.x];
        v *= 2.0;
        if (A.sat_const) v += A.sat_const[0];
        A.out[threadIdx.x] = v;
    }
    if (threadIdx.x == 0) A.cnt[2 * n_tiles] = 0;                      // ready for the next launch
}

// a1 + a2 for tile heights 32 and 64: N' of all recoil rows, once per call, in the fragment layout of the fold --
// block of 8 rows, 8-point group mb, lane (r, c): { N'[8 mb + r][8 blk + 2 c], N'[8 mb + r][8 blk + 2 c + 1] }.
// One CTA per 64 rows and period; thread (blk_local, lane), all mb.  Rows >= n_T and points >= Pb are zero.
__global__ void __launch_bounds__(256)
k_ridge_frag(const RidgeArgs A, const Kinds kd, const Consts cst, const int MB)
{
    __shared__ double sC[kRidgeMaxP * kCoefStride];
    __shared__ double sRate[kRidgeMaxP * RW_MAX_COMPONENTS];
    const int PP = 8 * MB, Pb = A.Pb, n_T = A.n_T, d = blockIdx.y;
    if (!A.wts) {
        if (A.param) {
            if ((int)threadIdx.x < PP) {
                double cc[kCoefStride], rr[RW_MAX_COMPONENTS];
                if ((int)threadIdx.x < Pb) {
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
            for (int q = threadIdx.x; q < PP * kCoefStride; q += 256) sC[q] = (q / kCoefStride < Pb) ? A.coef[q] : 0.0;
            for (int q = threadIdx.x; q < PP * RW_MAX_COMPONENTS; q += 256)
                sRate[q] = (q / RW_MAX_COMPONENTS < Pb && A.rate) ? A.rate[q] : 1.0;
        }
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, r = lane >> 2, c = lane & 3;
    const int blk = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (blk >= A.nblk8) return;
    const int ia = 8 * blk + 2 * c;
    const bool ok0 = ia < n_T, ok1 = ia + 1 < n_T;
    double2 *dst = reinterpret_cast<double2 *>(A.frag) + ((size_t)d * A.nblk8 + blk) * (MB * 32) + lane;
    if (A.wts) {
        const double n0 = ok0 ? A.N_mc[(size_t)d * n_T + ia] : 0.0, n1 = ok1 ? A.N_mc[(size_t)d * n_T + ia + 1] : 0.0;
        for (int mb = 0; mb < MB; ++mb) {
            const int p = 8 * mb + r;
            dst[mb * 32] = make_double2((p < Pb && ok0) ? A.wts[(size_t)p * n_T + ia] * n0 : 0.0,
                                        (p < Pb && ok1) ? A.wts[(size_t)p * n_T + ia + 1] * n1 : 0.0);
        }
        return;
    }
    const double *Wd = A.What + (size_t)d * kCoefStride * n_T;
    double w0[kNumTerms], w1[kNumTerms];
#pragma unroll
    for (int b = 0; b < kNumTerms; ++b) {
        w0[b] = ok0 ? __ldg(Wd + (size_t)b * n_T + ia) : 0.0;
        w1[b] = ok1 ? __ldg(Wd + (size_t)b * n_T + ia + 1) : 0.0;
    }
    const int cq0 = ok0 ? A.comp8[ia] : 0, cq1 = ok1 ? A.comp8[ia + 1] : 0;
    for (int mb = 0; mb < MB; ++mb) {
        const int p = 8 * mb + r;
        double v0 = 0.0, v1 = 0.0;
#pragma unroll
        for (int b = 0; b < kNumTerms; ++b) {
            const double cb = sC[p * kCoefStride + b];
            v0 = fma(cb, w0[b], v0);
            v1 = fma(cb, w1[b], v1);
        }
        dst[mb * 32] = make_double2(v0 * sRate[p * RW_MAX_COMPONENTS + cq0], v1 * sRate[p * RW_MAX_COMPONENTS + cq1]);   // rate_k of Eq. (17)
    }
}

template <int MB>
static cudaError_t launch_ridge_t(const RidgeArgs &A, const Kinds &kd, const Consts &cst, int grid, cudaStream_t s)
{
    // (the > 48 KB dynamic shared memory attribute is set by ridge_setup() at rw_create, for the device of the context)
    // cooperative: the contributors of a tile wait for one another, so the whole grid (one wave by construction,
    // ridge_grid) must be resident at once; the launch fails instead of hanging where it could not be
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(RidgeCfg<MB>::Threads);
    cfg.dynamicSmemBytes = RidgeCfg<MB>::Smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_fold_ridge<MB>, A, kd, cst);
}

template <int MB> static cudaError_t ridge_attr_t()
{
    return cudaFuncSetAttribute(k_fold_ridge<MB>, cudaFuncAttributeMaxDynamicSharedMemorySize, RidgeCfg<MB>::Smem);
}

// rw_create: the function attributes belong to the device that is current, not to the process -- a context on a
// second GPU of the same process needs them set again, so no "done once" flag.
int ridge_setup(rw_ctx *ctx)
{
    cudaError_t e = ridge_attr_t<1>();
    if (e == cudaSuccess) e = ridge_attr_t<2>();
    if (e == cudaSuccess) e = ridge_attr_t<3>();
    if (e == cudaSuccess) e = ridge_attr_t<4>();
    if (e == cudaSuccess) e = ridge_attr_t<5>();
    if (e == cudaSuccess) e = ridge_attr_t<6>();
    if (e == cudaSuccess) e = ridge_attr_t<7>();
    if (e == cudaSuccess) e = ridge_attr_t<8>();
    if (e != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "cudaFuncSetAttribute(k_fold_ridge): %s", cudaGetErrorString(e));
    return RW_OK;
}

// Grid of k_fold_ridge for tile height 8 << mb_log2 (mb_log2 >= 2: any of the heights 24 .. 64): one wave of the SM slots, but at least ~256 recoil rows of one
// strip per CTA (a smaller share is not worth a partial tile).  Host arithmetic only; also sizes the slot scratch.
int ridge_grid(int n_T, int n_rec, int D, int mb_log2, int num_sms, int *nblk_out)
{
    const int RS = (mb_log2 <= 1) ? 8 : 16;
    const int strips = (n_rec + kRgCols - 1) / kRgCols;
    const int nblk = (n_T + RS - 1) / RS;
    const long long U = (long long)strips * D * nblk;
    const int slots = num_sms * ((mb_log2 <= 1) ? 2 : 1);
    long long G = U / (256 / RS);
    if (G > slots) G = slots;                                          // <= 2 kRidgePlanSMs: s_slot[] in the kernel
    // a whole number of CTAs per strip when that still fills >= 95 % of the slots: the strips then advance through the
    // recoil rows in step, so that the 2 KB row segments in flight belong to few, complete 8 n_rec-byte rows of R
    // (measured on config 4, 4 / 16 points: 0.181 / 0.186 ms with 288 CTAs, 0.187 / 0.197 ms with 296)
    const long long n_tiles = (long long)strips * D;
    if (G == slots && n_tiles <= slots && (slots / n_tiles) * n_tiles * 20 >= (long long)slots * 19) G = (slots / n_tiles) * n_tiles;
    if (G < 1) G = 1;
    if (nblk_out) *nblk_out = nblk;
    return (int)G;
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
    if (Pb > L.ridge_max_p) return cudaErrorInvalidValue;               // the slot scratch is sized by max_batch (plan())
    const int MB = (Pb + 7) / 8;                                        // tile height 8 MB: the points rounded up to 8
    const int mbl = MB <= 1 ? 0 : MB == 2 ? 1 : 2;                      // geometry class: 2 CTAs per SM x 8-row stages | 1 x 16
    RidgeArgs A;
    A.R = ctx->R; A.R_period_stride = ctx->R_period_stride; A.ldR = ctx->ldR;
    A.n_T = ctx->n_T; A.n_rec = ctx->n_rec; A.D = ctx->D;
    A.coef = coef; A.param = param; A.wts = wts;
    A.rate = rate; A.comp8 = ctx->comp8;
    A.What = ctx->What; A.N_mc = ctx->N_mc; A.bkg = ctx->bkg; A.counts = ctx->counts;
    A.sat_const = full_eq18 ? ctx->sat_const : nullptr;
    A.Pb = Pb;
    A.n_strips = L.ridge_strips;
    // the slot scratch is sized for kRidgePlanSMs (plan() runs without a device); fewer SMs only shrink the grid
    const int grid = ridge_grid(ctx->n_T, ctx->n_rec, ctx->D, mbl, ctx->num_sms < kRidgePlanSMs ? ctx->num_sms : kRidgePlanSMs, &A.nblk);
    const int RS = (mbl <= 1) ? 8 : 16;
    A.zero_ring = (ctx->ldR - (L.ridge_strips - 1) * kRgCols < kRgCols) || (ctx->n_T % RS != 0);
    A.zero = 0;
    A.slots = ctx->ridge_slots; A.strip_part = ctx->ridge_part; A.cnt = ctx->ridge_cnt;
    A.out = out; A.out_mu = out_mu;
    A.frag = ctx->ridge_frag;
    A.nblk8 = (ctx->n_T + 7) / 8 + 8;
    Kinds none;
    none.k = 0;
    for (int a = 0; a < RW_N_KINDS; ++a) none.kind[a] = -1;
    const Kinds &k = kd ? *kd : none;
    cudaError_t e;
    {
        ProfScope prof(ctx, s);
        if (MB >= 3) {                   // tile heights 24 .. 64: N' once per call
            k_ridge_frag<<<dim3((unsigned)((A.nblk8 + 7) / 8), (unsigned)ctx->D), 256, 0, s>>>(A, k, ctx->cst, MB);
            ctx->launches++;
        }
        switch (MB) {
        case 1: e = launch_ridge_t<1>(A, k, ctx->cst, grid, s); break;
        case 2: e = launch_ridge_t<2>(A, k, ctx->cst, grid, s); break;
        case 3: e = launch_ridge_t<3>(A, k, ctx->cst, grid, s); break;
        case 4: e = launch_ridge_t<4>(A, k, ctx->cst, grid, s); break;
        case 5: e = launch_ridge_t<5>(A, k, ctx->cst, grid, s); break;
        case 6: e = launch_ridge_t<6>(A, k, ctx->cst, grid, s); break;
        case 7: e = launch_ridge_t<7>(A, k, ctx->cst, grid, s); break;
        default: e = launch_ridge_t<8>(A, k, ctx->cst, grid, s); break;
        }
    }
    if (e != cudaSuccess) return e;
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
