// rw_fold_gemm.cu -- steps a3 + a4 for batched points: the response fold as a dense FP64 contraction
//   mu[p][k] = sum_i N'[p][i] R[i][k] + bkg[k]      (Eq. 11 / Eq. 1)
// with the binned Poisson terms of Eq. (18) reduced in the epilogue, so mu never
// touches HBM.  This is the operation the paper names as its bottleneck.
//
// Blackwell has no FP64 path in tcgen05/TMEM; FP64 tensor work is the warp-level DMMA.8x8x4
// (mma.sync.m8n8k4.f64), measured at 37.1 TFLOP/s on B200.  Design:
//   * persistent CTAs (one per SM), (16 MB) x 128 output tiles with MB in {1,2,4,8} 8-point row blocks per
//     warp (tile heights 16/32/64/128 follow the batch size), BK = 16, TMA/mbarrier ring of 6-10 stages
//   * 8 DMMA warps (two per SM sub-partition) as 2 (points) x 4 (bins); lane 0 of warp 0 also issues the
//     TMA loads, kStages-2 stage-iterations ahead of the math
//   * an R tile arrives as ONE TMA box of 16 rows x 132 columns (1056-byte rows: long L2 requests instead of
//     128-byte swizzle atoms; the 4 extra columns make the row pitch = 32 mod 128 bytes, so the four
//     k-rows a quarter-warp reads fall in four different 32-byte bank groups); N' arrives as one 2-D box
//     of the 8x8-blocked A_packed (rw_coef.cu), whose blocks interleave k and k+4.  Every fragment load is one
//     conflict-free LDS.128 -- A gives the fragments of two k-steps, R gives two adjacent output columns.
//   * the next stage's full barrier is polled before the last DMMA block of a stage, so its latency is hidden
//   * fused epilogue: + bkg, Poisson term, sum over the thread's 4 adjacent columns, shuffle over the
//     4 lanes of a row, shared-memory sum over the 4 column warps, one partial per (row, n-tile)
//     written to partial[d][n_tile][row]; k_reduce adds tiles and periods in a fixed order.
//   * split-K for what does not fill the machine (small batches; the last partial wave of a large one):
//     a work item is (tile, k-range), the accumulators go to a per-item scratch tile, and
//     k_tile_deviance adds the k-ranges in a fixed order, then does the same + bkg / Poisson / row sum.
#include "rw_internal.h"

namespace rw {

constexpr int kBoxCols = kBN + 4;                      // columns per R box: 128 + 4 (pitch 1056 B = 32 mod 128)
constexpr int kRowBytesB = kBoxCols * 8;
constexpr int kStageBytesB = kBK * kRowBytesB;         // 16.5 KB of R per stage
constexpr int kKB = kBK / 8;                           // 8-bin groups per stage
static_assert(kBK == 16 && kBN == 128, "fragment indexing below assumes this tile");

template <int MB> struct GemmCfg {
    static constexpr int BM = 16 * MB;                              // points per tile
    static constexpr int StageBytesA = BM * kBK * 8;                // 2 KB x MB of N' per stage
    static constexpr int StageBytes = StageBytesA + kStageBytesB;
    static constexpr int Stages = (MB == 8) ? 6 : (MB == 4) ? 8 : 10;
    static constexpr int Prefetch = Stages - 2;                     // stage-iterations the TMA issue runs ahead
    static constexpr int SmemRed = 4 * BM * 8;                      // [4 column warps][BM rows]
    static constexpr int Smem = Stages * StageBytes + SmemRed + 2 * Stages * 8 + 1024;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
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
__device__ __forceinline__ uint32_t mbar_test(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

struct TileCoord { int m, n; };
__device__ __forceinline__ TileCoord tile_coord(int t, int tiles_m, int tiles_n)
{
    constexpr int GM = 8;     // m-tiles per raster group: a wave of 148 CTAs shares 8 N' and ~19 R panels in L2
    const int per_group = GM * tiles_n;
    const int g = t / per_group, rem = t - g * per_group;
    const int first_m = g * GM;
    const int gm = min(GM, tiles_m - first_m);
    TileCoord tc;
    tc.m = first_m + rem % gm;
    tc.n = rem / gm;
    return tc;
}

// One launch covers tiles [tile0, tile0 + n_tiles) of the (tiles_m x tiles_n) grid, each cut into S k-ranges of
// kps stage-iterations.  S == 1: fused Poisson epilogue.  S > 1: accumulators -> mu_tile[item][BM][128].
struct GemmWork {
    int n_T, n_rec, tiles_m, tiles_n, tile0, n_tiles, S, kps, D, d;
    int64_t Pc, part_stride;
    int zero;                 // 0, opaque to the compiler (release of a pipeline stage, tile heights 16..64)
    const double *bkg, *counts;
    double *partial, *out_mu, *mu_tile;
};

template <int MB>
__global__ void __launch_bounds__(kGemmThreads, 1)
k_fold_gemm(const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapR,
            const GemmWork W)
{
    using Cfg = GemmCfg<MB>;
    constexpr int BM = Cfg::BM, kStages = Cfg::Stages;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t sbase = smem_u32(smem);
    const uint32_t full_bar = sbase + kStages * Cfg::StageBytes + Cfg::SmemRed;
    const uint32_t empty_bar = full_bar + kStages * 8;
    double *red = reinterpret_cast<double *>(smem + kStages * Cfg::StageBytes);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full_bar + 8 * s, 1);
            mbar_init(empty_bar + 8 * s, kGemmConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int k_iters = (W.n_T + kBK - 1) / kBK;
    const int total_items = W.n_tiles * W.S;
    const int tiles_m = W.tiles_m, tiles_n = W.tiles_n, S = W.S, kps = W.kps;

    // ---------------------------------------------------------------------- TMA producer duty
    // Every warp tracks the load sequence (one load = one stage of one work item), Prefetch loads ahead of its
    // own math; load number q is issued by lane 0 of warp q % 8.  Rotating the duty keeps the eight warps'
    // work equal: with a fixed producer warp that warp is the slowest, the other seven run ahead until they
    // all wait on the load it has just issued, and the pipeline depth hides its lag instead of the latency.
    // (A dedicated producer warp would put three warps on one SM sub-partition and cap every thread at 168
    // registers; the 64x32 FP64 warp tile of MB = 8 needs ~236.)
    int p_item = blockIdx.x, p_kt = 0, p_kt1 = 0, p_stage = 0, p_seq = 0;
    uint32_t p_phase = 0;
    TileCoord p_tc = {0, 0};
    auto producer_open = [&]() {      // position the load sequence on item p_item
        if (p_item >= total_items) return;
        const int tl = p_item / S, ks = p_item - tl * S;
        p_tc = tile_coord(W.tile0 + tl, tiles_m, tiles_n);
        p_kt = ks * kps;
        p_kt1 = min(k_iters, p_kt + kps);
    };
    auto produce_step = [&]() {
        if (p_item >= total_items) return;
        if ((p_seq & (kGemmConsumerWarps - 1)) == warp && lane == 0) {
            mbar_wait(empty_bar + 8 * p_stage, p_phase ^ 1);
            const uint32_t fb = full_bar + 8 * p_stage;
            mbar_expect_tx(fb, Cfg::StageBytes);
            const uint32_t dstA = sbase + p_stage * Cfg::StageBytes;
            tma_load_2d(dstA, &tmapA, p_kt * kBK * 8, p_tc.m * (BM / 8), fb);
            tma_load_2d(dstA + Cfg::StageBytesA, &tmapR, p_tc.n * kBN, p_kt * kBK, fb);
        }
        ++p_seq;
        if (++p_stage == kStages) { p_stage = 0; p_phase ^= 1; }
        if (++p_kt == p_kt1) {
            p_item += gridDim.x;
            producer_open();
        }
    };
    producer_open();
#pragma unroll 1
    for (int q = 0; q < Cfg::Prefetch; ++q) produce_step();

    // ---------------------------------------------------------------------- DMMA consumers
    const int wm = warp >> 2, wn = warp & 3;
    const int r = lane >> 2, c = lane & 3;
    // A: block (MB wm + mb, kb) is 512 contiguous bytes, lane reads its 16 bytes
    const uint32_t a_off = (uint32_t)(wm * MB * kKB) * 512 + lane * 16;
    // R: row 8 kb + c + 4 s, columns 32 wn + 16 sj + 2 r + {0,1}
    uint32_t b_off[2];
#pragma unroll
    for (int s = 0; s < 2; ++s)
        b_off[s] = Cfg::StageBytesA + (uint32_t)(c + 4 * s) * kRowBytesB + (uint32_t)(32 * wn + 2 * r) * 8;

    int stage = 0, release = -1;   // `release`: the stage consumed in the previous iteration, not yet handed back
    uint32_t phase = 0;
    uint32_t ready = 0;      // result of the early poll of the next stage's full barrier
    for (int item = blockIdx.x; item < total_items; item += gridDim.x) {
        const int tl = item / S, ks = item - tl * S;
        const TileCoord tc = tile_coord(W.tile0 + tl, tiles_m, tiles_n);
        const int kt0 = ks * kps, kt1 = min(k_iters, kt0 + kps);
        double acc[MB][2][2][2];
#pragma unroll
        for (int mb = 0; mb < MB; ++mb)
#pragma unroll
            for (int sj = 0; sj < 2; ++sj)
#pragma unroll
                for (int nb = 0; nb < 2; ++nb) acc[mb][sj][nb][0] = acc[mb][sj][nb][1] = 0.0;

        for (int kt = kt0; kt < kt1; ++kt) {
            produce_step();
            if (!ready) mbar_wait(full_bar + 8 * stage, phase);
            const uint32_t st = sbase + stage * Cfg::StageBytes;
            uint32_t dep = 0;
#pragma unroll
            for (int kb = 0; kb < kKB; ++kb) {
                double2 a[MB], b[2][2];
#pragma unroll
                for (int mb = 0; mb < MB; ++mb)
                    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];"
                                 : "=d"(a[mb].x), "=d"(a[mb].y)
                                 : "r"(st + a_off + (uint32_t)(mb * kKB + kb) * 512));
#pragma unroll
                for (int sj = 0; sj < 2; ++sj)
#pragma unroll
                    for (int s = 0; s < 2; ++s)
                        asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];"
                                     : "=d"(b[sj][s].x), "=d"(b[sj][s].y)
                                     : "r"(st + b_off[s] + (uint32_t)sj * 128 + (uint32_t)kb * (8 * kRowBytesB)));
                if constexpr (MB < 8) {
#pragma unroll
                    for (int mb = 0; mb < MB; ++mb) dep |= (uint32_t)__double2hiint(a[mb].x);
                    dep |= (uint32_t)__double2hiint(b[0][0].x) | (uint32_t)__double2hiint(b[0][1].x) |
                           (uint32_t)__double2hiint(b[1][0].x) | (uint32_t)__double2hiint(b[1][1].x);
                }
                if (kb == kKB - 1) {
                    // poll the next stage's barrier now: the result is back by the time the last
                    // DMMA block of this stage has issued, so the wait above costs no pipe bubble
                    const int ns = (stage + 1 == kStages) ? 0 : stage + 1;
                    ready = mbar_test(full_bar + 8 * ns, (stage + 1 == kStages) ? (phase ^ 1) : phase);
                }
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int mb = 0; mb < MB; ++mb) {
                        const double av = s ? a[mb].y : a[mb].x;
#pragma unroll
                        for (int sj = 0; sj < 2; ++sj) {
                            dmma884(acc[mb][sj][0][0], acc[mb][sj][0][1], av, b[sj][s].x);
                            dmma884(acc[mb][sj][1][0], acc[mb][sj][1][1], av, b[sj][s].y);
                        }
                    }
            }
            // A stage may be handed back only when every fragment load of it has RETURNED: released right behind the
            // loop, ptxas places the arrive directly after the last LDS issue, and in k_fold_ridge the producer's refill
            // has been seen to overtake such a load (rw_fold_ridge.cu).  128-row tiles (no register to spare, deep
            // slack): one iteration late, behind the next stage's barrier wait -- every DMMA reading the stage has been
            // issued by then, and the TMA issue, Stages - 2 ahead, still finds its slot released an iteration earlier.
            // Smaller tiles (HBM-bound, every stage in flight counts): at once, the arrive's address depending on the
            // loaded registers (& 0 the compiler cannot see; lane 0's registers stand for the warp-wide LDS).
            __syncwarp();
            if constexpr (MB == 8) {
                if (lane == 0 && release >= 0) mbar_arrive(empty_bar + 8 * release);
                release = stage;
            } else {
                if (lane == 0) mbar_arrive(empty_bar + 8 * stage + (dep & (uint32_t)W.zero));
            }
            if (++stage == kStages) { stage = 0; phase ^= 1; }
        }

        const int lrow0 = wm * (8 * MB) + r;                    // row within the tile, + 8 mb
        const int lcol0 = wn * 32 + 4 * c;                      // column within the tile, + 16 sj + {0,1,2,3}
        if (S > 1) {
            // ---------------------------------------------------------------- split-K: park the accumulators
            double *dst = W.mu_tile + (size_t)item * (BM * kBN);
#pragma unroll
            for (int mb = 0; mb < MB; ++mb)
#pragma unroll
                for (int sj = 0; sj < 2; ++sj) {
                    double2 *q = reinterpret_cast<double2 *>(dst + (size_t)(lrow0 + 8 * mb) * kBN + lcol0 + 16 * sj);
                    q[0] = make_double2(acc[mb][sj][0][0], acc[mb][sj][1][0]);
                    q[1] = make_double2(acc[mb][sj][0][1], acc[mb][sj][1][1]);
                }
            continue;
        }
        // ------------------------------------------------------------------ fused epilogue
        const int row0 = tc.m * BM + lrow0;
        const int col0 = tc.n * kBN + lcol0;
        // columns >= n_rec: R is zero-filled there (TMA), so with bkg = n = 1/n = 0 their term is exactly 0
        double bk[2][4], cn[2][4], ci[2][4];
#pragma unroll
        for (int sj = 0; sj < 2; ++sj)
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int col = col0 + 16 * sj + q;
                const bool ok = col < W.n_rec;
                bk[sj][q] = ok ? __ldg(W.bkg + col) : 0.0;
                cn[sj][q] = ok ? __ldg(W.counts + col) : 0.0;
                ci[sj][q] = cn[sj][q] > 0.0 ? 1.0 / cn[sj][q] : 0.0;
            }
        if (W.out_mu) {
#pragma unroll
            for (int mb = 0; mb < MB; ++mb) {
                const int64_t row = row0 + 8 * mb;
#pragma unroll
                for (int sj = 0; sj < 2; ++sj)
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int col = col0 + 16 * sj + q;
                        if (row < W.Pc && col < W.n_rec)
                            W.out_mu[((size_t)row * W.D + W.d) * W.n_rec + col] = acc[mb][sj][q & 1][q >> 1] + bk[sj][q];
                    }
            }
        }
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) {
            double sum = 0.0;
#pragma unroll
            for (int sj = 0; sj < 2; ++sj)      // column q = 2 e + nb of the group holds acc[mb][sj][nb][e]
                sum += poisson_sum4(acc[mb][sj][0][0] + bk[sj][0], acc[mb][sj][1][0] + bk[sj][1],
                                    acc[mb][sj][0][1] + bk[sj][2], acc[mb][sj][1][1] + bk[sj][3],
                                    cn[sj][0], cn[sj][1], cn[sj][2], cn[sj][3],
                                    ci[sj][0], ci[sj][1], ci[sj][2], ci[sj][3]);
            sum += __shfl_xor_sync(0xffffffffu, sum, 1);
            sum += __shfl_xor_sync(0xffffffffu, sum, 2);
            if (c == 0) red[wn * BM + lrow0 + 8 * mb] = sum;
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (threadIdx.x < BM) {
            const int64_t row = (int64_t)tc.m * BM + threadIdx.x;
            const double v = (red[threadIdx.x] + red[BM + threadIdx.x]) +
                             (red[2 * BM + threadIdx.x] + red[3 * BM + threadIdx.x]);
            if (row < W.Pc) W.partial[(size_t)tc.n * W.part_stride + row] = v;
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
    }
}

// Split-K finish: mu = sum over the S k-ranges (fixed order) + bkg, Poisson term, row sum over the tile's 128
// columns -> partial[n_tile][row], exactly the slot the fused epilogue fills.  One CTA per tile, one warp per row.
__global__ void __launch_bounds__(256)
k_tile_deviance(const double *__restrict__ mu_tile, int BM, int S, int tile0, int tiles_m, int tiles_n,
                int n_rec, int64_t Pc, const double *__restrict__ bkg, const double *__restrict__ counts,
                double *__restrict__ partial, int64_t part_stride, double *__restrict__ out_mu, int D, int d)
{
    const TileCoord tc = tile_coord(tile0 + blockIdx.x, tiles_m, tiles_n);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int col = tc.n * kBN + 4 * lane;
    double bk[4], cn[4], ci[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const bool ok = col + q < n_rec;
        bk[q] = ok ? bkg[col + q] : 0.0;
        cn[q] = ok ? counts[col + q] : 0.0;
        ci[q] = cn[q] > 0.0 ? 1.0 / cn[q] : 0.0;
    }
    const double *base = mu_tile + (size_t)blockIdx.x * S * (BM * kBN);
    for (int lr = warp; lr < BM; lr += 8) {
        const int64_t row = (int64_t)tc.m * BM + lr;
        double m[4] = {0.0, 0.0, 0.0, 0.0};
        for (int s = 0; s < S; ++s) {
            const double2 *q = reinterpret_cast<const double2 *>(base + ((size_t)s * BM + lr) * kBN + 4 * lane);
            const double2 u = q[0], v = q[1];
            m[0] += u.x; m[1] += u.y; m[2] += v.x; m[3] += v.y;
        }
        if (out_mu && row < Pc) {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (col + q < n_rec) out_mu[((size_t)row * D + d) * n_rec + col + q] = m[q] + bk[q];
        }
        // columns >= n_rec hold 0 + 0 with n = 0: term 0
        double sum = poisson_sum4(m[0] + bk[0], m[1] + bk[1], m[2] + bk[2], m[3] + bk[3], cn[0], cn[1], cn[2], cn[3],
                                  ci[0], ci[1], ci[2], ci[3]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0 && row < Pc) partial[(size_t)tc.n * part_stride + row] = sum;
    }
}

// ------------------------------------------------------------------------------------ host side
typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                    CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                    CUtensorMapFloatOOBfill);

static PFN_encodeTiled get_encode()
{
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<PFN_encodeTiled>(p);
    }
    return fn;
}

int make_tensor_maps(rw_ctx *ctx)
{
    PFN_encodeTiled enc = get_encode();
    if (!enc) return fail(ctx, RW_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    const Layout &L = ctx->lay;
    for (int v = 0; v < 4; ++v) {            // one map of N' per tile height 16 << v (the box is part of the map)
        cuuint64_t dims[2] = {(cuuint64_t)L.KPAD * 8, (cuuint64_t)(L.MC / 8)};
        cuuint64_t strides[1] = {(cuuint64_t)L.A_pitch * sizeof(double)};
        cuuint32_t box[2] = {kBK * 8, (cuuint32_t)(2 << v)};
        cuuint32_t estr[2] = {1, 1};
        CUresult r = enc(&ctx->tmapA[v], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, ctx->A_packed, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(ctx, RW_ERR_CUDA, "cuTensorMapEncodeTiled(A) failed: %d", (int)r);
    }
    for (int d = 0; d < ctx->D; ++d) {
        cuuint64_t dims[2] = {(cuuint64_t)ctx->n_rec, (cuuint64_t)ctx->n_T};
        cuuint64_t strides[1] = {(cuuint64_t)ctx->ldR * sizeof(double)};
        cuuint32_t box[2] = {kBoxCols, kBK};
        cuuint32_t estr[2] = {1, 1};
        void *base = const_cast<double *>(ctx->R + (size_t)d * ctx->R_period_stride);
        CUresult r = enc(&ctx->tmapR[d], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, base, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(ctx, RW_ERR_CUDA, "cuTensorMapEncodeTiled(R[%d]) failed: %d", d, (int)r);
    }
    cudaError_t e = cudaFuncSetAttribute(k_fold_gemm<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmCfg<1>::Smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fold_gemm<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmCfg<2>::Smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fold_gemm<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmCfg<4>::Smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fold_gemm<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmCfg<8>::Smem);
    if (e != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
    return RW_OK;
}

template <int MB>
static void launch_gemm_t(rw_ctx *ctx, int d, const GemmWork &W, int grid, cudaStream_t s)
{
    ProfScope prof(ctx, s);
    k_fold_gemm<MB><<<grid, kGemmThreads, GemmCfg<MB>::Smem, s>>>(ctx->tmapA[MB == 1 ? 0 : MB == 2 ? 1 : MB == 4 ? 2 : 3],
                                                                  ctx->tmapR[d], W);
    ctx->launches++;
}

static void launch_gemm_any(rw_ctx *ctx, int MB, int d, const GemmWork &W, cudaStream_t s)
{
    const int items = W.n_tiles * W.S;
    const int grid = items < ctx->num_sms ? items : ctx->num_sms;
    switch (MB) {
    case 1: launch_gemm_t<1>(ctx, d, W, grid, s); break;
    case 2: launch_gemm_t<2>(ctx, d, W, grid, s); break;
    case 4: launch_gemm_t<4>(ctx, d, W, grid, s); break;
    default: launch_gemm_t<8>(ctx, d, W, grid, s); break;
    }
}

// Tile height for a chunk of Pc points: the smallest of 16/32/64/128 that holds it, 128 beyond.
int gemm_rows_per_warp_block(int64_t Pc) { return Pc <= 16 ? 1 : Pc <= 32 ? 2 : Pc <= 64 ? 4 : 8; }

// Split factor for `tail` tiles that do not fill the machine: the smallest S <= s_max whose S*tail work items
// use >= 90 % of the SM slots of the waves they occupy, else the best one.
int gemm_tail_split(int tail, int num_sms, int k_iters, int max_items)
{
    int s_max = k_iters / 8;
    if (s_max > 16) s_max = 16;
    if (s_max > max_items / tail) s_max = max_items / tail;
    if (s_max < 1) s_max = 1;
    int best = 1;
    double best_eff = 0.0;
    for (int S = 1; S <= s_max; ++S) {
        const int kps = (k_iters + S - 1) / S;
        if ((S - 1) * kps >= k_iters) continue;                       // an empty k-range
        const int items = tail * S;
        const double eff = (double)items / ((double)((items + num_sms - 1) / num_sms) * num_sms);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = S; }
        if (eff >= 0.9) break;
    }
    return best;
}

cudaError_t launch_fold_gemm(rw_ctx *ctx, int d, int64_t Pc, double *out_mu, int64_t /*mu_p0*/, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    const int MB = gemm_rows_per_warp_block(Pc);
    const int BM = 16 * MB;
    GemmWork W;
    W.n_T = ctx->n_T; W.n_rec = ctx->n_rec; W.D = ctx->D; W.d = d;
    W.tiles_m = (int)((Pc + BM - 1) / BM);
    W.tiles_n = L.n_tiles_n;
    W.zero = 0;
    W.Pc = Pc; W.part_stride = L.MC;
    W.bkg = ctx->bkg + (size_t)d * ctx->n_rec;
    W.counts = ctx->counts + (size_t)d * ctx->n_rec;
    W.partial = ctx->partial + (size_t)d * W.tiles_n * L.MC;
    W.out_mu = out_mu;
    W.mu_tile = ctx->mu_tile;
    const int k_iters = (ctx->n_T + kBK - 1) / kBK;
    const int total = W.tiles_m * W.tiles_n;
    int full = total / ctx->num_sms * ctx->num_sms;
    int tail = total - full;
    int S = tail ? gemm_tail_split(tail, ctx->num_sms, k_iters, L.mu_tile_items) : 1;
    if (S == 1) { full = total; tail = 0; }
    if (full) {
        W.tile0 = 0; W.n_tiles = full; W.S = 1; W.kps = k_iters;
        launch_gemm_any(ctx, MB, d, W, s);
    }
    if (tail) {
        W.tile0 = full; W.n_tiles = tail; W.S = S; W.kps = (k_iters + S - 1) / S;
        launch_gemm_any(ctx, MB, d, W, s);
        k_tile_deviance<<<tail, 256, 0, s>>>(ctx->mu_tile, BM, S, full, W.tiles_m, W.tiles_n, ctx->n_rec, Pc, W.bkg,
                                             W.counts, W.partial, W.part_stride, out_mu, ctx->D, d);
        ctx->launches++;
    }
    return cudaGetLastError();
}

}  // namespace rw
