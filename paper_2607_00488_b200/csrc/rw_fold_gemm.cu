// rw_fold_gemm.cu -- steps a3 + a4 for large batches: the response fold as a dense FP64 contraction
//   mu[p][k] = sum_i N'[p][i] R[i][k] + bkg[k]      (Eq. 11 / Eq. 1)
// with the binned Poisson terms of Eq. (18) reduced in the epilogue, so mu never
// touches HBM.  This is the operation the paper names as its bottleneck.
//
// Blackwell has no FP64 path in tcgen05/TMEM; FP64 tensor work is the warp-level DMMA.8x8x4
// (mma.sync.m8n8k4.f64), measured at 37.1 TFLOP/s on B200.  Design:
//   * persistent CTAs (one per SM), 128x128 output tile, BK = 16, 6-stage TMA/mbarrier pipeline
//   * 8 DMMA warps (two per SM sub-partition), 64x32 warp tiles; lane 0 of warp 0 also issues the
//     TMA loads, kStages-2 stage-iterations ahead of the math
//   * R tiles arrive by TMA as eight 16-column sub-tiles with the 128-byte swizzle; N' arrives as
//     one 2-D box of the 8x8-blocked A_packed (rw_coef.cu).  The contraction index inside every
//     group of 8 recoil bins is visited in the order {0,2,4,6},{1,3,5,7}: with that permutation
//     (legal because it is applied to both operands) every fragment load is one conflict-free
//     LDS.128 -- A gives the fragments of two k-steps, R gives two adjacent output columns.
//   * epilogue: + bkg, Poisson term, sum over the thread's 4 adjacent columns, shuffle over the
//     4 lanes of a row, shared-memory sum over the 4 column warps, one partial per (row, n-tile)
//     written to partial[d][n_tile][row]; k_reduce adds tiles and periods in a fixed order.
#include "rw_internal.h"

namespace rw {

constexpr int kStageBytesA = kBM * kBK * 8;            // 16 KB
constexpr int kStageBytesB = kBK * kBN * 8;            // 16 KB
constexpr int kStageBytes = kStageBytesA + kStageBytesB;
constexpr int kSubTileBytes = kBK * 128;               // one 16-column swizzled sub-tile
constexpr int kSmemRed = 4 * kBM * 8;                  // [4 column warps][128 rows]
constexpr int kSmemBars = 2 * kStages * 8;
constexpr int kGemmSmem = kStages * kStageBytes + kSmemRed + kSmemBars + 1024;
constexpr int kPrefetch = (kStages > 3) ? kStages - 2 : kStages - 1;                 // stage-iterations the TMA issue runs ahead
static_assert((kBK == 16 || kBK == 32) && kBM == 128 && kBN == 128, "fragment indexing below assumes this tile");
constexpr int kKB = kBK / 8;                           // 8-bin groups per stage

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

#ifdef RW_GEMM_STATS
__device__ unsigned long long g_gemm_stats[148 * 8];
__device__ __forceinline__ long long clk() { long long t; asm volatile("mov.u64 %0, %%clock64;" : "=l"(t)); return t; }
#endif

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

__global__ void __launch_bounds__(kGemmThreads, 1)
k_fold_gemm(const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapR,
            int n_T, int n_rec, int64_t Pc, int tiles_m, int tiles_n,
            const double *__restrict__ bkg, const double *__restrict__ counts,
            double *__restrict__ partial /*[tiles_n][part_stride]*/, int64_t part_stride,
            double *__restrict__ out_mu /*NULL or rows of this chunk, [.][D][n_rec]*/, int D, int d)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t sbase = smem_u32(smem);
    const uint32_t full_bar = sbase + kStages * kStageBytes + kSmemRed;
    const uint32_t empty_bar = full_bar + kStages * 8;
    double *red = reinterpret_cast<double *>(smem + kStages * kStageBytes);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full_bar + 8 * s, 1);
            mbar_init(empty_bar + 8 * s, kGemmConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int k_iters = (n_T + kBK - 1) / kBK;
    const int total_tiles = tiles_m * tiles_n;

    // ---------------------------------------------------------------------- TMA producer duty
    // Lane 0 of warp 0 runs kPrefetch stage-iterations ahead of the consumers.  (A dedicated
    // producer warp would put three warps on one SM sub-partition and cap every thread at 168
    // registers; the 64x32 FP64 warp tile needs ~230.)
    const bool is_producer = threadIdx.x == 0;
    int p_t = blockIdx.x, p_kt = 0, p_stage = 0;
    uint32_t p_phase = 0;
    TileCoord p_tc = tile_coord(p_t < total_tiles ? p_t : 0, tiles_m, tiles_n);
    auto produce_one = [&]() {
        if (p_t >= total_tiles) return;
        mbar_wait(empty_bar + 8 * p_stage, p_phase ^ 1);
        const uint32_t fb = full_bar + 8 * p_stage;
        mbar_expect_tx(fb, kStageBytes);
        const uint32_t dstA = sbase + p_stage * kStageBytes;
        tma_load_2d(dstA, &tmapA, p_kt * kBK * 8, p_tc.m * (kBM / 8), fb);
        const uint32_t dstB = dstA + kStageBytesA;
#pragma unroll
        for (int j = 0; j < kBN / 16; ++j)
            tma_load_2d(dstB + j * kSubTileBytes, &tmapR, p_tc.n * kBN + 16 * j, p_kt * kBK, fb);
        if (++p_stage == kStages) { p_stage = 0; p_phase ^= 1; }
        if (++p_kt == k_iters) {
            p_kt = 0;
            p_t += gridDim.x;
            if (p_t < total_tiles) p_tc = tile_coord(p_t, tiles_m, tiles_n);
        }
    };
    if (is_producer) {
#pragma unroll 1
        for (int q = 0; q < kPrefetch; ++q) produce_one();
    }

    // ---------------------------------------------------------------------- DMMA consumers
    const int wm = warp >> 2, wn = warp & 3;
    const int r = lane >> 2, c = lane & 3;
    // A: block (8 wm + mb, kb) is 512 contiguous bytes, lane reads its 16 bytes
    const uint32_t a_off = (uint32_t)(wm * 8 * kKB) * 512 + lane * 16;
    // R: sub-tile (2 wn + sj), row 8 kb + 2c + s, 16-byte chunk (r ^ (2c + s))
    uint32_t b_off[2];
#pragma unroll
    for (int s = 0; s < 2; ++s)
        b_off[s] = kStageBytesA + (uint32_t)(2 * wn) * kSubTileBytes + (uint32_t)(2 * c + s) * 128 +
                   (uint32_t)((r ^ (2 * c + s)) * 16);

    int stage = 0;
    uint32_t phase = 0;
    uint32_t ready = 0;      // result of the early poll of the next stage's full barrier
    for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
        const TileCoord tc = tile_coord(t, tiles_m, tiles_n);
        double acc[8][2][2][2];
#pragma unroll
        for (int mb = 0; mb < 8; ++mb)
#pragma unroll
            for (int sj = 0; sj < 2; ++sj)
#pragma unroll
                for (int nb = 0; nb < 2; ++nb) acc[mb][sj][nb][0] = acc[mb][sj][nb][1] = 0.0;

        for (int kt = 0; kt < k_iters; ++kt) {
            if (is_producer) produce_one();
#ifdef RW_GEMM_STATS
            {
                long long t0 = clk();
                mbar_wait(full_bar + 8 * stage, phase);
                long long dt = clk() - t0;
                if (threadIdx.x == 32 && blockIdx.x < 148) {
                    unsigned long long *st = g_gemm_stats + blockIdx.x * 8;
                    st[0] += dt; st[1] += 1;
                    if (dt > 500) st[2] += 1;
                    if (dt > 4000) st[3] += 1;
                    if ((unsigned long long)dt > st[4]) st[4] = dt;
                    if (kt < 4) st[5] += dt;
                }
            }
#else
            if (!ready) mbar_wait(full_bar + 8 * stage, phase);
#endif
            const uint32_t st = sbase + stage * kStageBytes;
#pragma unroll
            for (int kb = 0; kb < kKB; ++kb) {
                double2 a[8], b[2][2];
#pragma unroll
                for (int mb = 0; mb < 8; ++mb)
                    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];"
                                 : "=d"(a[mb].x), "=d"(a[mb].y)
                                 : "r"(st + a_off + (uint32_t)(mb * kKB + kb) * 512));
#pragma unroll
                for (int sj = 0; sj < 2; ++sj)
#pragma unroll
                    for (int s = 0; s < 2; ++s)
                        asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];"
                                     : "=d"(b[sj][s].x), "=d"(b[sj][s].y)
                                     : "r"(st + b_off[s] + (uint32_t)sj * kSubTileBytes + (uint32_t)kb * 1024));
                if (kb == kKB - 1) {
                    // poll the next stage's barrier now: the result is back by the time the last
                    // 64 DMMAs of this stage have issued, so the wait below costs no pipe bubble
                    const int ns = (stage + 1 == kStages) ? 0 : stage + 1;
                    ready = mbar_test(full_bar + 8 * ns, (stage + 1 == kStages) ? (phase ^ 1) : phase);
                }
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int mb = 0; mb < 8; ++mb) {
                        const double av = s ? a[mb].y : a[mb].x;
#pragma unroll
                        for (int sj = 0; sj < 2; ++sj) {
                            dmma884(acc[mb][sj][0][0], acc[mb][sj][0][1], av, b[sj][s].x);
                            dmma884(acc[mb][sj][1][0], acc[mb][sj][1][1], av, b[sj][s].y);
                        }
                    }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar + 8 * stage);
            if (++stage == kStages) { stage = 0; phase ^= 1; }
        }

        // ------------------------------------------------------------------ fused epilogue
        const int row0 = tc.m * kBM + wm * 64 + r;              // + 8 mb
        const int col0 = tc.n * kBN + wn * 32 + 4 * c;          // + 16 sj + {0,1,2,3}
        double bk[2][4], cn[2][4];
#pragma unroll
        for (int sj = 0; sj < 2; ++sj)
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int col = col0 + 16 * sj + q;
                const bool ok = col < n_rec;
                bk[sj][q] = ok ? __ldg(bkg + col) : 0.0;
                cn[sj][q] = ok ? __ldg(counts + col) : 0.0;
            }
#pragma unroll
        for (int mb = 0; mb < 8; ++mb) {
            double sum = 0.0;
#pragma unroll
            for (int sj = 0; sj < 2; ++sj)
#pragma unroll
                for (int e = 0; e < 2; ++e)
#pragma unroll
                    for (int nb = 0; nb < 2; ++nb) {
                        const int q = 2 * e + nb;
                        const double mu = acc[mb][sj][nb][e] + bk[sj][q];
                        const int col = col0 + 16 * sj + q;
                        if (col < n_rec) {
                            sum += poisson_term(mu, cn[sj][q]);
                            if (out_mu) {
                                const int64_t row = row0 + 8 * mb;
                                if (row < Pc) out_mu[((size_t)row * D + d) * n_rec + col] = mu;
                            }
                        }
                    }
            sum += __shfl_xor_sync(0xffffffffu, sum, 1);
            sum += __shfl_xor_sync(0xffffffffu, sum, 2);
            if (c == 0) red[wn * kBM + wm * 64 + 8 * mb + r] = sum;
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (threadIdx.x < kBM) {
            const int64_t row = (int64_t)tc.m * kBM + threadIdx.x;
            const double v = (red[threadIdx.x] + red[kBM + threadIdx.x]) +
                             (red[2 * kBM + threadIdx.x] + red[3 * kBM + threadIdx.x]);
            if (row < Pc) partial[(size_t)tc.n * part_stride + row] = v;
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
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

#ifdef RW_GEMM_STATS
extern "C" int rw_debug_gemm_stats(unsigned long long *host_out, int reset)
{
    cudaDeviceSynchronize();
    if (host_out) cudaMemcpyFromSymbol(host_out, g_gemm_stats, sizeof(unsigned long long) * 148 * 8);
    if (reset) { static unsigned long long z[148 * 8]; cudaMemcpyToSymbol(g_gemm_stats, z, sizeof(z)); }
    return 0;
}
#endif

int make_tensor_maps(rw_ctx *ctx)
{
    PFN_encodeTiled enc = get_encode();
    if (!enc) return fail(ctx, RW_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    const Layout &L = ctx->lay;
    {
        cuuint64_t dims[2] = {(cuuint64_t)L.KPAD * 8, (cuuint64_t)(L.MC / 8)};
        cuuint64_t strides[1] = {(cuuint64_t)L.A_pitch * sizeof(double)};
        cuuint32_t box[2] = {kBK * 8, kBM / 8};
        cuuint32_t estr[2] = {1, 1};
        CUresult r = enc(&ctx->tmapA, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, ctx->A_packed, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(ctx, RW_ERR_CUDA, "cuTensorMapEncodeTiled(A) failed: %d", (int)r);
    }
    for (int d = 0; d < ctx->D; ++d) {
        cuuint64_t dims[2] = {(cuuint64_t)ctx->n_rec, (cuuint64_t)ctx->n_T};
        cuuint64_t strides[1] = {(cuuint64_t)ctx->ldR * sizeof(double)};
        cuuint32_t box[2] = {16, kBK};
        cuuint32_t estr[2] = {1, 1};
        void *base = const_cast<double *>(ctx->R + (size_t)d * ctx->R_period_stride);
        CUresult r = enc(&ctx->tmapR[d], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, base, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(ctx, RW_ERR_CUDA, "cuTensorMapEncodeTiled(R[%d]) failed: %d", d, (int)r);
    }
    cudaError_t e = cudaFuncSetAttribute(k_fold_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem);
    if (e != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
    return RW_OK;
}

cudaError_t launch_fold_gemm(rw_ctx *ctx, int d, int64_t Pc, double *out_mu, int64_t /*mu_p0*/, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    const int tiles_m = (int)((Pc + kBM - 1) / kBM);
    const int tiles_n = L.n_tiles_n;
    const int total = tiles_m * tiles_n;
    const int grid = total < ctx->num_sms ? total : ctx->num_sms;
    double *part = ctx->partial + (size_t)d * tiles_n * L.MC;
    ProfScope prof(ctx, s);
    k_fold_gemm<<<grid, kGemmThreads, kGemmSmem, s>>>(
        ctx->tmapA, ctx->tmapR[d], ctx->n_T, ctx->n_rec, Pc, tiles_m, tiles_n,
        ctx->bkg + (size_t)d * ctx->n_rec, ctx->counts + (size_t)d * ctx->n_rec, part, L.MC, out_mu, ctx->D, d);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
