// rw_fold_tf32.cu -- opt-in RW_FP32 variant of the batched fold (`real_t` switch of
// PAPER.md:226; BASELINE north_star: "within 1e-5 relative for any opt-in FP32 variant").
//
// The fold mu[p][k] = sum_i N'[p][i] R[i][k] (Eq. 11) on the 5th-generation tensor cores:
// tcgen05.mma.kind::tf32 with FP32 accumulators in tensor memory.  TF32 keeps 11 significand bits, so each FP64
// operand is split in two TF32 pieces x = hi + lo (both rounded to nearest) and the product is
//     a b ~ a_hi b_hi + (a_hi b_lo + a_lo b_hi)            (the dropped a_lo b_lo is 2^-22 relative)
// i.e. three MMAs per k-step.  The tensor core adds into its FP32 accumulator with truncation, whose bias grows
// with the number of additions; so the contraction is cut into chunks of 128 recoil bins, each accumulated in
// TMEM from zero, and the chunk results are added in registers with round-to-nearest FP32 adds by the epilogue
// warps (3.8e-6 worst-case truncation bias per chunk, ~1e-6 typical; measured against the FP64 oracle in
// tests/test_gpu_fp32.py).  The Poisson terms of Eq. (18) are evaluated in FP64 on the converted mu.
//
// One CTA per SM, 192 threads: warp 0 = TMA producer (one lane), warp 1 = MMA issuer (one lane) and TMEM owner,
// warps 2-5 = epilogue (thread = one point row of the 128 x 128 tile: the row sum needs no cross-thread
// reduction).  Operands are K-major with the 128-byte swizzle: N' as [points][n_T] FP32 hi/lo written by
// k_gen_A32, R as a transposed FP32 hi/lo copy [n_rec][n_T] made once at rw_create.  A 3-stage ring of
// 4 x 16 KB tiles (32 recoil bins per stage); TMEM holds two (main, correction) accumulator pairs so the MMAs of
// chunk c+1 overlap the drain of chunk c.
#include "rw_internal.h"

namespace rw {

constexpr int kF32BK = 32;                      // recoil bins per stage: one 128-byte swizzle atom of FP32
constexpr int kF32Stages = 3;
constexpr int kF32TileBytes = 128 * kF32BK * 4; // 16 KB: 128 rows x 128 bytes
constexpr int kF32StageBytes = 4 * kF32TileBytes;       // A_hi, A_lo, B_hi, B_lo
constexpr int kF32ChunkStages = 4;              // 128 recoil bins per TMEM accumulation chunk
constexpr int kF32Threads = 192;
constexpr int kF32Smem = kF32Stages * kF32StageBytes + 3 * 128 * 8 + 256 + 1024;

__device__ __forceinline__ uint32_t f32_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void f32_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void f32_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void f32_mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void f32_mbar_wait(uint32_t bar, uint32_t parity)
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
__device__ __forceinline__ void f32_tma_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
// K-major operand tile, 128-byte swizzle: rows of 128 bytes, 8-row groups 1024 bytes apart (SBO), descriptor
// version 1 (sm_100), layout type 2 = SWIZZLE_128B.  A k-step of 8 TF32 advances the start address by 32 bytes.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr)
{
    return (uint64_t)((smem_addr & 0x3ffff) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// D[tmem] (+)= A[smem] B[smem], M = N = 128, K = 8, TF32 inputs, FP32 accumulate; issued by one thread.
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                          uint32_t accumulate)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
}

// round to the nearest TF32 (10 explicit significand bits), result held in an FP32 container
__device__ __forceinline__ float to_tf32(float x)
{
    return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
}
__device__ __forceinline__ void split_tf32(double x, float &hi, float &lo)
{
    hi = to_tf32((float)x);
    lo = to_tf32((float)(x - (double)hi));
}

// ---------------------------------------------------------------------------------------------- operand prep
// R[n_T][ldR] (FP64, rec index fastest) -> Rt_hi, Rt_lo [n_rec][KP] (FP32, recoil index fastest): the K-major
// B operand.  32 x 32 transpose tiles through shared memory; run once per period at rw_create.
__global__ void __launch_bounds__(256)
k_split_R(const double *__restrict__ R, int ldR, int n_T, int n_rec, int KP, float *__restrict__ hi,
          float *__restrict__ lo)
{
    __shared__ double tile[32][33];
    const int i0 = blockIdx.x * 32, k0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8) {
        const int i = i0 + r, k = k0 + tx;
        tile[r][tx] = (i < n_T && k < n_rec) ? R[(size_t)i * ldR + k] : 0.0;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int k = k0 + r, i = i0 + tx;
        if (k < n_rec && i < KP) {
            float h, l;
            split_tf32(tile[tx][r], h, l);
            hi[(size_t)k * KP + i] = h;
            lo[(size_t)k * KP + i] = l;
        }
    }
}

// N'[p][i] = sum_b coef[p][b] W^[b][i] in FP64 (steps a1 + a2, Eq. 14 / Eq. 1), split into TF32 hi/lo rows
// [rows_pad][KP]; rows >= Pc and bins >= n_T are zero.  8 points x 256 bins per CTA, W^ staged in shared memory.
__global__ void __launch_bounds__(256)
k_gen_A32(const double *__restrict__ coef, int64_t p0, int64_t Pc, const double *__restrict__ What, int n_T,
          int KP, const double *__restrict__ rate, const uint8_t *__restrict__ comp8, float *__restrict__ hi,
          float *__restrict__ lo)
{
    __shared__ double sW[kNumTerms][256];
    __shared__ double sC[8][kCoefStride];
    __shared__ double sRate[8][RW_MAX_COMPONENTS];
    if (threadIdx.x < 8 * RW_MAX_COMPONENTS) {
        const int r = threadIdx.x / RW_MAX_COMPONENTS, cq = threadIdx.x % RW_MAX_COMPONENTS;
        const int64_t row = (int64_t)blockIdx.x * 8 + r;
        sRate[r][cq] = (comp8 && row < Pc) ? rate[(p0 + row) * RW_MAX_COMPONENTS + cq] : 1.0;
    }
    const int i0 = blockIdx.y * 256;
    const int64_t row0 = (int64_t)blockIdx.x * 8;
    for (int q = threadIdx.x; q < kNumTerms * 256; q += 256) {
        const int b = q >> 8, ii = q & 255, i = i0 + ii;
        sW[b][ii] = (i < n_T) ? What[(size_t)b * n_T + i] : 0.0;
    }
    if (threadIdx.x < 8 * kCoefStride) {
        const int r = threadIdx.x / kCoefStride, b = threadIdx.x - r * kCoefStride;
        sC[r][b] = (row0 + r < Pc) ? coef[(p0 + row0 + r) * kCoefStride + b] : 0.0;
    }
    __syncthreads();
    const int i = i0 + threadIdx.x;
    if (i >= KP) return;
    const int cq = (comp8 && i < n_T) ? comp8[i] : 0;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        double v = 0.0;
#pragma unroll
        for (int b = 0; b < kNumTerms; ++b) v = fma(sC[r][b], sW[b][threadIdx.x], v);
        v *= sRate[r][cq];                                   // rate_k of Eq. (17); 1 with a single component
        float h, l;
        split_tf32(v, h, l);
        hi[(size_t)(row0 + r) * KP + i] = h;
        lo[(size_t)(row0 + r) * KP + i] = l;
    }
}

// ---------------------------------------------------------------------------------------------- the contraction
// Raster: groups of 8 m-tiles sweep n, so a wave of 148 CTAs shares 8 N' panels and ~19 R panels in L2 (with
// m fastest over the whole grid every n-tile re-streams all of N' from HBM: 290 GB per launch at config-4 size,
// HBM-bound at 5.5 TB/s -- ncu, round 1).
__device__ __forceinline__ void f32_tile_coord(int t, int tiles_m, int tiles_n, int &tm, int &tn)
{
    constexpr int GM = 8;
    const int per_group = GM * tiles_n;
    const int g = t / per_group, rem = t - g * per_group;
    const int first_m = g * GM;
    const int gm = min(GM, tiles_m - first_m);
    tm = first_m + rem % gm;
    tn = rem / gm;
}

struct F32Work {
    int n_T, n_rec, tiles_m, tiles_n, D, d;
    int64_t Pc, part_stride;
    const double *bkg, *counts;
    double *partial, *out_mu;
};

__global__ void __launch_bounds__(kF32Threads, 1)
k_fold_tf32(const __grid_constant__ CUtensorMap mapAhi, const __grid_constant__ CUtensorMap mapAlo,
            const __grid_constant__ CUtensorMap mapBhi, const __grid_constant__ CUtensorMap mapBlo, const F32Work W)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t sbase = f32_smem_u32(smem);
    double *s_bkg = reinterpret_cast<double *>(smem + kF32Stages * kF32StageBytes);       // [128] per tile
    double *s_cnt = s_bkg + 128, *s_inv = s_cnt + 128;
    const uint32_t bars = sbase + kF32Stages * kF32StageBytes + 3 * 128 * 8;
    const uint32_t full_bar = bars, empty_bar = bars + 8 * kF32Stages;
    const uint32_t tfull_bar = empty_bar + 8 * kF32Stages, tempty_bar = tfull_bar + 16;
    uint32_t *s_tmem = reinterpret_cast<uint32_t *>(smem + kF32Stages * kF32StageBytes + 3 * 128 * 8 + 128);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kF32Stages; ++s) { f32_mbar_init(full_bar + 8 * s, 1); f32_mbar_init(empty_bar + 8 * s, 1); }
        for (int b = 0; b < 2; ++b) { f32_mbar_init(tfull_bar + 8 * b, 1); f32_mbar_init(tempty_bar + 8 * b, 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {     // TMEM: all 512 columns = 2 buffers x (main, correction) x 128 FP32 columns
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(f32_smem_u32(s_tmem)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *s_tmem;

    const int k_stages = (W.n_T + kF32BK - 1) / kF32BK;                      // stages per tile
    const int n_chunks = (k_stages + kF32ChunkStages - 1) / kF32ChunkStages; // TMEM chunks per tile
    const int total_tiles = W.tiles_m * W.tiles_n;

    if (warp == 0) {
        // ------------------------------------------------------------------ TMA producer
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
                int tm, tn;
                f32_tile_coord(t, W.tiles_m, W.tiles_n, tm, tn);
                for (int ks = 0; ks < k_stages; ++ks) {
                    f32_mbar_wait(empty_bar + 8 * stage, phase ^ 1);
                    const uint32_t fb = full_bar + 8 * stage, dst = sbase + stage * kF32StageBytes;
                    f32_mbar_expect_tx(fb, kF32StageBytes);
                    f32_tma_2d(dst, &mapAhi, ks * kF32BK, tm * 128, fb);
                    f32_tma_2d(dst + kF32TileBytes, &mapAlo, ks * kF32BK, tm * 128, fb);
                    f32_tma_2d(dst + 2 * kF32TileBytes, &mapBhi, ks * kF32BK, tn * 128, fb);
                    f32_tma_2d(dst + 3 * kF32TileBytes, &mapBlo, ks * kF32BK, tn * 128, fb);
                    if (++stage == kF32Stages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer
        if (lane == 0) {
            // instruction descriptor: D = F32 (bits 4-5 = 1), A = B = TF32 (bits 7-9, 10-12 = 2), K-major both,
            // N >> 3 at bit 17, M >> 4 at bit 24
            const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
            int stage = 0; uint32_t phase = 0;
            uint32_t cseq = 0;                                   // chunk sequence number over the CTA's tiles
            for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
                for (int c = 0; c < n_chunks; ++c, ++cseq) {
                    const uint32_t buf = cseq & 1;
                    f32_mbar_wait(tempty_bar + 8 * buf, ((cseq >> 1) & 1) ^ 1);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t d_main = tmem_base + buf * 256, d_corr = d_main + 128;
                    const int s1 = min(k_stages, (c + 1) * kF32ChunkStages);
                    for (int ks = c * kF32ChunkStages; ks < s1; ++ks) {
                        f32_mbar_wait(full_bar + 8 * stage, phase);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t st = sbase + stage * kF32StageBytes;
#pragma unroll
                        for (int k = 0; k < kF32BK / 8; ++k) {
                            const uint64_t a_hi = umma_desc_sw128(st + k * 32);
                            const uint64_t a_lo = umma_desc_sw128(st + kF32TileBytes + k * 32);
                            const uint64_t b_hi = umma_desc_sw128(st + 2 * kF32TileBytes + k * 32);
                            const uint64_t b_lo = umma_desc_sw128(st + 3 * kF32TileBytes + k * 32);
                            const uint32_t acc = (ks > c * kF32ChunkStages || k > 0) ? 1u : 0u;
                            umma_tf32(d_main, a_hi, b_hi, idesc, acc);
                            umma_tf32(d_corr, a_hi, b_lo, idesc, acc);
                            umma_tf32(d_corr, a_lo, b_hi, idesc, 1u);
                        }
                        umma_commit(empty_bar + 8 * stage);      // frees the smem slot when these MMAs have read it
                        if (++stage == kF32Stages) { stage = 0; phase ^= 1; }
                    }
                    umma_commit(tfull_bar + 8 * buf);            // chunk accumulated: epilogue may drain it
                }
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue warps 2..5
        const int q = warp & 3;                                  // TMEM lane quarter this warp may read
        const int lrow = 32 * q + lane;                          // row of the tile = TMEM lane
        const int et = threadIdx.x - 64;                         // 0..127
        uint32_t cseq = 0;
        for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
            int tm, tn;
            f32_tile_coord(t, W.tiles_m, W.tiles_n, tm, tn);
            {   // per-tile column constants; columns >= n_rec get bkg = n = 1/n = 0 (their mu is 0: term 0)
                asm volatile("bar.sync 1, 128;" ::: "memory");
                const int col = tn * 128 + et;
                const bool ok = col < W.n_rec;
                const double n = ok ? W.counts[col] : 0.0;
                s_bkg[et] = ok ? W.bkg[col] : 0.0;
                s_cnt[et] = n;
                s_inv[et] = n > 0.0 ? 1.0 / n : 0.0;
                asm volatile("bar.sync 1, 128;" ::: "memory");
            }
            float sum[128];
#pragma unroll
            for (int j = 0; j < 128; ++j) sum[j] = 0.f;
            for (int c = 0; c < n_chunks; ++c, ++cseq) {
                const uint32_t buf = cseq & 1;
                f32_mbar_wait(tfull_bar + 8 * buf, (cseq >> 1) & 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t taddr = tmem_base + buf * 256 + ((uint32_t)(32 * q) << 16);
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    uint32_t v[32];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {                // h = 0: main accumulator, 1: correction
                        tmem_ld32(taddr + 128 * h + 32 * g, v);
                        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                        for (int j = 0; j < 32; ++j)             // round-to-nearest FP32 adds outside the tensor core
                            sum[32 * g + j] += __uint_as_float(v[j]);
                    }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) f32_mbar_arrive(tempty_bar + 8 * buf);
            }
            const int64_t row = (int64_t)tm * 128 + lrow;
            double tot = 0.0;
#pragma unroll
            for (int j = 0; j < 128; j += 4) {
                const double m0 = (double)sum[j] + s_bkg[j], m1 = (double)sum[j + 1] + s_bkg[j + 1];
                const double m2 = (double)sum[j + 2] + s_bkg[j + 2], m3 = (double)sum[j + 3] + s_bkg[j + 3];
                if (W.out_mu && row < W.Pc) {
                    double *dst = W.out_mu + ((size_t)row * W.D + W.d) * W.n_rec + tn * 128 + j;
                    if (tn * 128 + j < W.n_rec) dst[0] = m0;
                    if (tn * 128 + j + 1 < W.n_rec) dst[1] = m1;
                    if (tn * 128 + j + 2 < W.n_rec) dst[2] = m2;
                    if (tn * 128 + j + 3 < W.n_rec) dst[3] = m3;
                }
                tot += poisson_sum4(m0, m1, m2, m3, s_cnt[j], s_cnt[j + 1], s_cnt[j + 2], s_cnt[j + 3],
                                    s_inv[j], s_inv[j + 1], s_inv[j + 2], s_inv[j + 3]);
            }
            if (row < W.Pc) W.partial[(size_t)tn * W.part_stride + row] = tot;
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}

// ---------------------------------------------------------------------------------------------- host side
typedef CUresult (*PFN_encodeTiled32)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                      const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                      CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                      CUtensorMapFloatOOBfill);

static int encode_kmajor_f32(rw_ctx *ctx, CUtensorMap *map, float *base, int KP, int64_t rows)
{
    static PFN_encodeTiled32 enc = nullptr;
    if (!enc) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            return fail(ctx, RW_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
        enc = reinterpret_cast<PFN_encodeTiled32>(p);
    }
    cuuint64_t dims[2] = {(cuuint64_t)KP, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)KP * sizeof(float)};
    cuuint32_t box[2] = {kF32BK, 128};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, RW_ERR_CUDA, "cuTensorMapEncodeTiled(fp32 operand) failed: %d", (int)r);
    return RW_OK;
}

// rw_create with RW_CREATE_FP32: transposed TF32 hi/lo copy of every period's R, tensor maps, kernel attribute.
int tf32_setup(rw_ctx *ctx, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    const int KP = L.KP32;
    const size_t per = (size_t)ctx->n_rec * KP;
    for (int d = 0; d < ctx->D; ++d) {
        float *hi = ctx->R32 + (size_t)(2 * d) * per, *lo = hi + per;
        dim3 grid((KP + 31) / 32, (ctx->n_rec + 31) / 32);
        k_split_R<<<grid, 256, 0, s>>>(ctx->R + (size_t)d * ctx->R_period_stride, ctx->ldR, ctx->n_T, ctx->n_rec, KP, hi, lo);
        ctx->launches++;
        int rc = encode_kmajor_f32(ctx, &ctx->tmapB32[2 * d], hi, KP, ctx->n_rec);
        if (rc == RW_OK) rc = encode_kmajor_f32(ctx, &ctx->tmapB32[2 * d + 1], lo, KP, ctx->n_rec);
        if (rc != RW_OK) return rc;
    }
    if (cudaGetLastError() != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "k_split_R launch failed");
    float *a_hi = reinterpret_cast<float *>(ctx->A_packed), *a_lo = a_hi + (size_t)L.MC * KP;
    int rc = encode_kmajor_f32(ctx, &ctx->tmapA32[0], a_hi, KP, L.MC);
    if (rc == RW_OK) rc = encode_kmajor_f32(ctx, &ctx->tmapA32[1], a_lo, KP, L.MC);
    if (rc != RW_OK) return rc;
    cudaError_t e = cudaFuncSetAttribute(k_fold_tf32, cudaFuncAttributeMaxDynamicSharedMemorySize, kF32Smem);
    if (e != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "cudaFuncSetAttribute(k_fold_tf32): %s", cudaGetErrorString(e));
    return RW_OK;
}

// Steps a1-a4 for the Pc points at coef[p0..] and period d through the TF32 x 3 contraction.
cudaError_t launch_fold_tf32(rw_ctx *ctx, int d, int64_t p0, int64_t Pc, double *out_mu, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    const int KP = L.KP32;
    float *a_hi = reinterpret_cast<float *>(ctx->A_packed), *a_lo = a_hi + (size_t)L.MC * KP;
    const int64_t rows_pad = (Pc + 127) / 128 * 128;
    dim3 ggrid((unsigned)(rows_pad / 8), (unsigned)((KP + 255) / 256));
    k_gen_A32<<<ggrid, 256, 0, s>>>(ctx->coef, p0, Pc, ctx->What + (size_t)d * kCoefStride * ctx->n_T, ctx->n_T, KP,
                                    ctx->rate, ctx->comp8, a_hi, a_lo);
    ctx->launches++;
    F32Work W;
    W.n_T = ctx->n_T; W.n_rec = ctx->n_rec; W.D = ctx->D; W.d = d;
    W.tiles_m = (int)(rows_pad / 128); W.tiles_n = L.n_tiles_n;
    W.Pc = Pc; W.part_stride = L.MC;
    W.bkg = ctx->bkg + (size_t)d * ctx->n_rec;
    W.counts = ctx->counts + (size_t)d * ctx->n_rec;
    W.partial = ctx->partial + (size_t)d * W.tiles_n * L.MC;
    W.out_mu = out_mu;
    const int total = W.tiles_m * W.tiles_n;
    const int grid = total < ctx->num_sms ? total : ctx->num_sms;
    {
        ProfScope prof(ctx, s);
        k_fold_tf32<<<grid, kF32Threads, kF32Smem, s>>>(ctx->tmapA32[0], ctx->tmapA32[1], ctx->tmapB32[2 * d],
                                                        ctx->tmapB32[2 * d + 1], W);
    }
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
