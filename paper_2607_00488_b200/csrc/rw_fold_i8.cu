// rw_fold_i8.cu -- opt-in RW_SLICED variant of the batched fold ("FP64-by-slicing
// (Ozaki-style) on low-precision tensor cores as a way past the native FP64 peak while holding 1e-12").
//
// The fold mu[p][k] = sum_i N'[p][i] R[i][k] (Eq. 11) has only non-negative terms.  Each row of N'
// and each column of R is written in fixed point relative to its own power-of-two scale and cut into NS base-256
// digits ("slices"; NS = 8 for n_T <= 2048, else 7),
//     N'[p][i] = 2^(e_p - 7) sum_s a_s[p][i] 2^(-8 s),      R[i][k] = 2^(f_k - 7) sum_t b_t[i][k] 2^(-8 t),
// with BALANCED digits: a_0 in [0, 129] (unsigned; one spare bit keeps the carry), a_s in [-128, 127] for s > 0.
// The contraction becomes NS (NS + 1) / 2 INT8 tensor-core products with EXACT int32 accumulation (tcgen05.mma
// kind::i8, accumulators in TMEM; |digit product| <= 129 x 128, NS pairs per accumulator:
// 7 x 16512 x 18560 bins < 2^31 and 8 x 16512 x 8192 < 2^31; contractions longer than 16384 bins are accumulated in
// segments, drained and summed in FP64 by the epilogue):
//     mu[p][k] - bkg[k] = 2^(e_p + f_k - 14) sum_{d=0..NS-1} 2^(-8d) sum_{s+t=d} sum_i a_s[p][i] b_t[i][k].
// Balanced digits are what lets 8-bit slices through at n_T = 16384 (unsigned ones would need 7-bit slices, i.e.
// 8 slices and 36 products for the same 55 bits that 7 slices and 28 products give here).
// Before slicing, recoil bin i is rescaled by an exact power of two on both sides, N'[p][i] / 2^tau_i and
// R[i][k] 2^tau_i with 2^tau_i ~ N_mc[i]: the rows of N' then have the dynamic range of the WEIGHTS (Eq. 14) instead
// of that of the MC spectrum times the weights, which is what the fixed-point error is relative to.
// Pairs with s + t >= NS are below 2^-(8 NS - 1) of (row max x column max x N_T) and are dropped; the fixed-point
// values are rounded to nearest at 2^-(8 NS - 1) of the row / column maximum.  There is no rounding anywhere
// else, so the error is a bound in terms of the scales, not of the individual mu: for responses whose columns
// spread over many recoil bins (all BASELINE configurations) it is < 1e-13 of mu; see DESIGN.md section 3.3.
//
// CERTIFICATE.  With A_i = N'[p][i] 2^-tau_i < 2^e_p, B_i = R[i][k] 2^tau_i < 2^f_k, K'_k the number of recoil bins
// whose fixed-point R entry is non-zero and S_k = sum_i B_i 2^-f_k (<= K'_k):
//   rounding of A:  sum_i |A_i - A~_i| B_i   <= 2^(e_p - 8 NS) 2^f_k S_k          (half an ulp of 2^(e_p - 8 NS + 1) each)
//   rounding of B:  sum_i A~_i |B_i - B~_i|  <= 2^(f_k - 8 NS) 2^e_p K'_k + 2^e_p L_k,   L_k = the sum of the entries
//                   0 < B_i < 2^(f_k - 8 NS) that round to zero: they are not among the K'_k, and each loses all of
//                   A~_i B_i (a floor below the resolution over thousands of live bins, next to a few large entries
//                   that meet N' = 0, is otherwise certified while the column's whole signal is gone)
//   dropped pairs s + t >= NS (|digits| <= 129, 128; both digits are lower ones):
//                   K'_k 2^(e_p + f_k - 14) 16512 sum_{d >= NS} (2 NS - 1 - d) 2^(-8 d)  <=  1.01 NS K'_k 2^(e_p + f_k - 8 NS)
// so |mu~ - mu| <= 2^e_p g_k with the per-column constant g_k = 2^(f_k - 8 NS) (S_k + (1 + 1.01 NS) K'_k) + L_k, computed once
// at rw_create (k_col_bound); the fast mode adds the diagonals 4 .. NS - 1 it leaves out: 5.07 K'_k 2^(e_p + f_k - 32).
// The epilogue turns it into the certified relative error max_k delta / (mu~ - delta) (+ 2e-15 for its own FP64
// rounding) of every point, which rw_eval_certified returns and RW_SLICED_STRICT acts on (rw_api.cu).
//
// One CTA per SM, 320 threads (TMA warp, MMA warp, 8 epilogue warps), tile 128 points x 128 bins, 32 recoil bins per
// k-block.  The slices are stored in global memory already in the tensor core's canonical K-major no-swizzle layout
// (8 x 16-byte core matrices), all slices of a (tile, k-block) contiguous: a stage is plain bulk copies into a 64 KB
// slot.  One 128-column TMEM accumulator per diagonal s + t, four at a time (two passes, see k_fold_i8); the
// epilogue combines them in FP64 (Horner) and evaluates the Poisson terms of Eq. (18).
#include <limits.h>

#include "rw_internal.h"

namespace rw {

constexpr int kI8BM = 128, kI8BN = 128, kI8BK = 32;
constexpr int kI8SliceBytesA = kI8BM * kI8BK;                   // 4 KB
constexpr int kI8SliceBytesB = kI8BN * kI8BK;                   // 4 KB
constexpr int kI8Threads = 320;                                 // TMA warp, MMA warp, 8 epilogue warps
#ifndef RW_I8_STAGES
#define RW_I8_STAGES 3              // measured: 2 slots cost 0.7 %, a 4th does not fit
#endif
constexpr int kI8SlotBytes = 65536, kI8Stages = RW_I8_STAGES;   // a slot: N' slices in its first half, R slices in its second
constexpr int kI8Smem = kI8Stages * kI8SlotBytes + 5 * kI8BN * 8 + 256 + 1024;
constexpr int kI8SegKT = 512;       // k-blocks (16384 bins) accumulated in int32 before the epilogue drains TMEM:
                                    // 7 pairs x 129 x 128 x 16384 bins < 2^31; longer contractions go in segments
constexpr int kI8BadRow = INT_MAX;                              // exponent marker: the row holds a non-finite / negative value

// ---------------------------------------------------------------------------------------------- slicing
// Fixed point: q = round(x 2^(8 ns - 1 - e)) for 0 <= x < 2^e, so q <= 2^(8 ns - 1); scale2 = 2^(8 ns - 1 - e).
// Adding 0x80 to every digit below the top one and reading bytes gives the balanced digits: byte ^ 0x80 is the
// two's-complement int8 of (digit - 128 + carry handling done by the addition); the top byte (<= 129) stays unsigned.
__device__ __forceinline__ unsigned long long i8_fixed(double x, double scale2, int ns)
{
    const unsigned long long bias = 0x0080808080808080ull >> (8 * (8 - ns));
    return __double2ull_rn(x * scale2) + bias;
}
__device__ __forceinline__ uint32_t i8_digit(unsigned long long qb, int s, int ns)    // slice s (0 = top) as a byte
{
    const uint32_t u = (uint32_t)(qb >> (8 * (ns - 1 - s))) & 0xffu;
    return s == 0 ? u : (u ^ 0x80u);
}
__device__ __forceinline__ int i8_exponent(double vmax)          // smallest e with vmax < 2^e (0 for vmax == 0)
{
    if (!(vmax > 0.0)) return 0;
    int e;
    frexp(vmax, &e);                                             // vmax = m 2^e, m in [0.5, 1)
    return e;
}

// N'[p][i] = rate * sum_b coef[p][b] W^[b][i] (steps a1 + a2) for 16 points x all recoil bins per CTA, W^ staged
// 512 bins at a time.  PASS 0: row maximum -> exponent e_p.  PASS 1: slices, written 16 bytes at a time into
//   As[m-tile][k-block][slice][16-byte chunk c][row group g][row r8][16]     (canonical K-major core matrices)
// shared-memory column swizzle: a thread reads 16 consecutive bins (lane stride 128 bytes = one bank for the whole
// warp); XOR-ing the low 4 index bits with the 16-bin group number spreads 16 lanes over 16 banks
__device__ __forceinline__ int i8_sw(int ii) { return ii ^ ((ii >> 4) & 15); }

// SRC 1 (rw_eval_weights, rw_eval_pee): N'[p][i] = w[p][i] N_mc[i] from caller-visible weights instead (`What` is
// N_mc[n_T] of the period then, `coef` the weights of the chunk's first point).
constexpr int i8_slice_smem(int src)   // k_slice_A: two staging buffers + coefficient / rate rows
{
    return 2 * ((src == 0 ? kNumTerms : 1) * 512 * 8 + 1024) + 16 * (kCoefStride + RW_MAX_COMPONENTS) * 8;
}
constexpr int kI8SliceRows = 16;      // rows per CTA: 2 per warp, so that every staged W^ value read from shared memory serves two rows

// slice s (0 = top) of four fixed-point values as one 32-bit word of the operand: the digit is byte NS - 1 - s of
// each value, gathered with three byte permutes (NS is a template parameter so the selectors are immediates)
template <int NS>
__device__ __forceinline__ uint32_t i8_pack4(const unsigned long long (&q)[16], int j0, int s)
{
    const int bidx = NS - 1 - s, bsel = bidx & 3;
    const uint32_t sel = (uint32_t)bsel | ((uint32_t)(4 + bsel) << 4);
    uint32_t w[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) w[j] = bidx < 4 ? (uint32_t)q[j0 + j] : (uint32_t)(q[j0 + j] >> 32);
    const uint32_t t01 = __byte_perm(w[0], w[1], sel), t23 = __byte_perm(w[2], w[3], sel);
    const uint32_t r = __byte_perm(t01, t23, 0x5410);
    return s == 0 ? r : (r ^ 0x80808080u);
}

template <int PASS, int SRC, int NS>
__global__ void __launch_bounds__(256)
k_slice_A(const double *__restrict__ coef, const double *__restrict__ rate, const uint8_t *__restrict__ comp8 /*padded*/,
          int64_t p0, int64_t Pc, const double *__restrict__ What, const int8_t *__restrict__ tau /*[n_T], padded*/,
          int n_T, int KT, int ns_store /*slices written: NS, or 4 for the fast mode*/, int *__restrict__ e_row,
          uint8_t *__restrict__ As)
{
    constexpr int ns = NS;
    constexpr int RPW = kI8SliceRows / 8;
    constexpr int NW = (SRC == 0) ? kNumTerms : 1;               // staged rows of W^ (SRC 1: N_mc only)
    // dynamic shared memory: two staging buffers {W^ rows [NW][512], comp [512] bytes, tau [512] bytes}, filled with
    // cp.async one 512-bin chunk ahead of the arithmetic (the kernel was latency-bound on these loads)
    extern __shared__ __align__(16) uint8_t slice_smem[];
    constexpr int kBufBytes = NW * 512 * 8 + 512 + 512;
    double *sC = reinterpret_cast<double *>(slice_smem + 2 * kBufBytes);                  // [16][12]
    double *sRate = sC + kI8SliceRows * kCoefStride;                                      // [16][4]
    const int r0 = (threadIdx.x >> 5) * RPW, lane = threadIdx.x & 31;
    const int64_t row0 = (int64_t)blockIdx.x * kI8SliceRows + r0;
    if (SRC == 0 && threadIdx.x < kI8SliceRows * kCoefStride) {
        const int rr = threadIdx.x / kCoefStride, b = threadIdx.x - rr * kCoefStride;
        const int64_t q = (int64_t)blockIdx.x * kI8SliceRows + rr;
        sC[rr * kCoefStride + b] = (q < Pc) ? coef[(p0 + q) * kCoefStride + b] : 0.0;
    }
    if (SRC == 0 && threadIdx.x < kI8SliceRows * RW_MAX_COMPONENTS) {
        const int rr = threadIdx.x / RW_MAX_COMPONENTS, cq = threadIdx.x % RW_MAX_COMPONENTS;
        const int64_t q = (int64_t)blockIdx.x * kI8SliceRows + rr;
        sRate[rr * RW_MAX_COMPONENTS + cq] = (q < Pc) ? rate[(p0 + q) * RW_MAX_COMPONENTS + cq] : 1.0;
    }
    int e[RPW];
    double scale2[RPW], vmax[RPW];
    bool bad[RPW];
#pragma unroll
    for (int u = 0; u < RPW; ++u) {
        e[u] = (PASS == 1) ? e_row[row0 + u] : 0;
        scale2[u] = (PASS == 1 && e[u] != kI8BadRow) ? ldexp(1.0, 8 * ns - 1 - e[u]) : 0.0;
        vmax[u] = 0.0;
        bad[u] = false;
    }
    const int n_pad = KT * kI8BK;
    const double limit = ldexp(1.0, 8 * ns - 1);                  // q <= 2^(8 ns - 1) keeps the top digit <= 128
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(slice_smem);
    auto stage = [&](int i0, int buf) {          // chunk [i0, i0 + 512) -> buffer buf; bins >= n_T read as zero
        const uint32_t dW = sbase + buf * kBufBytes;
        for (int q = threadIdx.x; q < NW * 512; q += 256) {
            const int b = q >> 9, ii = q & 511, i = i0 + ii;
            const bool in = i < n_T;
            const double *src = What + (in ? (size_t)b * n_T + i : 0);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dW + (b * 512 + i8_sw(ii)) * 8), "l"(src),
                         "r"(in ? 8 : 0) : "memory");
        }
        if (threadIdx.x < 128) {                 // comp / tau bytes: padded to a multiple of 512 bins at rw_create
            const uint32_t dC = dW + NW * 512 * 8 + 4 * threadIdx.x;
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4, 4;" ::"r"(dC), "l"(comp8 + i0 + 4 * threadIdx.x) : "memory");
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4, 4;" ::"r"(dC + 512), "l"(tau + i0 + 4 * threadIdx.x) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    stage(0, 0);
    int buf = 0;
    for (int i0 = 0; i0 < n_pad; i0 += 512, buf ^= 1) {
        if (i0 > 0) __syncthreads();                               // everyone is done with the buffer refilled next
        if (i0 + 512 < n_pad) {
            stage(i0 + 512, buf ^ 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();                                           // chunk i0 is in buffer buf for every thread
        const double(*sW)[512] = reinterpret_cast<const double(*)[512]>(slice_smem + buf * kBufBytes);
        const uint8_t *sComp = slice_smem + buf * kBufBytes + NW * 512 * 8;
        const uint8_t *sTau = sComp + 512;
        const int ii0 = lane * 16, ibase = i0 + ii0;             // this thread: 16 consecutive bins of its rows
        if (ibase >= n_pad) continue;
        unsigned long long q16[RPW][16];
        const uint4 cw = *reinterpret_cast<const uint4 *>(sComp + ii0);
        const uint32_t cws[4] = {cw.x, cw.y, cw.z, cw.w};
        const uint4 tw = *reinterpret_cast<const uint4 *>(sTau + ii0);
        const uint32_t tws[4] = {tw.x, tw.y, tw.z, tw.w};
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int sj = i8_sw(ii0 + j);
            const int tj = (int)(int8_t)((tws[j >> 2] >> (8 * (j & 3))) & 0xffu);
            const double scl = __hiloint2double((1023 - tj) << 20, 0);       // 2^-tau_i, exact
            double v[RPW];
            if (SRC == 0) {
                double wv[kNumTerms];
#pragma unroll
                for (int b = 0; b < kNumTerms; ++b) wv[b] = sW[b][sj];
                const uint32_t cmp = (cws[j >> 2] >> (8 * (j & 3))) & 0xffu;
#pragma unroll
                for (int u = 0; u < RPW; ++u) {
                    double acc = 0.0;
#pragma unroll
                    for (int b = 0; b < kNumTerms; ++b) acc = fma(sC[(r0 + u) * kCoefStride + b], wv[b], acc);
                    v[u] = acc * sRate[(r0 + u) * RW_MAX_COMPONENTS + cmp] * scl;       // N' / 2^tau_i
                    // derivative rows of rw_eval_grad (slot 11 = 1): the positive part of the row, negatives -> 0
                    if (sC[(r0 + u) * kCoefStride + kCoefStride - 1] != 0.0) v[u] = fmax(v[u], 0.0);
                }
            } else {
                const double nm = sW[0][sj] * scl;
#pragma unroll
                for (int u = 0; u < RPW; ++u)
                    v[u] = (row0 + u < Pc && ibase + j < n_T) ? coef[(size_t)(row0 + u) * n_T + ibase + j] * nm : 0.0;
            }
#pragma unroll
            for (int u = 0; u < RPW; ++u) {
                if (PASS == 0) {
                    if (!(v[u] >= 0.0) || isinf(v[u])) bad[u] = true;
                    vmax[u] = fmax(vmax[u], v[u]);
                } else {
                    // the exponent may come from k_row_bound (an upper bound, never below the row maximum): a negative
                    // or non-finite N', or -- should the bound ever fail -- a value past 2^e, makes the row NaN
                    if (!(v[u] >= 0.0) || !(v[u] * scale2[u] <= limit)) bad[u] = e[u] != kI8BadRow;
                    q16[u][j] = i8_fixed((e[u] == kI8BadRow || bad[u]) ? 0.0 : v[u], scale2[u], ns);
                }
            }
        }
        if (PASS == 1) {
#pragma unroll
            for (int u = 0; u < RPW; ++u) {
                const int64_t row = row0 + u, mt = row >> 7;
                const int rr = (int)(row & 127), g = rr >> 3, r8 = rr & 7;
                const int kt = ibase >> 5, c = (ibase >> 4) & 1;
                uint8_t *base = As + ((size_t)(mt * KT + kt) * ns * 2 + c) * 2048 + g * 128 + r8 * 16;
#pragma unroll
                for (int s = 0; s < NS; ++s) {
                    if (s >= ns_store) break;
                    *reinterpret_cast<uint4 *>(base + (size_t)s * kI8SliceBytesA) =
                        make_uint4(i8_pack4<NS>(q16[u], 0, s), i8_pack4<NS>(q16[u], 4, s), i8_pack4<NS>(q16[u], 8, s),
                                   i8_pack4<NS>(q16[u], 12, s));
                }
            }
        }
    }
    if (PASS == 1) {
#pragma unroll
        for (int u = 0; u < RPW; ++u) {
            int bd = bad[u];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) bd |= __shfl_xor_sync(0xffffffffu, bd, o);
            if (bd && lane == 0) e_row[row0 + u] = kI8BadRow;    // read by the fold's epilogue: NaN for that point
        }
    }
    if (PASS == 0) {
#pragma unroll
        for (int u = 0; u < RPW; ++u) {
            double vm = vmax[u];
            int bd = bad[u];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                vm = fmax(vm, __shfl_xor_sync(0xffffffffu, vm, o));
                bd |= __shfl_xor_sync(0xffffffffu, bd, o);
            }
            if (lane == 0) e_row[row0 + u] = bd ? kI8BadRow : i8_exponent(vm);
        }
    }
}

// ---- row exponents of N' without a pass over N' (coefficient rows only) ----
// Per 32-bin block B and basis term b: hi / lo = max / min over the block of W^_b[i] 2^-tau_i; cmask = components
// present.  Then for a point   max_i N'[p][i] 2^-tau_i  <=  max_B rate_B(p) sum_b max(c_b hi_b[B], c_b lo_b[B]),
// a sum of maxima in place of the maximum of the sum: 16 x cheaper than evaluating N', and tight because all W^_b
// carry the same N_mc[i] / S_SM[i] factor (the exponent comes out one larger than the exact one in a few per cent
// of the rows: one bit of 55).
__global__ void __launch_bounds__(32)
k_block_tables(const double *__restrict__ What /*[12][n_T]*/, const int *__restrict__ tau, const uint8_t *__restrict__ comp8,
               int n_T, int n_blk, double *__restrict__ hi /*[11][n_blk]*/, double *__restrict__ lo, int *__restrict__ cmask)
{
    const int B = blockIdx.x, i = B * 32 + threadIdx.x;
    const bool in = i < n_T;
    const double scl = in ? ldexp(1.0, -tau[i]) : 0.0;
    for (int b = 0; b < kNumTerms; ++b) {
        const double v = in ? What[(size_t)b * n_T + i] * scl : 0.0;
        double h = in ? v : -INFINITY, l = in ? v : INFINITY;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            h = fmax(h, __shfl_xor_sync(0xffffffffu, h, o));
            l = fmin(l, __shfl_xor_sync(0xffffffffu, l, o));
        }
        if (threadIdx.x == 0) { hi[(size_t)b * n_blk + B] = h; lo[(size_t)b * n_blk + B] = l; }
    }
    int m = in ? (1 << comp8[i]) : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m |= __shfl_xor_sync(0xffffffffu, m, o);
    if (threadIdx.x == 0) cmask[B] = m;
}

// One warp per point of the chunk: e_row[p] from the bound above (NaN / infinite coefficients: bad row).
__global__ void __launch_bounds__(256)
k_row_bound(const double *__restrict__ coef, const double *__restrict__ rate, int64_t p0, int64_t Pc, int64_t rows_pad,
            const double *__restrict__ hi, const double *__restrict__ lo, const int *__restrict__ cmask, int n_blk,
            int *__restrict__ e_row)
{
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (row >= rows_pad) return;
    if (row >= Pc) { if (lane == 0) e_row[row] = 0; return; }      // padding rows of the last tile: all-zero slices
    double c[kNumTerms], r[RW_MAX_COMPONENTS];
#pragma unroll
    for (int b = 0; b < kNumTerms; ++b) c[b] = coef[(p0 + row) * kCoefStride + b];
#pragma unroll
    for (int q = 0; q < RW_MAX_COMPONENTS; ++q) r[q] = rate[(p0 + row) * RW_MAX_COMPONENTS + q];
    double vmax = 0.0;
    bool bad = false;
    for (int B = lane; B < n_blk; B += 32) {
        double sum = 0.0;
#pragma unroll
        for (int b = 0; b < kNumTerms; ++b) sum += fmax(c[b] * hi[(size_t)b * n_blk + B], c[b] * lo[(size_t)b * n_blk + B]);
        const int m = cmask[B];
        double rm = 0.0;
#pragma unroll
        for (int q = 0; q < RW_MAX_COMPONENTS; ++q)
            if (m >> q & 1) rm = fmax(rm, r[q]);
        const double v = sum * rm;
        if (!(v == v) || isinf(v) || !(rm == rm)) bad = true;
        vmax = fmax(vmax, v);
    }
#pragma unroll
    for (int b = 0; b < kNumTerms; ++b) bad = bad || !(c[b] == c[b]) || isinf(c[b]);
    int bd = bad;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        vmax = fmax(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
        bd |= __shfl_xor_sync(0xffffffffu, bd, o);
    }
    if (lane == 0) e_row[row] = bd ? kI8BadRow : i8_exponent(vmax * (1.0 + 1e-9));     // rounding slack of the 11-term sums
}

// Column maxima of R -> exponents f_k (one thread per column, rows read coalesced across the warp).
// tau_i = binary exponent of the mean of N_mc over the 33 bins around i (0 where that mean is 0): the per-bin
// rescaling shared by both operands.  The window keeps tau smooth: it follows the shape of the MC spectrum, which
// is what spans decades, without passing bin-to-bin noise of N_mc on to the columns of R.
__global__ void k_tau(const double *__restrict__ N_mc, int n_T, int *__restrict__ tau, int8_t *__restrict__ tau_b)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_T) return;
    double acc = 0.0;
    for (int j = max(0, i - 16); j <= min(n_T - 1, i + 16); ++j) acc += N_mc[j];
    tau[i] = max(-120, min(120, i8_exponent(acc / 33.0)));
    tau_b[i] = (int8_t)tau[i];                                   // byte copy, zero-padded to 512 bins, for k_slice_A's cp.async      // any tau is valid (shared by both operands); keep 2^-tau an FP32 normal
}

__global__ void k_colexp_B(const double *__restrict__ R, int ldR, int n_T, int n_rec, const int *__restrict__ tau,
                           int *__restrict__ f_col)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_rec) return;
    double vmax = 0.0;
    for (int i = 0; i < n_T; ++i) vmax = fmax(vmax, ldexp(R[(size_t)i * ldR + k], tau[i]));
    f_col[k] = i8_exponent(vmax);
}

// g_k of the certificate (header comment): per column, the number of recoil bins whose fixed-point entry is non-zero
// and the sum of the rescaled entries.  gcol[0][k]: full contraction, gcol[1][k]: fast mode.
__global__ void k_col_bound(const double *__restrict__ R, int ldR, int n_T, int n_rec, int ns, const int *__restrict__ tau,
                            const int *__restrict__ f_col, double *__restrict__ gcol /*[2][n_rec]*/)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_rec) return;
    const int f = f_col[k];
    const double scale2 = ldexp(1.0, 8 * ns - 1 - f);
    double sum = 0.0, cnt = 0.0, lost = 0.0;
    for (int i = 0; i < n_T; ++i) {
        const double v = ldexp(R[(size_t)i * ldR + k], tau[i]);
        sum += v;
        if (__double2ull_rn(v * scale2) != 0ull) cnt += 1.0;
        else lost += v;                                              // below the resolution: the whole entry is the error
    }
    const double S = ldexp(sum, -f) * (1.0 + 1e-9);                  // its own summation rounding
    const double full = (ldexp(S + (1.0 + 1.01 * ns) * cnt, f - 8 * ns) + lost) * (1.0 + 1e-6);
    gcol[k] = full;
    gcol[(size_t)n_rec + k] = full + ldexp(5.07 * cnt, f - 32);
}

// Slices of R in  Bs[n-tile][k-block][slice][chunk c][column group g][column r8][16]  (K-major core matrices,
// "rows" of the B operand are reconstructed bins).  Thread = (column, 16 consecutive recoil bins).
__global__ void __launch_bounds__(256)
k_slice_B(const double *__restrict__ R, int ldR, int n_T, int n_rec, int n_cols /*128 x column tiles*/, int KT, int ns,
          const int *__restrict__ tau, const int *__restrict__ f_col, uint8_t *__restrict__ Bs)
{
    const int k = blockIdx.x * 256 + threadIdx.x;                // column (padded columns carry zeros)
    const int ibase = blockIdx.y * 16;
    if (k >= n_cols) return;
    const int f = (k < n_rec) ? f_col[k] : 0;
    const double scale2 = ldexp(1.0, 8 * ns - 1 - f);
    unsigned long long q16[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const int i = ibase + j;
        const double v = (k < n_rec && i < n_T) ? ldexp(R[(size_t)i * ldR + k], tau[i]) : 0.0;     // exact: R 2^tau_i
        q16[j] = i8_fixed(v, scale2, ns);
    }
    const int nt = k >> 7, rr = k & 127, g = rr >> 3, r8 = rr & 7;
    const int kt = ibase >> 5, c = (ibase >> 4) & 1;
    uint8_t *base = Bs + ((size_t)((size_t)nt * KT + kt) * ns * 2 + c) * 2048 + g * 128 + r8 * 16;
#pragma unroll
    for (int t = 0; t < 8; ++t) {
        if (t >= ns) break;
        uint32_t w[4];
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            uint32_t x = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) x |= i8_digit(q16[4 * h + j], t, ns) << (8 * j);
            w[h] = x;
        }
        *reinterpret_cast<uint4 *>(base + (size_t)t * kI8SliceBytesB) = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

// ---------------------------------------------------------------------------------------------- the contraction
__device__ __forceinline__ uint32_t i8_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void i8_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void i8_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void i8_mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void i8_mbar_wait(uint32_t bar, uint32_t parity)
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
// contiguous global -> shared bulk copy (TMA engine, no tensor map), completion on an mbarrier
__device__ __forceinline__ void i8_bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// K-major operand, no swizzle: 8 rows x 16 bytes core matrices (128 contiguous bytes); SBO = distance between
// 8-row groups, LBO = distance between the two 16-byte K chunks of a 32-element k-step; descriptor version 1.
__device__ __forceinline__ uint64_t i8_desc(uint32_t smem_addr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((smem_addr & 0x3ffff) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) |
           ((uint64_t)(sbo_bytes >> 4) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                        uint32_t accumulate)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void i8_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
}

struct I8Work {
    int n_rec, KT, tiles_m, tiles_n, D, d;
    int64_t Pc, part_stride;
    const uint8_t *As, *Bs;
    const int *e_row, *f_col;
    const double *bkg, *counts;
    const double *gcol;       // [n_rec] certificate constants of this period and mode, or NULL
    double *partial, *out_mu;
    double *cert;             // [2 tiles_n][part_stride] certified relative error per (half tile, point), or NULL
};

__device__ __forceinline__ void i8_tile_coord(int t, int tiles_m, int tiles_n, int &tm, int &tn)
{
    constexpr int GM = 8;             // 8 point tiles sweep the column tiles: a wave shares their slices in L2
    const int per_group = GM * tiles_n;
    const int g = t / per_group, rem = t - g * per_group;
    const int first_m = g * GM;
    const int gm = min(GM, tiles_m - first_m);
    tm = first_m + rem % gm;
    tn = rem / gm;
}

// Horner step over one accumulator: v = v * 2^-8 + acc (exact int32 -> double), 16 columns
__device__ __forceinline__ void i8_horner16(uint32_t taddr, double (&v)[16], bool first)
{
    uint32_t a[16];
    tmem_ld16(taddr, a);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = first ? (double)(int)a[j] : fma(v[j], 0.00390625, (double)(int)a[j]);
}

// Tile = 128 points x 128 bins.  A product with N = 64 columns cannot be issued faster than every ~50 cycles (its
// tensor-pipe slot is 32), one with N = 128 fills its 64-cycle slot, so the tile is 128 columns wide and the NS
// diagonals (one 128-column int32 accumulator each; TMEM holds four) are done in TWO PASSES over the recoil bins:
// pass 0 the diagonals 0..3 (10 products per 32 bins, slices 0..3 of both operands), pass 1 the diagonals 4..NS-1
// (18 or 26 products, all slices).  Eight epilogue warps (lane quadrant x column half) keep the pass-0 Horner sums
// of their 64 columns in registers until pass 1 has drained.
// FAST (RW_SLICED_FAST): pass 0 only.  Balanced digits round to nearest at every truncation point, so the top four
// slices of the same operands are the 31-bit fixed-point values and the four diagonals kept are everything above
// 2^-32 of (row max x column max): an FP32-class result from 10 of the 28 / 36 products.
template <int NS, bool FAST>
__global__ void __launch_bounds__(kI8Threads, 1)
k_fold_i8(const I8Work W)
{
    constexpr int kSlot = kI8SlotBytes, kStages = kI8Stages, kBOff = kI8SlotBytes / 2;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const uint32_t sbase = i8_smem_u32(smem);
    double *s_bkg = reinterpret_cast<double *>(smem + kStages * kSlot);                // [128] per tile
    double *s_cnt = s_bkg + kI8BN, *s_inv = s_cnt + kI8BN, *s_scl = s_inv + kI8BN;    // counts, 1/counts, 2^f_k
    double *s_g = s_scl + kI8BN;                                                      // certificate constants g_k
    const uint32_t bars = sbase + kStages * kSlot + 5 * kI8BN * 8;
    const uint32_t full_bar = bars, empty_bar = bars + 8 * kStages;
    const uint32_t tfull_bar = empty_bar + 8 * kStages, tempty_bar = tfull_bar + 8;
    uint32_t *s_tmem = reinterpret_cast<uint32_t *>(smem + kStages * kSlot + 5 * kI8BN * 8 + 128);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) { i8_mbar_init(full_bar + 8 * s, 1); i8_mbar_init(empty_bar + 8 * s, 1); }
        i8_mbar_init(tfull_bar, 1);
        i8_mbar_init(tempty_bar, 8);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {     // TMEM: 4 accumulators x 128 int32 columns = all 512 columns
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(i8_smem_u32(s_tmem)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *s_tmem;
    const int total_tiles = W.tiles_m * W.tiles_n;
    const int KT = W.KT;
    constexpr size_t kPerKtA = (size_t)NS * kI8SliceBytesA, kPerKtB = (size_t)NS * kI8SliceBytesB;

    if (warp == 0) {
        // ------------------------------------------------------------------ producer: bulk copies, no tensor maps
        // pass 0: a stage is TWO 32-bin blocks (slices 0..3: 16 KB + 16 KB each); pass 1: one block, all slices
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
                int tm, tn;
                i8_tile_coord(t, W.tiles_m, W.tiles_n, tm, tn);
                const uint8_t *a = W.As + (size_t)tm * KT * kPerKtA;
                const uint8_t *b = W.Bs + (size_t)tn * KT * kPerKtB;
                for (int kt = 0; kt < KT; kt += 2) {
                    i8_mbar_wait(empty_bar + 8 * stage, phase ^ 1);
                    const uint32_t fb = full_bar + 8 * stage, dst = sbase + stage * kSlot;
                    const int nk = min(2, KT - kt);
                    i8_mbar_expect_tx(fb, nk * 8 * 4096);
                    for (int h = 0; h < nk; ++h) {
                        i8_bulk_g2s(dst + h * 16384, a + (size_t)(kt + h) * kPerKtA, 4 * kI8SliceBytesA, fb);
                        i8_bulk_g2s(dst + kBOff + h * 16384, b + (size_t)(kt + h) * kPerKtB, 4 * kI8SliceBytesB, fb);
                    }
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
                for (int kt = 0; kt < (FAST ? 0 : KT); ++kt) {
                    i8_mbar_wait(empty_bar + 8 * stage, phase ^ 1);
                    const uint32_t fb = full_bar + 8 * stage, dst = sbase + stage * kSlot;
                    i8_mbar_expect_tx(fb, (uint32_t)(kPerKtA + kPerKtB));
                    i8_bulk_g2s(dst, a + (size_t)kt * kPerKtA, (uint32_t)kPerKtA, fb);
                    i8_bulk_g2s(dst + kBOff, b + (size_t)kt * kPerKtB, (uint32_t)kPerKtB, fb);
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer
        if (lane == 0) {
            // D = S32 (bits 4-5 = 2), A / B format at bits 7-9 / 10-12 (0 = unsigned 8 bit: the top slice, 1 = signed:
            // the balanced lower slices), K-major, N >> 3 at bit 17, M >> 4 at bit 24
            const uint32_t idesc = (2u << 4) | ((uint32_t)(kI8BN >> 3) << 17) | ((uint32_t)(kI8BM >> 4) << 24);
            int stage = 0; uint32_t phase = 0, pseq = 0;
            for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
                // ---- pass 0: diagonals 0..3 into accumulators 0..3, one segment of <= 16384 bins at a time
                for (int k0 = 0; k0 < KT; k0 += kI8SegKT) {
                const int k1 = min(KT, k0 + kI8SegKT);
                i8_mbar_wait(tempty_bar, (pseq & 1) ^ 1);        // the epilogue has drained the previous segment / pass
                ++pseq;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                for (int kt = k0; kt < k1; kt += 2) {
                    i8_mbar_wait(full_bar + 8 * stage, phase);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const int nk = min(2, KT - kt);
                    for (int h = 0; h < nk; ++h) {
                        const uint32_t sa = sbase + stage * kSlot + h * 16384, sb = sa + kBOff;
#pragma unroll
                        for (int d = 0; d < 4; ++d)
#pragma unroll
                            for (int s = 0; s <= d; ++s)
                                umma_i8(tmem_base + d * kI8BN, i8_desc(sa + s * kI8SliceBytesA, 2048, 128),
                                        i8_desc(sb + (d - s) * kI8SliceBytesB, 2048, 128),
                                        idesc | (s > 0 ? 1u << 7 : 0u) | (d - s > 0 ? 1u << 10 : 0u),
                                        (kt + h > k0 || s > 0) ? 1u : 0u);
                    }
                    i8_commit(empty_bar + 8 * stage);
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
                i8_commit(tfull_bar);
                }
                // ---- pass 1: diagonals 4..NS-1 into accumulators 0..NS-5
                for (int k0 = 0; k0 < (FAST ? 0 : KT); k0 += kI8SegKT) {
                const int k1 = min(KT, k0 + kI8SegKT);
                i8_mbar_wait(tempty_bar, (pseq & 1) ^ 1);
                ++pseq;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                for (int kt = k0; kt < k1; ++kt) {
                    i8_mbar_wait(full_bar + 8 * stage, phase);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t sa = sbase + stage * kSlot, sb = sa + kBOff;
#pragma unroll
                    for (int d = 4; d < NS; ++d)
#pragma unroll
                        for (int s = 0; s <= d; ++s)
                            umma_i8(tmem_base + (d - 4) * kI8BN, i8_desc(sa + s * kI8SliceBytesA, 2048, 128),
                                    i8_desc(sb + (d - s) * kI8SliceBytesB, 2048, 128),
                                    idesc | (s > 0 ? 1u << 7 : 0u) | (d - s > 0 ? 1u << 10 : 0u), (kt > k0 || s > 0) ? 1u : 0u);
                    i8_commit(empty_bar + 8 * stage);
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
                i8_commit(tfull_bar);
                }
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue warps 2..9
        const int q = warp & 3;                                  // TMEM lane quadrant this warp may read
        const int half = (warp - 2) >> 2;                        // its 64 of the tile's 128 columns
        const int lrow = 32 * q + lane;
        const int et = threadIdx.x - 64;                         // 0..255
        uint32_t pseq = 0;
        for (int t = blockIdx.x; t < total_tiles; t += gridDim.x) {
            int tm, tn;
            i8_tile_coord(t, W.tiles_m, W.tiles_n, tm, tn);
            asm volatile("bar.sync 1, 256;" ::: "memory");
            if (et < kI8BN) {        // column constants; columns >= n_rec: all slices are zero, bkg = n = 1/n = 0
                const int col = tn * kI8BN + et;
                const bool ok = col < W.n_rec;
                const double n = ok ? W.counts[col] : 0.0;
                s_bkg[et] = ok ? W.bkg[col] : 0.0;
                s_cnt[et] = n;
                s_inv[et] = n > 0.0 ? 1.0 / n : 0.0;
                s_scl[et] = ok ? ldexp(1.0, W.f_col[col]) : 0.0;
                s_g[et] = (ok && W.gcol) ? W.gcol[col] : 0.0;
            }
            asm volatile("bar.sync 1, 256;" ::: "memory");
            const int64_t row = (int64_t)tm * kI8BM + lrow;
            const int e = W.e_row[row];
            const double rscale = (e == kI8BadRow) ? __longlong_as_double(0x7ff8000000000000LL) : ldexp(1.0, e - 14);
            const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + 64 * half;
            double v[4][16];
#pragma unroll
            for (int g = 0; g < 4; ++g)
#pragma unroll
                for (int j = 0; j < 16; ++j) v[g][j] = 0.0;
            // ---- pass 0: v = sum_{d=0..3} 2^(-8d) acc_d, kept in registers (summed over the <= 16384-bin segments)
            const int nseg = (KT + kI8SegKT - 1) / kI8SegKT;
            for (int seg = 0; seg < nseg; ++seg) {
                i8_mbar_wait(tfull_bar, pseq & 1);
                ++pseq;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    double u[16];
#pragma unroll
                    for (int d = 3; d >= 0; --d) i8_horner16(taddr + d * kI8BN + 16 * g, u, d == 3);
#pragma unroll
                    for (int j = 0; j < 16; ++j) v[g][j] += u[j];
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) i8_mbar_arrive(tempty_bar);
            }
            // ---- pass 1: v += 2^-32 sum_{d=4..NS-1} 2^(-8(d-4)) acc_(d-4)
            for (int seg = 0; seg < (FAST ? 0 : nseg); ++seg) {
                i8_mbar_wait(tfull_bar, pseq & 1);
                ++pseq;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    double u[16];
#pragma unroll
                    for (int d = NS - 1; d >= 4; --d) i8_horner16(taddr + (d - 4) * kI8BN + 16 * g, u, d == NS - 1);
#pragma unroll
                    for (int j = 0; j < 16; ++j) v[g][j] = fma(u[j], 2.3283064365386963e-10 /* 2^-32 */, v[g][j]);
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) i8_mbar_arrive(tempty_bar);       // the next tile's products run under the Poisson terms
            }
            double tot = 0.0, worst = 0.0;
            const double escale = (e == kI8BadRow) ? 0.0 : ldexp(1.0, e);      // delta_k = 2^e_p g_k
#pragma unroll
            for (int g = 0; g < 4; ++g) {
#pragma unroll
                for (int j = 0; j < 16; j += 4) {
                    const int c0 = 64 * half + 16 * g + j;
                    const double m0 = fma(v[g][j] * rscale, s_scl[c0], s_bkg[c0]);
                    const double m1 = fma(v[g][j + 1] * rscale, s_scl[c0 + 1], s_bkg[c0 + 1]);
                    const double m2 = fma(v[g][j + 2] * rscale, s_scl[c0 + 2], s_bkg[c0 + 2]);
                    const double m3 = fma(v[g][j + 3] * rscale, s_scl[c0 + 3], s_bkg[c0 + 3]);
                    if (W.cert) {        // certified |mu~ - mu| / mu <= delta / (mu~ - delta); +inf where delta >= mu~ > 0
                        const double mm[4] = {m0, m1, m2, m3};
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const double dl = escale * s_g[c0 + u];
                            const double rel = (dl > 0.0) ? ((mm[u] > dl) ? dl / (mm[u] - dl) : __longlong_as_double(0x7ff0000000000000LL)) : 0.0;
                            worst = fmax(worst, rel);
                        }
                    }
                    if (W.out_mu && row < W.Pc) {
                        const int col = tn * kI8BN + c0;
                        double *dst = W.out_mu + ((size_t)row * W.D + W.d) * W.n_rec + col;
                        if (col < W.n_rec) dst[0] = m0;
                        if (col + 1 < W.n_rec) dst[1] = m1;
                        if (col + 2 < W.n_rec) dst[2] = m2;
                        if (col + 3 < W.n_rec) dst[3] = m3;
                    }
                    tot += poisson_sum4(m0, m1, m2, m3, s_cnt[c0], s_cnt[c0 + 1], s_cnt[c0 + 2], s_cnt[c0 + 3],
                                        s_inv[c0], s_inv[c0 + 1], s_inv[c0 + 2], s_inv[c0 + 3]);
                }
            }
            if (row < W.Pc) W.partial[(size_t)(2 * tn + half) * W.part_stride + row] = tot;
            if (W.cert && row < W.Pc)       // a row that could not be sliced (NaN result) certifies nothing
                W.cert[(size_t)(2 * tn + half) * W.part_stride + row] =
                    (e == kI8BadRow) ? __longlong_as_double(0x7ff0000000000000LL) : worst + 2e-15;
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}

// ---------------------------------------------------------------------------------------------- host side
// rw_create with RW_CREATE_SLICED: column exponents and the eight slices of every period's R.
int i8_setup(rw_ctx *ctx, cudaStream_t s)
{
    const Layout &L = ctx->lay;
    const int KT = L.KT8, n_cols = L.NT8 * 64;                  // NT8 counts 64-column units and is even
    const size_t per = (size_t)(L.NT8 / 2) * KT * L.ns8 * kI8SliceBytesB;
    // zero-padded byte copies of tau and comp8 (k_slice_A stages them 512 bins at a time with cp.async)
    if (cudaMemsetAsync(ctx->tau8b, 0, (size_t)ctx->D * L.KP512, s) != cudaSuccess ||
        cudaMemsetAsync(ctx->comp8p, 0, (size_t)L.KP512, s) != cudaSuccess ||
        cudaMemcpyAsync(ctx->comp8p, ctx->comp8, (size_t)ctx->n_T, cudaMemcpyDeviceToDevice, s) != cudaSuccess)
        return fail(ctx, RW_ERR_CUDA, "slicing setup: %s", cudaGetErrorString(cudaGetLastError()));
    for (int d = 0; d < ctx->D; ++d) {
        const double *Rd = ctx->R + (size_t)d * ctx->R_period_stride;
        int *f = ctx->f_col8 + (size_t)d * ctx->n_rec, *tau = ctx->tau8 + (size_t)d * ctx->n_T;
        k_tau<<<(ctx->n_T + 255) / 256, 256, 0, s>>>(ctx->N_mc + (size_t)d * ctx->n_T, ctx->n_T, tau,
                                                     ctx->tau8b + (size_t)d * L.KP512);
        k_block_tables<<<KT, 32, 0, s>>>(ctx->What + (size_t)d * kCoefStride * ctx->n_T, tau, ctx->comp8, ctx->n_T, KT,
                                         ctx->blk_hl8 + (size_t)d * 2 * kNumTerms * KT,
                                         ctx->blk_hl8 + ((size_t)d * 2 + 1) * kNumTerms * KT, ctx->blk_cm8);
        ctx->launches++;
        k_colexp_B<<<(ctx->n_rec + 127) / 128, 128, 0, s>>>(Rd, ctx->ldR, ctx->n_T, ctx->n_rec, tau, f);
        k_col_bound<<<(ctx->n_rec + 127) / 128, 128, 0, s>>>(Rd, ctx->ldR, ctx->n_T, ctx->n_rec, L.ns8, tau, f,
                                                              ctx->gcol8 + (size_t)d * 2 * ctx->n_rec);
        dim3 grid((n_cols + 255) / 256, KT * 2);
        k_slice_B<<<grid, 256, 0, s>>>(Rd, ctx->ldR, ctx->n_T, ctx->n_rec, n_cols, KT, L.ns8, tau, f, ctx->B8 + (size_t)d * per);
        ctx->launches += 4;
    }
    if (cudaGetLastError() != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "slicing R failed at launch");
    cudaError_t e = cudaFuncSetAttribute(k_fold_i8<8, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kI8Smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fold_i8<7, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kI8Smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fold_i8<8, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kI8Smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fold_i8<7, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kI8Smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_slice_A<1, 0, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, i8_slice_smem(0));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_slice_A<1, 0, 7>, cudaFuncAttributeMaxDynamicSharedMemorySize, i8_slice_smem(0));
    if (e != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "cudaFuncSetAttribute(k_fold_i8): %s", cudaGetErrorString(e));
    return RW_OK;
}

// Steps a1-a4 for the Pc points at coef[p0..] and period d through the sliced INT8 contraction.
// With `w` (weights of the chunk's Pc points, [Pc][n_T]) the rows are N' = w N_mc instead of the coefficient rows.
cudaError_t launch_fold_i8(rw_ctx *ctx, int d, int64_t p0, int64_t Pc, double *out_mu, cudaStream_t s, const double *w,
                           bool fast, bool certify)
{
    const Layout &L = ctx->lay;
    const int KT = L.KT8;
    const int64_t rows_pad = (Pc + kI8BM - 1) / kI8BM * kI8BM;
    uint8_t *As = reinterpret_cast<uint8_t *>(ctx->A_packed);     // 8 slice bytes per (point, bin): fits the FP64 N'
    const double *What = ctx->What + (size_t)d * kCoefStride * ctx->n_T;
    const unsigned sgrid = (unsigned)(rows_pad / kI8SliceRows);
    const int8_t *tau_b = ctx->tau8b + (size_t)d * L.KP512;
    const int nst = fast ? 4 : L.ns8;
#define RW_SLICE_LAUNCH(PASS, SRC, NS, c0, r0, m0, pp, W0)                                                          \
    k_slice_A<PASS, SRC, NS><<<sgrid, 256, i8_slice_smem(SRC), s>>>(c0, r0, ctx->comp8p, pp, Pc, W0, tau_b, ctx->n_T, KT, \
                                                                    nst, ctx->e_row8, As)
    if (w) {
        const double *N_mc = ctx->N_mc + (size_t)d * ctx->n_T;
        if (L.ns8 == 8) { RW_SLICE_LAUNCH(0, 1, 8, w, nullptr, nullptr, 0, N_mc); RW_SLICE_LAUNCH(1, 1, 8, w, nullptr, nullptr, 0, N_mc); }
        else { RW_SLICE_LAUNCH(0, 1, 7, w, nullptr, nullptr, 0, N_mc); RW_SLICE_LAUNCH(1, 1, 7, w, nullptr, nullptr, 0, N_mc); }
    } else {
        k_row_bound<<<(unsigned)(rows_pad / 8), 256, 0, s>>>(ctx->coef, ctx->rate, p0, Pc, rows_pad,
                                                             ctx->blk_hl8 + (size_t)d * 2 * kNumTerms * KT,
                                                             ctx->blk_hl8 + ((size_t)d * 2 + 1) * kNumTerms * KT,
                                                             ctx->blk_cm8, KT, ctx->e_row8);
        if (L.ns8 == 8) RW_SLICE_LAUNCH(1, 0, 8, ctx->coef, ctx->rate, ctx->comp8, p0, What);
        else RW_SLICE_LAUNCH(1, 0, 7, ctx->coef, ctx->rate, ctx->comp8, p0, What);
    }
#undef RW_SLICE_LAUNCH
    ctx->launches += 2;
    I8Work W;
    W.n_rec = ctx->n_rec; W.KT = KT; W.D = ctx->D; W.d = d;
    W.tiles_m = (int)(rows_pad / kI8BM); W.tiles_n = L.NT8 / 2;
    W.Pc = Pc; W.part_stride = L.MC;
    W.As = As;
    W.Bs = ctx->B8 + (size_t)d * (L.NT8 / 2) * KT * L.ns8 * kI8SliceBytesB;
    W.e_row = ctx->e_row8;
    W.f_col = ctx->f_col8 + (size_t)d * ctx->n_rec;
    W.bkg = ctx->bkg + (size_t)d * ctx->n_rec;
    W.counts = ctx->counts + (size_t)d * ctx->n_rec;
    W.partial = ctx->partial + (size_t)d * L.NT8 * L.MC;       // [D][NT8][MC]: 64-column half tiles in this mode
    W.out_mu = out_mu;
    W.gcol = certify ? ctx->gcol8 + ((size_t)d * 2 + (fast ? 1 : 0)) * ctx->n_rec : nullptr;
    W.cert = certify ? ctx->cert_part + (size_t)d * L.NT8 * L.MC : nullptr;
    const int total = W.tiles_m * W.tiles_n;
    const int grid = total < ctx->num_sms ? total : ctx->num_sms;
    {
        ProfScope prof(ctx, s);
        if (L.ns8 == 8 && !fast) k_fold_i8<8, false><<<grid, kI8Threads, kI8Smem, s>>>(W);
        else if (L.ns8 == 8) k_fold_i8<8, true><<<grid, kI8Threads, kI8Smem, s>>>(W);
        else if (!fast) k_fold_i8<7, false><<<grid, kI8Threads, kI8Smem, s>>>(W);
        else k_fold_i8<7, true><<<grid, kI8Threads, kI8Smem, s>>>(W);
    }
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
