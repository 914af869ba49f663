// rw_noalloc.cu -- rw_fold_weights_static: one evaluation of steps a2-a4 that needs no context, no workspace and no
// device allocation of any kind (include/rw.h has the contract).
//
// Who this is for.  Every other entry point of this library works on a workspace the caller obtained from
// cudaMalloc (or from an allocator built on it).  Some callers cannot do that: a likelihood plugged into a host
// application that has already handed the whole device to its own memory pool and passes plugins nothing but
// input and output buffers; a fit running beside latency-critical streams, where cudaMalloc / cudaFree would
// synchronise the whole device; a process under a hard memory budget that was spent before the plugin was loaded.
// For them the scratch of the streaming fold (the per-row-range partial sums of mu and the "who finishes last"
// tickets of rw_fold_stream.cu) lives here in a file-scope __device__ array of fixed size that the CUDA module
// carries: every GPU that loads librw.so holds kStaticBytes (4 MiB + 512 B) of it until the process exits.
//
// The kernel is the single-point, single-period case of k_fold_stream with caller weights (Eq. 1, PAPER.md:35-38;
// Eq. 11; Eq. 18): a CTA streams a 512-column strip of a range of recoil rows, parks its
// partial sums, and the last CTA of a strip / the last strip finish the sums in a fixed order (results do not
// depend on which CTA happens to be last).
#include <mutex>

#include "rw_internal.h"

namespace rw {

constexpr int kStaticMaxRec = RW_STATIC_MAX_N_REC;          // columns the parked partial sums are sized for
constexpr int kStaticMaxSplits = 64;                        // row ranges per strip
constexpr int kStaticMaxStrips = kStaticMaxRec / kStreamCols;
constexpr int kStaticRC = 64;                               // recoil rows staged per iteration
constexpr size_t kOffPart = 0;                                                            // [splits][ld] doubles
constexpr size_t kOffStrip = kOffPart + (size_t)kStaticMaxSplits * kStaticMaxRec * 8;     // [strips] doubles
constexpr size_t kOffCnt = kOffStrip + 256;                                               // [strips] + 1 ints
constexpr size_t kStaticBytes = kOffCnt + 256;
static_assert(kStaticMaxStrips * 8 <= 256 && (kStaticMaxStrips + 1) * 4 <= 256, "scratch tail too small");

// The scratch itself.  In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device
// address and must never be handed to a kernel or to cudaMemsetAsync as it stands.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

struct StaticArgs {
    const double *w, *N_mc, *R, *bkg, *counts;
    int64_t ldR;
    int n_T, n_rec, rows_per_split, n_splits, ld;
    double *mu_part, *strip_part;
    int *cnt;
    double *out, *out_mu;
};

__global__ void __launch_bounds__(kStreamThreads)
k_fold_static(const StaticArgs A)
{
    __shared__ double sN[2][kStaticRC];
    __shared__ double red[kStreamThreads / 32];
    __shared__ int s_last;
    const int strip = blockIdx.x, split = blockIdx.y;
    const int col = strip * kStreamCols + 2 * threadIdx.x;
    const int i0 = split * A.rows_per_split, i1 = min(A.n_T, i0 + A.rows_per_split);
    const bool col_ok = col < A.n_rec;
    double acc0 = 0.0, acc1 = 0.0;

    auto stage = [&](int ic, int buf) {                     // a2: N'_i = w_i N_mc,i of 64 recoil rows
        if (threadIdx.x < kStaticRC) {
            const int i = ic + threadIdx.x;
            sN[buf][threadIdx.x] = (i < i1) ? A.w[i] * A.N_mc[i] : 0.0;
        }
    };
    if (i0 < i1) stage(i0, 0);
    int buf = 0;
    for (int ic = i0; ic < i1; ic += kStaticRC, buf ^= 1) {  // a3: this CTA's rows of its 512 columns
        __syncthreads();
        if (col_ok) {
            const double *Rp = A.R + (size_t)ic * A.ldR + col;
            const int nrows = min(kStaticRC, i1 - ic);
#pragma unroll 1
            for (int r0 = 0; r0 < nrows; r0 += 8) {
                double2 rv[8];
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    rv[u] = (r0 + u < nrows) ? __ldg(reinterpret_cast<const double2 *>(Rp + (size_t)(r0 + u) * A.ldR))
                                             : make_double2(0.0, 0.0);
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const double n = sN[buf][r0 + u];
                    acc0 = fma(n, rv[u].x, acc0);
                    acc1 = fma(n, rv[u].y, acc1);
                }
            }
        }
        if (ic + kStaticRC < i1) stage(ic + kStaticRC, buf ^ 1);
    }
    if (col_ok) __stcg(reinterpret_cast<double2 *>(A.mu_part + (size_t)split * A.ld + col), make_double2(acc0, acc1));

    // last CTA of this strip: row ranges in order, background, Poisson terms of the strip (a4)
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(A.cnt + strip, 1) == A.n_splits - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double t = 0.0;
    if (col_ok) {
        double m0 = 0.0, m1 = 0.0;
        for (int s = 0; s < A.n_splits; ++s) {
            const double2 v = __ldcg(reinterpret_cast<const double2 *>(A.mu_part + (size_t)s * A.ld + col));
            m0 += v.x;
            m1 += v.y;
        }
        const bool ok1 = col + 1 < A.n_rec;
        const double a0 = m0 + A.bkg[col], a1 = ok1 ? m1 + A.bkg[col + 1] : 0.0;
        if (A.out_mu) {
            A.out_mu[col] = a0;
            if (ok1) A.out_mu[col + 1] = a1;
        }
        t = poisson_term(a0, A.counts[col]) + (ok1 ? poisson_term(a1, A.counts[col + 1]) : 0.0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) red[warp] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
#pragma unroll
        for (int q = 0; q < kStreamThreads / 32; ++q) v += red[q];
        __stcg(A.strip_part + strip, v);
    }

    // last strip: strips in order, write the result, leave the tickets at zero
    const int n_strips = gridDim.x;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(A.cnt + n_strips, 1) == n_strips - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int q = 0; q < n_strips; ++q) v += __ldcg(A.strip_part + q);
        A.out[0] = 2.0 * v;
    }
    if (threadIdx.x <= n_strips) A.cnt[threadIdx.x] = 0;
}

// Device address of g_static_scratch on the CURRENT device, looked up once per device and remembered.
constexpr int kMaxDevices = 64;
static std::mutex g_static_mutex;
static unsigned char *g_static_ptr[kMaxDevices] = {};

static int static_scratch(unsigned char **ptr)
{
    int dev = -1;
    RW_CUDA(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices)
        return fail(nullptr, RW_ERR_UNSUPPORTED, "rw_fold_weights_static: device ordinal %d beyond %d", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void *p = nullptr;
        RW_CUDA(nullptr, cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return fail(nullptr, RW_ERR_CUDA, "rw_fold_weights_static: cudaGetSymbolAddress returned a null address");
        g_static_ptr[dev] = static_cast<unsigned char *>(p);
    }
    *ptr = g_static_ptr[dev];
    return RW_OK;
}

}  // namespace rw

extern "C" int rw_fold_weights_static(const double *w, const double *N_mc, const double *R, int64_t ldR, int32_t n_T,
                                      int32_t n_rec, const double *bkg, const double *counts, double *out_m2lnL,
                                      double *out_mu, void *cuda_stream)
{
    using namespace rw;
    const char *fn = "rw_fold_weights_static";
    if (n_T < 0 || n_rec < 0) return fail(nullptr, RW_ERR_INVALID, "%s: negative size (n_T %d, n_rec %d)", fn, n_T, n_rec);
    if (n_rec > kStaticMaxRec)
        return fail(nullptr, RW_ERR_INVALID,
                    "%s: n_rec = %d exceeds RW_STATIC_MAX_N_REC = %d, the size its built-in scratch was compiled for "
                    "(use rw_create + rw_eval_weights with a caller workspace instead)", fn, n_rec, kStaticMaxRec);
    if (!out_m2lnL) return fail(nullptr, RW_ERR_INVALID, "%s: out_m2lnL is NULL", fn);
    if (n_rec > 0 && (!bkg || !counts)) return fail(nullptr, RW_ERR_INVALID, "%s: bkg / counts is NULL", fn);
    if (n_rec > 0 && n_T > 0) {
        if (!w || !N_mc || !R) return fail(nullptr, RW_ERR_INVALID, "%s: w / N_mc / R is NULL", fn);
        if (ldR < n_rec || (ldR & 1) || (reinterpret_cast<uintptr_t>(R) & 15))
            return fail(nullptr, RW_ERR_INVALID, "%s: R must be 16-byte aligned with an even row pitch ldR >= n_rec (ldR %lld)",
                        fn, (long long)ldR);
    }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (n_rec == 0) {                                       // empty sum: -2lnL = 0 (all-zero bytes are 0.0)
        RW_CUDA(nullptr, cudaMemsetAsync(out_m2lnL, 0, sizeof(double), s));
        return RW_OK;
    }
    unsigned char *scr = nullptr;
    if (int rc = static_scratch(&scr)) return rc;

    StaticArgs A;
    A.w = w; A.N_mc = N_mc; A.R = R; A.bkg = bkg; A.counts = counts; A.ldR = ldR;
    A.n_T = n_T; A.n_rec = n_rec;
    const int strips = (n_rec + kStreamCols - 1) / kStreamCols;
    // about four CTAs per SM of a B200 in flight, at most kStaticMaxSplits row ranges, each a multiple of 64 rows
    int want = (4 * 148 + strips - 1) / strips;
    want = want < 1 ? 1 : (want > kStaticMaxSplits ? kStaticMaxSplits : want);
    int rows = ((n_T + want - 1) / want + kStaticRC - 1) / kStaticRC * kStaticRC;
    if (rows < kStaticRC) rows = kStaticRC;
    A.rows_per_split = rows;
    A.n_splits = n_T > 0 ? (n_T + rows - 1) / rows : 1;
    A.ld = (n_rec + 1) & ~1;
    A.mu_part = reinterpret_cast<double *>(scr + kOffPart);
    A.strip_part = reinterpret_cast<double *>(scr + kOffStrip);
    A.cnt = reinterpret_cast<int *>(scr + kOffCnt);
    A.out = out_m2lnL; A.out_mu = out_mu;
    // The array keeps whatever the previous call left.  The partial sums and strip sums are fully rewritten before
    // they are read; only the tickets must start at zero.  The kernel leaves them at zero, but a call that was
    // aborted would not have, so they are cleared on the stream every time.
    RW_CUDA(nullptr, cudaMemsetAsync(A.cnt, 0, (strips + 1) * sizeof(int), s));
    k_fold_static<<<dim3(strips, A.n_splits), kStreamThreads, 0, s>>>(A);
    RW_CUDA(nullptr, cudaGetLastError());
    return RW_OK;
}
