// rw_profile.cu -- profiled overall rate normalisation ("profiling an
// overall rate normalization at each scan point"; rate_k of Eq. 17; Gaussian constraint of
// Eq. 18).
//
// For one point the fold gives the signal prediction S_j = mu_j - B_j over the bins j of all periods.  With a
// free normalisation s >= 0,
//     mu_j(s) = s S_j + B_j,    f(s) = 2 sum_j [mu_j - n_j + n_j ln(n_j/mu_j)] + ((s - s0)/sigma)^2   (pull iff sigma > 0)
// is convex in s, so the profiled value is f at the root of
//     g(s) = f'(s)/2 = sum_j S_j (1 - n_j/mu_j) + (s - s0)/sigma^2
// (or at s = 0 when g(0) >= 0).  g is increasing and concave: Newton's iteration from the left of the root
// converges monotonically; a bracket [lo, hi] guards the steps taken from the right.
// One CTA per point; the point's S row (all periods) is cached in shared memory when it fits, every Newton
// step is one pass over it with a fixed-order block reduction of (g, g').
#include "rw_internal.h"

namespace rw {

constexpr int kProfThreads = 1024;   // a Newton step is a latency chain (pass + block reduction): keep the pass short
constexpr int kProfSmemRow = 20480;     // doubles of S cached in shared memory (160 KB); larger rows re-read HBM/L2

struct Pair { double a, b; };

__device__ __forceinline__ Pair block_sum2(double a, double b, double (*red)[2])
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();                       // red[] may still be read from the previous call
    if (lane == 0) { red[warp][0] = a; red[warp][1] = b; }
    __syncthreads();
    Pair r = {0.0, 0.0};
#pragma unroll
    for (int w = 0; w < kProfThreads / 32; ++w) { r.a += red[w][0]; r.b += red[w][1]; }
    return r;
}

template <bool CACHED>
__global__ void __launch_bounds__(kProfThreads)
k_profile(const double *__restrict__ mu_rows /*[rows][nb]: mu at s = 1*/, int nb,
          const double *__restrict__ bkg, const double *__restrict__ counts, double s0, double sigma,
          const double *__restrict__ sat_const /*NULL or the Eq. 18 constant*/,
          double *__restrict__ out, double *__restrict__ out_scale)
{
    extern __shared__ double sS[];
    __shared__ double red[kProfThreads / 32][2];
    const double *row = mu_rows + (size_t)blockIdx.x * nb;
    if (CACHED) {
        for (int j = threadIdx.x; j < nb; j += kProfThreads) sS[j] = row[j] - bkg[j];
        __syncthreads();
    }
    auto sig = [&](int j) { return CACHED ? sS[j] : row[j] - bkg[j]; };
    const double inv_var = (sigma > 0.0) ? 1.0 / (sigma * sigma) : 0.0;

    auto eval_g = [&](double s) {          // (g, g') at s
        double g = 0.0, dg = 0.0;
#pragma unroll 4
        for (int j = threadIdx.x; j < nb; j += kProfThreads) {
            const double S = sig(j), n = counts[j];
            if (S != 0.0) {
                if (n > 0.0) {
                    const double q = S / fma(s, S, bkg[j]);     // S/mu; +inf when mu = 0
                    g += S - n * q;
                    dg += n * q * q;
                } else {
                    g += S;
                }
            }
        }
        Pair r = block_sum2(g, dg, red);
        r.a += (s - s0) * inv_var;
        r.b += inv_var;
        return r;
    };

    double s_hat = 0.0;
    Pair r = eval_g(0.0);
    if (r.a < 0.0) {                       // interior minimum (NaN inputs fall through to the value pass)
        double lo = 0.0, hi = -1.0;        // hi < 0: no upper bracket yet
        double s = (sigma > 0.0 && s0 > 0.0) ? s0 : 1.0;
        for (int it = 0; it < 100; ++it) {
            r = eval_g(s);
            if (r.a == 0.0) break;
            if (r.a < 0.0) lo = s; else hi = s;
            double sn = s - r.a / r.b;
            if (sn == s) break;            // the step is below one ulp of s: converged (without this test a step
                                           // from the left with no upper bracket yet would be "rejected", s doubled,
                                           // and ~50 bisections spent coming back)
            const bool rejected = !(sn > lo) || (hi > 0.0 && !(sn < hi)) || !(r.b > 0.0);
            if (rejected) sn = (hi > 0.0) ? 0.5 * (lo + hi) : 2.0 * s;
            // Newton converges quadratically here: once a step is below 1e-12 relative, the point it lands on is
            // exact to rounding, so that step is the last one
            const bool done = (!rejected && fabs(sn - s) <= 1e-12 * fabs(sn)) || (hi > 0.0 && hi - lo <= 1e-15 * hi);
            s = sn;
            if (done) break;
        }
        s_hat = s;
    } else if (!(r.a >= 0.0)) {
        s_hat = r.a;                       // NaN propagates
    }

    double t = 0.0;
    for (int j = threadIdx.x; j < nb; j += kProfThreads)
        t += poisson_term(fma(s_hat, sig(j), bkg[j]), counts[j]);
    Pair v = block_sum2(t, 0.0, red);
    if (threadIdx.x == 0) {
        double f = 2.0 * v.a;
        if (sigma > 0.0) f += (s_hat - s0) * (s_hat - s0) * inv_var;
        if (sat_const) f += sat_const[0];
        out[blockIdx.x] = f;
        if (out_scale) out_scale[blockIdx.x] = s_hat;
    }
}

int profile_setup(rw_ctx *ctx)
{
    cudaError_t e = cudaFuncSetAttribute(k_profile<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         kProfSmemRow * 8);
    if (e != cudaSuccess) return fail(ctx, RW_ERR_CUDA, "cudaFuncSetAttribute(k_profile): %s", cudaGetErrorString(e));
    return RW_OK;
}

cudaError_t launch_profile(rw_ctx *ctx, const double *mu_rows, int64_t rows, double s0, double sigma,
                           bool full_eq18, double *out, double *out_scale, cudaStream_t s)
{
    const int nb = ctx->D * ctx->n_rec;
    const double *sat = full_eq18 ? ctx->sat_const : nullptr;
    if (nb <= kProfSmemRow)
        k_profile<true><<<(unsigned)rows, kProfThreads, (size_t)nb * 8, s>>>(mu_rows, nb, ctx->bkg, ctx->counts, s0,
                                                                            sigma, sat, out, out_scale);
    else
        k_profile<false><<<(unsigned)rows, kProfThreads, 0, s>>>(mu_rows, nb, ctx->bkg, ctx->counts, s0, sigma, sat,
                                                                 out, out_scale);
    ctx->launches++;
    return cudaGetLastError();
}

}  // namespace rw
