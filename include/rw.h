/*
 * rw.h -- C ABI of the B200-native spectrum-reweighting likelihood hot path
 * (arxiv/paper_2607_00488; citations are PAPER.md:<line> + equation).
 *
 * One context (rw_ctx) = the device-resident, theta-independent tables of one analysis
 * ("initialized once and remain resident on the target device throughout
 * the fit").  rw_eval_batch runs, for P parameter points, the four steps of one
 * likelihood call:
 *   a1  couplings g~ = g + eps (Eq. 6) -> recoil spectrum S_theta(T_i) (Eq. 12,
 *       PAPER.md:138; Eq. 4/8/9; cut T <= 2E^2/(m_e+2E))
 *   a2  weights w_i = S_theta/S_SM applied to the MC recoil spectrum (Eq. 14, Eq. 1;
 *       PAPER.md:151,35)
 *   a3  fold mu[p,d,k] = sum_i w_i N_mc[d,i] R[d,i,k] + bkg[d,k]  (Eq. 11)
 *   a4  binned Poisson -2lnL against the counts, summed over periods (Eq. 18)
 * Every step runs in CUDA kernels (sm_100a); there is no CPU fallback.
 *
 * Conventions
 *   - all functions return 0 (RW_OK) or a negative rw_status; no exception crosses the ABI;
 *     there is no global state; rw_last_error(ctx) gives a human-readable message.
 *   - "host"/"device" is stated for every pointer.  Arrays are row-major, FP64.
 *   - the library never allocates device memory: the caller passes one workspace
 *     (rw_workspace_bytes) which the context owns until rw_destroy.
 *   - rw_eval_batch is asynchronous and stream-ordered: it only enqueues work on
 *     `cuda_stream` (a cudaStream_t, NULL = legacy default stream) and never synchronises
 *     (RW_PARAM_HOST / RW_OUT_HOST copies are enqueued on the same stream: pinned memory => still
 *     async).  The one exception is the opt-in RW_SLICED_STRICT / RW_FP32, see the flag.
 *   - one context must not be used from two streams at once; several contexts may coexist.
 */
#ifndef RW_H_
#define RW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rw_ctx rw_ctx; /* opaque; created by rw_create, freed by rw_destroy */

typedef enum {
    RW_OK = 0,
    RW_ERR_INVALID = -1,     /* bad argument / input table (see rw_last_error) */
    RW_ERR_WORKSPACE = -2,   /* workspace NULL, misaligned or too small */
    RW_ERR_CUDA = -3,        /* a CUDA runtime/driver call failed */
    RW_ERR_UNSUPPORTED = -4, /* e.g. not an sm_100 device */
    RW_ERR_NOMEM = -5        /* host allocation failed */
} rw_status;

/* parameter kinds: which new-physics parameter a column of param[P][k] holds.
 * eps_{alpha alpha}^{eL,R} of Eq. (6); mu_nu in Bohr magnetons. */
enum {
    RW_EPS_EE_L = 0, RW_EPS_EE_R = 1,
    RW_EPS_MM_L = 2, RW_EPS_MM_R = 3,
    RW_EPS_TT_L = 4, RW_EPS_TT_R = 5,
    RW_MU_NU = 6,
    RW_RATE_0 = 7,          /* RW_RATE_0 + c: rate scale of signal component c (rate_k of Eq. 17); */
    RW_RATE_1 = 8,          /* multiplies that component's reweighted MC content; absent => 1.  c < n_comp <= 4 */
    RW_RATE_2 = 9,
    RW_RATE_3 = 10,
    RW_N_KINDS = 11
};
enum { RW_MAX_COMPONENTS = 4 };

enum { RW_MEM_HOST = 0, RW_MEM_DEVICE = 1 };

/* rw_eval_batch flags */
enum {
    RW_DEVIANCE    = 0u,       /* default: 2 sum [mu - n + n ln(n/mu)] (Eq. 18 minus its saturated value) */
    RW_FULL_EQ18   = 1u << 0,  /* literal first sum of Eq. (18): 2 sum [mu - n ln mu + lnGamma(n+1)] */
    RW_MODE_AUTO   = 0u,       /* 1 point: one-launch streaming path; 2..64: streaming DMMA kernel, tile height = the points
                                  rounded up to 8 (one launch up to 16 points, two above: N' is written first); more: tiled
                                  DMMA batched contraction (on large responses the last P mod 128 <= 96 points of a batch go
                                  through the streaming DMMA kernel instead of a partly filled row of tiles; when that takes
                                  two calls they share the points evenly, e.g. 65 = 40 + 25).  The
                                  streaming DMMA kernel is a cooperative launch (its CTAs share out the epilogue of a
                                  column strip and wait for one another); it can be captured in a CUDA graph */
    RW_MODE_STREAM = 1u << 4,  /* force the HBM-streaming fold (any P, groups of 16 points per launch) */
    RW_MODE_GEMM   = 2u << 4,  /* force the tiled FP64 tensor-core (DMMA) contraction */
    RW_MODE_COLLAPSED = 3u << 4, /* opt-in: rank-K prefolded templates (exact, O(K n_rec) per point); see below */
    RW_MODE_RIDGE  = 4u << 4,  /* force the streaming DMMA kernel (any P, groups of 64 points per launch): R is read
                                  from HBM once per group and contracted on the FP64 tensor cores in the same pass */
    RW_MODE_MASK   = 7u << 4,
    RW_PARAM_HOST  = 1u << 8,  /* `param` is a host pointer (copied H2D on the stream) */
    RW_OUT_HOST    = 1u << 9,  /* `out_m2lnL` (and `out_mu`) are host pointers (copied D2H on the stream) */
    RW_FP32        = 1u << 10, /* opt-in reduced precision for the batched contraction (rw_eval_batch / rw_eval_profile, dense
                                  fold of more than 4 points): mu within 1e-5 relative of the FP64 path, GUARANTEED -- it is
                                  RW_SLICED_FAST | RW_SLICED_STRICT: the top four 8-bit slices of both operands on the INT8
                                  tensor cores, and any point whose certified error exceeds 1e-5 is recomputed in FP64.
                                  Needs a context created with RW_CREATE_FP32 or RW_CREATE_SLICED.  (Round 1 had a separate
                                  TF32 x 3 kernel here; the fast sliced contraction is 1.7x faster and more accurate.) */
    RW_SLICED      = 1u << 11, /* opt-in FP64-by-slicing for the batched contraction: rows of N' and columns of R in fixed point
                                  (8 balanced base-256 digits for n_T <= 2048, else 7: 63 / 55 bits below their own maximum),
                                  36 / 28 INT8 tensor-core products per 32 recoil bins with exact int32 accumulation.  The error
                                  is bounded in terms of (row max)(column max), not of mu: ~1e-13 of mu for responses spread
                                  over many recoil bins; the certified per-point bound is what
                                  rw_eval_certified returns, and RW_SLICED_STRICT enforces 1e-12.
                                  Needs RW_CREATE_SLICED; non-negative finite N' (else NaN for that point, or the FP64 result
                                  under RW_SLICED_STRICT).  Accepted by rw_eval_batch, rw_eval_certified, rw_eval_profile,
                                  rw_eval_weights, rw_eval_pee and rw_eval_grad (dense fold only; the streaming, ridge and
                                  collapsed regimes ignore it). */
    RW_SLICED_FAST = 1u << 12, /* opt-in reduced precision on the same slices: only their top four (31-bit fixed point) and
                                  the four leading diagonals, 10 INT8 products per 32 recoil bins.  Error
                                  ~1e-9 (row max)(column max) n_T per bin: mu within 1e-5 relative wherever RW_SLICED
                                  holds 1e-12 (the FP32 bar of this library).  Same requirements and scope as RW_SLICED,
                                  which it excludes. */
    RW_SLICED_STRICT = 1u << 13 /* with RW_SLICED / RW_SLICED_FAST: never silently less accurate than promised.  Every point
                                  carries a rigorous bound on max_k |mu~ - mu| / mu from the fixed-point scales (rw_fold_i8.cu);
                                  a point whose bound exceeds 1e-12 (RW_SLICED) or 1e-5 (RW_SLICED_FAST) is recomputed by the
                                  FP64 DMMA path, so every result meets the bar of its mode whatever the response looks like.
                                  The library reads the number of such points back: ONE stream synchronisation per chunk of
                                  <= 32768 points (the only calls that synchronise; they cannot be captured in a CUDA graph). */
};

/* rw_inputs.create_flags */
enum {
    RW_CREATE_FP32 = 1u << 0,  /* same as RW_CREATE_SLICED (RW_FP32 runs on the INT8 slices) */
    RW_CREATE_SLICED = 1u << 1 /* also keep R cut into 8 (n_T <= 2048) or 7 INT8 slices (at most the bytes of R) and the
                                  per-column certificate constants, for RW_SLICED / RW_SLICED_FAST / RW_FP32 */
};

/* Physical constants.  The paper prints symbols only; any field that is 0
 * takes the default: sin2_theta_w 0.23121, m_e 0.51099895 MeV, G_F 1.1663788e-11 MeV^-2,
 * alpha_em 1/137.035999084.  Natural units, MeV. */
typedef struct {
    double sin2_theta_w, m_e_MeV, G_F_MeV2, alpha_em;
} rw_constants;

typedef struct {
    int32_t n_E;            /* flux-grid entries: continuum cells + lines */
    const double *E_MeV;    /* [n_E] neutrino energies, > 0 */
    const double *flux_w;   /* [n_E] phi(E_j)*dE_j >= 0; a line is one entry with its integrated flux */
    const double *P_e;      /* [n_E] nu_e survival probability in [0,1] */
    const double *P_mu;     /* [n_E] or NULL -> (1-P_e)(1-f_tau) */
    const double *P_tau;    /* [n_E] or NULL -> (1-P_e) f_tau */
    double f_tau;           /* used only when P_mu/P_tau are NULL */
    int32_t n_T;            /* recoil bins */
    const double *T_MeV;    /* [n_T] representative recoil energy per bin, > 0 */
    int32_t n_rec;          /* reconstructed-observable bins */
    int32_t n_periods;      /* data periods D (>= 1), -2lnL is summed over them */
    const double *N_mc;     /* [D][n_T]  MC recoil spectrum under the SM, >= 0 */
    const double *R;        /* [D][n_T][n_rec] conditional response P(rec k | T_i), rec index fastest,
                               >= 0, sum_k R[i][k] = efficiency_i */
    const double *bkg;      /* [D][n_rec] theta-independent background, >= 0 */
    const double *counts;   /* [D][n_rec] observed counts as doubles (Asimov allowed), >= 0 */
    rw_constants consts;
    int32_t mem_kind;       /* RW_MEM_HOST: all arrays are host pointers, copied into the workspace.
                               RW_MEM_DEVICE: all arrays are device pointers; R is borrowed (caller keeps
                               it alive until rw_destroy) when 16-byte aligned with even n_rec, the
                               small tables are copied. */
    uint32_t create_flags;  /* 0, RW_CREATE_FP32 and/or RW_CREATE_SLICED */
    int32_t n_comp;         /* signal components (Eq. 17; Sec. IV B); 0 or 1: one.
                               With n_comp > 1, flux_w, P_e (and P_mu, P_tau) are [n_comp][n_E] tables on the shared
                               E grid, and the recoil bins of all components are concatenated along n_T. */
    const int32_t *comp_of_T; /* [n_T] component of every recoil bin (same memory kind as the other arrays);
                               ignored (may be NULL) when n_comp <= 1. */
} rw_inputs;

/* Bytes of device workspace rw_create needs for these inputs and batches of up to max_batch points.
 * Only the sizes, n_periods, mem_kind and create_flags fields of `in` are read. */
int rw_workspace_bytes(const rw_inputs *in, int64_t max_batch, size_t *bytes);

/* Validate inputs, place tables in the workspace, run the setup kernels (basis spectra, S_SM,
 * pre-scaled basis W^, saturated constant) on `cuda_stream`, and synchronise that stream once.
 * dev_workspace: device pointer, 256-byte aligned, >= rw_workspace_bytes; owned by ctx until destroy.
 * max_batch (an addition to the north_star signature): the library never allocates device memory, so the per-call
 * scratch (coefficients, the reweighted spectrum of a chunk, partial sums) is part of the workspace and has to be
 * sized when the workspace is; it must equal the value given to rw_workspace_bytes.  Calls with more points are
 * processed in slices of max_batch. */
int rw_create(const rw_inputs *in, int64_t max_batch, void *dev_workspace, size_t workspace_bytes,
              void *cuda_stream, rw_ctx **out);

/* Replace the observed counts ([D][n_rec], host or device per mem_kind); for toys / Asimov rescans. */
int rw_set_counts(rw_ctx *ctx, const double *counts, int32_t mem_kind, void *cuda_stream);

/* -2lnL for P points.
 *   param       [P][k] row-major, device pointer (host if RW_PARAM_HOST)
 *   param_kind  host [k], distinct values in RW_EPS_EE_L..RW_MU_NU (absent: 0) and RW_RATE_0 + c, c < n_comp (absent: 1)
 *   out_m2lnL   [P] device pointer (host if RW_OUT_HOST)
 *   out_mu      NULL, or [P][D][n_rec] predicted counts mu (same memory kind as out_m2lnL); with RW_OUT_HOST it is staged
 *               through the workspace in slices and copied D2H on the stream
 * P may be 0 (no-op) and may exceed max_batch (processed in slices).  Per-point numerical outcomes
 * are values, not errors: mu_k = 0 with n_k > 0 gives +inf; non-finite parameters give NaN. */
int rw_eval_batch(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                  double *out_m2lnL, double *out_mu, uint32_t flags, void *cuda_stream);

/* rw_eval_certified: rw_eval_batch for the sliced contractions (flags must hold RW_SLICED, RW_SLICED_FAST or RW_FP32;
 * DEVICE pointers only, no out_mu) that also returns, per point, the certified bound
 *     out_bound[p] >= max over bins and periods of |mu~ - mu| / mu
 * of what the INT8 contraction computed (0 for points that went through an FP64 path: calls of up to 64 points, which
 * RW_MODE_AUTO gives to the streaming kernels, or points recomputed under RW_SLICED_STRICT; +inf where a bin's bound reaches its mu or the row could not be sliced).
 * The bound is rigorous for the arithmetic of rw_fold_i8.cu and pessimistic by 10-100x on smooth inputs. */
int rw_eval_certified(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                      double *out_m2lnL, double *out_bound, uint32_t flags, void *cuda_stream);

/* Points recomputed in FP64 by strict sliced calls of this context so far (instrumentation, like rw_launch_count). */
int64_t rw_strict_fallback_count(const rw_ctx *ctx);

/* RW_MODE_COLLAPSED (rw_eval_batch only).  Eq. (4) is quadratic in the couplings, Eq. (8)
 * linear in mu_nu^2 and the fold of Eq. (11) linear in the spectrum, so
 *   mu[p][d][k] - bkg[d][k] = sum_q rate_q sum_b c_b(theta_p) G[d][q][b][k],   G[d][q][b][k] = sum_{i in component q} W^[d][b][i] R[d][i][k]
 * exactly (up to rounding order).  rw_create folds the 11 templates G of every component once; this mode then evaluates a point
 * in O(11 n_rec D) instead of O(n_T n_rec D).  It is NOT what RW_MODE_AUTO/STREAM/GEMM run (those execute the
 * full fold for every point, which is the only valid path once weights are not low-rank -- rw_eval_weights).
 *
 * rw_eval_weights: steps a3 + a4 for caller-supplied weights (Eq. 1, with an arbitrary
 * diag(r)): mu[p][d][k] = sum_i w[p][i] N_mc[d][i] R[d][i][k] + bkg[d][k], then Eq. (18).  For per-point
 * nuisances that make the weights something other than the spectrum ratio of Eq. (14) (oscillation
 * parameters, flux shapes: PAPER.md:220).
 *   w          [P][n_T] row-major DEVICE pointer, finite and >= 0 (not validated; garbage in, garbage out)
 *   out_m2lnL  [P] device pointer;  out_mu NULL or [P][D][n_rec] device pointer
 *   flags      RW_FULL_EQ18, RW_MODE_AUTO/STREAM/RIDGE/GEMM, RW_SLICED / RW_SLICED_FAST (+ RW_SLICED_STRICT: a chunk
 *              with an uncertified point is recomputed as a whole in FP64)
 *              (COLLAPSED, RW_FP32, RW_PARAM_HOST, RW_OUT_HOST: RW_ERR_UNSUPPORTED)
 * Asynchronous and stream-ordered like rw_eval_batch; P may be 0 and may exceed max_batch. */
int rw_eval_weights(rw_ctx *ctx, const double *w, int64_t P, double *out_m2lnL, double *out_mu,
                    uint32_t flags, void *cuda_stream);

/* rw_eval_pee: the path with a survival-probability table per point (the "physics update" of PAPER.md:220 evaluates
 * the oscillation probabilities for every parameter vector; here they arrive tabulated on the flux grid).
 *     w[p][i] = S_theta_p(T_i; P_e_pts[p]) / S_SM(T_i; nominal tables)       (Eq. 12 / Eq. 14; the MC sample and the SM
 * reference stay those of the nominal tables given to rw_create, reading R16).  The rest 1 - P_e of a point goes
 * to nu_mu and nu_tau by f_tau, or -- in a context created with explicit P_mu / P_tau -- in the nominal tables' mu : tau
 * ratio at every energy (reading R17).  These weights are not low-rank; they are built per point from three suffix sums
 * over the flux grid sorted by T_max (O(n_E + n_T) per point, rw_pee.cu) and folded by the dense path of rw_eval_weights.
 *   param, param_kind, P, k   as rw_eval_batch (DEVICE param; kinds RW_EPS_* and RW_MU_NU only)
 *   P_e_pts                   [P][n_comp][n_E] device pointer ([P][n_E] for one component), values in [0,1] (not validated)
 *   out_m2lnL [P], out_mu NULL or [P][D][n_rec]   device pointers
 *   flags                     RW_FULL_EQ18, RW_MODE_AUTO/STREAM/RIDGE/GEMM, RW_SLICED / RW_SLICED_FAST (+ RW_SLICED_STRICT)
 * Several components or explicit tables need n_E <= ~8500 (the scans live in shared memory).  Asynchronous, stream-ordered. */
int rw_eval_pee(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                const double *P_e_pts, double *out_m2lnL, double *out_mu, uint32_t flags, void *cuda_stream);

/* rw_eval_profile: -2lnL with the overall rate normalisation of the signal profiled out per point (PAPER.md:309,
 * "profiling an overall rate normalization at each scan point"; rate_k of Eq. 17; the Gaussian
 * constraint of Eq. 18, on that one nuisance).  With S = mu - bkg the fold of the point at unit
 * normalisation, over the bins of all periods,
 *     out[p]   = min over s >= 0 of  2 sum [mu_s - n + n ln(n/mu_s)] + ((s - s0)/sigma)^2,   mu_s = s S + bkg
 *     scale[p] = the minimiser s^ (0 when the data want no signal)
 * The objective is convex in s; the minimiser is found by a bracketed Newton iteration to double precision.
 *   param, param_kind, P, k   as rw_eval_batch (DEVICE param only)
 *   s0, sigma                 centre and width of the Gaussian pull on s; sigma <= 0 or +inf-like: no pull
 *   out_m2lnL [P], out_scale [P] or NULL   device pointers
 *   flags                     RW_FULL_EQ18; RW_MODE_AUTO/STREAM/RIDGE/GEMM (dense fold) or RW_MODE_COLLAPSED; RW_FP32,
 *                             RW_SLICED, RW_SLICED_FAST (+ RW_SLICED_STRICT) select the contraction as in rw_eval_batch
 * Asynchronous and stream-ordered; P may exceed max_batch. */
int rw_eval_profile(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                    double s0, double sigma, double *out_m2lnL, double *out_scale, uint32_t flags,
                    void *cuda_stream);

/* rw_eval_grad: -2lnL and its gradient with respect to the k scanned parameters, for gradient-based minimisers
 * (the paper minimises Eq. 18 with MIGRAD).  The path is linear in the coefficient vector of
 * Eq. (4)/(8) and in the rates of Eq. (17), so d mu / d theta_m is the same fold applied to derivative coefficients;
 *     out_grad[p][m] = sum over bins and periods of 2 (1 - n/mu) d mu / d theta_m      (n = 0: 2 d mu / d theta_m).
 * A point costs 1 + k rows of the batched fold.  DEVICE pointers only; flags: RW_FULL_EQ18 (value only), the fold
 * modes, and RW_SLICED / RW_SLICED_FAST: a derivative row changes sign along the recoil bins and the sliced contraction
 * wants non-negative rows, so there it is folded as its positive and its negative part (1 + 2k rows per point) and the
 * two folds are subtracted; each part carries the contraction's error relative to its own size.  RW_SLICED_STRICT and
 * RW_FP32: RW_ERR_UNSUPPORTED (a difference of two folds has no per-point certificate).  max_batch must be >= 1 + k
 * (1 + 2k with the sliced flags).  Asynchronous and stream-ordered; P may exceed max_batch. */
int rw_eval_grad(rw_ctx *ctx, const double *param, int64_t P, int32_t k, const int32_t *param_kind,
                 double *out_m2lnL, double *out_grad /*[P][k]*/, uint32_t flags, void *cuda_stream);

/* Device pointers to setup tables, for inspection/tests (valid until rw_destroy):
 *   RW_TABLE_S_SM   [n_T]        SM recoil spectrum S_SM(T_i) (Eq. 12 at theta = 0)
 *   RW_TABLE_BASIS  [10][n_T]    basis spectra A_e,B_e,C_e,A_mu,...,C_tau,D
 *   RW_TABLE_WHAT   [D][12][n_T] pre-scaled basis W^ = basis * N_mc / S_SM (+ dead-bin row)
 *   RW_TABLE_G      [D][n_comp][12][ldG] prefolded templates G (ldG = n_rec rounded up to even; rows 11 unused) */
enum { RW_TABLE_S_SM = 0, RW_TABLE_BASIS = 1, RW_TABLE_WHAT = 2, RW_TABLE_G = 3 };
int rw_get_table(const rw_ctx *ctx, int32_t which, const double **dev_ptr, int64_t *n_elems);

/* Number of kernels this context has launched so far (setup + eval); for bench accounting. */
int64_t rw_launch_count(const rw_ctx *ctx);

/* Measurement hooks (bench.py roofline): between begin and end every fold-kernel launch
 * (k_fold_gemm / k_fold_stream, the dominant kernels) is bracketed by CUDA events recorded on the
 * launching stream.  rw_profile_end synchronises those events and returns the summed kernel time
 * in ms and the number of launches timed (at most 32768; later launches are not bracketed). */
int rw_profile_begin(rw_ctx *ctx);
int rw_profile_end(rw_ctx *ctx, double *fold_ms_total, int64_t *fold_launches);

int rw_destroy(rw_ctx *ctx);

/* rw_fold_weights_static: steps a2 + a3 + a4 for ONE point and ONE period on caller weights, for callers that cannot
 * allocate device memory at all -- so cannot even provide the workspace rw_create wants.  Examples: a likelihood
 * plugged into a host application whose own memory pool already owns the device and which hands a plugin only its
 * input and output buffers; a fit next to latency-critical streams that a cudaMalloc / cudaFree (both synchronise the
 * device) would stall; a process whose memory budget was fixed before this library was loaded.
 *     mu[k]  = sum_i w[i] N_mc[i] R[i][k] + bkg[k]           (Eq. 1; Eq. 11)
 *     out    = 2 sum_k [mu_k - n_k + n_k ln(n_k / mu_k)]     (Eq. 18, relative to its saturated value)
 * the same numbers as rw_eval_weights with P = 1, D = 1, RW_MODE_STREAM (up to the order of the row-range sums).
 * No rw_ctx, no workspace: the call and everything under it uses no cudaMalloc, cudaFree or allocating library
 * routine.  The scratch of the streaming fold (partial sums per row range, completion tickets) is a fixed
 * 4 MiB + 512 B __device__ array inside librw.so; every GPU that loads the library holds it until the process exits.
 *   w [n_T], N_mc [n_T], bkg [n_rec], counts [n_rec]   DEVICE pointers, FP64
 *   R                    DEVICE pointer, [n_T] rows of pitch ldR doubles, rec index fastest; 16-byte aligned, ldR even
 *                        and >= n_rec
 *   out_m2lnL            DEVICE pointer to one double;  out_mu: NULL or DEVICE [n_rec]
 *   n_rec <= RW_STATIC_MAX_N_REC (the scratch is compiled for that many columns): larger => RW_ERR_INVALID with a
 *   message saying so (rw_last_error(NULL)); n_T is not limited.  n_T = 0 gives mu = bkg, n_rec = 0 gives 0.
 * Asynchronous and stream-ordered on `cuda_stream`, never synchronises.  Numerical outcomes are values as in
 * rw_eval_batch (mu_k = 0 < n_k: +inf; NaN in: NaN out).
 * First call on a device: looks up the device address of the built-in array (cudaGetSymbolAddress, once per device,
 * for the device that is current at the call) -- make that first call outside any stream capture.
 * One array per GPU serves every call and keeps what the previous call left in it; the call clears the tickets it
 * needs at zero on the stream before the kernel.  Two calls of this process that can overlap on one GPU (issued on
 * different streams, or from different host threads without ordering) race on it and give garbage: keep all calls
 * on a GPU ordered one after the other.  Other processes have their own copy of the array. */
enum { RW_STATIC_MAX_N_REC = 8192 };
int rw_fold_weights_static(const double *w, const double *N_mc, const double *R, int64_t ldR, int32_t n_T,
                           int32_t n_rec, const double *bkg, const double *counts, double *out_m2lnL,
                           double *out_mu, void *cuda_stream);

const char *rw_strerror(int status);
const char *rw_last_error(const rw_ctx *ctx); /* ctx may be NULL: the last failure without a context (rw_create,
                                                 rw_fold_weights_static, a NULL ctx) of the CALLING THREAD -- that one
                                                 buffer is thread-local state, the only state outside contexts besides
                                                 the built-in scratch of rw_fold_weights_static */

#ifdef __cplusplus
}
#endif
#endif /* RW_H_ */
