/*
 * rw_oracle.c -- CPU ORACLE for the spectrum-reweighting likelihood hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA path in
 * paper_2607_00488_b200/csrc; neither side includes or imports the other.
 *
 * What it is: the plain definitions of arxiv/paper_2607_00488 written
 * out as loops -- no basis decomposition, no blocking, no BLAS, no reordering.
 * Inputs and outputs are IEEE binary64; every intermediate and accumulator is
 * `long double` (x87 80-bit, 64-bit significand on x86-64) so that the oracle is
 * more accurate than the 1e-12 parity tolerance by several orders of magnitude.
 * The single exception is the kinematic cut, which is *specified* in binary64
 * (reading R2) so that both sides take the same yes/no decision.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`), per function:
 *   orc_tmax          closed form + textbook Compton edges (7Be 665 keV, pp 261 keV)
 *   orc_sm_couplings  Eq. (2)-(3) values, tests/golden/sm_couplings.txt
 *   orc_dsigma_weak   antiderivative closed form vs adaptive quadrature; textbook
 *                     sigma_e/E, sigma_mu/E high-energy slopes; sigma_0
 *   orc_dsigma_mm     antiderivative ln(T2/T1)-(T2-T1)/E vs quadrature; zero at T=E
 *   orc_spectrum      single-line reduction to dsigma; continuum limit vs scipy
 *                     dblquad-free closed form; exact quadratic/linear structure in
 *                     (eps, mu_nu^2); chirality sign-flip symmetry; mpmath brute force
 *   orc_weights       theta=0 => w == 1 bit-exactly
 *   orc_fold          identity / rank-1 responses; numpy matmul on random inputs;
 *                     folded total = sum_i w_i N_i eff_i
 *   orc_deviance      n == mu => 0; vs scipy.stats.poisson.logpmf; small-d expansion
 *   orc_eq18          vs -2*sum(scipy.stats.poisson.logpmf)
 *   orc_eval_batch    composition of the above; Asimov injection-recovery
 *                     (PAPER.md:309-311); rank-K prefold identity
 *   orc_profile_scale closed form s^ = sum n / sum S (no background, no pull); Asimov data at s* => s^ = s*,
 *                     value 0; scipy.optimize.minimize_scalar on a numpy objective;
 *                     pull limits sigma -> 0 (s^ -> s0) and sigma -> inf; boundary s^ = 0
 *   orc_eval_components  n_comp = 1 reproduces orc_eval_batch; identical tables split over two components
 *                     reproduce it too; mu - bkg is linear in the per-component rates with the single-component
 *                     predictions as coefficients; a component's bins get the weights of its own flux table
 *   orc_eval_grad     central finite differences (Richardson) of orc_eval_components in every parameter kind;
 *                     zero gradient at an Asimov point; value output identical to orc_eval_components
 *   orc_eval_pee      reference P_ee for every point reproduces orc_eval_batch; equals orc_eval_weights fed
 *                     the spectrum ratio computed with orc_spectrum on the point's table; P_ee = 1 / 0 on a
 *                     single line give the pure nu_e / nu_mu,tau cross-section ratio of Eq. (4)
 *   orc_eval_pee_components  single component without explicit tables reproduces orc_eval_pee; the nominal
 *                     tables for every point reproduce orc_eval_components (explicit tables included, so the rho
 *                     split returns exactly P_mu, P_tau); a component's bins follow its own table only
 *   orc_eval_weights  equals orc_eval_batch when fed orc_weights(theta); numpy matmul +
 *                     scipy Poisson on random weights; w == 1 gives the SM prediction
 * No function here is "parity unpinned".
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC rw_oracle.c -o librw_oracle.so -lm
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <float.h>
#include <stdlib.h>

#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double xreal; /* extended working precision */

typedef struct {
    double sin2_theta_w; /* weak mixing angle, Eq. (2)-(3) PAPER.md:56-58 */
    double m_e;          /* electron mass [MeV] */
    double G_F;          /* Fermi constant [MeV^-2] */
    double alpha_em;     /* fine-structure constant, Eq. (8) */
} orc_consts;

/* parameter kinds (values fixed by DESIGN.md "param_kind" table, not by a shared header) */
enum {
    ORC_EPS_EE_L = 0, ORC_EPS_EE_R = 1,
    ORC_EPS_MM_L = 2, ORC_EPS_MM_R = 3,
    ORC_EPS_TT_L = 4, ORC_EPS_TT_R = 5,
    ORC_MU_NU    = 6,  /* mu_nu in Bohr magnetons */
    ORC_N_KINDS  = 7
};

/* The paper gives no numerical constants (symbols only);
 * DESIGN.md reading R1 fixes PDG-style values, natural units, MeV. */
void orc_default_consts(orc_consts *c)
{
    c->sin2_theta_w = 0.23121;
    c->m_e          = 0.51099895;
    c->G_F          = 1.1663788e-11;
    c->alpha_em     = 1.0 / 137.035999084;
}

int orc_long_double_mant_dig(void) { return LDBL_MANT_DIG; }

/* Kinematic limit of the recoil energy for neutrino energy E: T <= 2E^2/(m_e+2E).
 * Not printed in PAPER.md; fixed by BASELINE.json north_star (reading R2).
 * Evaluated in binary64, one expression, exactly as written. */
double orc_tmax(double E, double m_e)
{
    volatile double num = 2.0 * E * E;
    volatile double den = m_e + 2.0 * E;
    return num / den;
}

/* Eq. (2)-(3).  Flavour order: 0=e, 1=mu, 2=tau. */
void orc_sm_couplings(const orc_consts *c, double gL[3], double gR[3])
{
    gL[0] = 0.5 + c->sin2_theta_w;   gR[0] = c->sin2_theta_w;
    gL[1] = -0.5 + c->sin2_theta_w;  gR[1] = c->sin2_theta_w;
    gL[2] = -0.5 + c->sin2_theta_w;  gR[2] = c->sin2_theta_w;
}

/* Eq. (4) / Eq. (7), PAPER.md:65,83:
 *   dsigma/dT = (2 G_F^2 m_e / pi) [ gL^2 + gR^2 (1 - T/E)^2 - gL gR m_e T / E^2 ]
 * (no kinematic cut applied here). */
static xreal xdsigma_weak(const orc_consts *c, xreal E, xreal T, xreal gL, xreal gR)
{
    const xreal pi = acosl(-1.0L);
    xreal pref = 2.0L * (xreal)c->G_F * (xreal)c->G_F * (xreal)c->m_e / pi;
    xreal one_m = 1.0L - T / E;
    return pref * (gL * gL + gR * gR * one_m * one_m - gL * gR * (xreal)c->m_e * T / (E * E));
}

/* Eq. (8):  dsigma^MM/dT = (pi alpha^2 / m_e^2) (mu_nu/mu_B)^2 (1/T - 1/E). */
static xreal xdsigma_mm(const orc_consts *c, xreal E, xreal T, xreal mu_nu)
{
    const xreal pi = acosl(-1.0L);
    xreal pref = pi * (xreal)c->alpha_em * (xreal)c->alpha_em / ((xreal)c->m_e * (xreal)c->m_e);
    return pref * mu_nu * mu_nu * (1.0L / T - 1.0L / E);
}

double orc_dsigma_weak(const orc_consts *c, double E, double T, double gL, double gR)
{
    return (double)xdsigma_weak(c, E, T, gL, gR);
}

double orc_dsigma_mm(const orc_consts *c, double E, double T, double mu_nu)
{
    return (double)xdsigma_mm(c, E, T, mu_nu);
}

/* theta[7] indexed by the ORC_* kinds above. */
static void xspectrum(const orc_consts *c, int n_E, const double *E, const double *flux_w,
                      const double *P_e, const double *P_mu, const double *P_tau,
                      int n_T, const double *T, const double *theta, xreal *S)
{
    double gL0[3], gR0[3];
    xreal gL[3], gR[3];
    orc_sm_couplings(c, gL0, gR0);
    /* Eq. (6): g -> g + eps_{alpha alpha}^{eL,R} */
    gL[0] = (xreal)gL0[0] + (xreal)theta[ORC_EPS_EE_L];
    gR[0] = (xreal)gR0[0] + (xreal)theta[ORC_EPS_EE_R];
    gL[1] = (xreal)gL0[1] + (xreal)theta[ORC_EPS_MM_L];
    gR[1] = (xreal)gR0[1] + (xreal)theta[ORC_EPS_MM_R];
    gL[2] = (xreal)gL0[2] + (xreal)theta[ORC_EPS_TT_L];
    gR[2] = (xreal)gR0[2] + (xreal)theta[ORC_EPS_TT_R];
    xreal mu_nu = (xreal)theta[ORC_MU_NU];

    /* Eq. (12) with the flavour sum of Eq. (5) and the incoherent MM term of Eq. (9),
     * PAPER.md:138-140, 69-71, 102.  flux_w[j] = phi(E_j) * dE_j; a line is one entry. */
    for (int i = 0; i < n_T; ++i) {
        xreal acc = 0.0L;
        for (int j = 0; j < n_E; ++j) {
            if (!(T[i] <= orc_tmax(E[j], c->m_e))) continue; /* kinematic cut (R2) */
            xreal Ej = E[j], Ti = T[i];
            xreal weak = (xreal)P_e[j]   * xdsigma_weak(c, Ej, Ti, gL[0], gR[0])
                       + (xreal)P_mu[j]  * xdsigma_weak(c, Ej, Ti, gL[1], gR[1])
                       + (xreal)P_tau[j] * xdsigma_weak(c, Ej, Ti, gL[2], gR[2]);
            /* MM term is flavour independent; sum_alpha P_alpha = 1 */
            xreal mm = xdsigma_mm(c, Ej, Ti, mu_nu);
            acc += (xreal)flux_w[j] * (weak + mm);
        }
        S[i] = acc;
    }
}

void orc_spectrum(const orc_consts *c, int n_E, const double *E, const double *flux_w,
                  const double *P_e, const double *P_mu, const double *P_tau,
                  int n_T, const double *T, const double *theta, double *S_out)
{
    xreal *S = (xreal *)malloc(sizeof(xreal) * (size_t)(n_T > 0 ? n_T : 1));
    xspectrum(c, n_E, E, flux_w, P_e, P_mu, P_tau, n_T, T, theta, S);
    for (int i = 0; i < n_T; ++i) S_out[i] = (double)S[i];
    free(S);
}

/* Bin-to-bin weights, Eq. (14) in the un-normalised north_star form w_i = S_theta/S_SM
 * (readings R5, R9: w := 1 where S_SM == 0). */
static void xweights(int n_T, const xreal *S, const xreal *S_sm, xreal *w)
{
    for (int i = 0; i < n_T; ++i)
        w[i] = (S_sm[i] == 0.0L) ? 1.0L : S[i] / S_sm[i];
}

void orc_weights(const orc_consts *c, int n_E, const double *E, const double *flux_w,
                 const double *P_e, const double *P_mu, const double *P_tau,
                 int n_T, const double *T, const double *theta, double *w_out)
{
    static const double zero[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
    size_t n = (size_t)(n_T > 0 ? n_T : 1);
    xreal *S = (xreal *)malloc(sizeof(xreal) * 3 * n), *S0 = S + n, *w = S0 + n;
    xspectrum(c, n_E, E, flux_w, P_e, P_mu, P_tau, n_T, T, theta, S);
    xspectrum(c, n_E, E, flux_w, P_e, P_mu, P_tau, n_T, T, zero, S0);
    xweights(n_T, S, S0, w);
    for (int i = 0; i < n_T; ++i) w_out[i] = (double)w[i];
    free(S);
}

/* Eq. (1)/(11): mu_k = sum_i R[i][k] * (w_i * N_mc,i) + bkg_k.
 * R row-major [n_T][n_rec], conditional response (sum_k R[i][k] = efficiency_i). */
static void xfold(int n_T, int n_rec, const xreal *w, const double *N_mc, const double *R,
                  const double *bkg, xreal *mu)
{
    for (int k = 0; k < n_rec; ++k) {
        xreal acc = 0.0L;
        for (int i = 0; i < n_T; ++i)
            acc += (w[i] * (xreal)N_mc[i]) * (xreal)R[(size_t)i * n_rec + k];
        mu[k] = acc + (xreal)bkg[k];
    }
}

void orc_fold(int n_T, int n_rec, const double *w, const double *N_mc, const double *R,
              const double *bkg, double *mu_out)
{
    xreal *xw = (xreal *)malloc(sizeof(xreal) * (size_t)(n_T + n_rec + 1)), *mu = xw + n_T;
    for (int i = 0; i < n_T; ++i) xw[i] = w[i];
    xfold(n_T, n_rec, xw, N_mc, R, bkg, mu);
    for (int k = 0; k < n_rec; ++k) mu_out[k] = (double)mu[k];
    free(xw);
}

/* Poisson deviance = Eq. (18) first sum minus its saturated value (reading R7):
 *   2 sum_k [ mu - n + n ln(n/mu) ];  n = 0 => 2 mu;  mu = 0 < n => +inf  (R8). */
static xreal xdeviance(int n_rec, const xreal *mu, const double *n)
{
    xreal acc = 0.0L;
    for (int k = 0; k < n_rec; ++k) {
        xreal nk = n[k], mk = mu[k];
        if (nk > 0.0L) {
            if (mk > 0.0L) {
                xreal d = mk - nk;
                acc += d - nk * log1pl(d / nk);
            } else {
                acc += (xreal)INFINITY;
            }
        } else {
            acc += mk;
        }
    }
    return 2.0L * acc;
}

/* Literal first sum of Eq. (18): 2 sum [mu - n ln mu + lnGamma(n+1)]. */
static xreal xeq18(int n_rec, const xreal *mu, const double *n)
{
    xreal acc = 0.0L;
    for (int k = 0; k < n_rec; ++k) {
        xreal nk = n[k], mk = mu[k];
        xreal t = mk + lgammal(nk + 1.0L);
        if (nk > 0.0L) t -= nk * logl(mk);
        acc += t;
    }
    return 2.0L * acc;
}

double orc_deviance(int n_rec, const double *mu, const double *n)
{
    xreal *xmu = (xreal *)malloc(sizeof(xreal) * (size_t)(n_rec > 0 ? n_rec : 1));
    for (int k = 0; k < n_rec; ++k) xmu[k] = mu[k];
    double r = (double)xdeviance(n_rec, xmu, n);
    free(xmu);
    return r;
}

double orc_eq18(int n_rec, const double *mu, const double *n)
{
    xreal *xmu = (xreal *)malloc(sizeof(xreal) * (size_t)(n_rec > 0 ? n_rec : 1));
    for (int k = 0; k < n_rec; ++k) xmu[k] = mu[k];
    double r = (double)xeq18(n_rec, xmu, n);
    free(xmu);
    return r;
}

/* Whole path for a batch of points (one "likelihood call" per point).
 *   params  [P][k] row-major, kinds[k] in ORC_* (absent kinds are 0)
 *   N_mc    [n_periods][n_T];  R [n_periods][n_T][n_rec];  bkg, counts [n_periods][n_rec]
 *   out     [P] deviance (or literal Eq. 18 sum if full_eq18 != 0), summed over periods
 *   mu_out  NULL or [P][n_periods][n_rec]
 *   abs_out NULL or [P]: sum_k 2|term_k| (conditioning scale for the tolerance, reading T)
 * The SM denominator is computed once per call by the same spectrum routine at theta = 0
 * ("computed once during initialization").  Returns 0, or -1 on bad kinds. */
int orc_eval_batch(const orc_consts *c, int n_E, const double *E, const double *flux_w,
                   const double *P_e, const double *P_mu, const double *P_tau,
                   int n_T, const double *T, int n_rec, int n_periods,
                   const double *N_mc, const double *R, const double *bkg, const double *counts,
                   int64_t P, int k, const int32_t *kinds, const double *params,
                   double *out, double *mu_out, double *abs_out, int full_eq18, int nthreads)
{
    static const double zero[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
    for (int a = 0; a < k; ++a) {
        if (kinds[a] < 0 || kinds[a] >= ORC_N_KINDS) return -1;
        for (int b = 0; b < a; ++b) if (kinds[a] == kinds[b]) return -1;
    }
    xreal *S0 = (xreal *)malloc(sizeof(xreal) * (size_t)(n_T > 0 ? n_T : 1));
    xspectrum(c, n_E, E, flux_w, P_e, P_mu, P_tau, n_T, T, zero, S0);
    if (nthreads < 1) nthreads = 1;

#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int64_t p = 0; p < P; ++p) {
        double theta[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
        for (int a = 0; a < k; ++a) theta[kinds[a]] = params[p * k + a];
        xreal *S = (xreal *)malloc(sizeof(xreal) * (size_t)(2 * n_T + n_rec + 1));
        xreal *w = S + n_T, *mu = w + n_T;
        xspectrum(c, n_E, E, flux_w, P_e, P_mu, P_tau, n_T, T, theta, S);
        xweights(n_T, S, S0, w);
        xreal total = 0.0L, total_abs = 0.0L;
        for (int d = 0; d < n_periods; ++d) {
            const double *Nd = N_mc + (size_t)d * n_T;
            const double *Rd = R + (size_t)d * n_T * n_rec;
            const double *Bd = bkg + (size_t)d * n_rec;
            const double *Cd = counts + (size_t)d * n_rec;
            xfold(n_T, n_rec, w, Nd, Rd, Bd, mu);
            total += full_eq18 ? xeq18(n_rec, mu, Cd) : xdeviance(n_rec, mu, Cd);
            if (mu_out)
                for (int q = 0; q < n_rec; ++q)
                    mu_out[((size_t)p * n_periods + d) * n_rec + q] = (double)mu[q];
            if (abs_out)
                for (int q = 0; q < n_rec; ++q) {
                    xreal one = xdeviance(1, mu + q, Cd + q);
                    total_abs += fabsl(one);
                }
        }
        out[p] = (double)total;
        if (abs_out) abs_out[p] = (double)total_abs;
        free(S);
    }
    free(S0);
    return 0;
}

/* Profiled overall rate normalisation (Sec. VI B: "profiling an overall rate normalization at
 * each scan point"; rate_k of Eq. 17; Gaussian constraint of Eq. 18).
 * Given the signal prediction S[j] >= 0 (fold at unit normalisation, background removed), background B[j] and
 * counts n[j] over all bins of all periods:
 *     mu_j(s) = s S_j + B_j,   f(s) = 2 sum_j [mu_j - n_j + n_j ln(n_j/mu_j)] + ((s - s0)/sigma)^2   (pull iff sigma > 0)
 * returns s^ = argmin_{s >= 0} f(s) and f(s^).  f is convex in s (reading R13), so the minimiser is
 * the root of f' (or 0 when f'(0) >= 0); it is bracketed by doubling and found by bisection in long double.
 * With full_eq18 the value is the literal Eq. (18) sum at s^ instead of the deviance (same minimiser). */
static xreal xprofile_dfds(int n, const xreal *S, const double *B, const double *cnt, xreal s, xreal s0, xreal sigma)
{
    xreal acc = 0.0L;
    for (int j = 0; j < n; ++j) {
        xreal mu = s * S[j] + (xreal)B[j];
        if (cnt[j] > 0.0) {
            if (S[j] != 0.0L) acc += S[j] * (1.0L - (xreal)cnt[j] / mu);   /* mu = 0 => -inf: pushes s up */
        } else {
            acc += S[j];
        }
    }
    acc *= 2.0L;
    if (sigma > 0.0L) acc += 2.0L * (s - s0) / (sigma * sigma);
    return acc;
}

static xreal xprofile_scale(int n, const xreal *S, const double *B, const double *cnt, xreal s0, xreal sigma,
                            int full_eq18, xreal *f_min)
{
    xreal s_hat;
    xreal lo = 0.0L, hi = 1.0L;
    if (!(xprofile_dfds(n, S, B, cnt, 0.0L, s0, sigma) < 0.0L)) {
        s_hat = 0.0L;                                  /* f increasing on s >= 0: boundary minimum */
    } else {
        int guard = 0;
        while (xprofile_dfds(n, S, B, cnt, hi, s0, sigma) < 0.0L && guard++ < 4000) { lo = hi; hi *= 2.0L; }
        for (int it = 0; it < 200; ++it) {
            xreal mid = 0.5L * (lo + hi);
            if (xprofile_dfds(n, S, B, cnt, mid, s0, sigma) < 0.0L) lo = mid; else hi = mid;
        }
        s_hat = 0.5L * (lo + hi);
    }
    xreal *mu = (xreal *)malloc(sizeof(xreal) * (size_t)(n > 0 ? n : 1));
    for (int j = 0; j < n; ++j) mu[j] = s_hat * S[j] + (xreal)B[j];
    xreal f = full_eq18 ? xeq18(n, mu, cnt) : xdeviance(n, mu, cnt);
    if (sigma > 0.0L) f += (s_hat - s0) * (s_hat - s0) / (sigma * sigma);
    free(mu);
    *f_min = f;
    return s_hat;
}

/* Stand-alone entry for the pins: S, B, cnt of length n. */
double orc_profile_scale(int n, const double *S, const double *B, const double *cnt, double s0, double sigma,
                         int full_eq18, double *f_min)
{
    xreal *xS = (xreal *)malloc(sizeof(xreal) * (size_t)(n > 0 ? n : 1));
    for (int j = 0; j < n; ++j) xS[j] = S[j];
    xreal f;
    xreal s = xprofile_scale(n, xS, B, cnt, s0, sigma, full_eq18, &f);
    free(xS);
    *f_min = (double)f;
    return (double)s;
}

/* Whole path with the normalisation profiled per point: steps a1-a3 as in orc_eval_batch (signal S = fold
 * without background, kept in long double), then orc_profile_scale over the bins of all periods.
 *   out [P] profiled -2lnL;  scale_out [P] s^;  abs_out NULL or [P] sum 2|term| at s^. */
int orc_eval_profile(const orc_consts *c, int n_E, const double *E, const double *flux_w,
                     const double *P_e, const double *P_mu, const double *P_tau,
                     int n_T, const double *T, int n_rec, int n_periods,
                     const double *N_mc, const double *R, const double *bkg, const double *counts,
                     int64_t P, int k, const int32_t *kinds, const double *params, double s0, double sigma,
                     double *out, double *scale_out, double *abs_out, int full_eq18, int nthreads)
{
    static const double zero[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
    for (int a = 0; a < k; ++a) {
        if (kinds[a] < 0 || kinds[a] >= ORC_N_KINDS) return -1;
        for (int b = 0; b < a; ++b) if (kinds[a] == kinds[b]) return -1;
    }
    xreal *S0 = (xreal *)malloc(sizeof(xreal) * (size_t)(n_T > 0 ? n_T : 1));
    xspectrum(c, n_E, E, flux_w, P_e, P_mu, P_tau, n_T, T, zero, S0);
    double *zero_bkg = (double *)calloc((size_t)(n_rec > 0 ? n_rec : 1), sizeof(double));
    if (nthreads < 1) nthreads = 1;
    const int nb = n_periods * n_rec;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int64_t p = 0; p < P; ++p) {
        double theta[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
        for (int a = 0; a < k; ++a) theta[kinds[a]] = params[p * k + a];
        xreal *Sp = (xreal *)malloc(sizeof(xreal) * (size_t)(2 * n_T + nb + 1));
        xreal *w = Sp + n_T, *sig = w + n_T;
        xspectrum(c, n_E, E, flux_w, P_e, P_mu, P_tau, n_T, T, theta, Sp);
        xweights(n_T, Sp, S0, w);
        for (int d = 0; d < n_periods; ++d)
            xfold(n_T, n_rec, w, N_mc + (size_t)d * n_T, R + (size_t)d * n_T * n_rec, zero_bkg, sig + (size_t)d * n_rec);
        xreal f;
        xreal s_hat = xprofile_scale(nb, sig, bkg, counts, s0, sigma, full_eq18, &f);
        out[p] = (double)f;
        if (scale_out) scale_out[p] = (double)s_hat;
        if (abs_out) {
            xreal tot = 0.0L;
            for (int j = 0; j < nb; ++j) {
                xreal mu = s_hat * sig[j] + (xreal)bkg[j];
                tot += fabsl(xdeviance(1, &mu, counts + j));
            }
            abs_out[p] = (double)tot;
        }
        free(Sp);
    }
    free(S0);
    free(zero_bkg);
    return 0;
}

/* Steps a3 + a4 for caller-supplied weights: Eq. (1), E_obs = R diag(r) E_true with an
 * arbitrary per-point weight vector r = w[p][.] (the case where a per-point nuisance -- oscillation
 * parameters, flux shape, PAPER.md:220 -- makes the weights something other than the spectrum
 * ratio of Eq. 14), then Eq. (18).  The same w is applied to every period's MC spectrum.
 *   w [P][n_T];  out [P];  mu_out NULL or [P][n_periods][n_rec];  abs_out NULL or [P]. */
int orc_eval_weights(int n_T, int n_rec, int n_periods, const double *N_mc, const double *R,
                     const double *bkg, const double *counts, int64_t P, const double *w,
                     double *out, double *mu_out, double *abs_out, int full_eq18, int nthreads)
{
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int64_t p = 0; p < P; ++p) {
        xreal *xw = (xreal *)malloc(sizeof(xreal) * (size_t)(n_T + n_rec + 1));
        xreal *mu = xw + n_T;
        for (int i = 0; i < n_T; ++i) xw[i] = (xreal)w[(size_t)p * n_T + i];
        xreal total = 0.0L, total_abs = 0.0L;
        for (int d = 0; d < n_periods; ++d) {
            const double *Cd = counts + (size_t)d * n_rec;
            xfold(n_T, n_rec, xw, N_mc + (size_t)d * n_T, R + (size_t)d * n_T * n_rec,
                  bkg + (size_t)d * n_rec, mu);
            total += full_eq18 ? xeq18(n_rec, mu, Cd) : xdeviance(n_rec, mu, Cd);
            if (mu_out)
                for (int q = 0; q < n_rec; ++q)
                    mu_out[((size_t)p * n_periods + d) * n_rec + q] = (double)mu[q];
            if (abs_out)
                for (int q = 0; q < n_rec; ++q) total_abs += fabsl(xdeviance(1, mu + q, Cd + q));
        }
        out[p] = (double)total;
        if (abs_out) abs_out[p] = (double)total_abs;
        free(xw);
    }
    return 0;
}

/* Several signal components (Eq. 17: mu_j = MT M_j sum_k rate_k f^(k)(j; eps); Sec. IV B a-b,
 * every neutrino component has its own flux, survival probability, recoil spectrum and
 * response).  The recoil bins of all components are concatenated along the contraction index: bin i belongs to
 * component comp_of_T[i], its spectrum (Eq. 12) and SM reference use that component's flux table
 * flux_w[comp][.], P_alpha[comp][.] on the shared E grid, its response rows are R[.][i][.], and a per-point
 * rate scale multiplies its reweighted MC content.  Parameter kinds 0..6 as orc_eval_batch; kind 7 + c is the
 * rate scale of component c (absent => 1).  n_comp <= 4. */
int orc_eval_components(const orc_consts *c, int n_E, const double *E, int n_comp, const double *flux_w,
                        const double *P_e, const double *P_mu, const double *P_tau,
                        int n_T, const double *T, const int32_t *comp_of_T, int n_rec, int n_periods,
                        const double *N_mc, const double *R, const double *bkg, const double *counts,
                        int64_t P, int k, const int32_t *kinds, const double *params,
                        double *out, double *mu_out, double *abs_out, int full_eq18, int nthreads)
{
    static const double zero[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
    if (n_comp < 1 || n_comp > 4) return -1;
    for (int a = 0; a < k; ++a) {
        if (kinds[a] < 0 || kinds[a] >= ORC_N_KINDS + n_comp) return -1;
        for (int b = 0; b < a; ++b) if (kinds[a] == kinds[b]) return -1;
    }
    for (int i = 0; i < n_T; ++i) if (comp_of_T[i] < 0 || comp_of_T[i] >= n_comp) return -1;
    size_t nT = (size_t)(n_T > 0 ? n_T : 1);
    xreal *S0 = (xreal *)malloc(sizeof(xreal) * nT * 2), *tmp0 = S0 + nT;
    for (int q = 0; q < n_comp; ++q) {      /* SM reference of every bin from its own component's table */
        xspectrum(c, n_E, E, flux_w + (size_t)q * n_E, P_e + (size_t)q * n_E, P_mu + (size_t)q * n_E,
                  P_tau + (size_t)q * n_E, n_T, T, zero, tmp0);
        for (int i = 0; i < n_T; ++i) if (comp_of_T[i] == q) S0[i] = tmp0[i];
    }
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int64_t p = 0; p < P; ++p) {
        double theta[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
        double rate[4] = {1.0, 1.0, 1.0, 1.0};
        for (int a = 0; a < k; ++a) {
            if (kinds[a] < ORC_N_KINDS) theta[kinds[a]] = params[p * k + a];
            else rate[kinds[a] - ORC_N_KINDS] = params[p * k + a];
        }
        xreal *S = (xreal *)malloc(sizeof(xreal) * (3 * nT + (size_t)n_rec + 1));
        xreal *tmp = S + nT, *w = tmp + nT, *mu = w + nT;
        for (int q = 0; q < n_comp; ++q) {
            xspectrum(c, n_E, E, flux_w + (size_t)q * n_E, P_e + (size_t)q * n_E, P_mu + (size_t)q * n_E,
                      P_tau + (size_t)q * n_E, n_T, T, theta, tmp);
            for (int i = 0; i < n_T; ++i) if (comp_of_T[i] == q) S[i] = tmp[i];
        }
        xweights(n_T, S, S0, w);
        for (int i = 0; i < n_T; ++i) w[i] *= (xreal)rate[comp_of_T[i]];      /* rate_k of Eq. (17) */
        xreal total = 0.0L, total_abs = 0.0L;
        for (int d = 0; d < n_periods; ++d) {
            const double *Cd = counts + (size_t)d * n_rec;
            xfold(n_T, n_rec, w, N_mc + (size_t)d * n_T, R + (size_t)d * n_T * n_rec, bkg + (size_t)d * n_rec, mu);
            total += full_eq18 ? xeq18(n_rec, mu, Cd) : xdeviance(n_rec, mu, Cd);
            if (mu_out)
                for (int q = 0; q < n_rec; ++q) mu_out[((size_t)p * n_periods + d) * n_rec + q] = (double)mu[q];
            if (abs_out)
                for (int q = 0; q < n_rec; ++q) total_abs += fabsl(xdeviance(1, mu + q, Cd + q));
        }
        out[p] = (double)total;
        if (abs_out) abs_out[p] = (double)total_abs;
        free(S);
    }
    free(S0);
    return 0;
}

/* Gradient of -2lnL with respect to the scanned parameters (for gradient-based minimisers; the paper fits
 * Eq. 18 with MIGRAD).  Written from the derivatives of the definitions:
 *   d/dgL of Eq. (4) bracket = 2 gL - gR m_e T/E^2,   d/dgR = 2 gR (1 - T/E)^2 - gL m_e T/E^2
 *   d/dmu_nu of Eq. (8) = 2 mu_nu (pi alpha^2/m_e^2)(1/T - 1/E)
 *   d mu_j = sum_i R_ij N_mc,i rate_c(i) dS_i/S_SM,i  (rate parameter: the component's own prediction / rate)
 *   d(-2lnL)/dtheta = sum_j 2 (1 - n_j/mu_j) dmu_j/dtheta                        (Eq. 18; n_j = 0: 2 dmu_j)
 * grad_out [P][k] in the order of `kinds`; out [P] as orc_eval_components. */
static xreal xdspectrum_bin(const orc_consts *c, int n_E, const double *E, const double *flux_w, const double *P_e,
                            const double *P_mu, const double *P_tau, double Ti, const double *theta, int kind)
{
    double gL0[3], gR0[3];
    orc_sm_couplings(c, gL0, gR0);
    const xreal pi = acosl(-1.0L);
    const xreal pref = 2.0L * (xreal)c->G_F * (xreal)c->G_F * (xreal)c->m_e / pi;
    const xreal pmm = pi * (xreal)c->alpha_em * (xreal)c->alpha_em / ((xreal)c->m_e * (xreal)c->m_e);
    xreal acc = 0.0L;
    for (int j = 0; j < n_E; ++j) {
        if (!(Ti <= orc_tmax(E[j], c->m_e))) continue;
        xreal Ej = E[j], T = Ti, d;
        if (kind == ORC_MU_NU) {
            d = 2.0L * (xreal)theta[ORC_MU_NU] * pmm * (1.0L / T - 1.0L / Ej);
        } else {
            const int fl = kind / 2;                       /* 0 e, 1 mu, 2 tau */
            const double *Pf = fl == 0 ? P_e : (fl == 1 ? P_mu : P_tau);
            xreal gL = (xreal)gL0[fl] + (xreal)theta[2 * fl], gR = (xreal)gR0[fl] + (xreal)theta[2 * fl + 1];
            xreal one_m = 1.0L - T / Ej, x = (xreal)c->m_e * T / (Ej * Ej);
            d = (kind % 2 == 0) ? (2.0L * gL - gR * x) : (2.0L * gR * one_m * one_m - gL * x);
            d *= pref * (xreal)Pf[j];
        }
        acc += (xreal)flux_w[j] * d;
    }
    return acc;
}

int orc_eval_grad(const orc_consts *c, int n_E, const double *E, int n_comp, const double *flux_w,
                  const double *P_e, const double *P_mu, const double *P_tau,
                  int n_T, const double *T, const int32_t *comp_of_T, int n_rec, int n_periods,
                  const double *N_mc, const double *R, const double *bkg, const double *counts,
                  int64_t P, int k, const int32_t *kinds, const double *params,
                  double *out, double *grad_out, int nthreads)
{
    static const double zero[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
    if (n_comp < 1 || n_comp > 4) return -1;
    for (int a = 0; a < k; ++a) {
        if (kinds[a] < 0 || kinds[a] >= ORC_N_KINDS + n_comp) return -1;
        for (int b = 0; b < a; ++b) if (kinds[a] == kinds[b]) return -1;
    }
    size_t nT = (size_t)(n_T > 0 ? n_T : 1);
    xreal *S0 = (xreal *)malloc(sizeof(xreal) * nT * 2), *tmp0 = S0 + nT;
    for (int q = 0; q < n_comp; ++q) {
        xspectrum(c, n_E, E, flux_w + (size_t)q * n_E, P_e + (size_t)q * n_E, P_mu + (size_t)q * n_E,
                  P_tau + (size_t)q * n_E, n_T, T, zero, tmp0);
        for (int i = 0; i < n_T; ++i) if (comp_of_T[i] == q) S0[i] = tmp0[i];
    }
    double *zero_bkg = (double *)calloc((size_t)(n_rec > 0 ? n_rec : 1), sizeof(double));
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int64_t p = 0; p < P; ++p) {
        double theta[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
        double rate[4] = {1.0, 1.0, 1.0, 1.0};
        for (int a = 0; a < k; ++a) {
            if (kinds[a] < ORC_N_KINDS) theta[kinds[a]] = params[p * k + a];
            else rate[kinds[a] - ORC_N_KINDS] = params[p * k + a];
        }
        xreal *S = (xreal *)malloc(sizeof(xreal) * (4 * nT + 2 * (size_t)n_rec * (size_t)n_periods + 2));
        xreal *tmp = S + nT, *w = tmp + nT, *dw = w + nT, *mu = dw + nT, *dmu = mu + (size_t)n_rec * n_periods;
        for (int q = 0; q < n_comp; ++q) {
            xspectrum(c, n_E, E, flux_w + (size_t)q * n_E, P_e + (size_t)q * n_E, P_mu + (size_t)q * n_E,
                      P_tau + (size_t)q * n_E, n_T, T, theta, tmp);
            for (int i = 0; i < n_T; ++i) if (comp_of_T[i] == q) S[i] = tmp[i];
        }
        xweights(n_T, S, S0, w);                           /* unscaled weights S_theta/S_SM (1 in dead bins) */
        for (int i = 0; i < n_T; ++i) tmp[i] = w[i] * (xreal)rate[comp_of_T[i]];
        xreal total = 0.0L;
        for (int d = 0; d < n_periods; ++d) {
            xfold(n_T, n_rec, tmp, N_mc + (size_t)d * n_T, R + (size_t)d * n_T * n_rec, bkg + (size_t)d * n_rec,
                  mu + (size_t)d * n_rec);
            total += xdeviance(n_rec, mu + (size_t)d * n_rec, counts + (size_t)d * n_rec);
        }
        out[p] = (double)total;
        for (int a = 0; a < k; ++a) {
            for (int i = 0; i < n_T; ++i) {
                const int q = comp_of_T[i];
                if (kinds[a] >= ORC_N_KINDS) {             /* rate of one component: its own unscaled content */
                    dw[i] = (q == kinds[a] - ORC_N_KINDS) ? w[i] : 0.0L;
                } else if (S0[i] == 0.0L) {
                    dw[i] = 0.0L;                          /* dead bin: w = 1 for every theta */
                } else {
                    dw[i] = (xreal)rate[q] * xdspectrum_bin(c, n_E, E, flux_w + (size_t)q * n_E, P_e + (size_t)q * n_E,
                                                            P_mu + (size_t)q * n_E, P_tau + (size_t)q * n_E, T[i],
                                                            theta, kinds[a]) / S0[i];
                }
            }
            xreal g = 0.0L;
            for (int d = 0; d < n_periods; ++d) {
                xfold(n_T, n_rec, dw, N_mc + (size_t)d * n_T, R + (size_t)d * n_T * n_rec, zero_bkg, dmu);
                for (int j = 0; j < n_rec; ++j) {
                    xreal m = mu[(size_t)d * n_rec + j], n = counts[(size_t)d * n_rec + j];
                    g += 2.0L * (n > 0.0L ? (1.0L - n / m) : 1.0L) * dmu[j];
                }
            }
            grad_out[p * k + a] = (double)g;
        }
        free(S);
    }
    free(S0);
    free(zero_bkg);
    return 0;
}

/* Per-point survival probabilities (the "physics update" of PAPER.md:220 evaluates the oscillation
 * probabilities for every parameter vector; here they arrive as a table P_e_pts[p][.] per point).  The MC sample
 * and the SM reference stay those of the nominal table P_e (the denominator is computed once), so
 *     w_i(p) = S_theta(T_i; P_e_pts[p]) / S_SM(T_i; P_e)          (Eq. 12 / Eq. 14; reading R16)
 * with P_mu, P_tau = (1 - P_e)(1 - f_tau), (1 - P_e) f_tau for the point's and the nominal table alike.  These
 * weights are not a low-rank function of theta: the dense fold is required.  Single component. */
int orc_eval_pee(const orc_consts *c, int n_E, const double *E, const double *flux_w, const double *P_e,
                 double f_tau, int n_T, const double *T, int n_rec, int n_periods,
                 const double *N_mc, const double *R, const double *bkg, const double *counts,
                 int64_t P, int k, const int32_t *kinds, const double *params, const double *P_e_pts,
                 double *out, double *mu_out, double *abs_out, int full_eq18, int nthreads)
{
    static const double zero[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
    for (int a = 0; a < k; ++a) {
        if (kinds[a] < 0 || kinds[a] >= ORC_N_KINDS) return -1;
        for (int b = 0; b < a; ++b) if (kinds[a] == kinds[b]) return -1;
    }
    size_t nE = (size_t)(n_E > 0 ? n_E : 1);
    double *Pm0 = (double *)malloc(sizeof(double) * 2 * nE), *Pt0 = Pm0 + nE;
    for (int j = 0; j < n_E; ++j) { Pm0[j] = (1.0 - P_e[j]) * (1.0 - f_tau); Pt0[j] = (1.0 - P_e[j]) * f_tau; }
    xreal *S0 = (xreal *)malloc(sizeof(xreal) * (size_t)(n_T > 0 ? n_T : 1));
    xspectrum(c, n_E, E, flux_w, P_e, Pm0, Pt0, n_T, T, zero, S0);
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int64_t p = 0; p < P; ++p) {
        double theta[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
        for (int a = 0; a < k; ++a) theta[kinds[a]] = params[p * k + a];
        const double *Pp = P_e_pts + (size_t)p * n_E;
        double *Pm = (double *)malloc(sizeof(double) * 2 * nE), *Pt = Pm + nE;
        for (int j = 0; j < n_E; ++j) { Pm[j] = (1.0 - Pp[j]) * (1.0 - f_tau); Pt[j] = (1.0 - Pp[j]) * f_tau; }
        xreal *S = (xreal *)malloc(sizeof(xreal) * (size_t)(2 * n_T + n_rec + 1));
        xreal *w = S + n_T, *mu = w + n_T;
        xspectrum(c, n_E, E, flux_w, Pp, Pm, Pt, n_T, T, theta, S);
        xweights(n_T, S, S0, w);
        xreal total = 0.0L, total_abs = 0.0L;
        for (int d = 0; d < n_periods; ++d) {
            const double *Cd = counts + (size_t)d * n_rec;
            xfold(n_T, n_rec, w, N_mc + (size_t)d * n_T, R + (size_t)d * n_T * n_rec, bkg + (size_t)d * n_rec, mu);
            total += full_eq18 ? xeq18(n_rec, mu, Cd) : xdeviance(n_rec, mu, Cd);
            if (mu_out)
                for (int q = 0; q < n_rec; ++q) mu_out[((size_t)p * n_periods + d) * n_rec + q] = (double)mu[q];
            if (abs_out)
                for (int q = 0; q < n_rec; ++q) total_abs += fabsl(xdeviance(1, mu + q, Cd + q));
        }
        out[p] = (double)total;
        if (abs_out) abs_out[p] = (double)total_abs;
        free(S);
        free(Pm);
    }
    free(S0);
    free(Pm0);
    return 0;
}

/* Per-point survival probabilities with several signal components and / or explicit nominal nu_mu, nu_tau tables
 * (Eq. 17, on top of the per-point physics update of PAPER.md:220).  P_e_pts[p][q][.] is the nu_e
 * survival probability of point p for component q on the shared E grid.  The paper does not say how the rest,
 * 1 - P_e, of a point is shared between nu_mu and nu_tau when the analysis was set up with explicit tables:
 * DESIGN.md reading R17 keeps the nominal tables' mu : tau ratio at every energy,
 *     P_mu^p(E) = (1 - P_e^p(E)) P_mu(E) / (P_mu(E) + P_tau(E)),   P_tau^p likewise
 * (where P_mu + P_tau = 0, and when no explicit tables were given: the f_tau split of reading R3).  The SM reference of
 * a bin is computed from the NOMINAL tables of its component (reading R16).  Single-component calls without
 * explicit tables reduce to orc_eval_pee. */
int orc_eval_pee_components(const orc_consts *c, int n_E, const double *E, int n_comp, const double *flux_w,
                            const double *P_e, const double *P_mu, const double *P_tau, int have_mu_tau, double f_tau,
                            int n_T, const double *T, const int32_t *comp_of_T, int n_rec, int n_periods,
                            const double *N_mc, const double *R, const double *bkg, const double *counts,
                            int64_t P, int k, const int32_t *kinds, const double *params, const double *P_e_pts,
                            double *out, double *mu_out, double *abs_out, int full_eq18, int nthreads)
{
    static const double zero[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
    if (n_comp < 1 || n_comp > 4) return -1;
    for (int a = 0; a < k; ++a) {
        if (kinds[a] < 0 || kinds[a] >= ORC_N_KINDS) return -1;
        for (int b = 0; b < a; ++b) if (kinds[a] == kinds[b]) return -1;
    }
    for (int i = 0; i < n_T; ++i) if (comp_of_T[i] < 0 || comp_of_T[i] >= n_comp) return -1;
    size_t nT = (size_t)(n_T > 0 ? n_T : 1), nE = (size_t)(n_E > 0 ? n_E : 1);
    /* nominal nu_mu / nu_tau tables (given, or the f_tau split) and the share rho of 1 - P_e each flavour takes */
    double *Pm0 = (double *)malloc(sizeof(double) * 4 * nE * (size_t)n_comp);
    double *Pt0 = Pm0 + nE * n_comp, *rho_m = Pt0 + nE * n_comp, *rho_t = rho_m + nE * n_comp;
    for (size_t j = 0; j < nE * (size_t)n_comp; ++j) {
        if (have_mu_tau) { Pm0[j] = P_mu[j]; Pt0[j] = P_tau[j]; }
        else { Pm0[j] = (1.0 - P_e[j]) * (1.0 - f_tau); Pt0[j] = (1.0 - P_e[j]) * f_tau; }
        double sum = Pm0[j] + Pt0[j];
        if (have_mu_tau && sum > 0.0) { rho_m[j] = Pm0[j] / sum; rho_t[j] = Pt0[j] / sum; }
        else { rho_m[j] = 1.0 - f_tau; rho_t[j] = f_tau; }
    }
    xreal *S0 = (xreal *)malloc(sizeof(xreal) * nT * 2), *tmp0 = S0 + nT;
    for (int q = 0; q < n_comp; ++q) {
        xspectrum(c, n_E, E, flux_w + (size_t)q * n_E, P_e + (size_t)q * n_E, Pm0 + (size_t)q * n_E,
                  Pt0 + (size_t)q * n_E, n_T, T, zero, tmp0);
        for (int i = 0; i < n_T; ++i) if (comp_of_T[i] == q) S0[i] = tmp0[i];
    }
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int64_t p = 0; p < P; ++p) {
        double theta[ORC_N_KINDS] = {0, 0, 0, 0, 0, 0, 0};
        for (int a = 0; a < k; ++a) theta[kinds[a]] = params[p * k + a];
        double *Pm = (double *)malloc(sizeof(double) * 2 * nE), *Pt = Pm + nE;
        xreal *S = (xreal *)malloc(sizeof(xreal) * (3 * nT + (size_t)n_rec + 1));
        xreal *tmp = S + nT, *w = tmp + nT, *mu = w + nT;
        for (int q = 0; q < n_comp; ++q) {
            const double *Pp = P_e_pts + ((size_t)p * n_comp + q) * n_E;
            for (int j = 0; j < n_E; ++j) {
                Pm[j] = (1.0 - Pp[j]) * rho_m[(size_t)q * n_E + j];
                Pt[j] = (1.0 - Pp[j]) * rho_t[(size_t)q * n_E + j];
            }
            xspectrum(c, n_E, E, flux_w + (size_t)q * n_E, Pp, Pm, Pt, n_T, T, theta, tmp);
            for (int i = 0; i < n_T; ++i) if (comp_of_T[i] == q) S[i] = tmp[i];
        }
        xweights(n_T, S, S0, w);
        xreal total = 0.0L, total_abs = 0.0L;
        for (int d = 0; d < n_periods; ++d) {
            const double *Cd = counts + (size_t)d * n_rec;
            xfold(n_T, n_rec, w, N_mc + (size_t)d * n_T, R + (size_t)d * n_T * n_rec, bkg + (size_t)d * n_rec, mu);
            total += full_eq18 ? xeq18(n_rec, mu, Cd) : xdeviance(n_rec, mu, Cd);
            if (mu_out)
                for (int q = 0; q < n_rec; ++q) mu_out[((size_t)p * n_periods + d) * n_rec + q] = (double)mu[q];
            if (abs_out)
                for (int q = 0; q < n_rec; ++q) total_abs += fabsl(xdeviance(1, mu + q, Cd + q));
        }
        out[p] = (double)total;
        if (abs_out) abs_out[p] = (double)total_abs;
        free(S);
        free(Pm);
    }
    free(S0);
    free(Pm0);
    return 0;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
