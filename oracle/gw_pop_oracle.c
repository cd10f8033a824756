/*
 * gw_pop_oracle.c -- CPU oracle of the population ("recycling") likelihood.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, section IV):
 *
 *   Eq. 3:   L_tot({d_i} | Lambda, R)  proportional to  R^N e^{-R VT(Lambda)}
 *                                                       prod_{i=1..N} sum_{j=1..n_i} p(theta_ij | Lambda) / p(theta_ij | 0)
 *
 * with theta_ij the j-th posterior sample of event i, p(theta | 0) the prior the single-event analysis sampled with
 * and p(theta | Lambda) the population model.  The paper's own benchmark ignores VT ("For
 * the benchmarking performed in this work, we ignore this quantity") and draws an equal number n of samples per event
 * ("a single N x n_i array"); the rate R enters only through the dropped prefactor.  So the oracle
 * returns, Eq. 3 taken literally without that prefactor,
 *
 *   ln L(Lambda) = sum_i ln [ sum_j p(theta_ij | Lambda) / p(theta_ij | 0) ]
 *
 * (the Monte-Carlo mean 1/n would add the constant -N ln n; Eq. 3 prints none; reading P2).
 *
 * PAPER.md names the population models only by citation (mass [37], spin magnitude [39], spin tilt
 * [33]) and prints no formula.  The closed forms below are the reading DESIGN.md section 14 takes (P1): literature
 * forms restated, each normalised in closed form:
 *
 *   theta  = (m1, q, a1, a2, c1, c2): primary mass [Msun], mass ratio m2/m1 in (0,1], spin magnitudes in [0,1],
 *            cosines of the two spin tilts in [-1,1].
 *   Lambda = (alpha, m_min, m_max, lam, m_pp, sig_pp, beta_q, alpha_chi, beta_chi, xi, sig_1, sig_2).
 *
 *   mass   p(m1)      = (1 - lam) PL(m1; -alpha, [m_min, m_max]) + lam TN(m1; m_pp, sig_pp, [m_min, m_max])
 *                       ("power law + peak", no low-mass smoothing), zero outside [m_min, m_max];
 *   ratio  p(q | m1)  = (1 + beta_q) q^beta_q / (1 - (m_min/m1)^(1+beta_q))   for m_min/m1 <= q <= 1, else zero;
 *   spin   p(a)       = a^(alpha_chi-1) (1-a)^(beta_chi-1) / B(alpha_chi, beta_chi)   (Beta distribution), iid a1, a2;
 *   tilt   p(c1, c2)  = (1 - xi)/4 + xi TN(c1; 1, sig_1, [-1,1]) TN(c2; 1, sig_2, [-1,1])
 *                       (isotropic + preferentially aligned mixture).
 *
 *   PL(x; -alpha, [lo,hi]) = x^-alpha / int_lo^hi t^-alpha dt;  TN = normal density truncated and renormalised.
 *
 * The oracle writes every density in its natural form (pow, exp, erf, lgamma of libm), one factor after the other, sums
 * over j and over i in index order with Neumaier compensation, and shares no code with the CUDA path (which works on
 * precomputed logarithms and merged exponents).  fp64 throughout.  Pins: tests/test_oracle_population.py.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call this.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { T_M1 = 0, T_Q, T_A1, T_A2, T_C1, T_C2, GWPO_NTHETA = 6 };
enum { L_ALPHA = 0, L_MMIN, L_MMAX, L_LAM, L_MPP, L_SIGPP, L_BETAQ, L_ACHI, L_BCHI, L_XI, L_SIG1, L_SIG2, GWPO_NLAMBDA = 12 };

#define GWPO_PI 3.14159265358979323846

/* normalised power law x^-alpha on [lo, hi] */
double gwpo_powerlaw_pdf(double x, double alpha, double lo, double hi)
{
    if (!(x >= lo && x <= hi)) return 0.0;
    double norm;
    if (fabs(1.0 - alpha) < 1e-12) norm = log(hi / lo);
    else                           norm = (pow(hi, 1.0 - alpha) - pow(lo, 1.0 - alpha)) / (1.0 - alpha);
    return pow(x, -alpha) / norm;
}

/* normal density N(mu, sigma) truncated to [lo, hi] and renormalised */
double gwpo_truncnorm_pdf(double x, double mu, double sigma, double lo, double hi)
{
    if (!(x >= lo && x <= hi)) return 0.0;
    const double z = (x - mu) / sigma;
    const double gauss = exp(-0.5 * z * z) / (sigma * sqrt(2.0 * GWPO_PI));
    const double cdf_hi = 0.5 * (1.0 + erf((hi - mu) / (sigma * sqrt(2.0))));
    const double cdf_lo = 0.5 * (1.0 + erf((lo - mu) / (sigma * sqrt(2.0))));
    return gauss / (cdf_hi - cdf_lo);
}

/* primary mass: power law + Gaussian peak on [m_min, m_max] */
double gwpo_mass_pdf(double m1, const double *L)
{
    const double pl = gwpo_powerlaw_pdf(m1, L[L_ALPHA], L[L_MMIN], L[L_MMAX]);
    const double pk = gwpo_truncnorm_pdf(m1, L[L_MPP], L[L_SIGPP], L[L_MMIN], L[L_MMAX]);
    return (1.0 - L[L_LAM]) * pl + L[L_LAM] * pk;
}

/* mass ratio given the primary mass: power law q^beta on [m_min/m1, 1] */
double gwpo_ratio_pdf(double q, double m1, const double *L)
{
    const double qlo = L[L_MMIN] / m1;
    if (!(qlo < 1.0)) return 0.0;                 /* m1 <= m_min: no room for a secondary */
    return gwpo_powerlaw_pdf(q, -L[L_BETAQ], qlo, 1.0);
}

/* spin magnitude: Beta(alpha_chi, beta_chi) on [0, 1] */
double gwpo_beta_pdf(double a, double alpha_chi, double beta_chi)
{
    if (!(a >= 0.0 && a <= 1.0)) return 0.0;
    const double ln_b = lgamma(alpha_chi) + lgamma(beta_chi) - lgamma(alpha_chi + beta_chi);
    return pow(a, alpha_chi - 1.0) * pow(1.0 - a, beta_chi - 1.0) / exp(ln_b);
}

/* spin tilts: isotropic + aligned mixture on [-1, 1]^2 */
double gwpo_tilt_pdf(double c1, double c2, const double *L)
{
    if (!(c1 >= -1.0 && c1 <= 1.0 && c2 >= -1.0 && c2 <= 1.0)) return 0.0;
    const double aligned = gwpo_truncnorm_pdf(c1, 1.0, L[L_SIG1], -1.0, 1.0) * gwpo_truncnorm_pdf(c2, 1.0, L[L_SIG2], -1.0, 1.0);
    return (1.0 - L[L_XI]) * 0.25 + L[L_XI] * aligned;
}

/* 1 if Lambda is inside the model's domain */
int gwpo_lambda_valid(const double *L)
{
    for (int k = 0; k < GWPO_NLAMBDA; ++k) if (!isfinite(L[k])) return 0;
    return L[L_MMIN] > 0.0 && L[L_MMAX] > L[L_MMIN] && L[L_LAM] >= 0.0 && L[L_LAM] <= 1.0 && L[L_SIGPP] > 0.0 &&
           L[L_ACHI] > 0.0 && L[L_BCHI] > 0.0 && L[L_XI] >= 0.0 && L[L_XI] <= 1.0 && L[L_SIG1] > 0.0 && L[L_SIG2] > 0.0;
}

/* p(theta | Lambda): the product of the four factors */
double gwpo_population_pdf(const double *theta, const double *L)
{
    const double pm = gwpo_mass_pdf(theta[T_M1], L);
    const double pq = gwpo_ratio_pdf(theta[T_Q], theta[T_M1], L);
    const double pa = gwpo_beta_pdf(theta[T_A1], L[L_ACHI], L[L_BCHI]) * gwpo_beta_pdf(theta[T_A2], L[L_ACHI], L[L_BCHI]);
    const double pt = gwpo_tilt_pdf(theta[T_C1], theta[T_C2], L);
    return pm * pq * pa * pt;
}

static void neumaier_add(double *sum, double *comp, double x)
{
    const double t = *sum + x;
    if (fabs(*sum) >= fabs(x)) *comp += (*sum - t) + x;
    else                       *comp += (x - t) + *sum;
    *sum = t;
}

/* Eq. 3 without the R^N e^{-R VT} prefactor:  lnl[b] = sum_i ln sum_j p(theta_ij | Lambda_b) / prior_ij.
 * samples [n_events][n_samples][6], prior [n_events][n_samples] (> 0), lambdas [n_lambda][12];
 * per_event (nullable) [n_lambda][n_events] receives the inner sums.  An invalid Lambda gives NaN; an event whose
 * samples all have zero weight gives -inf.  Returns the threads used.                                             */
int gwpo_lnl(int64_t n_events, int64_t n_samples, const double *samples, const double *prior, int64_t n_lambda,
             const double *lambdas, int n_threads, double *lnl, double *per_event)
{
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
#endif
    const int64_t n_work = n_lambda * n_events;
    double *inner = (double *)malloc(sizeof(double) * (size_t)(n_work > 0 ? n_work : 1));
    if (!inner) return -1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t w = 0; w < n_work; ++w) {
        const int64_t b = w / n_events, i = w % n_events;
        const double *L = lambdas + b * GWPO_NLAMBDA;
        double s = 0.0, c = 0.0;
        if (!gwpo_lambda_valid(L)) { inner[w] = NAN; continue; }
        for (int64_t j = 0; j < n_samples; ++j) {
            const double *th = samples + (i * n_samples + j) * GWPO_NTHETA;
            neumaier_add(&s, &c, gwpo_population_pdf(th, L) / prior[i * n_samples + j]);
        }
        inner[w] = s + c;
    }
    for (int64_t b = 0; b < n_lambda; ++b) {
        double s = 0.0, c = 0.0;
        int empty = 0, bad = 0;                   /* an event without support: ln 0 = -inf; an invalid Lambda: NaN */
        for (int64_t i = 0; i < n_events; ++i) {
            const double v = inner[b * n_events + i];
            if (per_event) per_event[b * n_events + i] = v;
            if (v != v) bad = 1;
            else if (v == 0.0) empty = 1;
            else neumaier_add(&s, &c, log(v));
        }
        lnl[b] = bad ? NAN : (empty ? -INFINITY : s + c);
    }
    free(inner);
    return used;
}
