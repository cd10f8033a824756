/*
 * gw_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` leg may build, load or call this file.  The CUDA library
 * (paper_1904_02863_b200/csrc) shares no code, header, table or constant
 * generator with it, and neither includes nor links the other.
 *
 * What it is: the plain definition of the single-event hot path, written out
 * bin by bin in IEEE fp64 with libm, no blocking, no fusion, no reordering:
 *
 *   lnL(theta) = sum_det [ Re<d|h(theta)> - 1/2 <h(theta)|h(theta)> ],
 *   <a|b>      = 4 df sum_f a(f) conj(b(f)) / S_n(f)
 *
 * which is the theta-dependent part of the paper's Eq. 1 (PAPER.md line 63,
 * section III: exponent -(2/T)|d-h|^2/S = -1/2 * 4 df |d-h|^2/S with df=1/T);
 * the frequency-domain time shift exp(-2 i pi f dt_det) is PAPER.md line 69,
 * section III; "the template for the response of the detector" is PAPER.md
 * line 65.  PAPER.md gives no formula for the waveform; BASELINE.json's
 * north_star fixes it to the TaylorF2 stationary-phase inspiral (3.5PN phase,
 * Newtonian amplitude, aligned spins at 1.5PN spin-orbit and 2PN spin-spin),
 * written out here in the notation of SURVEY.md section 8(c), steps O1..O7,
 * and of DESIGN.md section 3 (the readings A1..A20).
 *
 * Arithmetic: every function below uses the "v-form" of the phase,
 *   v = (pi M f)^(1/3),  Psi = ... + 3/(128 eta) v^-5 sum_k (phi_k + phil_k ln v) v^k,
 * with libm cbrt/pow/log/cexp, one bin at a time.  (The CUDA path uses a
 * different algebraic form, tables in f^(1/3) and a Horner scheme in turns; a
 * transcription slip in one cannot hide in the other.)  Sums over bins are
 * Neumaier-compensated, in ascending bin order.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): phi_k rationals
 * and anchors (P1a), stationary-phase re-derivation from the 3.5PN energy and
 * flux (P1b), Newtonian chirp time (P1c), two codings of the spin terms
 * (P1d), <h|h> closed form and quadrature (P2), d=0 / noiseless identities and
 * Cauchy-Schwarz (P3), shift identities (P4), antenna-pattern invariants and a
 * closed-form special case (P5), light-travel-time bounds (P6), 40-digit
 * mpmath spot values (P7), a hand-expanded tiny case (P8), bin independence
 * (P9); the tidal option (NEXT-1): Lambda~ form against the per-body form, re-derivation from the tidal
 * energy and flux, equal-mass special case, 40-digit spot values (P10, tests/test_oracle_tidal.py); spin_order 2:
 * re-derivation of the 2.5/3/3.5PN spin-orbit terms from the spin-orbit energy and flux, (chi_s, chi_a) coding,
 * special cases (P11, tests/test_oracle_spin35.py).
 * The digits of the H1/L1/V1 geometry are input data, not oracle
 * arithmetic; they are pinned by invariants only.
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- constants (SURVEY.md 8(c) "Constants": all from exactly defined values) ---- */
#define GWO_PI      3.14159265358979323846
#define GWO_C_SI    299792458.0                       /* m/s, exact                     */
#define GWO_GMSUN   1.3271244e20                      /* m^3/s^2, IAU 2015 nominal      */
#define GWO_AU      149597870700.0                    /* m, exact                       */
#define GWO_EULER   0.57721566490153286061            /* Euler-Mascheroni               */

static double gwo_tsun(void)  { return GWO_GMSUN / (GWO_C_SI * GWO_C_SI * GWO_C_SI); }  /* s   */
static double gwo_mpc_s(void) { return 1.0e6 * (648000.0 / GWO_PI) * GWO_AU / GWO_C_SI; } /* s */

/* theta layout: the GW_P_* order of SURVEY.md 8(b) (restated, not included) */
enum { T_MC = 0, T_Q, T_CHI1, T_CHI2, T_DL, T_TC, T_PHIC, T_COSI, T_RA, T_DEC, T_PSI, T_N = 11 };

/* detector row layout used by this oracle (13 doubles; its own, not the library's struct):
 *   [0] kind (0 geometric, 1 fixed)   [1..3] vertex r (m)   [4..6] x arm   [7..9] y arm
 *   [10] F+ (fixed)   [11] Fx (fixed)   [12] dt (fixed, s)                                  */
enum { D_KIND = 0, D_VTX = 1, D_XARM = 4, D_YARM = 7, D_FP = 10, D_FC = 11, D_DT = 12, D_N = 13 };

void gwo_constants(double *out4)
{
    out4[0] = gwo_tsun();
    out4[1] = gwo_mpc_s();
    out4[2] = GWO_C_SI;
    out4[3] = GWO_EULER;
}

/* ---- O1: masses -------------------------------------------------------------------- */
/* q = m2/m1 in (0,1]; eta = q/(1+q)^2; M = Mc eta^(-3/5); M_s = M T_sun; mu1 = 1/(1+q), mu2 = q/(1+q). */
void gwo_masses(double mc_msun, double q, double *eta, double *mtot_s, double *mu1, double *mu2)
{
    *eta    = q / ((1.0 + q) * (1.0 + q));
    *mtot_s = mc_msun * pow(*eta, -3.0 / 5.0) * gwo_tsun();
    *mu1    = 1.0 / (1.0 + q);
    *mu2    = q / (1.0 + q);
}

/* ---- O2: TaylorF2 phase coefficients (readings A5, A7, A8) ---- */
/* phi[k] multiplies v^k, phil[k] multiplies v^k ln v, k = 0..7; phi[1] = 0.
 * spin_order 0: beta = sigma = 0;  1: 1.5PN spin-orbit beta and 2PN spin-spin sigma;
 * 2 (NEXT-1 option, reading A22): in addition the spin-orbit terms
 *   linear in the spins at 2.5PN, 3PN and 3.5PN, in the variables
 *     S_l = mu1^2 chi1 + mu2^2 chi2,   dS_l = (mu1 - mu2)(mu2 chi2 - mu1 chi1):
 *     gamma   = (554345/1134 + 110/9 eta) S_l + (13915/84 - 10/3 eta) dS_l
 *     phi_5  -= gamma,  phil_5 -= 3 gamma
 *     phi_6  += pi (3760 S_l + 1490 dS_l)/3
 *     phi_7  += (-8980424995/762048 + 6586595/756 eta - 305/36 eta^2) S_l
 *               - (170978035/48384 - 2876425/672 eta - 4735/144 eta^2) dS_l
 *   (terms quadratic in the spins beyond 2PN are not included).                              */
void gwo_phase_coefficients(double eta, double mu1, double mu2, double chi1, double chi2,
                            int spin_order, double *phi, double *phil)
{
    const double pi = GWO_PI;
    double beta = 0.0, sigma = 0.0;
    if (spin_order >= 1) {
        beta  = (113.0 / 12.0 * mu1 * mu1 + 25.0 / 4.0 * eta) * chi1
              + (113.0 / 12.0 * mu2 * mu2 + 25.0 / 4.0 * eta) * chi2;
        sigma = 79.0 / 8.0 * eta * chi1 * chi2
              + 81.0 / 16.0 * (mu1 * mu1 * chi1 * chi1 + mu2 * mu2 * chi2 * chi2);
    }
    for (int k = 0; k < 8; ++k) { phi[k] = 0.0; phil[k] = 0.0; }
    phi[0] = 1.0;
    phi[2] = 3715.0 / 756.0 + 55.0 / 9.0 * eta;
    phi[3] = -16.0 * pi + 4.0 * beta;
    phi[4] = 15293365.0 / 508032.0 + 27145.0 / 504.0 * eta + 3085.0 / 72.0 * eta * eta - 10.0 * sigma;
    phi[5] = pi * (38645.0 / 756.0 - 65.0 / 9.0 * eta);
    phil[5] = 3.0 * pi * (38645.0 / 756.0 - 65.0 / 9.0 * eta);
    phi[6] = 11583231236531.0 / 4694215680.0 - 640.0 / 3.0 * pi * pi - 6848.0 / 21.0 * GWO_EULER
           + eta * (-15737765635.0 / 3048192.0 + 2255.0 / 12.0 * pi * pi)
           + 76055.0 / 1728.0 * eta * eta - 127825.0 / 1296.0 * eta * eta * eta
           - 6848.0 / 21.0 * log(4.0);
    phil[6] = -6848.0 / 21.0;
    phi[7] = pi * (77096675.0 / 254016.0 + 378515.0 / 1512.0 * eta - 74045.0 / 756.0 * eta * eta);
    if (spin_order >= 2) {
        const double sl  = mu1 * mu1 * chi1 + mu2 * mu2 * chi2;
        const double dsl = (mu1 - mu2) * (mu2 * chi2 - mu1 * chi1);
        const double gamma = (554345.0 / 1134.0 + 110.0 / 9.0 * eta) * sl + (13915.0 / 84.0 - 10.0 / 3.0 * eta) * dsl;
        phi[5]  -= gamma;
        phil[5] -= 3.0 * gamma;
        phi[6]  += pi * (3760.0 * sl + 1490.0 * dsl) / 3.0;
        phi[7]  += (-8980424995.0 / 762048.0 + 6586595.0 / 756.0 * eta - 305.0 / 36.0 * eta * eta) * sl
                 - (170978035.0 / 48384.0 - 2876425.0 / 672.0 * eta - 4735.0 / 144.0 * eta * eta) * dsl;
    }
}

/* ---- NEXT-1 option: tidal phase terms ------------------------ */
/* Point-mass TaylorF2 plus the adiabatic quadrupolar tidal terms, for the neutron-star workloads C2/C3
 * (the paper's motivation includes the neutron-star equation of state; the formula is not in
 * PAPER.md -- literature closed form, reading A21).  With Lambda_A = (2/3) k2_A (R_A/m_A)^5 the dimensionless
 * tidal deformability of body A (body 1 is the heavier one, q = m2/m1 <= 1),
 *   Lambda~  = (8/13) [ (1 + 7 eta - 31 eta^2)(L1 + L2) + sqrt(1-4 eta)(1 + 9 eta - 11 eta^2)(L1 - L2) ]
 *   dLambda~ = (1/2) [ sqrt(1-4 eta)(1 - 13272/1319 eta + 8944/1319 eta^2)(L1 + L2)
 *                     + (1 - 15910/1319 eta + 32850/1319 eta^2 + 3380/1319 eta^3)(L1 - L2) ]
 *   phi_10 = -(39/2) Lambda~                                            (5PN, tidal_order >= 1)
 *   phi_12 = -(3115/64) Lambda~ + (6595/364) sqrt(1-4 eta) dLambda~     (6PN, tidal_order >= 2)
 * in the same units as phi_0..phi_7: Psi += 3/(128 eta) v^-5 (phi_10 v^10 + phi_12 v^12).
 * tidal_order 0: both are zero.                                                                     */
void gwo_tidal_coefficients(double eta, double lambda1, double lambda2, int tidal_order,
                            double *phi10, double *phi12)
{
    *phi10 = 0.0;
    *phi12 = 0.0;
    if (tidal_order <= 0) return;
    const double root = sqrt(fmax(0.0, 1.0 - 4.0 * eta));
    const double ls = lambda1 + lambda2, la = lambda1 - lambda2;
    const double lam_t = 8.0 / 13.0 * ((1.0 + 7.0 * eta - 31.0 * eta * eta) * ls
                                       + root * (1.0 + 9.0 * eta - 11.0 * eta * eta) * la);
    const double dlam_t = 0.5 * (root * (1.0 - 13272.0 / 1319.0 * eta + 8944.0 / 1319.0 * eta * eta) * ls
                                 + (1.0 - 15910.0 / 1319.0 * eta + 32850.0 / 1319.0 * eta * eta
                                    + 3380.0 / 1319.0 * eta * eta * eta) * la);
    *phi10 = -39.0 / 2.0 * lam_t;
    if (tidal_order >= 2) *phi12 = -3115.0 / 64.0 * lam_t + 6595.0 / 364.0 * root * dlam_t;
}

/* ---- O3: phase at one frequency ------------------------------------------------------- */
/* Psi(f) = 2 pi f t_c - phi_c - pi/4 + 3/(128 eta) v^-5 sum_k (phi_k + phil_k ln v) v^k,
 * v = (pi M_s f)^(1/3).  No cut-off at f_ISCO (reading A6).
 * The per-proposal quantities (eta, M_s, phi_k, phil_k) do not depend on f; callers that loop
 * over bins compute them once per proposal and pass them in.                                 */
typedef struct {
    double eta, mtot_s, phi[8], phil[8], tc, phic;
    double phi10, phi12;          /* tidal option; zero otherwise */
} gwo_source;

static gwo_source source_of(const double *theta, int spin_order)
{
    gwo_source s;
    double mu1, mu2;
    gwo_masses(theta[T_MC], theta[T_Q], &s.eta, &s.mtot_s, &mu1, &mu2);
    gwo_phase_coefficients(s.eta, mu1, mu2, theta[T_CHI1], theta[T_CHI2], spin_order, s.phi, s.phil);
    s.tc = theta[T_TC];
    s.phic = theta[T_PHIC];
    s.phi10 = 0.0;
    s.phi12 = 0.0;
    return s;
}

/* the same with the tidal option: lambdas = (Lambda_1, Lambda_2) of this proposal, or NULL */
static gwo_source source_of_tidal(const double *theta, int spin_order, const double *lambdas, int tidal_order)
{
    gwo_source s = source_of(theta, spin_order);
    if (lambdas && tidal_order > 0)
        gwo_tidal_coefficients(s.eta, lambdas[0], lambdas[1], tidal_order, &s.phi10, &s.phi12);
    return s;
}

static double phase_of(const gwo_source *s, double f)
{
    double v   = cbrt(GWO_PI * s->mtot_s * f);
    double lnv = log(v);
    double series = 0.0, vk = 1.0;                 /* vk = v^k */
    for (int k = 0; k < 8; ++k) {
        series += (s->phi[k] + s->phil[k] * lnv) * vk;
        vk *= v;
    }
    if (s->phi10 != 0.0 || s->phi12 != 0.0)        /* tidal option: v^10 and v^12 terms */
        series += s->phi10 * pow(v, 10.0) + s->phi12 * pow(v, 12.0);
    return 2.0 * GWO_PI * f * s->tc - s->phic - GWO_PI / 4.0
         + 3.0 / (128.0 * s->eta) * pow(v, -5.0) * series;
}

double gwo_phase(double f, const double *theta, int spin_order)
{
    gwo_source s = source_of(theta, spin_order);
    return phase_of(&s, f);
}

double gwo_phase_tidal(double f, const double *theta, int spin_order, const double *lambdas, int tidal_order)
{
    gwo_source s = source_of_tidal(theta, spin_order, lambdas, tidal_order);
    return phase_of(&s, f);
}

/* ---- NEXT-1 option: inspiral cut-off ---------------------- */
/* f_ISCO = 1 / (6^(3/2) pi M_s): the gravitational-wave frequency of the innermost stable circular orbit of
 * a Schwarzschild hole of the total mass; with isco_cut the template is zero for f > f_ISCO (bins with
 * f <= f_ISCO are kept).  Off by default (reading A6).                                                 */
double gwo_f_isco(double mc_msun, double q)
{
    double eta, mtot_s, mu1, mu2;
    gwo_masses(mc_msun, q, &eta, &mtot_s, &mu1, &mu2);
    return 1.0 / (6.0 * sqrt(6.0) * GWO_PI * mtot_s);
}

/* ---- O4: Newtonian amplitude ------------------------------------------------------------ */
/* A0 = sqrt(5/24) pi^(-2/3) (Mc T_sun)^(5/6) / (D Mpc/c)   [s^(-1/6)];  h0(f) = A0 f^(-7/6) exp(-i Psi). */
double gwo_amplitude(double mc_msun, double dl_mpc)
{
    return sqrt(5.0 / 24.0) * pow(GWO_PI, -2.0 / 3.0) * pow(mc_msun * gwo_tsun(), 5.0 / 6.0)
         / (dl_mpc * gwo_mpc_s());
}

/* ---- O6: antenna patterns and geocentric delay -------------------------------------------- */
static double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* a^T D b with D = (x (x) x - y (x) y)/2 */
static double bilinear_D(const double *xarm, const double *yarm, const double *a, const double *b)
{
    return 0.5 * (dot3(a, xarm) * dot3(xarm, b) - dot3(a, yarm) * dot3(yarm, b));
}

void gwo_antenna(const double *det, double ra, double dec, double psi, double gmst,
                 double *fplus, double *fcross, double *dt_s)
{
    if (det[D_KIND] != 0.0) {          /* FIXED response (config C0) */
        *fplus = det[D_FP]; *fcross = det[D_FC]; *dt_s = det[D_DT];
        return;
    }
    const double g = gmst - ra;
    const double X[3] = { -cos(psi) * sin(g) - sin(psi) * cos(g) * sin(dec),
                          -cos(psi) * cos(g) + sin(psi) * sin(g) * sin(dec),
                           sin(psi) * cos(dec) };
    const double Y[3] = {  sin(psi) * sin(g) - cos(psi) * cos(g) * sin(dec),
                           sin(psi) * cos(g) + cos(psi) * sin(g) * sin(dec),
                           cos(psi) * cos(dec) };
    const double *xa = det + D_XARM, *ya = det + D_YARM;
    *fplus  = bilinear_D(xa, ya, X, X) - bilinear_D(xa, ya, Y, Y);
    *fcross = bilinear_D(xa, ya, X, Y) + bilinear_D(xa, ya, Y, X);
    const double n[3] = { cos(dec) * cos(ra - gmst), cos(dec) * sin(ra - gmst), sin(dec) };
    *dt_s = -dot3(det + D_VTX, n) / GWO_C_SI;      /* reading A13 */
}

/* exposes X, Y, n for the orthonormality pins (P5) */
void gwo_sky_frame(double ra, double dec, double psi, double gmst, double *X, double *Y, double *n)
{
    const double g = gmst - ra;
    X[0] = -cos(psi) * sin(g) - sin(psi) * cos(g) * sin(dec);
    X[1] = -cos(psi) * cos(g) + sin(psi) * sin(g) * sin(dec);
    X[2] =  sin(psi) * cos(dec);
    Y[0] =  sin(psi) * sin(g) - cos(psi) * cos(g) * sin(dec);
    Y[1] =  sin(psi) * cos(g) + cos(psi) * sin(g) * sin(dec);
    Y[2] =  cos(psi) * cos(dec);
    n[0] = cos(dec) * cos(ra - gmst);
    n[1] = cos(dec) * sin(ra - gmst);
    n[2] = sin(dec);
}

/* ---- O4..O6: detector-frame waveform at one (theta, detector, frequency) ------------------- */
/* h_I(f) = [F+ 1/2(1+cos^2 i) - i Fx cos i] * A0 f^(-7/6) exp(-i Psi(f)) * exp(-2 pi i f dt_I) */
static double complex h_det_at(double f, const gwo_source *src, double cosi,
                               double a0, double fplus, double fcross, double dt_s, double f_cut)
{
    if (f_cut > 0.0 && f > f_cut) return 0.0;      /* NEXT-1 option isco_cut: h = 0 above f_ISCO */
    double complex h0     = a0 * pow(f, -7.0 / 6.0) * cexp(CMPLX(0.0, -phase_of(src, f)));    /* O4 */
    double complex hplus  = 0.5 * (1.0 + cosi * cosi) * h0;                 /* O5 */
    double complex hcross = CMPLX(0.0, -cosi) * h0;                         /* O5 */
    double complex shift  = cexp(CMPLX(0.0, -2.0 * GWO_PI * f * dt_s));
    return (fplus * hplus + fcross * hcross) * shift;
}

/* h_out[n_prop][n_det][n_bins][2] (re, im) */
/* lambdas: NULL, or [n_prop][2] = (Lambda_1, Lambda_2) per proposal, used when tidal_order > 0 */
void gwo_waveform_tidal(int64_t n_bins, const double *freqs, int n_det, const double *dets, double gmst,
                        int64_t n_prop, const double *theta, int spin_order, int isco_cut,
                        const double *lambdas, int tidal_order, double *h_out)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t b = 0; b < n_prop; ++b) {
        const double *th = theta + b * T_N;
        const double a0 = gwo_amplitude(th[T_MC], th[T_DL]);
        const gwo_source src = source_of_tidal(th, spin_order, lambdas ? lambdas + 2 * b : NULL, tidal_order);
        const double f_cut = isco_cut ? gwo_f_isco(th[T_MC], th[T_Q]) : 0.0;
        for (int i = 0; i < n_det; ++i) {
            double fp, fc, dt;
            gwo_antenna(dets + (size_t)i * D_N, th[T_RA], th[T_DEC], th[T_PSI], gmst, &fp, &fc, &dt);
            double *row = h_out + (((size_t)b * n_det + i) * (size_t)n_bins) * 2;
            for (int64_t j = 0; j < n_bins; ++j) {
                double complex h = h_det_at(freqs[j], &src, th[T_COSI], a0, fp, fc, dt, f_cut);
                row[2 * j]     = creal(h);
                row[2 * j + 1] = cimag(h);
            }
        }
    }
}

/* Neumaier-compensated accumulation: (sum, comp) += x */
static void neumaier_add(double *sum, double *comp, double x)
{
    double t = *sum + x;
    if (fabs(*sum) >= fabs(x)) *comp += (*sum - t) + x;
    else                       *comp += (x - t) + *sum;
    *sum = t;
}

/* ---- O7: inner products and lnL -------------------------------------------------------------- */
/* data_ri[n_det][n_bins][2], psd[n_det][n_bins]; lnl[n_prop]; parts[n_prop][n_det][3] =
 * (Re<d|h>, Im<d|h>, <h|h>) (parts may be NULL).  n_threads <= 0: OpenMP default.
 * Returns the number of threads the proposal loop used.                                        */
int gwo_lnl_tidal(int64_t n_bins, const double *freqs, double delta_f, int n_det,
                  const double *data_ri, const double *psd, const double *dets, double gmst,
                  int64_t n_prop, const double *theta, int spin_order, int isco_cut,
                  const double *lambdas, int tidal_order, int n_threads, double *lnl, double *parts)
{
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
    used = omp_get_max_threads();
    if ((int64_t)used > n_prop) used = (int)(n_prop > 0 ? n_prop : 1);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t b = 0; b < n_prop; ++b) {
        const double *th = theta + b * T_N;
        const double a0 = gwo_amplitude(th[T_MC], th[T_DL]);
        const gwo_source src = source_of_tidal(th, spin_order, lambdas ? lambdas + 2 * b : NULL, tidal_order);
        const double f_cut = isco_cut ? gwo_f_isco(th[T_MC], th[T_Q]) : 0.0;
        double total = 0.0;
        for (int i = 0; i < n_det; ++i) {
            double fp, fc, dt;
            gwo_antenna(dets + (size_t)i * D_N, th[T_RA], th[T_DEC], th[T_PSI], gmst, &fp, &fc, &dt);
            const double *d = data_ri + ((size_t)i * (size_t)n_bins) * 2;
            const double *S = psd + (size_t)i * (size_t)n_bins;
            double dh_re = 0, dh_re_c = 0, dh_im = 0, dh_im_c = 0, hh = 0, hh_c = 0;
            for (int64_t j = 0; j < n_bins; ++j) {
                double complex h  = h_det_at(freqs[j], &src, th[T_COSI], a0, fp, fc, dt, f_cut);
                double complex dj = CMPLX(d[2 * j], d[2 * j + 1]);
                double complex t  = dj * conj(h) / S[j];
                neumaier_add(&dh_re, &dh_re_c, creal(t));
                neumaier_add(&dh_im, &dh_im_c, cimag(t));
                neumaier_add(&hh, &hh_c, (creal(h) * creal(h) + cimag(h) * cimag(h)) / S[j]);
            }
            const double dh_r = 4.0 * delta_f * (dh_re + dh_re_c);
            const double dh_i = 4.0 * delta_f * (dh_im + dh_im_c);
            const double h_h  = 4.0 * delta_f * (hh + hh_c);
            if (parts) {
                double *p = parts + ((size_t)b * n_det + i) * 3;
                p[0] = dh_r; p[1] = dh_i; p[2] = h_h;
            }
            total += dh_r - 0.5 * h_h;
        }
        lnl[b] = total;
    }
    return used;
}

/* the point-mass entry points (no tidal terms) */
void gwo_waveform_opt(int64_t n_bins, const double *freqs, int n_det, const double *dets, double gmst,
                      int64_t n_prop, const double *theta, int spin_order, int isco_cut, double *h_out)
{
    gwo_waveform_tidal(n_bins, freqs, n_det, dets, gmst, n_prop, theta, spin_order, isco_cut, NULL, 0, h_out);
}
int gwo_lnl_opt(int64_t n_bins, const double *freqs, double delta_f, int n_det,
                const double *data_ri, const double *psd, const double *dets, double gmst,
                int64_t n_prop, const double *theta, int spin_order, int isco_cut, int n_threads,
                double *lnl, double *parts)
{
    return gwo_lnl_tidal(n_bins, freqs, delta_f, n_det, data_ri, psd, dets, gmst, n_prop, theta, spin_order,
                         isco_cut, NULL, 0, n_threads, lnl, parts);
}

/* the default (no cut-off) entry points, as pinned by tests/test_oracle_*.py */
void gwo_waveform(int64_t n_bins, const double *freqs, int n_det, const double *dets, double gmst,
                  int64_t n_prop, const double *theta, int spin_order, double *h_out)
{
    gwo_waveform_opt(n_bins, freqs, n_det, dets, gmst, n_prop, theta, spin_order, 0, h_out);
}
int gwo_lnl(int64_t n_bins, const double *freqs, double delta_f, int n_det,
            const double *data_ri, const double *psd, const double *dets, double gmst,
            int64_t n_prop, const double *theta, int spin_order, int n_threads,
            double *lnl, double *parts)
{
    return gwo_lnl_opt(n_bins, freqs, delta_f, n_det, data_ri, psd, dets, gmst, n_prop, theta, spin_order, 0,
                       n_threads, lnl, parts);
}

/* ---- NEXT-1 option: likelihood marginalised over the coalescence phase --------------------------------- */
/* h depends on phi_c only through the factor exp(+i phi_c) (O3/O4), so with a uniform prior on phi_c
 *   L_marg = (1/2 pi) int_0^{2 pi} exp( Re[ e^{-i phi} sum_I <d|h>_I ] - 1/2 sum_I <h|h>_I ) d phi
 *          = I0(|sum_I <d|h>_I|) exp(-1/2 sum_I <h|h>_I),
 * where <d|h>_I is evaluated at any phi_c.  ln I0 is computed from its integral definition
 *   I0(x) = (1/pi) int_0^pi exp(x cos t) dt  =>  ln I0(x) = x + ln[(1/pi) int_0^pi exp(x (cos t - 1)) dt]
 * by the trapezoid rule on n points (exponentially convergent for this periodic, even integrand; n is chosen
 * from x so that the Gaussian peak of width ~1/sqrt(x) is resolved).                                       */
double gwo_log_bessel_i0(double x)
{
    x = fabs(x);
    long n = 64 + (long)(64.0 * sqrt(x));                 /* >= 64 points per peak width */
    if (n > 4000000) n = 4000000;
    double s = 0, c = 0;
    for (long k = 0; k <= n; ++k) {
        double t = GWO_PI * (double)k / (double)n;
        double w = (k == 0 || k == n) ? 0.5 : 1.0;
        neumaier_add(&s, &c, w * exp(x * (cos(t) - 1.0)));
    }
    return x + log((s + c) / (double)n);
}

/* lnl_marg[b] = ln I0(|sum_I (parts[b][I][0] + i parts[b][I][1])|) - 1/2 sum_I parts[b][I][2] */
void gwo_lnl_phase_marginal(int64_t n_prop, int n_det, const double *parts, double *lnl_marg)
{
    for (int64_t b = 0; b < n_prop; ++b) {
        double re = 0, im = 0, hh = 0;
        for (int i = 0; i < n_det; ++i) {
            const double *p = parts + ((size_t)b * n_det + i) * 3;
            re += p[0]; im += p[1]; hh += p[2];
        }
        lnl_marg[b] = gwo_log_bessel_i0(hypot(re, im)) - 0.5 * hh;
    }
}

/* generic noise-weighted inner product <a|b> = 4 df sum a conj(b)/S for one detector (pins P3) */
void gwo_inner(int64_t n_bins, double delta_f, const double *a_ri, const double *b_ri,
               const double *psd, double *out_re, double *out_im)
{
    double re = 0, re_c = 0, im = 0, im_c = 0;
    for (int64_t j = 0; j < n_bins; ++j) {
        double complex a = CMPLX(a_ri[2 * j], a_ri[2 * j + 1]);
        double complex b = CMPLX(b_ri[2 * j], b_ri[2 * j + 1]);
        double complex t = a * conj(b) / psd[j];
        neumaier_add(&re, &re_c, creal(t));
        neumaier_add(&im, &im_c, cimag(t));
    }
    *out_re = 4.0 * delta_f * (re + re_c);
    *out_im = 4.0 * delta_f * (im + im_c);
}

/* I7 = 4 df sum_j f_j^(-7/3) / S_j : the phase-independent norm of pin P2 */
double gwo_norm_i7(int64_t n_bins, const double *freqs, double delta_f, const double *psd)
{
    double s = 0, c = 0;
    for (int64_t j = 0; j < n_bins; ++j)
        neumaier_add(&s, &c, pow(freqs[j], -7.0 / 3.0) / psd[j]);
    return 4.0 * delta_f * (s + c);
}
