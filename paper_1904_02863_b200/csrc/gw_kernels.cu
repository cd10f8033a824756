// gw_kernels.cu -- the CUDA kernels of the hot path (sm_100a) and their launchers.
//
//   K0 precompute_kernel / norm_kernel : per-bin tables, once per context       (DESIGN.md 6.K0; a0)
//   K1 setup_kernel                    : theta_b -> per-proposal record         (DESIGN.md 6.K1; a1)
//   K2 waveform_kernel                 : complex128 h(f) to HBM                 (DESIGN.md 6.K2; a6)
//   K3 fused_kernel                    : phase + projection + <d|h>, fixed-order finish (6.K3; a2..a5)
//
// Phase convention: everything is carried in units of 1/kPhaseScale turns (quarter turns).  With x = f^(1/3), L = ln f
// and the per-bin basis b = (x^-5, x^-3, x^-2, x^-1, L, x, xL, x^2),
//     Phi'(f) = c5 + c0 b0 + c2 b1 + c3 b2 + c4 b3 + cL5 b4 + c6 b5 + cL6 b6 + c7 b7          [turns]
// is the TaylorF2 phase WITHOUT the 2 pi f t_c term; t_c is merged with the detector delay,
// tau_I = t_c + dt_I.  The waveform kernel adds f tau_I per detector.  The fused kernel adds f tau_0 (detector
// 0 is the time reference) and applies the remaining exp(+2 pi i f (tau_I - tau_0)), I >= 1, by a Horner-style
// recurrence on the uniform grid.  Shares nothing with oracle/.
#include <cmath>
#include <cstdio>

#include "gw_internal.h"
#include "gw_math.cuh"

namespace gw {

// =====================================================================================================
// K0: per-bin precompute (north_star item (2))
// =====================================================================================================
__global__ void precompute_kernel(int64_t n_bins, int64_t n_pad, int n_det, double f0, double delta_f,
                                  const double *__restrict__ freqs, const double *__restrict__ data_ri,
                                  const double *__restrict__ psd, double *__restrict__ planes)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_pad) return;
    double2 *pl = reinterpret_cast<double2 *>(planes);
    if (j < n_bins) {
        const double f   = freqs[j];
        const double x   = cbrt(f);
        const double xi  = 1.0 / x;
        const double fi  = 1.0 / f;
        const double xm2 = xi * xi;
        const double L   = log(f);
        pl[0 * n_pad + j] = make_double2(fi * xm2, fi);      // x^-5, x^-3
        pl[1 * n_pad + j] = make_double2(xm2, xi);           // x^-2, x^-1
        pl[2 * n_pad + j] = make_double2(L, x);              // ln f, x
        pl[3 * n_pad + j] = make_double2(x * L, x * x);      // x ln f, x^2
        const double a = 1.0 / (f * sqrt(x));                // f^(-7/6)
        pl[4 * n_pad + j] = make_double2(f, a);              // f, f^(-7/6)
        for (int i = 0; i < n_det; ++i) {
            const double w  = 4.0 * delta_f / psd[(int64_t)i * n_bins + j];
            const double wa = w * a;
            const double *d = data_ri + ((int64_t)i * n_bins + j) * 2;
            pl[(int64_t)(kBasisPlanes + i) * n_pad + j] = make_double2(wa * d[0], wa * d[1]);
        }
    } else {                                                 // padding: finite and inert
        pl[0 * n_pad + j] = make_double2(1.0, 1.0);
        pl[1 * n_pad + j] = make_double2(1.0, 1.0);
        pl[2 * n_pad + j] = make_double2(0.0, 1.0);
        pl[3 * n_pad + j] = make_double2(0.0, 1.0);
        pl[4 * n_pad + j] = make_double2(f0 + (double)j * delta_f, 0.0);
        for (int i = 0; i < n_det; ++i) pl[(int64_t)(kBasisPlanes + i) * n_pad + j] = make_double2(0.0, 0.0);
    }
}

// I7_I = sum_j (4 df / S_Ij) f_j^(-7/3): one CTA per detector, compensated per-thread sums over a fixed
// strided slice, then a fixed shared-memory tree (deterministic).
__global__ void __launch_bounds__(1024) norm_kernel(int64_t n_bins, double delta_f,
                                                    const double *__restrict__ psd,
                                                    const double2 *__restrict__ f_amp, double *__restrict__ i7)
{
    __shared__ double sh[1024];
    const int i = blockIdx.x;
    double s = 0.0, c = 0.0;
    for (int64_t j = threadIdx.x; j < n_bins; j += 1024) {
        const double a = f_amp[j].y;                          // f^(-7/6)
        const double v = (4.0 * delta_f / psd[(int64_t)i * n_bins + j]) * (a * a);
        const double t = s + v;                               // terms are positive: |s| >= |v| after the first
        c += (fabs(s) >= fabs(v)) ? ((s - t) + v) : ((v - t) + s);
        s = t;
    }
    sh[threadIdx.x] = s + c;
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) i7[i] = sh[0];
}

// isco_cut only: inclusive prefix sums cum[i][j] = sum_{k <= j} (4 df / S_Ik) f_k^(-7/3).  One CTA per detector;
// each thread sums a contiguous slice, the slice totals are scanned in thread order by one thread, and the
// slice is swept again: the order of additions is fixed by (M, 1024) alone.
__global__ void __launch_bounds__(1024) norm_cum_kernel(int64_t n_bins, int64_t n_pad, double delta_f,
                                                        const double *__restrict__ psd,
                                                        const double2 *__restrict__ f_amp, double *__restrict__ cum)
{
    __shared__ double sh[1024];
    const int i = blockIdx.x, t = threadIdx.x;
    const int64_t len = (n_bins + 1023) / 1024;
    const int64_t lo = (int64_t)t * len, hi = (lo + len < n_bins) ? lo + len : n_bins;
    double s = 0.0;
    for (int64_t j = lo; j < hi; ++j) {
        const double a = f_amp[j].y;
        s += (4.0 * delta_f / psd[(int64_t)i * n_bins + j]) * (a * a);
    }
    sh[t] = s;
    __syncthreads();
    if (t == 0) {
        double run = 0.0;
        for (int k = 0; k < 1024; ++k) { const double v = sh[k]; sh[k] = run; run += v; }   // exclusive scan
    }
    __syncthreads();
    double run = sh[t];
    for (int64_t j = lo; j < hi; ++j) {
        const double a = f_amp[j].y;
        run += (4.0 * delta_f / psd[(int64_t)i * n_bins + j]) * (a * a);
        cum[(int64_t)i * n_pad + j] = run;
    }
}

cudaError_t launch_precompute(const Tables &t, const double *freqs_dev, const double *data_dev,
                              const double *psd_dev, double *i7_dev, cudaStream_t s, int64_t *launches)
{
    const int threads = 256;
    const unsigned blocks = (unsigned)((t.n_pad + threads - 1) / threads);
    precompute_kernel<<<blocks, threads, 0, s>>>(t.n_bins, t.n_pad, t.n_det, t.f0, t.delta_f, freqs_dev,
                                                 data_dev, psd_dev, t.planes);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    norm_kernel<<<t.n_det, 1024, 0, s>>>(t.n_bins, t.delta_f, psd_dev,
                                         reinterpret_cast<const double2 *>(t.planes) + 4 * t.n_pad, i7_dev);
    *launches += 2;
    if (t.isco_cut) {
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        norm_cum_kernel<<<t.n_det, 1024, 0, s>>>(t.n_bins, t.n_pad, t.delta_f, psd_dev,
                                                 reinterpret_cast<const double2 *>(t.planes) + 4 * t.n_pad, t.i7cum);
        *launches += 1;
    }
    return cudaGetLastError();
}

// =====================================================================================================
// K1: per-proposal setup (step a1).  Four warps share 32 proposals by role; record fields are stored SoA
// (rec[field * rec_stride + b]) so that the thread-per-proposal kernels read them coalesced.
//   fields 0..8 : c0 c2 c3 c4 c5 cL5 c6 cL6 c7    (phase coefficients in turns, see file header)
//   per detector I (base 9 + 5 I): tau_I = t_c + dt_I ; CA_I = A0 * C_I (re, im) ;
//                                  rot_I = exp(-2 pi i rot_stride_hz tau_I) (re, im)
// An out-of-domain theta poisons CA with NaN (boundary contract in gwlnl.h).
// =====================================================================================================
struct SetupArgs {
    DetSet  dets;
    double  gmst;
    int     n_det, spin_order;
    int     n_param, tidal_order;   // doubles per theta row; NEXT-1 tidal option (0 | 1 | 2)
    int     stage_theta;            // 1: theta is pinned host memory read in place (stage rows through shared memory)
    int     isco_cut;               // 0: f_ISCO and the cut index are not needed
    double  band_xi, band_x1, band_l1;   // f_min^(-1/3), f_max^(1/3), max |ln f| at the band edges (phase-domain bound)
    double  max_dt;                      // max_I |dt_I| over the detectors [s]: the phase carries f (t_c + dt_I)
    int64_t n_prop, rec_stride;
    const double *theta;
    double *rec;
    double  rot_stride_hz;
    int     relative_tau;     // 1: tau_I (I >= 1) and rot_I are relative to detector 0 (fused kernel); 0: absolute
    const double2 *f_amp;     // basis plane 4: (f_j, f_j^-7/6), for the f_ISCO bin search
    int64_t n_bins;
    double  f0, delta_f, f_max;
};

// A CTA of 128 threads serves 32 proposals; warp w takes role w for proposal (block*32 + lane), so the four
// parts of the record are computed concurrently and no warp diverges:
//   role 0: masses and the nine phase coefficients (O1-O3)
//   role 1..3: amplitude, sky frame and the detector block(s) (O4-O6): role r takes detector r-1, and role 3
//              also detector 3 when n_det = 4.  Each detector role recomputes the (cheap) amplitude and frame.
__global__ void __launch_bounds__(128) setup_kernel(const SetupArgs a)
{
    pdl_launch_dependents();          // the dependent kernel may start its table prefetch now
    // Host variant with a pinned theta buffer (stage_theta): the CTA's 32 rows are contiguous, so they are staged with
    // coalesced loads over the host link (one pass over the rows) and every role reads its columns from shared
    // memory.  Device-resident theta is read directly (the staging round trip would cost ~1 us per call).
    __shared__ double s_theta[32 * GW_NPARAM_TIDAL];
    if (a.stage_theta) {
        const int64_t b_first = (int64_t)blockIdx.x * 32;
        const int64_t rows = a.n_prop - b_first < 32 ? a.n_prop - b_first : 32;
        const int n_load = (int)rows * a.n_param;
        const double *src = a.theta + b_first * a.n_param;
        for (int i = threadIdx.x; i < n_load; i += 128) s_theta[i] = src[i];
        __syncthreads();
    }
    const int role = threadIdx.x >> 5;
    const int64_t b = (int64_t)blockIdx.x * 32 + (threadIdx.x & 31);
    if (b >= a.n_prop) return;
    const double *th = a.stage_theta ? s_theta + (threadIdx.x & 31) * a.n_param : a.theta + b * a.n_param;
    double *r = a.rec + b;
    const int64_t S = a.rec_stride;
    const double mc = th[GW_P_MC];

    if (role == 0) {
        const double q = th[GW_P_Q], chi1 = th[GW_P_CHI1], chi2 = th[GW_P_CHI2], phic = th[GW_P_PHIC];
        // O1: masses.  kappa = (pi M)^(1/3) = (pi Mc)^(1/3) eta^(-1/5)
        const double opq   = 1.0 + q;
        const double eta   = q / (opq * opq);
        const double delta = (1.0 - q) / opq;                    // mu1 - mu2
        const double kc    = cbrt(kPi * mc * kTsun);             // (pi Mc)^(1/3): the 0PN term depends on Mc only
        const double ln_eta = log(eta);
        const double kap   = kc * exp(-0.2 * ln_eta);
        const double lnk   = log(kc) - 0.2 * ln_eta;
        const double ikap  = 1.0 / kap;
        // O2: phase coefficients; spin terms in the chi_s / chi_a coding
        double four_beta = 0.0, m10_sigma = 0.0;
        if (a.spin_order >= 1) {
            const double xs = 0.5 * (chi1 + chi2), xa = 0.5 * (chi1 - chi2);
            four_beta = (113.0 / 3.0 - 76.0 / 3.0 * eta) * xs + 113.0 / 3.0 * delta * xa;
            m10_sigma = (-405.0 / 8.0 + 2.5 * eta) * xs * xs + (-405.0 / 8.0 + 200.0 * eta) * xa * xa -
                        405.0 / 4.0 * delta * xs * xa;
        }
        const double eta2 = eta * eta;
        const double phi2 = 3715.0 / 756.0 + 55.0 / 9.0 * eta;
        const double phi3 = -16.0 * kPi + four_beta;
        const double phi4 = 15293365.0 / 508032.0 + 27145.0 / 504.0 * eta + 3085.0 / 72.0 * eta2 + m10_sigma;
        // NEXT-1 option spin_order 2: spin-orbit terms linear in the spins at 2.5PN, 3PN, 3.5PN, in the
        // (chi_s, chi_a) coding:  S_l = (1 - 2 eta) chi_s + delta chi_a,  dS_l = -(1 - 4 eta) chi_s - delta chi_a
        double so5 = 0.0, so6 = 0.0, so7 = 0.0;
        if (a.spin_order >= 2) {
            const double xs = 0.5 * (chi1 + chi2), xa = 0.5 * (chi1 - chi2);
            const double sl  = (1.0 - 2.0 * eta) * xs + delta * xa;
            const double dsl = -(1.0 - 4.0 * eta) * xs - delta * xa;
            so5 = -((554345.0 / 1134.0 + 110.0 / 9.0 * eta) * sl + (13915.0 / 84.0 - 10.0 / 3.0 * eta) * dsl);
            so6 = kPi * (3760.0 * sl + 1490.0 * dsl) / 3.0;
            so7 = (-8980424995.0 / 762048.0 + eta * (6586595.0 / 756.0 - 305.0 / 36.0 * eta)) * sl -
                  (170978035.0 / 48384.0 - eta * (2876425.0 / 672.0 + 4735.0 / 144.0 * eta)) * dsl;
        }
        const double phi5 = kPi * (38645.0 / 756.0 - 65.0 / 9.0 * eta) + so5;
        const double ph5l = 3.0 * phi5;
        constexpr double k6const = 11583231236531.0 / 4694215680.0 - 640.0 / 3.0 * kPi * kPi -
                                   6848.0 / 21.0 * (kEulerG + kLn4);
        const double phi6 = k6const + eta * (-15737765635.0 / 3048192.0 + 2255.0 / 12.0 * kPi * kPi) +
                            76055.0 / 1728.0 * eta2 - 127825.0 / 1296.0 * eta2 * eta + so6;
        constexpr double ph6l = -6848.0 / 21.0;
        const double phi7 = kPi * (77096675.0 / 254016.0 + 378515.0 / 1512.0 * eta - 74045.0 / 756.0 * eta2) + so7;
        // x-form, in turns: prefactor 3/(128 eta) / (2 pi); kappa^(k-5) x^(k-5)
        const double pref = 3.0 / (128.0 * eta) / kTwoPi;
        const double kc2  = kc * kc;
        const double ik2  = ikap * ikap;
        r[0 * S] = kPhaseScale * ((3.0 / 128.0 / kTwoPi) / (kc2 * kc2 * kc));                       // c0  * x^-5
        r[1 * S] = kPhaseScale * (pref * phi2 * ik2 * ikap);                                        // c2  * x^-3
        r[2 * S] = kPhaseScale * (pref * phi3 * ik2);                                               // c3  * x^-2
        r[3 * S] = kPhaseScale * (pref * phi4 * ikap);                                              // c4  * x^-1
        r[4 * S] = kPhaseScale * (pref * (phi5 + ph5l * lnk) - (phic + 0.25 * kPi) / kTwoPi);       // c5  (constant)
        r[5 * S] = kPhaseScale * (pref * ph5l / 3.0);                                               // cL5 * ln f
        r[6 * S] = kPhaseScale * (pref * kap * (phi6 + ph6l * lnk));                                // c6  * x
        r[7 * S] = kPhaseScale * (pref * kap * ph6l / 3.0);                                         // cL6 * x ln f
        r[8 * S] = kPhaseScale * (pref * kap * kap * phi7);                                         // c7  * x^2
        // NEXT-1 option tidal_order: 5PN and 6PN adiabatic tidal terms in the per-body coding,
        //   phi_10 = -sum_A 24 (12 - 11 X_A) X_A^4 Lambda_A,
        //   phi_12 = -sum_A (5/28)(3179 - 919 X_A - 2286 X_A^2 + 260 X_A^3) X_A^4 Lambda_A,   X_A = m_A / M,
        // as coefficients of x^5 and x^7 (v = kappa x).  Lambda_A must be finite and >= 0.
        double t10 = 0.0, t12 = 0.0;
        bool tidal_ok = true;
        if (a.tidal_order >= 1) {
            const double lam[2] = {th[GW_P_LAMBDA1], th[GW_P_LAMBDA2]};
            const double X[2]   = {1.0 / opq, q / opq};
            double p10 = 0.0, p12 = 0.0;
#pragma unroll
            for (int A = 0; A < 2; ++A) {
                const double x = X[A], x2 = x * x, w = x2 * x2 * lam[A];
                p10 -= 24.0 * (12.0 - 11.0 * x) * w;
                p12 -= (5.0 / 28.0) * (3179.0 + x * (-919.0 + x * (-2286.0 + x * 260.0))) * w;
                tidal_ok = tidal_ok && (lam[A] >= 0.0) && isfinite(lam[A]);
            }
            const double k2 = kap * kap, k5 = k2 * k2 * kap;
            t10 = kPhaseScale * (pref * p10 * k5);                                                  // t10 * x^5
            if (a.tidal_order >= 2) t12 = kPhaseScale * (pref * p12 * k5 * k2);                     // t12 * x^7
        }
        r[(int64_t)rec_field_t10(a.n_det) * S] = t10;
        r[(int64_t)rec_field_t12(a.n_det) * S] = t12;
        {   // domain of the integer range reduction (cis_quarter_turns: |phase| < 2^31 quarter turns): bound the
            // phase over the band by its terms at the band edges; beyond 1e9 phase units the proposal is poisoned
            const double xi = a.band_xi, x1 = a.band_x1, l1 = a.band_l1, tc = th[GW_P_TC];
            const double bound = fabs(r[0 * S]) * (xi * xi) * (xi * xi) * xi + fabs(r[1 * S]) * (xi * xi * xi) +
                                 fabs(r[2 * S]) * (xi * xi) + fabs(r[3 * S]) * xi + fabs(r[4 * S]) +
                                 fabs(r[5 * S]) * l1 + fabs(r[6 * S]) * x1 + fabs(r[7 * S]) * x1 * l1 +
                                 fabs(r[8 * S]) * x1 * x1 + kPhaseScale * (fabs(tc) + a.max_dt + 1.0) * a.f_max +
                                 (fabs(t10) + fabs(t12) * x1 * x1) * (x1 * x1) * (x1 * x1) * x1;
            if (!(bound < 1.0e9) || !tidal_ok) r[4 * S] = __longlong_as_double(0x7ff8000000000000LL);
        }
        // NEXT-1 option isco_cut: f_ISCO = 1/(6^(3/2) pi M) and the last bin with f_j <= f_ISCO (-1: none).
        // The decision is taken in fp64 against the same f_j the oracle compares with.
        if (!a.isco_cut) return;                                                    // the two fields are read by nobody
        const double f_isco = 1.0 / (6.0 * sqrt(6.0) * (kap * kap * kap));         // kappa^3 = pi M
        double jc = floor((f_isco - a.f0) / a.delta_f);
        int64_t j = jc < -1.0 ? -1 : (jc > (double)(a.n_bins - 1) ? a.n_bins - 1 : (int64_t)jc);
        while (j + 1 < a.n_bins && a.f_amp[j + 1].x <= f_isco) ++j;
        while (j >= 0 && a.f_amp[j].x > f_isco) --j;
        if (!(f_isco == f_isco)) j = -1;                                            // NaN masses: nothing kept
        r[(int64_t)rec_field_fisco(a.n_det) * S] = f_isco;
        r[(int64_t)rec_field_jcut(a.n_det) * S]  = (double)j;
        return;
    }

    // ---- detector roles ----
    const int i_first = role - 1;
    const int i_last  = (role == 3 && a.n_det > 3) ? a.n_det - 1 : i_first;
    if (i_first >= a.n_det) return;
    const double q = th[GW_P_Q], chi1 = th[GW_P_CHI1], chi2 = th[GW_P_CHI2];
    const double dl = th[GW_P_DL], tc = th[GW_P_TC], phic = th[GW_P_PHIC], cosi = th[GW_P_COSI];
    const double ra = th[GW_P_RA], dec = th[GW_P_DEC], psi = th[GW_P_PSI];
    bool ok = (mc > 0.0) && (q > 0.0) && (q <= 1.0) && (dl > 0.0) && (fabs(cosi) <= 1.0) &&
              (fabs(chi1) <= 1.0) && (fabs(chi2) <= 1.0);
    ok = ok && isfinite(mc) && isfinite(dl) && isfinite(tc) && isfinite(phic) && isfinite(ra) &&
         isfinite(dec) && isfinite(psi);

    // O4: Newtonian amplitude A0 = sqrt(5/24) pi^(-2/3) (Mc Tsun)^(5/6) / (D Mpc/c)
    const double u  = mc * kTsun;
    constexpr double kAmp = 0.212787510139663399157865621657;      // sqrt(5/24) pi^(-2/3)
    double a0 = kAmp * (sqrt(u) * cbrt(u)) / (dl * kMpcSec);
    if (!ok) a0 = __longlong_as_double(0x7ff8000000000000LL);

    // O6: sky frame
    double sg, cg, sd, cd, sp, cp;
    sincos(a.gmst - ra, &sg, &cg);
    sincos(dec, &sd, &cd);
    sincos(psi, &sp, &cp);
    const double X[3] = {-cp * sg - sp * cg * sd, -cp * cg + sp * sg * sd, sp * cd};
    const double Y[3] = {sp * sg - cp * cg * sd, sp * cg + cp * sg * sd, cp * cd};
    const double n[3] = {cd * cg, -cd * sg, sd};             // cos(ra - gmst) = cg, sin(ra - gmst) = -sg
    const double pol_plus = 0.5 * (1.0 + cosi * cosi);

    auto delay_of = [&](const DetGeom &g) {
        return g.kind == GW_DET_FIXED ? g.dt_s : -(g.rc[0] * n[0] + g.rc[1] * n[1] + g.rc[2] * n[2]);
    };
    const double tau0 = tc + delay_of(a.dets.d[0]);
    for (int i = i_first; i <= i_last; ++i) {
        const DetGeom &g = a.dets.d[i];
        double fp, fc;
        if (g.kind == GW_DET_FIXED) {
            fp = g.fplus; fc = g.fcross;
        } else {
            // D symmetric: (xx, xy, xz, yy, yz, zz)
            const double DX[3] = {g.D[0] * X[0] + g.D[1] * X[1] + g.D[2] * X[2],
                                  g.D[1] * X[0] + g.D[3] * X[1] + g.D[4] * X[2],
                                  g.D[2] * X[0] + g.D[4] * X[1] + g.D[5] * X[2]};
            const double DY[3] = {g.D[0] * Y[0] + g.D[1] * Y[1] + g.D[2] * Y[2],
                                  g.D[1] * Y[0] + g.D[3] * Y[1] + g.D[4] * Y[2],
                                  g.D[2] * Y[0] + g.D[4] * Y[1] + g.D[5] * Y[2]};
            fp = (X[0] * DX[0] + X[1] * DX[1] + X[2] * DX[2]) - (Y[0] * DY[0] + Y[1] * DY[1] + Y[2] * DY[2]);
            fc = 2.0 * (X[0] * DY[0] + X[1] * DY[1] + X[2] * DY[2]);
        }
        double tau = tc + delay_of(g);
        if (i > 0 && a.relative_tau) tau -= tau0;
        double rc_, rs_;
        cis_turns_of_product(-a.rot_stride_hz, tau, rc_, rs_);
        double *ri = r + (int64_t)(9 + kRecPerDet * i) * S;
        ri[0 * S] = kPhaseScale * tau;                       // in phase units (exact scaling)
        ri[1 * S] = a0 * (fp * pol_plus);                    // Re(A0 C_I),  C_I = F+ (1+cos^2 i)/2 - i Fx cos i
        ri[2 * S] = a0 * (-fc * cosi);                       // Im(A0 C_I)
        ri[3 * S] = rc_;
        ri[4 * S] = rs_;
    }
}

cudaError_t launch_setup(const Tables &t, const DetSet &dets, double gmst, int spin_order, int64_t n_prop,
                         const double *theta_dev, double *rec, int64_t rec_stride, double rot_stride_hz,
                         int relative_tau, int stage_theta, cudaStream_t s, int64_t *launches)
{
    SetupArgs a;
    a.stage_theta = stage_theta;
    a.isco_cut = t.isco_cut;
    a.dets = dets; a.gmst = gmst; a.n_det = t.n_det; a.spin_order = spin_order;
    a.n_param = t.n_param; a.tidal_order = t.tidal_order;
    a.n_prop = n_prop; a.rec_stride = rec_stride; a.theta = theta_dev; a.rec = rec;
    a.rot_stride_hz = rot_stride_hz; a.relative_tau = relative_tau;
    a.f_amp = reinterpret_cast<const double2 *>(t.planes) + 4 * t.n_pad;
    a.n_bins = t.n_bins; a.f0 = t.f0; a.delta_f = t.delta_f;
    a.f_max = t.f0 + (double)(t.n_bins - 1) * t.delta_f;
    a.band_xi = 1.0 / cbrt(t.f0); a.band_x1 = cbrt(a.f_max);
    a.band_l1 = fmax(fabs(log(t.f0)), fabs(log(a.f_max)));
    a.max_dt = 0.0;                      // FIXED: the given delay; GEOMETRIC: |dt| <= |r| / c
    for (int i = 0; i < t.n_det; ++i) {
        const DetGeom &g = dets.d[i];
        const double m = g.kind == GW_DET_FIXED ? fabs(g.dt_s)
                                                : sqrt(g.rc[0] * g.rc[0] + g.rc[1] * g.rc[1] + g.rc[2] * g.rc[2]);
        a.max_dt = fmax(a.max_dt, m);
    }
    const unsigned blocks = (unsigned)((n_prop + 31) / 32);
    setup_kernel<<<blocks, 128, 0, s>>>(a);
    *launches += 1;
    return cudaGetLastError();
}

// =====================================================================================================
// shared by K2/K3: the phase dot product (8 FMA)
// =====================================================================================================
struct PhaseCoef { double c0, c2, c3, c4, c5, cL5, c6, cL6, c7; };

__device__ __forceinline__ PhaseCoef load_coef(const double *rec, int64_t S, int64_t b)
{
    PhaseCoef k;
    const double *r = rec + b;
    k.c0 = r[0 * S]; k.c2 = r[1 * S]; k.c3 = r[2 * S]; k.c4 = r[3 * S]; k.c5 = r[4 * S];
    k.cL5 = r[5 * S]; k.c6 = r[6 * S]; k.cL6 = r[7 * S]; k.c7 = r[8 * S];
    return k;
}
__device__ __forceinline__ double phase_turns(const PhaseCoef &k, double2 b01, double2 b23, double2 b45,
                                              double2 b67)
{
    double p = __fma_rn(k.c0, b01.x, k.c5);
    p = __fma_rn(k.c2, b01.y, p);
    p = __fma_rn(k.c3, b23.x, p);
    p = __fma_rn(k.c4, b23.y, p);
    p = __fma_rn(k.cL5, b45.x, p);
    p = __fma_rn(k.c6, b45.y, p);
    p = __fma_rn(k.cL6, b67.x, p);
    p = __fma_rn(k.c7, b67.y, p);
    return p;
}

// =====================================================================================================
// K2: waveform-only kernel (north_star item (3); step a6).  Lanes run along bins so that every store is
// a 16-byte element of a 512-byte contiguous warp segment; each thread keeps its bin's basis in
// registers and walks props_per_cta proposals, so table reads are amortised and HBM traffic is the
// 16 B/element store stream.
//     h_I(f) = CA_I f^(-7/6) exp(-2 pi i (Phi'(f) + f tau_I))
// =====================================================================================================
#ifndef GW_WF_PROPS
#define GW_WF_PROPS 16
#endif
#ifndef GW_WF_BINS
#define GW_WF_BINS 2
#endif
#ifndef GW_WF_MIN_CTAS
#define GW_WF_MIN_CTAS 1
#endif
constexpr int kWfProps = GW_WF_PROPS;     // proposals per CTA while the five basis planes stay L2-resident
constexpr int kWfPropsLong = 64;          // ... and for long signals, whose planes stream from HBM once per proposal
                                          // block: 80 B of table reads per bin against 48 N_det B stored per proposal
constexpr int64_t kWfLongBins = 400000;   // 5 planes x 16 B x 400k bins = 32 MB: beyond this the planes do not stay in L2
constexpr int kWfBins  = GW_WF_BINS;      // bins per thread (kThreads * kWfBins bins per CTA)

struct WaveArgs {
    const double *planes, *rec;
    int64_t n_pad, n_bins, n_prop, rec_stride;
    int     bin_blocks, isco_cut;
    int     props_per_cta;   // kWfProps | kWfPropsLong
    double *h;
};

template <int NDET, bool TIDAL>
__global__ void __launch_bounds__(kThreads, GW_WF_MIN_CTAS) waveform_kernel(const WaveArgs a)
{
    constexpr int NT = 10 + 4 * NDET;            // index of the tidal pair (t10, t12) of a staged record
    constexpr int NF = NT + (TIDAL ? 2 : 0);     // doubles per staged record: 9 coefs + f_ISCO, (tau, pad, CAre, CAim) per det
    __shared__ __align__(16) double srec[kWfPropsLong][NF];
    const int     tid     = threadIdx.x;
    const int     bin_blk = blockIdx.x % a.bin_blocks;
    const int64_t p_blk   = blockIdx.x / a.bin_blocks;
    const double2 *pl = reinterpret_cast<const double2 *>(a.planes);
    double2 b01[kWfBins], b23[kWfBins], b45[kWfBins], b67[kWfBins];
    double  amp[kWfBins], f[kWfBins];
    double  x5[kWfBins], x7[kWfBins];            // TIDAL: x^5, x^7 of the thread's bins (x = f^(1/3))
    int64_t j[kWfBins];
    bool    in[kWfBins];
#pragma unroll
    for (int u = 0; u < kWfBins; ++u) {
        j[u]  = ((int64_t)bin_blk * kWfBins + u) * kThreads + tid;
        in[u] = j[u] < a.n_bins;
        const int64_t jc = in[u] ? j[u] : a.n_bins - 1;
        b01[u] = pl[0 * a.n_pad + jc]; b23[u] = pl[1 * a.n_pad + jc];
        b45[u] = pl[2 * a.n_pad + jc]; b67[u] = pl[3 * a.n_pad + jc];
        const double2 fa = pl[4 * a.n_pad + jc];
        f[u] = fa.x; amp[u] = fa.y;
        if (TIDAL) {
            const double x2 = b67[u].y;
            x5[u] = (x2 * x2) * b45[u].y;
            x7[u] = x5[u] * x2;
        }
    }
    pdl_wait_primary();                          // the records come from the setup kernel
    const int64_t b0 = p_blk * a.props_per_cta;
    const int     np = (int)((b0 + a.props_per_cta < a.n_prop) ? a.props_per_cta : a.n_prop - b0);
    for (int idx = tid; idx < np * NF; idx += kThreads) {
        const int p = idx / NF, fld = idx % NF;
        double v = 0.0;
        if (fld < 9) v = a.rec[(int64_t)fld * a.rec_stride + b0 + p];
        else if (fld == 9) v = a.isco_cut ? a.rec[(int64_t)rec_field_fisco(NDET) * a.rec_stride + b0 + p] : 1.0e308;
        else if (TIDAL && fld >= NT) v = a.rec[(int64_t)(rec_field_t10(NDET) + (fld - NT)) * a.rec_stride + b0 + p];
        else {
            const int i = (fld - 10) >> 2, w = (fld - 10) & 3;          // w: 0 tau, 2 CAre, 3 CAim
            if (w != 1) v = a.rec[(int64_t)(9 + kRecPerDet * i + (w == 0 ? 0 : w - 1)) * a.rec_stride + b0 + p];
        }
        srec[p][fld] = v;
    }
    __syncthreads();
    double2 *h = reinterpret_cast<double2 *>(a.h);
    for (int p = 0; p < np; ++p) {
        const double2 *r2 = reinterpret_cast<const double2 *>(srec[p]);  // warp-broadcast LDS.128
        const double2 k01 = r2[0], k23 = r2[1], k45 = r2[2], k67 = r2[3], k8 = r2[4];
        PhaseCoef k;
        k.c0 = k01.x; k.c2 = k01.y; k.c3 = k23.x; k.c4 = k23.y; k.c5 = k45.x; k.cL5 = k45.y;
        k.c6 = k67.x; k.cL6 = k67.y; k.c7 = k8.x;
        double ph[kWfBins];
#pragma unroll
        for (int u = 0; u < kWfBins; ++u) ph[u] = phase_turns(k, b01[u], b23[u], b45[u], b67[u]);
        if (TIDAL) {                                                     // NEXT-1 option: + t10 x^5 + t12 x^7
            const double2 tt = r2[NT / 2];
#pragma unroll
            for (int u = 0; u < kWfBins; ++u) ph[u] = __fma_rn(tt.y, x7[u], __fma_rn(tt.x, x5[u], ph[u]));
        }
        const double f_cut = k8.y;                                       // f_ISCO, or 1e308 without the cut-off
        double2 *row = h + ((b0 + p) * NDET) * a.n_bins;
#pragma unroll
        for (int i = 0; i < NDET; ++i) {
            const double2 t_ = r2[5 + 2 * i], ca = r2[6 + 2 * i];      // (tau, -), (CAre, CAim)
#pragma unroll
            for (int u = 0; u < kWfBins; ++u) {
                double c, s;
                cis_phase(__fma_rn(f[u], t_.x, ph[u]), c, s);
                const double kr = ca.x * amp[u], ki = ca.y * amp[u];
                // (kr + i ki)(c - i s)
                double2 out = make_double2(__fma_rn(kr, c, ki * s), __fma_rn(ki, c, -(kr * s)));
                if (f[u] > f_cut) out = make_double2(0.0, 0.0);            // NEXT-1 option isco_cut
                if (in[u]) __stcs(row + j[u], out);
            }
            row += a.n_bins;
        }
    }
}

template <int NDET, bool TIDAL>
static cudaError_t launch_waveform_t(const WaveArgs &a, int64_t blocks, cudaStream_t s)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks); cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, waveform_kernel<NDET, TIDAL>, a);
}

cudaError_t launch_waveform(const Tables &t, int64_t n_prop, const double *rec, int64_t rec_stride,
                            double *h_out, cudaStream_t s, int64_t *launches)
{
    WaveArgs a;
    a.planes = t.planes; a.rec = rec;
    a.n_pad = t.n_pad; a.n_bins = t.n_bins; a.n_prop = n_prop; a.rec_stride = rec_stride;
    a.bin_blocks = (int)((t.n_bins + kThreads * kWfBins - 1) / (kThreads * kWfBins));
    a.isco_cut = t.isco_cut;
    a.h = h_out;
    a.props_per_cta = t.n_bins > kWfLongBins ? kWfPropsLong : kWfProps;
    const int64_t p_blocks = (n_prop + a.props_per_cta - 1) / a.props_per_cta;
    const int64_t blocks = p_blocks * a.bin_blocks;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    *launches += 1;
    const bool tidal = t.tidal_order > 0;
    switch (t.n_det) {
    case 1: return tidal ? launch_waveform_t<1, true>(a, blocks, s) : launch_waveform_t<1, false>(a, blocks, s);
    case 2: return tidal ? launch_waveform_t<2, true>(a, blocks, s) : launch_waveform_t<2, false>(a, blocks, s);
    case 3: return tidal ? launch_waveform_t<3, true>(a, blocks, s) : launch_waveform_t<3, false>(a, blocks, s);
    case 4: return tidal ? launch_waveform_t<4, true>(a, blocks, s) : launch_waveform_t<4, false>(a, blocks, s);
    case 5: return tidal ? launch_waveform_t<5, true>(a, blocks, s) : launch_waveform_t<5, false>(a, blocks, s);
    case 6: return tidal ? launch_waveform_t<6, true>(a, blocks, s) : launch_waveform_t<6, false>(a, blocks, s);
    case 7: return tidal ? launch_waveform_t<7, true>(a, blocks, s) : launch_waveform_t<7, false>(a, blocks, s);
    case 8: return tidal ? launch_waveform_t<8, true>(a, blocks, s) : launch_waveform_t<8, false>(a, blocks, s);
    default: return cudaErrorInvalidValue;
    }
}

// =====================================================================================================
// K3: fused waveform + projection + inner product (north_star item (4); steps a2..a5)
//
// The (proposal tile, bin) pairs of a call form one flattened space, tile-major; CTA k of n_cta sweeps the contiguous
// range [k work / n_cta, (k+1) work / n_cta) of it (gw_internal.h, struct Plan): one SEGMENT per tile the range touches,
// i.e. kThreads threads = (kThreads / lpp) proposals x the bins [j0, j1) of that tile.  Every CTA gets the same number of
// bins whatever the batch size, so no SM idles and no partial second wave exists.
// lpp = lanes per proposal: 1 for sampler-sized batches (each thread owns one proposal and sweeps the
// chunk; the tables are read from shared memory as warp broadcasts), 2..32 for small batches (the lanes
// of a proposal interleave over the bins; a fixed xor-shuffle tree combines them).
// A segment is streamed through a kStages-deep ring of kStageBins-bin stages by bulk async copies (TMA
// engine) completing on mbarriers.  Per (proposal, bin): 9 FMA phase (incl. f tau_0), 12-op sincos (cis_phase_lnl) giving
// E = e^{+2 pi i (Phi' + f tau_0)}, detector 0: Z_0 += g_0j E (4 FMA), and per detector I >= 1
//     Z_I <- Z_I * rot_I + g_Ij * E                                                  (8 fp64 ops)
// where rot_I = exp(-2 pi i lpp df (tau_I - tau_0)): after the sweep Z_I * exp(+2 pi i f_last (tau_I - tau_0))
// equals sum_j g_Ij exp(+2 pi i (Phi'_j + f_j tau_I)), i.e. the time shift of PAPER.md:69 costs no sincos.
// <h|h>_I = |CA_I|^2 I7_I exactly for this waveform, so only <d|h> is accumulated.
// Cross-segment: partials to the workspace, a per-tile ticket, and the last CTA of a tile sums the tile's segments in
// ascending bin order (deterministic: the order is a function of (n_tiles, n_bins, n_cta) alone) and writes lnL and parts.
// =====================================================================================================
struct FusedArgs {
    const double *planes, *rec;
    int64_t n_pad, n_bins, n_prop, rec_stride;
    int64_t tile_len;        // n_bins + boundary bins: positions per tile in the flattened space (gw_internal.h, segment_at)
    int64_t work;            // flattened_work(n_tiles, n_bins, vbins): size of the flattened (tile, bin) space
    int64_t n_cta;           // CTAs of the grid: CTA k sweeps [k work / n_cta, (k+1) work / n_cta)
    int     lpp;
    int     gmax;            // groups per tile of the two-level finish (stride of gpartial / gtickets)
    int     cluster;         // > 0: the chunks of a tile are one thread-block cluster of this size (multi-lane layouts)
    double  f0, delta_f;
    double  i7[GW_MAX_DET];
    const double *i7cum;     // isco_cut: [NDET][n_pad] prefix sums of the norm
    int     phase_marginal;
    double *partial;         // [slot][2 NDET][PT] segment sums, slot = cta + tile
    unsigned int *tickets;   // [tile]
    double *gpartial;        // [tile][group][2 NDET][PT] group sums
    unsigned int *gtickets;  // [tile][group]
    double *lnl, *parts;
};

// ln I0(x), x >= 0: library I0 up to 500, then the asymptotic series e^x/sqrt(2 pi x) (1 + 1/8x + 9/128x^2 + ...)
// whose 8-term truncation error is below 1e-20 there.
__device__ __forceinline__ double log_bessel_i0(double x)
{
    if (x < 500.0) return log(cyl_bessel_i0(x));
    const double y = 1.0 / x;
    double s = 1.0 + y * (0.125 + y * (0.0703125 + y * (0.0732421875 + y * (0.112152099609375 +
               y * (0.22710800170898438 + y * (0.5725014209747314 + y * 1.7277275025844574))))));
    return x - 0.5 * log(kTwoPi * x) + log(s);
}

// The record fields the finish stage needs (CA_I and the cut index).  The cross-chunk finish loads them before the
// ticket round trip so that their L2 latency is not added to the last CTA's serial chain.
// ---- per-CTA timeline (diagnostic build only: -DGW_TIMELINE, csrc/build.py build_timeline, timeline.py) ----------------
// Thread 0 of every CTA stores the nanosecond globaltimer (and, for the first eight stamps, clock64) into a caller-given
// buffer of 32 words per CTA: 0 kernel entry, 1 sweep start / 2 sweep end / 3 ticket taken of the CTA's first segment,
// 4 exit, 5-7 the same three for its last later segment, 8..23 stage starts of the first segment; 24..31 clock64 at
// stamps 0..7.  Every stamp is stored at once, so no register is held across the sweep (ptxas: no spill, the hot loop
// unchanged).  The product build compiles GW_STAMP to nothing.
#ifndef GW_MULTI_UNROLL
#define GW_MULTI_UNROLL 5
#endif
constexpr int kMultiUnroll = GW_MULTI_UNROLL;   // bins per unrolled trip of the lanes-interleaved sweep
#ifdef GW_TIMELINE
__device__ unsigned long long *g_timeline = nullptr;
__device__ __forceinline__ unsigned long long timeline_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define GW_STAMP(k)                                                                                        \
    do {                                                                                                   \
        if (threadIdx.x == 0) {                                                                            \
            unsigned long long *p_ = g_timeline;                                                           \
            if (p_) {                                                                                      \
                p_[(size_t)blockIdx.x * 32 + (k)] = timeline_ns();                                         \
                if ((k) < 8) p_[(size_t)blockIdx.x * 32 + 24 + (k)] = (unsigned long long)clock64();       \
            }                                                                                              \
        }                                                                                                  \
    } while (0)
#else
#define GW_STAMP(k) do { } while (0)
#endif

template <int NDET>
struct FinishRec { double car[NDET], cai[NDET]; int64_t jcut; };

template <int NDET, bool ISCO>
__device__ __forceinline__ FinishRec<NDET> load_finish_rec(const FusedArgs &a, int64_t b)
{
    FinishRec<NDET> f;
    f.jcut = 0;
    if (ISCO) f.jcut = (int64_t)a.rec[(int64_t)rec_field_jcut(NDET) * a.rec_stride + b];
#pragma unroll
    for (int i = 0; i < NDET; ++i) {
        const double *ri = a.rec + (int64_t)(9 + kRecPerDet * i) * a.rec_stride + b;
        f.car[i] = ri[a.rec_stride];
        f.cai[i] = ri[2 * a.rec_stride];
    }
    return f;
}

template <int NDET, bool ISCO>
__device__ __forceinline__ void finish_proposal(const FusedArgs &a, int64_t b, const FinishRec<NDET> &f,
                                                const double (&zr)[NDET], const double (&zi)[NDET])
{
    double lnl = 0.0, sum_re = 0.0, sum_im = 0.0, sum_hh = 0.0;
    const int64_t jcut = f.jcut;
#pragma unroll
    for (int i = 0; i < NDET; ++i) {
        const double car = f.car[i], cai = f.cai[i];
        const double dh_re = __fma_rn(car, zr[i], cai * zi[i]);      // conj(CA) * Z
        const double dh_im = __fma_rn(car, zi[i], -(cai * zr[i]));
        const double norm  = ISCO ? (jcut >= 0 ? a.i7cum[(int64_t)i * a.n_pad + jcut] : 0.0) : a.i7[i];
        const double hh    = __fma_rn(car, car, cai * cai) * norm;
        lnl += dh_re - 0.5 * hh;
        sum_re += dh_re; sum_im += dh_im; sum_hh += hh;
        if (a.parts) {
            double *p = a.parts + (b * NDET + i) * 3;
            p[0] = dh_re; p[1] = dh_im; p[2] = hh;
        }
    }
    if (a.phase_marginal) lnl = log_bessel_i0(hypot(sum_re, sum_im)) - 0.5 * sum_hh;   // NEXT-1 option
    a.lnl[b] = lnl;
}

// One segment: bins [seg.j0, seg.j1) of proposal tile seg.tile.  `g` is the CTA's running position in the stage ring
// (stages issued so far): stage s of the segment uses buffer (g + s) % kStages and completes phase (g + s) / kStages of
// its mbarrier, so the ring carries on from segment to segment without re-initialisation.
template <int NDET, bool MULTI, bool ISCO, bool TIDAL>
__device__ __forceinline__ void fused_segment(const FusedArgs &a, const Segment &seg, uint32_t &g, const bool first,
                                              unsigned char *smem_raw, unsigned int &s_ticket, int &s_relmax)
{
    constexpr int NP = kBasisPlanes + NDET;                  // planes per stage
    double2  *sm   = reinterpret_cast<double2 *>(smem_raw);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + (size_t)kStages * NP * kStageBins * sizeof(double2));

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lpp = MULTI ? a.lpp : 1;
    const int ppw = 32 / lpp;
    const int PT  = kThreads / lpp;
    const int64_t tile = seg.tile;
    const int pic = MULTI ? warp * ppw + lane / lpp : tid;   // proposal slot in this CTA
    const int sub = MULTI ? lane % lpp : 0;                  // lane's position among the proposal's lanes
    int64_t b = tile * PT + pic;
    const bool live = b < a.n_prop;
    if (!live) b = a.n_prop - 1;

    const int64_t j0 = seg.j0;
    const int n = (int)(seg.j1 - seg.j0);
    const int n_stage = (n + kStageBins - 1) / kStageBins;
    const int n_issued0 = min(kStages, n_stage);             // stages prefetched before the records are known

    auto issue_stage = [&](int s) {
        const int buf = (int)((g + (uint32_t)s) % kStages);
        const int cnt = min(kStageBins, n - s * kStageBins);
        const uint32_t bytes = (uint32_t)cnt * (uint32_t)sizeof(double2);
        mbar_arrive_expect_tx(&bars[buf], bytes * NP);
        const double2 *src = reinterpret_cast<const double2 *>(a.planes) + j0 + (int64_t)s * kStageBins;
#pragma unroll
        for (int p = 0; p < NP; ++p)
            bulk_g2s(sm + (size_t)(buf * NP + p) * kStageBins, src + (int64_t)p * a.n_pad, bytes, &bars[buf]);
    };

    if (tid == 0) {
        if (ISCO) s_relmax = -1;
        for (int s = 0; s < n_issued0; ++s) issue_stage(s);   // tables do not depend on K1
    }
    if (first) pdl_wait_primary();                           // records come from the setup kernel
    const PhaseCoef k = load_coef(a.rec, a.rec_stride, b);
    double t10 = 0.0, t12 = 0.0;                             // NEXT-1 option: tidal terms t10 x^5 + t12 x^7
    if (TIDAL) {
        t10 = a.rec[(int64_t)rec_field_t10(NDET) * a.rec_stride + b];
        t12 = a.rec[(int64_t)rec_field_t12(NDET) * a.rec_stride + b];
    }
    double tau[NDET], rr[NDET], ri_[NDET], zr[NDET], zi[NDET];
#pragma unroll
    for (int i = 0; i < NDET; ++i) {
        const double *r = a.rec + (int64_t)(9 + kRecPerDet * i) * a.rec_stride + b;
        tau[i] = r[0];
        rr[i]  = r[3 * a.rec_stride];
        ri_[i] = r[4 * a.rec_stride];
        zr[i] = 0.0; zi[i] = 0.0;
    }

    int jrel = 0;                                            // isco_cut: last kept bin relative to j0 (may be < 0 or >= n)
    int n_run = n_stage;                                     // stages this segment sweeps
    int n_issued = n_stage;                                  // stages whose copies are issued (>= n_run)
    if (ISCO) {
        // Stages wholly above the cut-off of every proposal of the CTA contribute nothing: they are neither loaded
        // (beyond the prefetched ones) nor swept.  The rotation recurrence stops with the last swept bin, which is
        // the f_last of the seed below.
        const int64_t jcut = (int64_t)a.rec[(int64_t)rec_field_jcut(NDET) * a.rec_stride + b];
        jrel = (int)max((int64_t)-1, min(jcut - j0, (int64_t)n));
        int rel = min(jrel, n - 1);
        rel = __reduce_max_sync(0xffffffffu, rel);
        __syncthreads();                                     // s_relmax = -1 of this segment is in place
        if (lane == 0) atomicMax(&s_relmax, rel);
        __syncthreads();
        n_run = s_relmax < 0 ? 0 : s_relmax / kStageBins + 1;
        n_issued = max(n_run, n_issued0);
    }
    int iters_total = 0;
    GW_STAMP(first ? 1 : 5);
    for (int s = 0; s < n_stage; ++s) {
        const int buf = (int)((g + (uint32_t)s) % kStages);
        const uint32_t parity = ((g + (uint32_t)s) / kStages) & 1u;
        const int cnt = min(kStageBins, n - s * kStageBins);
        if (ISCO && s >= n_run) {                            // drain the prefetched stages, then stop
            if (s >= n_issued) break;
            mbar_wait(&bars[buf], parity);
            continue;
        }
        mbar_wait(&bars[buf], parity);
        if (first) GW_STAMP(8 + (s < 15 ? s : 15));
        const double2 *P = sm + (size_t)buf * NP * kStageBins;
        const int iters = MULTI ? (cnt + lpp - 1) / lpp : cnt;
        // last kept bin of this proposal relative to the stage (isco_cut), in [-1, kStageBins]
        const int cut_local = ISCO ? max(-1, min(jrel - s * kStageBins, kStageBins)) : 0;
        int it = 0;
        if (!MULTI) {
            // kUnroll bins per trip, written plane by plane ("k-major"): consecutive fp64 instructions then
            // share a register operand in the same slot (the coefficient across bins, c/s across detectors,
            // z across the re/im pair), which the operand-reuse cache serves.  A DFMA with three fresh
            // register operands issues at 2/3 rate on B200 (profiles/dfma_operand_probe).
            // E(it0): phase and sincos of kUnroll bins; U(it0): their detector updates (ascending bin order).
            auto compute_e = [&](int it, double (&cs)[kUnroll], double (&sn)[kUnroll]) {
                double ph[kUnroll];
                {
                    double2 v[kUnroll];
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) v[u] = P[0 * kStageBins + it + u];
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(k.c0, v[u].x, k.c5);
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(k.c2, v[u].y, ph[u]);
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) v[u] = P[1 * kStageBins + it + u];
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(k.c3, v[u].x, ph[u]);
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(k.c4, v[u].y, ph[u]);
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) v[u] = P[2 * kStageBins + it + u];
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(k.cL5, v[u].x, ph[u]);
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(k.c6, v[u].y, ph[u]);
                    double x1[kUnroll];                              // TIDAL: x = f^(1/3) of the bins
                    if (TIDAL) {
#pragma unroll
                        for (int u = 0; u < kUnroll; ++u) x1[u] = v[u].y;
                    }
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) v[u] = P[3 * kStageBins + it + u];
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(k.cL6, v[u].x, ph[u]);
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(k.c7, v[u].y, ph[u]);
                    if (TIDAL) {                                     // + x^5 (t10 + t12 x^2): 4 more fp64 instructions
                        double x5[kUnroll], tt[kUnroll];
#pragma unroll
                        for (int u = 0; u < kUnroll; ++u) x5[u] = v[u].y * v[u].y;
#pragma unroll
                        for (int u = 0; u < kUnroll; ++u) tt[u] = __fma_rn(t12, v[u].y, t10);
#pragma unroll
                        for (int u = 0; u < kUnroll; ++u) x5[u] *= x1[u];
#pragma unroll
                        for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(tt[u], x5[u], ph[u]);
                    }
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) v[u] = P[4 * kStageBins + it + u];
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) ph[u] = __fma_rn(tau[0], v[u].x, ph[u]);   // + f tau_0
                }
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) cis_phase_lnl(ph[u], cs[u], sn[u]);
                if (ISCO) {                                      // h = 0 above f_ISCO: the bin contributes nothing
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u)
                        if (it + u > cut_local) { cs[u] = 0.0; sn[u] = 0.0; }
                }
            };
            auto update_z = [&](int it, const double (&cs)[kUnroll], const double (&sn)[kUnroll]) {
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) {              // bins in ascending order: the Z recurrence
#pragma unroll
                    for (int i = 0; i < NDET; ++i) {
                        const double2 g = P[(kBasisPlanes + i) * kStageBins + it + u];
                        if (i == 0) {                                         // reference detector: no rotation
                            zr[0] = __fma_rn(-g.y, sn[u], __fma_rn(g.x, cs[u], zr[0]));
                            zi[0] = __fma_rn(g.y, cs[u], __fma_rn(g.x, sn[u], zi[0]));
                            continue;
                        }
                        const double t1 = g.y * sn[u];
                        const double t2 = g.y * cs[u];
                        const double a2 = __fma_rn(g.x, cs[u], -t1);          // Re g e^{+i 2 pi Phi'}
                        const double b2 = __fma_rn(g.x, sn[u], t2);           // Im
                        const double a3 = __fma_rn(zi[i], -ri_[i], a2);
                        const double b3 = __fma_rn(zi[i], rr[i], b2);
                        const double nr = __fma_rn(zr[i], rr[i], a3);
                        const double ni = __fma_rn(zr[i], ri_[i], b3);
                        zr[i] = nr; zi[i] = ni;
                    }
                }
            };
#if GW_PIPELINE
            // software pipeline: the sincos of the next kUnroll bins is issued together with the detector
            // updates of the current ones (two independent instruction streams in one basic block)
            if (iters >= kUnroll) {
                double cs[kUnroll], sn[kUnroll];
                compute_e(0, cs, sn);
                for (; it + 2 * kUnroll <= iters; it += kUnroll) {
                    double cn[kUnroll], sm_[kUnroll];
                    compute_e(it + kUnroll, cn, sm_);
                    update_z(it, cs, sn);
#pragma unroll
                    for (int u = 0; u < kUnroll; ++u) { cs[u] = cn[u]; sn[u] = sm_[u]; }
                }
                update_z(it, cs, sn);
                it += kUnroll;
            }
#else
            for (; it + kUnroll <= iters; it += kUnroll) {
                double cs[kUnroll], sn[kUnroll];
                compute_e(it, cs, sn);
                update_z(it, cs, sn);
            }
#endif
        }
#pragma unroll (MULTI ? kMultiUnroll : 1)
        for (; it < iters; ++it) {
            int jj = MULTI ? sub + it * lpp : it;
            bool masked = false;
            if (MULTI) { masked = jj >= cnt; jj = masked ? cnt - 1 : jj; }
            double ph = phase_turns(k, P[0 * kStageBins + jj], P[1 * kStageBins + jj],
                                    P[2 * kStageBins + jj], P[3 * kStageBins + jj]);
            if (TIDAL) {
                const double x = P[2 * kStageBins + jj].y, x2 = P[3 * kStageBins + jj].y;
                ph = __fma_rn(__fma_rn(t12, x2, t10), (x2 * x2) * x, ph);
            }
            ph = __fma_rn(tau[0], P[4 * kStageBins + jj].x, ph);
            double c, sn;
            cis_phase_lnl(ph, c, sn);
            if (ISCO && jj > cut_local) { c = 0.0; sn = 0.0; }
#pragma unroll
            for (int i = 0; i < NDET; ++i) {
                double2 g = P[(kBasisPlanes + i) * kStageBins + jj];
                if (MULTI && masked) g = make_double2(0.0, 0.0);
                if (i == 0) {
                    zr[0] = __fma_rn(-g.y, sn, __fma_rn(g.x, c, zr[0]));
                    zi[0] = __fma_rn(g.y, c, __fma_rn(g.x, sn, zi[0]));
                    continue;
                }
                const double wr = __fma_rn(g.x, c, -(g.y * sn));     // g * e^{+i 2 pi Phi'}
                const double wi = __fma_rn(g.x, sn, g.y * c);
                const double nr = __fma_rn(zr[i], rr[i], __fma_rn(-zi[i], ri_[i], wr));
                const double ni = __fma_rn(zr[i], ri_[i], __fma_rn(zi[i], rr[i], wi));
                zr[i] = nr; zi[i] = ni;
            }
        }
        iters_total += iters;
        __syncthreads();                                     // every warp is done with this buffer
        if (tid == 0 && s + kStages < n_run) issue_stage(s + kStages);   // n_run <= n_stage
    }

    GW_STAMP(first ? 2 : 6);
    // seed (detectors >= 1): multiply by exp(+2 pi i f_last (tau_I - tau_0)), f_last = frequency of this
    // thread's last iteration
    {
        const int64_t j_last = j0 + sub + (int64_t)(iters_total - 1) * lpp;
        const double f_last = __fma_rn((double)j_last, a.delta_f, a.f0);
#pragma unroll
        for (int i = 1; i < NDET; ++i) {
            double c, sn;
            cis_turns_of_product(f_last, tau[i] * (1.0 / kPhaseScale), c, sn);
            const double nr = __fma_rn(zr[i], c, -(zi[i] * sn));
            const double ni = __fma_rn(zr[i], sn, zi[i] * c);
            zr[i] = nr; zi[i] = ni;
        }
    }
    g += (uint32_t)n_issued;                                 // every issued stage has been waited for
    if (MULTI) {                                             // fixed xor tree over the proposal's lanes
        for (int o = lpp >> 1; o > 0; o >>= 1) {
#pragma unroll
            for (int i = 0; i < NDET; ++i) {
                zr[i] += __shfl_xor_sync(0xffffffffu, zr[i], o);
                zi[i] += __shfl_xor_sync(0xffffffffu, zi[i], o);
            }
        }
    }

    const int n_seg = seg.count;                             // segments of this tile, summed in ascending bin order
    if (n_seg == 1) {
        if (sub == 0 && live) finish_proposal<NDET, ISCO>(a, b, load_finish_rec<NDET, ISCO>(a, b), zr, zi);
        return;
    }
    if (MULTI && a.cluster > 0) {
        // The n_seg chunks of this tile are one thread-block cluster (aligned grid, n_seg = cluster size <= 16): the
        // partial sums go to each CTA's own (now idle) stage buffers, and CTA 0 of the cluster gathers them through
        // distributed shared memory in one round trip and adds them in chunk order -- no global partials, no fence, no
        // ticket.  Same additions in the same order as the ticket path below, so the bits are identical.
        double *sh = reinterpret_cast<double *>(smem_raw);
        const int blk = 2 * NDET * PT;                       // doubles per CTA
        if (sub == 0) {
#pragma unroll
            for (int i = 0; i < NDET; ++i) { sh[(2 * i) * PT + pic] = zr[i]; sh[(2 * i + 1) * PT + pic] = zi[i]; }
        }
        const int64_t b_fin = tile * PT + (tid < PT ? tid : 0);
        const FinishRec<NDET> frec = load_finish_rec<NDET, ISCO>(a, b_fin < a.n_prop ? b_fin : a.n_prop - 1);
        cluster_sync();                                      // every CTA's block is in place
        if (cluster_ctarank() == 0) {
            double *gather = sh + blk;
            const int nvals = blk * n_seg;
            for (int i = tid; i < nvals; i += kThreads) gather[i] = ld_dsmem_f64(sh + (i % blk), (uint32_t)(i / blk));
        }
        cluster_sync();                                      // CTA 0 has read everybody's block: the others may leave
        if (cluster_ctarank() != 0) return;
        __syncthreads();
        if (tid < PT) {
            const int64_t bb = tile * PT + tid;
            if (bb < a.n_prop) {
                const double *gather = sh + blk;
                double sr[NDET], si[NDET];
#pragma unroll
                for (int i = 0; i < NDET; ++i) { sr[i] = 0.0; si[i] = 0.0; }
                for (int c = 0; c < n_seg; ++c) {
#pragma unroll
                    for (int i = 0; i < NDET; ++i) {
                        sr[i] += gather[(c * 2 * NDET + 2 * i) * PT + tid];
                        si[i] += gather[(c * 2 * NDET + 2 * i + 1) * PT + tid];
                    }
                }
                finish_proposal<NDET, ISCO>(a, bb, frec, sr, si);
            }
        }
        return;
    }
    // stage 1 -> workspace: partial[(slot*2*NDET + comp)*PT + pic], slot = cta + tile (consecutive along the tile)
    const int64_t slot0 = seg.first_cta + tile;              // slot of the tile's first segment
    double *part = a.partial + (seg.slot * (int64_t)(2 * NDET)) * PT;
    if (sub == 0) {
#pragma unroll
        for (int i = 0; i < NDET; ++i) {
            part[(2 * i) * PT + pic]     = zr[i];
            part[(2 * i + 1) * PT + pic] = zi[i];
        }
    }
    // Ordered sum of `count` entries (segments or groups) of one proposal: entry e, component q at base[(e*2*NDET+q)*PT].
    // Loads of kFinishBatch entries are issued together (the sum is latency-bound on L2 otherwise); the additions
    // stay in index order, so the result does not depend on the batching.
    auto ordered_sum = [&](const double *base, int count, double (&sr)[NDET], double (&si)[NDET]) {
        constexpr int kFinishBatch = NDET <= 4 ? 8 : 2;       // 2 * NDET * kFinishBatch doubles in flight per thread
        for (int c = 0; c < count; c += kFinishBatch) {
            // the last batch may be short: its loads are clamped to the last entry and its additions masked, so that
            // a remainder costs one round trip to L2 like a full batch (the finish is a chain of L2 latencies)
            double v[kFinishBatch][2 * NDET];
#pragma unroll
            for (int u = 0; u < kFinishBatch; ++u) {
                const int e = min(c + u, count - 1);
#pragma unroll
                for (int q = 0; q < 2 * NDET; ++q)
                    v[u][q] = __ldcg(base + ((int64_t)e * 2 * NDET + q) * PT);
            }
#pragma unroll
            for (int u = 0; u < kFinishBatch; ++u) {
                if (c + u < count) {
#pragma unroll
                    for (int i = 0; i < NDET; ++i) { sr[i] += v[u][2 * i]; si[i] += v[u][2 * i + 1]; }
                }
            }
        }
    };
    // finish-stage record of the proposal this thread would finish (tid < PT), issued ahead of the ticket
    const int64_t b_fin = tile * PT + (tid < PT ? tid : 0);
    const FinishRec<NDET> frec = load_finish_rec<NDET, ISCO>(a, b_fin < a.n_prop ? b_fin : a.n_prop - 1);
    __threadfence();
    __syncthreads();
    const int n_groups = n_seg >= kFinishTwoLevelFrom ? (n_seg + kFinishGroup - 1) / kFinishGroup : 1;
    unsigned int last_ticket = (unsigned)(n_seg - 1);
    if (n_groups > 1) {
        // Two-level finish for many segments (a single CTA summing hundreds of partials is bound by one SM's L2
        // bandwidth): the last CTA of each group of kFinishGroup segments sums that group in order, and the
        // last group to finish sums the group sums in group order.  The order is fixed by (n_seg, kFinishGroup).
        const int group = seg.index / kFinishGroup;
        const int gsize = min(kFinishGroup, n_seg - group * kFinishGroup);
        unsigned int *gt = a.gtickets + tile * a.gmax + group;
        if (tid == 0) s_ticket = atomicAdd(gt, 1u);
        __syncthreads();
        if (s_ticket != (unsigned)(gsize - 1)) return;
        __threadfence();
        if (tid < PT) {
            double sr[NDET], si[NDET];
#pragma unroll
            for (int i = 0; i < NDET; ++i) { sr[i] = 0.0; si[i] = 0.0; }
            ordered_sum(a.partial + ((slot0 + (int64_t)group * kFinishGroup) * (int64_t)(2 * NDET)) * PT + tid, gsize, sr, si);
            double *gp = a.gpartial + ((tile * a.gmax + group) * (int64_t)(2 * NDET)) * PT + tid;
#pragma unroll
            for (int i = 0; i < NDET; ++i) { gp[(2 * i) * PT] = sr[i]; gp[(2 * i + 1) * PT] = si[i]; }
        }
        if (tid == 0) *gt = 0u;
        __threadfence();
        __syncthreads();
        last_ticket = (unsigned)(n_groups - 1);
    }
    if (tid == 0) s_ticket = atomicAdd(&a.tickets[tile], 1u);
    GW_STAMP(first ? 3 : 7);
    __syncthreads();
    if (s_ticket != last_ticket) return;
    // stage 2 (last CTA of the tile): segments (or group sums) added in index order
    __threadfence();
    {   // Small tiles (multi-lane layouts): all threads pull the tile's partials into the now idle stage buffers in
        // one round trip to L2, and the ordered sums read shared memory.  Same additions in the same order as the
        // direct path below, so the bits do not depend on which path runs.
        const int nvals = PT * 2 * NDET * n_seg;
        if (MULTI && n_groups == 1 && nvals <= kStages * NP * kStageBins * 2) {
            double *sh = reinterpret_cast<double *>(smem_raw);
            const double *src = a.partial + (slot0 * (int64_t)(2 * NDET)) * PT;
            for (int i = tid; i < nvals; i += kThreads) sh[i] = __ldcg(src + i);
            __syncthreads();
            if (tid < PT) {
                const int64_t bb = tile * PT + tid;
                if (bb < a.n_prop) {
                    double sr[NDET], si[NDET];
#pragma unroll
                    for (int i = 0; i < NDET; ++i) { sr[i] = 0.0; si[i] = 0.0; }
                    for (int c = 0; c < n_seg; ++c) {
#pragma unroll
                        for (int i = 0; i < NDET; ++i) {
                            sr[i] += sh[(c * 2 * NDET + 2 * i) * PT + tid];
                            si[i] += sh[(c * 2 * NDET + 2 * i + 1) * PT + tid];
                        }
                    }
                    finish_proposal<NDET, ISCO>(a, bb, frec, sr, si);
                }
            }
            if (tid == 0) a.tickets[tile] = 0u;
            __syncthreads();                                 // the stage buffers are free again for the next segment
            return;
        }
    }
    if (tid < PT) {
        const int64_t bb = tile * PT + tid;
        if (bb < a.n_prop) {
            double sr[NDET], si[NDET];
#pragma unroll
            for (int i = 0; i < NDET; ++i) { sr[i] = 0.0; si[i] = 0.0; }
            if (n_groups > 1)
                ordered_sum(a.gpartial + (tile * a.gmax * (int64_t)(2 * NDET)) * PT + tid, n_groups, sr, si);
            else
                ordered_sum(a.partial + (slot0 * (int64_t)(2 * NDET)) * PT + tid, n_seg, sr, si);
            finish_proposal<NDET, ISCO>(a, bb, frec, sr, si);
        }
    }
    if (tid == 0) a.tickets[tile] = 0u;                      // self-reset for the next call
}

template <int NDET, bool MULTI, bool ISCO, bool TIDAL>
__global__ void __launch_bounds__(kThreads, NDET > 4 ? 1 : kMinCtas) fused_kernel(const FusedArgs a)
{
    constexpr int NP = kBasisPlanes + NDET;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + (size_t)kStages * NP * kStageBins * sizeof(double2));
    __shared__ unsigned int s_ticket;
    __shared__ int s_relmax;

    GW_STAMP(0);
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    // this CTA's range of the flattened (tile, bin) space, one segment per tile it touches
    const int64_t cta = blockIdx.x;
    const int64_t w_end = work_begin(cta + 1, a.work, a.n_cta);
    uint32_t g = 0;
    bool first = true;
    for (int64_t w = work_begin(cta, a.work, a.n_cta); w < w_end;) {
        const Segment seg = segment_at(w, w_end, cta, a.n_bins, a.tile_len, a.work, a.n_cta);
        fused_segment<NDET, MULTI, ISCO, TIDAL>(a, seg, g, first, smem_raw, s_ticket, s_relmax);
        w += seg.len;
        first = false;
        if (w < w_end) __syncthreads();                      // s_ticket / s_relmax / stage buffers change hands
    }
    if (first) pdl_wait_primary();                           // an empty range still orders itself after the setup kernel
    GW_STAMP(4);
}

size_t fused_smem_bytes(int n_det)
{
    return (size_t)kStages * (kBasisPlanes + n_det) * kStageBins * sizeof(double2) + kStages * sizeof(uint64_t);
}

// A grid of at most one CTA per SM must not land two CTAs on one SM while another kernel (the setup kernel under
// programmatic dependent launch, or the previous call's tail) still holds some SMs: the doubled-up SMs would take
// twice as long.  Asking for more than half of an SM's shared memory makes the placement one per SM.
size_t fused_smem_bytes_exclusive(int n_det)
{
    const size_t need = fused_smem_bytes(n_det), half = (size_t)kExclusiveSmemBytes;
    return need > half ? need : half;
}

template <int NDET, bool MULTI, bool ISCO, bool TIDAL>
static cudaError_t launch_fused_t(const FusedArgs &a, int64_t blocks, bool exclusive, cudaStream_t s)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks); cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = exclusive ? fused_smem_bytes_exclusive(NDET) : fused_smem_bytes(NDET); cfg.stream = s;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    if (MULTI && a.cluster > 0) {                            // the chunks of a tile form one cluster
        at[1].id = cudaLaunchAttributeClusterDimension;
        at[1].val.clusterDim.x = (unsigned)a.cluster; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelEx(&cfg, fused_kernel<NDET, MULTI, ISCO, TIDAL>, a);
}

cudaError_t launch_fused(const Tables &t, const Plan &plan, int64_t n_prop, const double *rec,
                         int64_t rec_stride, double *partial, unsigned int *tickets, double *gpartial,
                         unsigned int *gtickets, double *lnl_out, double *parts_out, cudaStream_t s, int64_t *launches)
{
    FusedArgs a;
    a.planes = t.planes; a.rec = rec; a.n_pad = t.n_pad; a.n_bins = t.n_bins; a.n_prop = n_prop;
    a.rec_stride = rec_stride; a.lpp = plan.lpp; a.f0 = t.f0; a.delta_f = t.delta_f;
    a.tile_len = t.n_bins + plan.vbins; a.work = flattened_work(plan.n_tiles, t.n_bins, plan.vbins);
    a.n_cta = plan.n_cta; a.gmax = plan.gmax; a.cluster = plan.cluster;
    for (int i = 0; i < GW_MAX_DET; ++i) a.i7[i] = t.i7[i];
    a.partial = partial; a.tickets = tickets; a.lnl = lnl_out; a.parts = parts_out;
    a.gpartial = gpartial; a.gtickets = gtickets;
    const int64_t blocks = plan.n_cta;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    *launches += 1;
    a.i7cum = t.i7cum; a.phase_marginal = t.phase_marginal;
    const int variant = (plan.lpp > 1 ? 1 : 0) + (t.isco_cut ? 2 : 0) + (t.tidal_order > 0 ? 4 : 0);
    const bool ex = plan.exclusive != 0;
#define GW_DISPATCH(N)                                                                      \
    switch (variant) {                                                                      \
    case 0: return launch_fused_t<N, false, false, false>(a, blocks, ex, s);                \
    case 1: return launch_fused_t<N, true, false, false>(a, blocks, ex, s);                 \
    case 2: return launch_fused_t<N, false, true, false>(a, blocks, ex, s);                 \
    case 3: return launch_fused_t<N, true, true, false>(a, blocks, ex, s);                  \
    case 4: return launch_fused_t<N, false, false, true>(a, blocks, ex, s);                 \
    case 5: return launch_fused_t<N, true, false, true>(a, blocks, ex, s);                  \
    case 6: return launch_fused_t<N, false, true, true>(a, blocks, ex, s);                  \
    default: return launch_fused_t<N, true, true, true>(a, blocks, ex, s);                  \
    }
    switch (t.n_det) {
    case 1: GW_DISPATCH(1)
    case 2: GW_DISPATCH(2)
    case 3: GW_DISPATCH(3)
    case 4: GW_DISPATCH(4)
    case 5: GW_DISPATCH(5)
    case 6: GW_DISPATCH(6)
    case 7: GW_DISPATCH(7)
    case 8: GW_DISPATCH(8)
    default: return cudaErrorInvalidValue;
    }
#undef GW_DISPATCH
}

static int g_ctas_per_sm[GW_MAX_DET + 1] = {0};
static int g_cluster_ok[GW_MAX_DET + 1] = {0};

template <int NDET>
static cudaError_t configure_one()
{
    const int smem = (int)fused_smem_bytes_exclusive(NDET);
    cudaError_t e;
    const void *variants[8] = {
        (const void *)fused_kernel<NDET, false, false, false>, (const void *)fused_kernel<NDET, true, false, false>,
        (const void *)fused_kernel<NDET, false, true, false>,  (const void *)fused_kernel<NDET, true, true, false>,
        (const void *)fused_kernel<NDET, false, false, true>,  (const void *)fused_kernel<NDET, true, false, true>,
        (const void *)fused_kernel<NDET, false, true, true>,   (const void *)fused_kernel<NDET, true, true, true>};
    for (int v = 0; v < 8; ++v) {
        e = cudaFuncSetAttribute(variants[v], cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (v & 1) {                                         // multi-lane variants: clusters of up to 16 chunks
            e = cudaFuncSetAttribute(variants[v], cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (e != cudaSuccess) return e;
        }
    }
    int n = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fused_kernel<NDET, false, false, false>, kThreads, fused_smem_bytes(NDET));
    if (e != cudaSuccess) return e;
    g_ctas_per_sm[NDET] = n > 0 ? n : 1;
    // can a cluster of kMaxCluster exclusive CTAs (one per SM) be co-scheduled at all on this device?
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(kMaxCluster); cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = (size_t)smem;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = kMaxCluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int n_clusters = 0;
        const cudaError_t ec = cudaOccupancyMaxActiveClusters(&n_clusters, fused_kernel<NDET, true, false, false>, &cfg);
        if (ec != cudaSuccess) cudaGetLastError();
        g_cluster_ok[NDET] = (ec == cudaSuccess && n_clusters > 0) ? 1 : 0;
    }
    return cudaSuccess;
}

cudaError_t configure_kernels(int *out)
{
    cudaError_t e;

    if ((e = configure_one<1>()) != cudaSuccess) return e;
    if ((e = configure_one<2>()) != cudaSuccess) return e;
    if ((e = configure_one<3>()) != cudaSuccess) return e;
    if ((e = configure_one<4>()) != cudaSuccess) return e;
    if ((e = configure_one<5>()) != cudaSuccess) return e;
    if ((e = configure_one<6>()) != cudaSuccess) return e;
    if ((e = configure_one<7>()) != cudaSuccess) return e;
    if ((e = configure_one<8>()) != cudaSuccess) return e;
    if (out) for (int i = 0; i <= GW_MAX_DET; ++i) out[i] = g_ctas_per_sm[i];
    return cudaSuccess;
}
int fused_ctas_per_sm(int n_det) { return (n_det >= 1 && n_det <= GW_MAX_DET) ? g_ctas_per_sm[n_det] : 0; }
int fused_cluster_ok(int n_det) { return (n_det >= 1 && n_det <= GW_MAX_DET) ? g_cluster_ok[n_det] : 0; }

} // namespace gw

#ifdef GW_TIMELINE
// Diagnostic build only: the buffer (32 unsigned 64-bit words per CTA of the largest grid, device memory, zeroed by the
// caller) the fused kernel's CTAs stamp into; NULL switches the stamps off.  Returns the cudaError_t.
extern "C" int gw_timeline_set_buffer(unsigned long long *dev_ptr)
{
    return (int)cudaMemcpyToSymbol(gw::g_timeline, &dev_ptr, sizeof(dev_ptr));
}
#endif
