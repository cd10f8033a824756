/*
 * gwlnl.h -- C-ABI boundary of the B200-native (sm_100a) batched TaylorF2 waveform +
 * detector projection + Gaussian noise-weighted likelihood library.
 *
 * What the library computes (PAPER.md = /root/reference/PAPER.md, "Parallelized Inference for
 * Gravitational-Wave Astronomy", arXiv:1904.02863):
 *
 *   lnL(theta) = sum_det [ Re<d|h(theta)> - 1/2 <h(theta)|h(theta)> ],
 *   <a|b>      = 4 df sum_f a(f) conj(b(f)) / S_n(f),
 *
 * the theta-dependent part of the paper's single-event likelihood, Eq. 1 (section III:
 * exponent -(2/T)|d-h|^2/S with df = 1/T), for a BATCH of sampler proposals theta per call.  The
 * template h is "the template for the response of the detector", each detector's copy
 * "multiplied by a factor of exp(-2 i pi f dt_det)" (section III); "the value at each
 * frequency can be evaluated independently" (section II).  PAPER.md prints no waveform
 * formula; BASELINE.json's north_star fixes it to the TaylorF2 stationary-phase inspiral (3.5PN phase,
 * Newtonian amplitude, aligned spins at 1.5PN spin-orbit + 2PN spin-spin), written out in DESIGN.md
 * section 2 (steps O1..O7) with the readings of DESIGN.md section 3.
 *
 * Conventions common to every entry point
 *   - Every function returns an int: GW_OK (0) or a negative GW_ERR_* code.  Nothing throws, aborts
 *     or prints.  gw_strerror() names a code; gw_last_cuda_error() returns the CUDA error behind the
 *     most recent GW_ERR_CUDA of a context.
 *   - "dev" pointers are CUDA device pointers on the context's device; "host" pointers are ordinary
 *     host memory.  gw_ctx_create accepts either kind for its three arrays (it asks the CUDA runtime).
 *   - Ownership: the caller owns everything it passes in and every output buffer.  The context owns
 *     its tables and workspace and frees them in gw_ctx_destroy.  gw_ctx_create copies its inputs.
 *   - Asynchrony: the *_batch calls enqueue on `cuda_stream` (a cudaStream_t passed as void*, NULL =
 *     the legacy default stream) and return without synchronising, allocating or copying between
 *     host and device (the paper's reusable-buffer lesson).  The *_host variants
 *     copy in, compute, copy out and synchronise the stream before returning.
 *   - A context may be used from one stream at a time (it owns one workspace).
 *   - A context belongs to the device that was current in gw_ctx_create; later calls make that device current
 *     for their duration and restore the caller's.
 *   - Determinism: same context, same theta, same n_prop, same build, same GPU model => bit-identical
 *     outputs (fixed-order reductions only; no floating-point atomics).
 *   - theta lives on the device and is not validated on the host.  A proposal with Mc <= 0, q outside
 *     (0, 1], D <= 0, |cos iota| > 1, |chi| > 1 or any non-finite entry yields NaN in that proposal's
 *     outputs and does not affect other proposals.  So does a proposal whose phase could exceed 2.5e8 turns
 *     anywhere in the band (e.g. Mc < ~2e-3 Msun from 10 Hz), the domain of the integer range reduction.
 *   - All arithmetic is IEEE fp64; complex numbers are interleaved (re, im) pairs of doubles.
 */
#ifndef GWLNL_H
#define GWLNL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GW_ABI_VERSION 5

enum {
    GW_OK              =  0,
    GW_ERR_INVALID_ARG = -1,   /* NULL, bad size, non-uniform grid, non-positive PSD, n_prop > reserved ... */
    GW_ERR_ALLOC       = -2,   /* host or device allocation failed                                          */
    GW_ERR_CUDA        = -3,   /* a CUDA runtime call failed; see gw_last_cuda_error                         */
    GW_ERR_ARCH        = -4    /* the current device is not compute capability 10.x (sm_100a code only)      */
};

/* Detector description (step O6).
 * GW_DET_GEOMETRIC: antenna patterns F+, Fx(ra, dec, psi, gmst) and the geocentric delay are computed
 *   per proposal from the vertex position and the two arm directions (Earth-fixed frame):
 *   detector tensor D = (x (x) x - y (x) y)/2, delay dt = -(r . n)/c.
 * GW_DET_FIXED: F+, Fx, dt are the three given numbers for every proposal (BASELINE.json configs[0]:
 *   "optimally oriented, F+=1, Fx=0, dt=0").                                                            */
enum { GW_DET_GEOMETRIC = 0, GW_DET_FIXED = 1 };

typedef struct gw_detector {
    int    kind;                 /* GW_DET_GEOMETRIC | GW_DET_FIXED                                       */
    double vertex_m[3];          /* GEOMETRIC: vertex, Earth-fixed Cartesian, metres                      */
    double xarm[3], yarm[3];     /* GEOMETRIC: unit vectors along the arms, Earth-fixed                   */
    double fplus, fcross, dt_s;  /* FIXED: response and time delay (seconds)                              */
} gw_detector;

typedef struct gw_options {      /* NULL => { spin_order 1, isco_cut 0, max_batch 4096, phase_marginal 0, tidal_order 0 } */
    int     spin_order;          /* 0: no spin terms; 1: 1.5PN spin-orbit + 2PN spin-spin (A7);
                                    2 (NEXT-1 option): also the spin-orbit terms linear
                                    in the spins at 2.5PN, 3PN and 3.5PN                                   */
    int     isco_cut;            /* 0 (default, A6): every bin of the band is evaluated;
                                    1 (NEXT-1 option): h = 0 for f > f_ISCO =
                                    1/(6^(3/2) pi M) of the proposal's total mass                         */
    int64_t max_batch;           /* workspace reservation in proposals (>= 1); grow with gw_ctx_reserve   */
    int     phase_marginal;      /* 0: lnL at the proposal's phi_c; 1 (NEXT-1 option): lnl_out holds the
                                    likelihood marginalised over phi_c with a uniform prior,
                                    ln I0(|sum_I <d|h>_I|) - 1/2 sum_I <h|h>_I; parts are unchanged        */
    int     tidal_order;         /* 0: point masses; 1 | 2 (NEXT-1 option): 5PN | 5PN + 6PN
                                    adiabatic tidal phase terms; theta rows then have GW_NPARAM_TIDAL columns  */
} gw_options;

/* Column order of one proposal theta[GW_NPARAM] (units: Msun, -, -, -, Mpc, s, rad, -, rad, rad, rad):
 * chirp mass, mass ratio q = m2/m1 in (0,1], aligned spins chi1, chi2, luminosity distance,
 * geocentric coalescence time measured from the segment start, coalescence phase, cos(inclination),
 * right ascension, declination, polarisation angle.                                                     */
enum { GW_P_MC = 0, GW_P_Q, GW_P_CHI1, GW_P_CHI2, GW_P_DL, GW_P_TC, GW_P_PHIC,
       GW_P_COSI, GW_P_RA, GW_P_DEC, GW_P_PSI, GW_NPARAM = 11 };
/* A context created with tidal_order > 0 reads GW_NPARAM_TIDAL columns per proposal: the eleven above, then the
 * dimensionless tidal deformabilities Lambda_1 (of the heavier body, mass m1) and Lambda_2, each finite and >= 0
 * (else that proposal's outputs are NaN).  The phase gains 3/(128 eta) v^-5 (phi_10 v^10 + phi_12 v^12) with
 * phi_10 = -sum_A 24 (12 - 11 X_A) X_A^4 Lambda_A, phi_12 = -sum_A (5/28)(3179 - 919 X_A - 2286 X_A^2 +
 * 260 X_A^3) X_A^4 Lambda_A, X_A = m_A/M (phi_12 only for tidal_order 2).  "theta [n_prop][GW_NPARAM]" below reads
 * "[n_prop][gw_ctx_n_param(ctx)]" for such a context.                                                      */
enum { GW_P_LAMBDA1 = 11, GW_P_LAMBDA2 = 12, GW_NPARAM_TIDAL = 13 };

#define GW_MAX_DET 8             /* detectors per context (the fused kernel is specialised per count; 1..4 keep two
                                  * CTAs per SM, 5..8 run one CTA per SM with the larger register budget)       */

typedef struct gw_ctx gw_ctx;    /* opaque */

/* Create a context: validate and copy the inputs, then run the per-bin precompute kernel (DESIGN.md
 * section 6, kernel K0; north_star item (2)) that builds the tables the batch calls read:
 * f^(k/3) powers, ln f, f^(-7/6), the 4 df / S_n weights folded into g = (4 df/S) d f^(-7/6), and the
 * per-detector norm I7 = sum_f (4 df/S) f^(-7/3).  Synchronises `cuda_stream` before returning.
 *   out        receives the context (set to NULL on error)
 *   n_bins     M >= 2
 *   freqs_hz   [M] host or dev; strictly positive, ascending, uniform to rounding
 *              (|f_j - f_0 - j df| <= 1e-9 df + 8 ulp(f_max): the time shift is applied by a recurrence on the grid);
 *              df is taken as (f[M-1] - f[0])/(M-1)
 *   n_det      1..GW_MAX_DET
 *   data_ri    [n_det][M][2] host or dev; one-sided continuous-normalised transform d(f), strain/Hz, finite
 *   psd        [n_det][M] host or dev; one-sided S_n(f), strain^2/Hz, finite and > 0
 *   dets       [n_det] host; GEOMETRIC arms must be unit vectors to 1e-6
 *   gmst_rad   Greenwich mean sidereal time of the segment (frozen for the segment)
 *   opt        nullable
 * Errors: GW_ERR_INVALID_ARG, GW_ERR_ALLOC, GW_ERR_CUDA, GW_ERR_ARCH.                                    */
int gw_ctx_create(gw_ctx **out, int64_t n_bins, const double *freqs_hz, int n_det,
                  const double *data_ri, const double *psd, const gw_detector *dets,
                  double gmst_rad, const gw_options *opt, void *cuda_stream);

/* Grow the workspace so that batch calls accept up to `max_batch` proposals.  The only call besides
 * create/destroy that allocates; synchronises the device.  Never shrinks.                              */
int gw_ctx_reserve(gw_ctx *ctx, int64_t max_batch);

/* h(f) for a batch of proposals (north_star item (3); DESIGN.md kernel K2): TaylorF2 carrier, detector
 * projection and time shift, written as complex128.
 *   theta_dev  [n_prop][GW_NPARAM] dev
 *   h_out_dev  [n_prop][n_det][M][2] dev, 16-byte aligned
 * n_prop == 0 is GW_OK and writes nothing; n_prop > reserved is GW_ERR_INVALID_ARG.                     */
int gw_waveform_batch(gw_ctx *ctx, int64_t n_prop, const double *theta_dev, double *h_out_dev,
                      void *cuda_stream);

/* lnL for a batch of proposals (north_star item (4); DESIGN.md kernels K1 + K3): waveform, projection
 * and both inner products fused; h(f) never touches HBM.
 *   theta_dev      [n_prop][GW_NPARAM] dev
 *   lnl_out_dev    [n_prop] dev
 *   parts_out_dev  nullable; [n_prop][n_det][3] dev = Re<d|h>, Im<d|h>, <h|h> per detector              */
int gw_lnl_batch(gw_ctx *ctx, int64_t n_prop, const double *theta_dev, double *lnl_out_dev,
                 double *parts_out_dev, void *cuda_stream);

/* Host-buffer variants: theta_host -> (ctx-owned device staging) -> kernels -> outputs copied back to
 * host; the stream is synchronised before returning.  Pinned host memory makes the copies asynchronous
 * with respect to the host but is not required.  When theta_host is pinned and n_prop >= 2048 the setup kernel reads it
 * in place over the host link (coalesced loads, no staged copy).  When lnl_out_host is pinned (cudaHostAlloc / cudaHostRegister /
 * torch pin_memory) the kernel's finish stage stores lnL straight into it over the host link instead of a staged
 * device-to-host copy; the values are valid when the call returns either way.  The waveform variant processes the
 * batch in slabs of at most 512 MiB through a device staging buffer it allocates on first use.           */
int gw_lnl_batch_host(gw_ctx *ctx, int64_t n_prop, const double *theta_host, double *lnl_out_host,
                      double *parts_out_host, void *cuda_stream);
int gw_waveform_batch_host(gw_ctx *ctx, int64_t n_prop, const double *theta_host, double *h_out_host,
                           void *cuda_stream);

/* Destroy a context and free everything it owns.  NULL is a no-op returning GW_OK.                      */
int gw_ctx_destroy(gw_ctx *ctx);

/* Introspection.  Any output pointer may be NULL.                                                       */
int gw_ctx_info(const gw_ctx *ctx, int64_t *n_bins, int *n_det, double *delta_f, int64_t *max_batch);

/* Doubles per theta row this context reads: GW_NPARAM, or GW_NPARAM_TIDAL with the tidal option; -1 for NULL. */
int gw_ctx_n_param(const gw_ctx *ctx);

/* The launch shape gw_lnl_batch would use for n_prop proposals (what bench.py reports and what fixes
 * the summation order): lanes per proposal, proposals per CTA, number of frequency chunks, CTAs.  The aids that pin
 * this shape or time the kernels individually are declared in gwlnl_tuning.h, outside this boundary.          */
int gw_ctx_plan(const gw_ctx *ctx, int64_t n_prop, int *lanes_per_prop, int *props_per_cta,
                int *n_chunks, int64_t *n_ctas);

/* I7[n_det], the per-detector norm the precompute kernel produced (for tests of kernel K0).            */
int gw_ctx_norms(const gw_ctx *ctx, double *i7_host);

/* Number of kernel launches the library has enqueued through this context so far.                      */
int64_t gw_ctx_launch_count(const gw_ctx *ctx);

const char *gw_strerror(int code);
int gw_last_cuda_error(const gw_ctx *ctx);      /* a cudaError_t value, 0 if none                         */
int gw_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GWLNL_H */
