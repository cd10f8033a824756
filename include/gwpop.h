/*
 * gwpop.h -- C-ABI of the population ("recycling") likelihood, the paper's second GPU workload.
 * Implemented in csrc/gw_pop.cu, exported by csrc/libgwlnl.so.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, section IV): Eq. 3
 *
 *   L_tot({d_i} | Lambda, R)  proportional to  R^N e^{-R VT(Lambda)} prod_i sum_j p(theta_ij | Lambda) / p(theta_ij | 0)
 *
 * without the rate / selection prefactor, which the paper's own benchmark leaves out ("For the
 * benchmarking performed in this work, we ignore this quantity"):
 *
 *   lnL(Lambda) = sum_{i=1..N} ln [ sum_{j=1..n} p(theta_ij | Lambda) / p(theta_ij | 0) ]
 *
 * for a BATCH of hyper-parameter proposals Lambda per call.  Data flow as in the paper: the N x n
 * arrays of posterior samples (an equal number n per event) are moved to the GPU once, at context creation; a call
 * evaluates the probabilities, the sums and the logarithms there and returns one number per Lambda.
 *
 * PAPER.md cites its population models without printing them; the closed forms are DESIGN.md section
 * 14, reading P1:
 *   theta  = (m1 [Msun], q = m2/m1, a1, a2, cos tilt_1, cos tilt_2)                         GW_POP_T_* below
 *   Lambda = (alpha, m_min, m_max, lam, m_pp, sig_pp, beta_q, alpha_chi, beta_chi, xi, sig_1, sig_2)  GW_POP_L_*
 *   p(m1)     = (1 - lam) PL(m1; -alpha, [m_min, m_max]) + lam TN(m1; m_pp, sig_pp, [m_min, m_max])
 *   p(q | m1) = PL(q; +beta_q, [m_min / m1, 1])
 *   p(a)      = Beta(a; alpha_chi, beta_chi) for a1 and for a2
 *   p(c1, c2) = (1 - xi)/4 + xi TN(c1; 1, sig_1, [-1, 1]) TN(c2; 1, sig_2, [-1, 1])
 * (PL: normalised power law; TN: truncated, renormalised normal density).
 *
 * Conventions: those of gwlnl.h -- int return codes GW_OK / GW_ERR_*, opaque context that owns its device memory,
 * "dev" / "host" pointers, batch calls enqueue on `cuda_stream` without synchronising, allocating or copying between
 * host and device, fixed-order reductions only (bit-reproducible), IEEE fp64.  Lambda lives on the device and is not
 * validated on the host: a Lambda outside the model's domain (non-finite entry, m_min <= 0, m_max <= m_min, lam or xi
 * outside [0, 1], a non-positive sigma, alpha_chi or beta_chi) yields NaN for that Lambda only; a Lambda under which
 * some event has no sample inside the support yields -inf.  Whether a sample lies inside the support is decided as
 * m_min <= m1 <= m_max and ln q >= ln m_min - ln m1 in fp64.
 */
#ifndef GWPOP_H
#define GWPOP_H

#include <stdint.h>

#include "gwlnl.h"

#ifdef __cplusplus
extern "C" {
#endif

enum { GW_POP_T_M1 = 0, GW_POP_T_Q, GW_POP_T_A1, GW_POP_T_A2, GW_POP_T_C1, GW_POP_T_C2, GW_POP_NTHETA = 6 };
enum { GW_POP_L_ALPHA = 0, GW_POP_L_MMIN, GW_POP_L_MMAX, GW_POP_L_LAM, GW_POP_L_MPP, GW_POP_L_SIGPP, GW_POP_L_BETAQ,
       GW_POP_L_ALPHACHI, GW_POP_L_BETACHI, GW_POP_L_XI, GW_POP_L_SIG1, GW_POP_L_SIG2, GW_POP_NLAMBDA = 12 };

typedef struct gw_pop_ctx gw_pop_ctx;    /* opaque */

/* Create a context: validate and copy the samples, then run the precompute kernel that builds the per-sample planes
 * the batch calls stream (ln m1, m1, ln q, ln a1 + ln a2, ln(1-a1) + ln(1-a2), (c1-1)^2, (c2-1)^2, -ln prior).
 * Synchronises `cuda_stream` before returning.
 *   n_events   N >= 1;  n_samples  n >= 1 (the same for every event)
 *   samples    [N][n][GW_POP_NTHETA] host or dev; m1 > 0, 0 < q <= 1, 0 < a1, a2 < 1, |c1|, |c2| <= 1, all finite
 *   prior      [N][n] host or dev; p(theta_ij | 0) > 0, finite
 *   max_batch  hyper-parameter proposals per call the workspace is reserved for (>= 1)
 * Errors: GW_ERR_INVALID_ARG, GW_ERR_ALLOC, GW_ERR_CUDA, GW_ERR_ARCH.                                        */
int gw_pop_ctx_create(gw_pop_ctx **out, int64_t n_events, int64_t n_samples, const double *samples,
                      const double *prior, int64_t max_batch, void *cuda_stream);

/* lnL for a batch of hyper-parameter proposals.
 *   lambda_dev   [n_lambda][GW_POP_NLAMBDA] dev
 *   lnl_out_dev  [n_lambda] dev
 * n_lambda == 0 is GW_OK and writes nothing; n_lambda > max_batch is GW_ERR_INVALID_ARG.                     */
int gw_pop_lnl_batch(gw_pop_ctx *ctx, int64_t n_lambda, const double *lambda_dev, double *lnl_out_dev,
                     void *cuda_stream);

/* Host-buffer variant: copies Lambda in, computes, copies lnL out and synchronises the stream.              */
int gw_pop_lnl_batch_host(gw_pop_ctx *ctx, int64_t n_lambda, const double *lambda_host, double *lnl_out_host,
                          void *cuda_stream);

/* Destroy a context and free everything it owns.  NULL is a no-op returning GW_OK.                          */
int gw_pop_ctx_destroy(gw_pop_ctx *ctx);

/* Introspection.  Any output pointer may be NULL.  chunks_per_event: first-stage partial sums per event, which
 * (with n_samples) fixes the summation order.                                                               */
int gw_pop_ctx_info(const gw_pop_ctx *ctx, int64_t *n_events, int64_t *n_samples, int64_t *max_batch,
                    int *chunks_per_event);

/* Number of kernel launches enqueued through this context so far.                                           */
int64_t gw_pop_ctx_launch_count(const gw_pop_ctx *ctx);

/* Measurement aid (as gw_ctx_kernel_timing in gwlnl_tuning.h): record CUDA events around the main kernel of each
 * batch call; gw_pop_ctx_last_kernel_ms waits for the most recent call and returns the setup, main (map + first-stage
 * reduce) and finish kernel durations.                                                                      */
int gw_pop_ctx_kernel_timing(gw_pop_ctx *ctx, int enable);
int gw_pop_ctx_last_kernel_ms(gw_pop_ctx *ctx, double *setup_ms, double *main_ms, double *finish_ms);

/* ---- The no-allocation entry point ---------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): Eq. 3 for a batch of Lambda straight from device-resident samples, WITHOUT a context.  gw_pop_lnl_static calls
 * no cudaMalloc, cudaFree or other allocating routine, never synchronises and never copies between host and device:
 * it enqueues one 256-byte memset and five kernels on `cuda_stream` -- the kernels of gw_pop_lnl_batch (precompute,
 * setup, map-reduce, finish: same grids, same summation order, so the same bits) plus a one-line flag check.  All of
 * its scratch -- the 8 per-sample planes, the Lambda records, the first-stage partial sums, the bad-sample flag -- lives
 * in ONE file-scope `static __device__` array of GW_POP_STATIC_SCRATCH_DOUBLES doubles (16 MiB) inside the library;
 * every GPU that loads the library holds that array until the process exits.
 *   samples_dev  [N][n][GW_POP_NTHETA] dev (same domain as gw_pop_ctx_create);  prior_dev  [N][n] dev
 *   lambda_dev   [n_lambda][GW_POP_NLAMBDA] dev;  lnl_out_dev  [n_lambda] dev
 *   All four must be device memory of the CURRENT device; the caller owns them and keeps them alive until the stream
 *   has run the call.
 * Limit: gw_pop_static_need(N, n, n_lambda) = 32 + r32(16 n_lambda) + r32(n_lambda N ceil(n / 1024)) + 8 N n doubles
 * (r32 rounds up to a multiple of 32) must not exceed GW_POP_STATIC_SCRATCH_DOUBLES: about 2.6e5 samples in total
 * (PAPER.md:119's GWTC-1 catalogue of 10 x 20000 fits with 64 Lambda; PAPER.md:115's 4e6 samples do not -- use a
 * context).  A larger problem is rejected with GW_POP_ERR_TOO_LARGE before anything is enqueued.
 * Samples cannot be validated on the host without a synchronisation: if any sample or prior value is outside the
 * documented domain, every lnL of that call is NaN (gw_pop_ctx_create returns GW_ERR_INVALID_ARG instead).
 * The array is shared by every call on a device and keeps the last call's contents.  Nothing in it has to survive
 * between calls; the one word that must start at zero (the bad-sample flag) is cleared by the call itself.  Calls
 * enqueued on ONE stream are ordered and safe; calls that overlap on the GPU (different streams, or different host
 * threads on different streams) RACE on the array and return garbage -- serialise them.  The first call on each
 * device looks up the array's device address (once per device; make that call outside stream capture).
 * Errors: GW_ERR_INVALID_ARG (NULL, bad size, a pointer that is not device memory of the current device),
 * GW_POP_ERR_TOO_LARGE, GW_ERR_ARCH, GW_ERR_CUDA (gw_pop_static_last_cuda_error has the cudaError).
 * n_lambda == 0 is GW_OK and enqueues nothing.                                                              */
#define GW_POP_STATIC_SCRATCH_DOUBLES 2097152      /* 16 MiB per GPU                                          */
#define GW_POP_ERR_TOO_LARGE (-16)                 /* the problem needs more scratch than the static array has  */
int gw_pop_lnl_static(int64_t n_events, int64_t n_samples, const double *samples_dev, const double *prior_dev,
                      int64_t n_lambda, const double *lambda_dev, double *lnl_out_dev, void *cuda_stream);

/* Doubles of static scratch a problem of this size needs (host arithmetic only), or -1 for sizes that
 * gw_pop_lnl_static rejects as GW_ERR_INVALID_ARG (N < 1, n < 1, n_lambda < 0 or > 2^24, N n > 4e9).          */
int64_t gw_pop_static_need(int64_t n_events, int64_t n_samples, int64_t n_lambda);

/* cudaError of the most recent GW_ERR_CUDA return of gw_pop_lnl_static in this process (0 if none).         */
int gw_pop_static_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GWPOP_H */
