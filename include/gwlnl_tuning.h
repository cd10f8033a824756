/*
 * gwlnl_tuning.h -- testing / tuning / measurement aids exported by csrc/libgwlnl.so next to the product boundary
 * of gwlnl.h.  They are not part of the surface SURVEY.md 8(b) lists: the tests use them to force every launch shape
 * of the fused kernel, bench.py to time the kernels one by one.  Same conventions as gwlnl.h (int return codes,
 * opaque context, no allocation in the batch path).
 */
#ifndef GWLNL_TUNING_H
#define GWLNL_TUNING_H

#include "gwlnl.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Testing / tuning aid: pin the launch shape gw_lnl_batch uses (lanes_per_prop in {1,2,4,8,16,32}, n_chunks >= 1
 * frequency chunks per proposal tile); 0 leaves that choice to the planner.  A pinned shape whose partial sums do not
 * fit the reserved workspace makes gw_lnl_batch return GW_ERR_INVALID_ARG.                              */
int gw_ctx_force_plan(gw_ctx *ctx, int lanes_per_prop, int n_chunks);

/* Testing / tuning aid: pin the grid instead -- n_ctas CTAs share the flattened (proposal tile, bin) space equally,
 * whatever the tile count (n_ctas >= 1; 0 leaves the choice to the planner; overrides a pinned n_chunks).       */
int gw_ctx_force_grid(gw_ctx *ctx, int lanes_per_prop, int64_t n_ctas);

/* Testing / tuning aid: multi-lane grids of 2..16 chunks per tile launch every tile as one thread-block cluster and add
 * the chunk sums through distributed shared memory (default, enable = 1); 0 sends them through the global partial sums
 * and the per-tile ticket like every other grid.  Both paths add the same numbers in the same order (identical bits).  */
int gw_ctx_cluster_finish(gw_ctx *ctx, int enable);

/* Testing / tuning aid: gw_lnl_batch_host sends batches of up to 512 proposals through a library-owned CUDA graph (one
 * launch per call; default, enable = 1); 0 makes it enqueue the copy and the two kernels one by one like larger batches. */
int gw_ctx_host_graph(gw_ctx *ctx, int enable);

/* Host-only (no CUDA call): the segments that CTA `cta` of a grid of n_ctas CTAs sweeps when n_tiles proposal tiles
 * of n_bins bins, separated by boundary_bins positions without work (gw_ctx_boundary_bins; 0 = none), are shared
 * equally -- the same arithmetic the fused kernel runs (csrc/gw_internal.h, segment_at).  A range that only touches
 * boundary positions of a tile yields a row with j0 == j1 == n_bins (a segment of no bins).
 * Writes up to max_rows rows of 6 values (tile, j0, j1, index of the segment within its tile, segments of that tile,
 * partial-sum slot) and returns the number of segments of the CTA, or GW_ERR_INVALID_ARG.                     */
int gw_plan_cta_segments(int64_t n_tiles, int64_t n_bins, int64_t boundary_bins, int64_t n_ctas, int64_t cta, int max_rows,
                         int64_t *rows6);

/* Testing / tuning aid: on balanced grids (n_ctas not a multiple of the tile count) consecutive tiles are separated by
 * boundary positions without work in the flattened space, so that a CTA whose range crosses a tile boundary -- and pays
 * a segment end and a second prologue -- sweeps that many bins less and finishes with the others (default 30 per lane;
 * 0 = plain equal shares).  gw_ctx_plan_boundary_bins reports the value a batch size's plan uses (0 on aligned grids). */
int gw_ctx_boundary_bins(gw_ctx *ctx, int boundary_bins);
int gw_ctx_plan_boundary_bins(const gw_ctx *ctx, int64_t n_prop, int *boundary_bins);

/* Measurement aid: when enabled, the *_batch calls record CUDA events on their stream before the setup
 * kernel, between the setup kernel and the main (fused or waveform) kernel, and after it.  The event between
 * the two launches removes their programmatic overlap, so enable it only for kernel-level timing.
 * gw_ctx_last_kernel_ms waits for the most recent call and returns the two durations.                  */
int gw_ctx_kernel_timing(gw_ctx *ctx, int enable);
int gw_ctx_last_kernel_ms(gw_ctx *ctx, double *setup_ms, double *main_ms);

#ifdef __cplusplus
}
#endif
#endif /* GWLNL_TUNING_H */
