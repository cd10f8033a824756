// gw_internal.h -- host-side structs shared by gw_api.cu (C-ABI + host logic) and gw_kernels.cu
// (kernels + launchers).  Not part of the public boundary (include/gwlnl.h).  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/gwlnl.h"

namespace gw {

// Tunables (compile-time; build.py may override them with -D for sweeps).
#ifndef GW_THREADS
#define GW_THREADS 256
#endif
#ifndef GW_MIN_CTAS
#define GW_MIN_CTAS 2
#endif
#ifndef GW_UNROLL
#define GW_UNROLL 5
#endif
#ifndef GW_PIPELINE
#define GW_PIPELINE 1
#endif
#ifndef GW_STAGE_BINS
#define GW_STAGE_BINS 160
#endif
#ifndef GW_STAGES
#define GW_STAGES 3
#endif
constexpr int kThreads    = GW_THREADS;     // threads per CTA of the fused and waveform kernels
constexpr int kMinCtas    = GW_MIN_CTAS;    // __launch_bounds__ residency target of the fused kernel
constexpr int kStageBins  = GW_STAGE_BINS;  // bins per shared-memory stage of the fused kernel
constexpr int kStages     = GW_STAGES;      // stage ring depth
constexpr int kUnroll     = GW_UNROLL;      // bins per unrolled trip of the fused hot loop
// The lanes-interleaved sweep keeps each lane's bins at stride lpp <= 32 across stage boundaries, and every stage
// plane is one bulk copy of 16-byte elements.
static_assert(kStageBins % 32 == 0, "GW_STAGE_BINS must be a multiple of 32 (lanes-interleaved sweep, f_last seed)");
static_assert((kStageBins * 16) % 128 == 0, "stage planes must keep the 128-byte alignment of the bulk copies");
static_assert(kStages >= 2 && kThreads % 32 == 0 && kThreads <= 1024, "stage ring / CTA shape");
constexpr int kBasis      = 8;     // per-bin phase basis values (4 planes of 2)
constexpr int kBasisPlanes = 5;    // (x^-5,x^-3) (x^-2,x^-1) (ln f,x) (x ln f,x^2) (f,f^-7/6)
constexpr int kFinishGroup = 16;   // chunks per group of the two-level finish
constexpr int kFinishTwoLevelFrom = 33;  // n_chunks from which the finish is two-level
constexpr int kMaxCluster = 16;          // chunks per tile up to which they are launched as one cluster (non-portable size)
constexpr int kExclusiveSmemBytes = 120 * 1024;   // > half of an SM's 228 KB: at most one such CTA per SM
constexpr int kRecFixed   = 10;    // record fields before the per-detector block
constexpr int kRecPerDet  = 5;     // tau, Cre, Cim, rot_re, rot_im
// record fields: 0..8 phase coefficients, then kRecPerDet per detector, then f_ISCO and the index of the last
// bin with f_j <= f_ISCO (as a double), then the two tidal coefficients (of x^5 and x^7; zero without the option)
__host__ __device__ constexpr int rec_field_fisco(int n_det) { return 9 + kRecPerDet * n_det; }
__host__ __device__ constexpr int rec_field_jcut(int n_det)  { return 10 + kRecPerDet * n_det; }
__host__ __device__ constexpr int rec_field_t10(int n_det)   { return 11 + kRecPerDet * n_det; }
__host__ __device__ constexpr int rec_field_t12(int n_det)   { return 12 + kRecPerDet * n_det; }
__host__ __device__ constexpr int rec_fields(int n_det)      { return 13 + kRecPerDet * n_det; }

// One detector as the kernels see it (built on the host from gw_detector).
struct DetGeom {
    int    kind;          // GW_DET_GEOMETRIC | GW_DET_FIXED
    double D[6];          // detector tensor (xx, xy, xz, yy, yz, zz) = (x(x)x - y(x)y)/2
    double rc[3];         // vertex / c  [s]
    double fplus, fcross, dt_s;
};
struct DetSet { DetGeom d[GW_MAX_DET]; };

// Device tables of a context (all owned by the context).
struct Tables {
    int64_t n_bins;       // M
    int64_t n_pad;        // allocated bins per plane (>= M, multiple of 32)
    int     n_det;
    double  f0, delta_f;
    double *planes;       // [5 + n_det][n_pad][2]: the five basis planes above, then g_I (re,im) per detector
    double  i7[GW_MAX_DET];   // host copy of I7_I = sum_j (4 df/S_Ij) f_j^(-7/3)
    double *i7cum;        // isco_cut only: [n_det][n_pad] inclusive prefix sums of (4 df/S_Ij) f_j^(-7/3)
    int     isco_cut, phase_marginal;
    int     tidal_order;  // 0 | 1 (5PN) | 2 (5PN + 6PN): NEXT-1 option
    int     n_param;      // doubles per theta row: GW_NPARAM, or GW_NPARAM_TIDAL with the tidal option
};

// Launch shape of one gw_lnl_batch call (a pure function of n_prop and the context; fixes summation order).
// The (tile, bin) pairs of a call form one flattened space of work = n_tiles * n_bins positions, tile-major; CTA k of
// n_cta sweeps the contiguous range [k work / n_cta, (k+1) work / n_cta).  Where a range crosses a tile boundary the
// CTA sweeps two (or more) SEGMENTS, one per tile; a tile's segments are summed in ascending bin order.  With
// n_cta = n_tiles * n_chunks the ranges are the n_chunks equal chunks of every tile (the round-1 shape, and what
// gw_ctx_force_plan pins); with n_cta = SMs x resident CTAs every CTA gets the same number of bins whatever the
// shape -- no idle SMs, no second partial wave.
struct Plan {
    int     lpp;          // lanes per proposal (1,2,4,...,32)
    int     props_per_cta;// kThreads / lpp
    int64_t n_tiles;      // ceil(n_prop / props_per_cta)
    int64_t n_cta;        // CTAs of the grid
    int     max_seg;      // upper bound of segments per tile (what gw_ctx_plan reports as n_chunks)
    int     gmax;         // groups per tile of the two-level finish: stride of the group workspace (>= 1)
    int     exclusive;    // 1: the grid has at most one CTA per SM and is launched so that no SM takes two
    int     cluster;      // > 0: aligned multi-lane grid whose n_chunks (= cluster) chunks per tile form a thread-block cluster
    int     vbins;        // boundary bins between consecutive tiles in the flattened space (0 on aligned grids; see segment_at)
};

// ---- flattened work ranges (shared by the kernel, the planner and the CPU tests of the host logic) --------------
// first flattened position of CTA k
__host__ __device__ inline int64_t work_begin(int64_t k, int64_t work, int64_t n_cta) { return (k * work) / n_cta; }
// the CTA whose range holds flattened position p: the largest k with floor(k work / n_cta) <= p
__host__ __device__ inline int64_t cta_of_position(int64_t p, int64_t work, int64_t n_cta)
{
    return ((p + 1) * n_cta + work - 1) / work - 1;
}
// size of the flattened space: n_tiles tiles of n_bins bins with vbins boundary positions between consecutive tiles
__host__ __device__ inline int64_t flattened_work(int64_t n_tiles, int64_t n_bins, int64_t vbins)
{
    return n_tiles * (n_bins + vbins) - vbins;
}
// One segment = the part of a CTA's range that lies in one tile.
// Boundary bins: a CTA whose range crosses a tile boundary pays a segment end (seed, partial store, fence, ticket) and a
// second prologue, about as long as sweeping 30 bins.  So that such a CTA still finishes with the others, every tile but
// the last is n_bins + vbins = tile_len positions long in the flattened space: the vbins positions behind a tile's last
// bin hold no work, and a range that crosses them has that many bins less to sweep.  A range that only touches a tile's
// boundary positions is a segment of no bins (j0 = j1 = n_bins): it contributes zeros and takes its ticket like any
// other -- the hot kernel has no branch around a segment (a branch there costs the hot loop 5 % through ptxas's register
// allocation).  vbins = 0 gives plain equal shares.
struct Segment {
    int64_t tile, j0, j1;  // bins [j0, j1) of proposal tile `tile`
    int64_t len;           // flattened positions of the range that lie in this tile (>= j1 - j0)
    int64_t first_cta;     // the CTA that holds the tile's first bin
    int     index;         // position among the tile's segments (ascending bins) = cta - first_cta
    int     count;         // segments of the tile
    int64_t slot;          // partial-sum slot = cta + tile: consecutive along a tile, unique over the grid
};
__host__ __device__ inline Segment segment_at(int64_t w, int64_t w_end, int64_t cta, int64_t n_bins, int64_t tile_len,
                                              int64_t work, int64_t n_cta)
{
    Segment s;
    s.tile = w / tile_len;
    const int64_t p0 = w - s.tile * tile_len;                 // position within the tile, boundary positions included
    const int64_t left = w_end - w;
    const int64_t p1 = (tile_len - p0 < left) ? tile_len : p0 + left;
    s.len = p1 - p0;
    s.j0 = p0 < n_bins ? p0 : n_bins;
    s.j1 = p1 < n_bins ? p1 : n_bins;
    s.first_cta = cta_of_position(s.tile * tile_len, work, n_cta);
    const int64_t t_end = s.tile * tile_len + tile_len;       // one past the tile's last position (boundary positions included)
    const int64_t last_cta = cta_of_position((t_end < work ? t_end : work) - 1, work, n_cta);
    s.index = (int)(cta - s.first_cta);
    s.count = (int)(last_cta - s.first_cta + 1);
    s.slot = cta + s.tile;
    return s;
}

struct Workspace {
    int64_t max_batch;    // reserved proposals
    int64_t rec_stride;   // proposals per record field (>= max_batch, multiple of 32)
    double *rec;          // [kRecFixed + kRecPerDet*n_det][rec_stride]
    double *partial;      // chunk partials, size partial_doubles
    int64_t partial_doubles;
    unsigned int *tickets;// [max tiles]
    int64_t n_tickets;
    double *gpartial;     // group sums of the two-level finish, gpartial_doubles
    int64_t gpartial_doubles;
    unsigned int *gtickets;
    int64_t n_gtickets;
    double *theta_stage;  // [max_batch][n_param]     (host-variant staging)
    double *lnl_stage;    // [max_batch]
    double *parts_stage;  // [max_batch][n_det][3]
    double *h_stage;      // waveform slab staging (host variant), h_stage_doubles
    int64_t h_stage_doubles;
};

// ---- launchers (gw_kernels.cu).  All return the cudaError_t of the launch. ------------------------------
cudaError_t launch_precompute(const Tables &t, const double *freqs_dev, const double *data_dev,
                              const double *psd_dev, double *i7_dev, cudaStream_t s, int64_t *launches);
cudaError_t launch_setup(const Tables &t, const DetSet &dets, double gmst, int spin_order, int64_t n_prop,
                         const double *theta_dev, double *rec, int64_t rec_stride, double rot_stride_hz,
                         int relative_tau, int stage_theta, cudaStream_t s, int64_t *launches);
cudaError_t launch_fused(const Tables &t, const Plan &plan, int64_t n_prop, const double *rec,
                         int64_t rec_stride, double *partial, unsigned int *tickets, double *gpartial,
                         unsigned int *gtickets, double *lnl_out, double *parts_out, cudaStream_t s, int64_t *launches);
// chunk partial sums: one slot of 2 n_det props_per_cta doubles per segment
inline int64_t plan_partial_slots(const Plan &p) { return p.n_cta + p.n_tiles; }
cudaError_t launch_waveform(const Tables &t, int64_t n_prop, const double *rec, int64_t rec_stride,
                            double *h_out, cudaStream_t s, int64_t *launches);
cudaError_t configure_kernels(int *fused_ctas_per_sm);      // smem attributes + occupancy query (per n_det below)
int         fused_ctas_per_sm(int n_det);
int         fused_cluster_ok(int n_det);       // 1: clusters of kMaxCluster fused CTAs can be scheduled on this device
size_t      fused_smem_bytes(int n_det);

} // namespace gw
