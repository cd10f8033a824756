// gw_api.cu -- the C-ABI of include/gwlnl.h: context lifetime, input validation, launch planning and the
// batch entry points.  Every step of the hot path runs in the kernels of gw_kernels.cu; this file only
// validates, allocates (create/reserve only) and launches.  There is no CPU fallback.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "gw_internal.h"
#include "../../include/gwlnl_tuning.h"

using namespace gw;

struct gw_ctx {
    int          device;
    int          n_sm;
    int          ctas_per_sm;      // resident fused CTAs per SM for this n_det
    int          spin_order;
    double       gmst;
    DetSet       dets;
    Tables       t;
    Workspace    w;
    int          last_cuda_error;
    int64_t      launches;
    int          force_lpp, force_chunks;   // gw_ctx_force_plan (0 = planner's choice)
    int64_t      force_ctas;       // gw_ctx_force_grid (0 = planner's choice)
    int          cluster_finish;   // 1 (default): multi-lane aligned grids of <= 16 chunks reduce through thread-block clusters
    int64_t      plan_n[4];        // batch sizes of the cached plans (0 = empty): a sampler calls with few distinct sizes
    Plan         plan_of[4];       // make_plan is a pure function of n_prop for a given context and pinned shape
    int          plan_next;
    // Small synchronous host calls (gw_lnl_batch_host, n_prop <= kHostGraphMax) replay a library-owned CUDA graph of the two
    // kernels: theta goes through a pinned, mapped staging buffer that the setup kernel reads in place, lnL and parts come
    // back through pinned, mapped buffers the finish stage stores to, so the call is one graph launch and one synchronise.
    double      *pin_theta, *pin_lnl, *pin_parts;        // host addresses (cudaHostAlloc, mapped)
    double      *pin_theta_dev, *pin_lnl_dev, *pin_parts_dev;
    int64_t      pin_cap;                                 // proposals the pinned buffers hold
    cudaStream_t capture_stream;                          // graphs are captured here and launched on the caller's stream
    int64_t      graph_n[4];       // batch size of a cached graph (0 = empty), with or without parts
    int          graph_parts[4];
    cudaGraphExec_t graph_exec[4];
    int          graph_next;
    int          host_graph;       // 1 (default): use the graph path; gw_ctx_host_graph switches it
    int          boundary_bins;    // per lane: bins a range that crosses a tile boundary is shortened by on balanced grids (gw_ctx_boundary_bins)
    int          timing;           // gw_ctx_kernel_timing: record events around K1 and the main kernel
    cudaEvent_t  ev[3];            // before K1, between K1 and main, after main
};

namespace {

constexpr int64_t kHStageMaxDoubles = (int64_t)1 << 26;       // 512 MiB waveform slab for the host variant
#ifndef GW_HOST_GRAPH_MAX
#define GW_HOST_GRAPH_MAX 512
#endif
constexpr int64_t kHostGraphMax = GW_HOST_GRAPH_MAX;          // largest batch the host variant sends through its graph

int cuda_fail(gw_ctx *ctx, cudaError_t e)
{
    if (ctx) ctx->last_cuda_error = (int)e;
    return e == cudaErrorMemoryAllocation ? GW_ERR_ALLOC : GW_ERR_CUDA;
}

bool is_device_ptr(const void *p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

// device alias of pinned (mapped) host memory, or nullptr for pageable host memory
double *mapped_alias(const void *host_ptr)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, host_ptr) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return at.type == cudaMemoryTypeHost ? static_cast<double *>(at.devicePointer) : nullptr;
}

// ---- launch planning -----------------------------------------------------------------------------------
// Cost model: a CTA sweeps ceil(chunk/lpp) bins per thread plus a fixed prologue /
// epilogue worth ~kProBins bins; an SM runs its resident CTAs concurrently and the fp64 pipe saturates at
// about kSatWarps warps per scheduler.  The plan is a pure function of (n_prop, M, n_det, device), which is
// what makes the summation order reproducible.
constexpr double kProBins  = 14.0;
#ifndef GW_ZERO_COPY_LNL
#define GW_ZERO_COPY_LNL 1
#endif
// host variant: between these batch sizes K1 reads a pinned theta buffer in place (measured: below, the small staged
// copy is as quick and K1 is ~1 us shorter without its staging pass; at 65536 proposals in-place reads took 1.90 ms
// per call in both repeats against 1.90 - 2.2 ms with the staged copy)
#ifndef GW_ZERO_COPY_THETA_MIN
#define GW_ZERO_COPY_THETA_MIN 2048
#endif
#ifndef GW_ZERO_COPY_THETA_MAX
#define GW_ZERO_COPY_THETA_MAX 1048576
#endif
#ifndef GW_SAT_WARPS
#define GW_SAT_WARPS 2.0
#endif
#ifndef GW_EXCLUSIVE_PLANS
#define GW_EXCLUSIVE_PLANS 1
#endif
constexpr double kSatWarps = GW_SAT_WARPS;   // one 8-warp CTA per SM nearly saturates the fp64 pipe (brute-force sweep)
constexpr double kCoResidentGain = 0.985;
constexpr double kCoResidentGainMulti = 0.90;   // the lanes-interleaved loop (shuffles, short chunks) gains more from a second CTA (C0)
constexpr int    kMaxChunks = 4096;
constexpr int64_t kMaxWaves = 8;
#ifndef GW_MULTI_PENALTY
#define GW_MULTI_PENALTY 1.35
#endif
constexpr double kMultiPenalty = GW_MULTI_PENALTY;     // the lanes-interleaved loop costs this much more per bin (measured, C2)
constexpr double kTwoLevelHop = 16.0;      // the second fence + ticket round of the two-level finish (~2 us; C4 B = 1, 16)
#ifndef GW_CLUSTER_FINISH_COST
#define GW_CLUSTER_FINISH_COST 4.0
#endif
#ifndef GW_CLUSTER_MAX_CTAS
#define GW_CLUSTER_MAX_CTAS 32
#endif
constexpr int64_t kClusterMaxCtas = GW_CLUSTER_MAX_CTAS;    // grids up to this many CTAs may be launched as clusters
constexpr double kClusterFinish = GW_CLUSTER_FINISH_COST;   // cluster barrier + one distributed-shared-memory round trip, in bin sweeps
#ifndef GW_BOUNDARY_BINS
#define GW_BOUNDARY_BINS 30
#endif
constexpr int kBoundaryBins = GW_BOUNDARY_BINS;   // a segment end plus a second prologue, in bin sweeps of a one-lane CTA (timeline of C1: 3.3-3.8 us at 0.12 us per bin)
constexpr double kFinishPerChunk = 1.0;    // serial additions of the finish stage, in bin-sweep equivalents each (calibrated on C4 B = 256, 512)

// exact maximum of segments per tile for a grid of n_cta CTAs over n_tiles tiles of M bins
int max_segments_per_tile(int64_t n_tiles, int64_t M, int64_t vbins, int64_t n_cta)
{
    const int64_t L = M + vbins, work = flattened_work(n_tiles, M, vbins);
    if (vbins == 0 && n_cta % n_tiles == 0) return (int)(n_cta / n_tiles);   // aligned grid: every tile in n_cta / n_tiles chunks
    int64_t best = 1;
    for (int64_t t = 0; t < n_tiles; ++t) {
        const int64_t t_end = t * L + L < work ? t * L + L : work;            // boundary positions belong to the tile (segment_at)
        const int64_t c = cta_of_position(t_end - 1, work, n_cta) - cta_of_position(t * L, work, n_cta) + 1;
        if (c > best) best = c;
    }
    return (int)best;
}

Plan make_plan(const gw_ctx *ctx, int64_t n_prop)
{
    const int64_t M = ctx->t.n_bins;
    const int slots_per_sm = ctx->ctas_per_sm > 0 ? ctx->ctas_per_sm : 1;
    const int n_sm = ctx->n_sm > 0 ? ctx->n_sm : 148;
    const int64_t slots = (int64_t)n_sm * slots_per_sm;
    Plan best = {1, kThreads, (n_prop + kThreads - 1) / kThreads, (n_prop + kThreads - 1) / kThreads, 1, 1, 0, 0, 0};
    const int64_t stage_doubles = (int64_t)kStages * (kBasisPlanes + ctx->t.n_det) * kStageBins * 2;   // a CTA's idle stage ring
    double best_cost = 1e300;
    for (int lpp = 1; lpp <= 32; lpp *= 2) {
        if (ctx->force_lpp > 0 && lpp != ctx->force_lpp) continue;
        const int pt = kThreads / lpp;
        const int64_t tiles = (n_prop + pt - 1) / pt;
        const int64_t work = tiles * M;
        int64_t max_chunks = M / ((int64_t)8 * lpp);          // at least 8 iterations per thread
        const int64_t by_waves = (kMaxWaves * slots) / tiles; // no more than kMaxWaves waves of CTAs
        if (max_chunks > by_waves) max_chunks = by_waves;
        if (max_chunks > kMaxChunks) max_chunks = kMaxChunks;
        if (max_chunks < 1) max_chunks = 1;
        int64_t nc_first = 1;
        if (ctx->force_chunks > 0) { nc_first = max_chunks = (ctx->force_chunks < M ? ctx->force_chunks : M); }
        // candidate grids: the aligned ones (every tile in nc equal chunks), and -- unless a shape is pinned -- the two
        // balanced ones (one or all resident CTAs per SM, whatever the tile count)
        int64_t n_aligned = max_chunks - nc_first + 1;
        int64_t n_cand = n_aligned + (ctx->force_chunks > 0 ? 0 : 2);
        if (ctx->force_ctas > 0) { n_aligned = 0; n_cand = 1; }                 // a pinned grid is the only candidate
        for (int64_t ci = 0; ci < n_cand; ++ci) {
            int64_t ctas;
            bool aligned = ci < n_aligned;
            if (ctx->force_ctas > 0) {
                ctas = ctx->force_ctas < work ? ctx->force_ctas : work;
                aligned = ctas % tiles == 0;
            } else if (aligned) ctas = tiles * (nc_first + ci);
            else {
                ctas = (ci == n_aligned) ? n_sm : slots;
                if (ctas % tiles == 0) continue;                                // already among the aligned grids
                if (work / ctas < (int64_t)8 * lpp) continue;                    // at least 8 iterations per thread
            }
            const double bins_per_cta = (double)work / (double)ctas;
            const double sweep = std::ceil(bins_per_cta / lpp) * (lpp > 1 ? kMultiPenalty : 1.0);
            // segments a CTA sweeps: one, plus one per tile boundary inside its range (each costs a prologue / epilogue)
            const double segs = aligned ? 1.0 : 1.0 + std::fmin(1.0, (double)(tiles - 1) / (double)ctas) + std::floor(bins_per_cta / (double)M);
            const double pro = (kProBins + (lpp > 1 ? 2.0 : 0.0)) * segs;
            const int64_t per_sm = (ctas + n_sm - 1) / n_sm;                  // CTAs an SM must run
            const int64_t waves = (per_sm + slots_per_sm - 1) / slots_per_sm;
            const double resident = (double)per_sm / (double)waves;           // average co-resident CTAs
            const double warps_per_sched = resident * (kThreads / 32) / 4.0;
            double slowdown = warps_per_sched > kSatWarps ? warps_per_sched / kSatWarps : 1.0;
            if (resident >= 2.0) slowdown *= (lpp > 1 ? kCoResidentGainMulti : kCoResidentGain);  // a second CTA hides the first one's stage boundaries
            const int64_t nseg = aligned ? ctas / tiles : (ctas + tiles - 1) / tiles + 1;   // segments per tile
            // Multi-lane aligned grids of 2..16 chunks per tile launch every tile as one thread-block cluster and reduce the
            // chunk sums through distributed shared memory (no global partials, fence or ticket): a short, flat finish.
            // Only for grids of a few clusters: many clusters of 9-16 CTAs wait for whole groups of free SMs in one GPC
            // (measured: B = 64, 256 and C0 lose 5-9 us with clusters, B = 1 and 16 gain 2 us).
            const bool clustered = ctx->cluster_finish && lpp > 1 && aligned && nseg >= 2 && nseg <= kMaxCluster && ctas <= kClusterMaxCtas &&
                                   (int64_t)(2 * ctx->t.n_det) * pt * (nseg + 1) <= stage_doubles;
            const double finish_len = clustered ? kClusterFinish
                                    : nseg >= kFinishTwoLevelFrom ? kTwoLevelHop + (double)(kFinishGroup + (nseg + kFinishGroup - 1) / kFinishGroup)
                                                                  : (double)nseg;   // serial additions of the finish
            // lanes-interleaved CTAs have short sweeps and a latency-bound prologue that a co-resident CTA covers
            const double per_cta = lpp > 1 ? sweep * slowdown + pro : (sweep + pro) * slowdown;
            // SMs that run one CTA more than the others set the time of an unbalanced grid
            const double cost = (double)waves * per_cta + kFinishPerChunk * finish_len;
            if (cost < best_cost) {
                best_cost = cost;
                best.lpp = lpp; best.props_per_cta = pt; best.n_cta = ctas; best.n_tiles = tiles;
                // a grid that fits one CTA per SM is launched so that no SM takes two (launch_fused)
                best.exclusive = (GW_EXCLUSIVE_PLANS && ctas <= n_sm) ? 1 : 0;
                best.cluster = clustered ? (int)nseg : 0;
                // ranges that cross a tile boundary get vbins bins less (gw_internal.h, segment_at); aligned grids have none
                best.vbins = (aligned || tiles < 2 || work / ctas < 4 * (int64_t)ctx->boundary_bins * lpp) ? 0 : ctx->boundary_bins * lpp;
            }
        }
        if (tiles >= slots && ctx->force_lpp == 0) break;     // enough proposals to fill the GPU: keep this lpp
    }
    best.max_seg = max_segments_per_tile(best.n_tiles, M, best.vbins, best.n_cta);
    best.gmax = best.max_seg >= kFinishTwoLevelFrom ? (best.max_seg + kFinishGroup - 1) / kFinishGroup : 1;
    return best;
}

void drop_host_graphs(gw_ctx *ctx)
{
    for (int i = 0; i < 4; ++i) {
        if (ctx->graph_exec[i]) cudaGraphExecDestroy(ctx->graph_exec[i]);
        ctx->graph_exec[i] = nullptr;
        ctx->graph_n[i] = 0;
    }
}

// make_plan through a four-entry cache (the planner's search costs several microseconds of host time per call)
Plan cached_plan(gw_ctx *ctx, int64_t n_prop)
{
    for (int i = 0; i < 4; ++i)
        if (ctx->plan_n[i] == n_prop) return ctx->plan_of[i];
    const Plan p = make_plan(ctx, n_prop);
    const int slot = ctx->plan_next;
    ctx->plan_next = (slot + 1) & 3;
    ctx->plan_n[slot] = n_prop;
    ctx->plan_of[slot] = p;
    return p;
}

// upper bound of partial_need over every plan make_plan can return for n_prop <= max_batch
int64_t partial_bound(const gw_ctx *ctx, int64_t max_batch)
{
    const int slots_per_sm = ctx->ctas_per_sm > 0 ? ctx->ctas_per_sm : 1;
    const int n_sm = ctx->n_sm > 0 ? ctx->n_sm : 148;
    const int64_t ctas = kMaxWaves * (int64_t)n_sm * slots_per_sm + 2 * ((max_batch + kThreads - 1) / kThreads) + 4;   // n_cta + n_tiles slots
    return ctas * kThreads * (int64_t)(2 * ctx->t.n_det);
}

int64_t partial_need(const gw_ctx *ctx, const Plan &p)
{
    return (p.max_seg > 1 && !p.cluster) ? plan_partial_slots(p) * (int64_t)(2 * ctx->t.n_det) * p.props_per_cta : 0;
}

void free_workspace(Workspace &w)
{
    cudaFree(w.rec); cudaFree(w.partial); cudaFree(w.tickets); cudaFree(w.gpartial); cudaFree(w.gtickets);
    cudaFree(w.theta_stage);
    cudaFree(w.lnl_stage); cudaFree(w.parts_stage); cudaFree(w.h_stage);
    std::memset(&w, 0, sizeof(w));
}

int reserve_impl(gw_ctx *ctx, int64_t max_batch)
{
    if (max_batch <= ctx->w.max_batch) return GW_OK;
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    const int64_t need_partial = partial_bound(ctx, max_batch);
    const int64_t need_tickets = max_batch / (kThreads / 32) + 2;   // tiles at lpp = 32
    Workspace w;
    std::memset(&w, 0, sizeof(w));
    w.max_batch = max_batch;
    w.rec_stride = (max_batch + 31) / 32 * 32;
    const int n_det = ctx->t.n_det;
    const int64_t n_rec = rec_fields(n_det);
    w.partial_doubles = need_partial > 0 ? need_partial : 1;
    w.n_tickets = need_tickets;
    // two-level finish: n_groups <= n_chunks / 8 whenever it is used (n_chunks >= 33, groups of 16)
    w.gpartial_doubles = w.partial_doubles / 8 + 1;
    w.n_gtickets = need_partial / ((int64_t)kThreads * 2 * n_det) / 8 + need_tickets + 1;
    w.h_stage_doubles = 0;                                    // the host waveform variant allocates its slab on first use
    bool ok = true;
    ok = ok && (e = cudaMalloc(&w.rec, sizeof(double) * n_rec * w.rec_stride)) == cudaSuccess;
    ok = ok && (e = cudaMalloc(&w.partial, sizeof(double) * w.partial_doubles)) == cudaSuccess;
    ok = ok && (e = cudaMalloc(&w.tickets, sizeof(unsigned int) * w.n_tickets)) == cudaSuccess;
    ok = ok && (e = cudaMalloc(&w.gpartial, sizeof(double) * w.gpartial_doubles)) == cudaSuccess;
    ok = ok && (e = cudaMalloc(&w.gtickets, sizeof(unsigned int) * w.n_gtickets)) == cudaSuccess;
    ok = ok && (e = cudaMemset(w.gtickets, 0, sizeof(unsigned int) * w.n_gtickets)) == cudaSuccess;
    ok = ok && (e = cudaMalloc(&w.theta_stage, sizeof(double) * max_batch * ctx->t.n_param)) == cudaSuccess;
    ok = ok && (e = cudaMalloc(&w.lnl_stage, sizeof(double) * max_batch)) == cudaSuccess;
    ok = ok && (e = cudaMalloc(&w.parts_stage, sizeof(double) * max_batch * n_det * 3)) == cudaSuccess;
    ok = ok && (e = cudaMemset(w.tickets, 0, sizeof(unsigned int) * w.n_tickets)) == cudaSuccess;
    if (!ok) {
        free_workspace(w);
        cudaGetLastError();
        return cuda_fail(ctx, e);
    }
    drop_host_graphs(ctx);                                   // cached graphs hold pointers into the old workspace
    double *old_h = ctx->w.h_stage;
    const int64_t old_h_doubles = ctx->w.h_stage_doubles;
    ctx->w.h_stage = nullptr;
    free_workspace(ctx->w);
    ctx->w = w;
    ctx->w.h_stage = old_h;
    ctx->w.h_stage_doubles = old_h_doubles;
    // The two memsets above ran on the legacy default stream, which is not ordered against non-blocking streams:
    // the zeroed ticket counters must be in place before any batch call on any stream can read them.
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return cuda_fail(ctx, e);
    return GW_OK;
}

bool finite_pos(double v) { return std::isfinite(v) && v > 0.0; }

// Makes the context's device current for the duration of a call and restores the caller's device afterwards
// (a no-op when it is current already, which is the one-process-per-GPU case).
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const gw_ctx *ctx)
    {
        if (ctx && cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device)
            switched = cudaSetDevice(ctx->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

int check_batch_args(gw_ctx *ctx, int64_t n_prop, const void *theta, const void *out)
{
    if (!ctx || n_prop < 0) return GW_ERR_INVALID_ARG;
    if (n_prop == 0) return GW_OK;
    if (!theta || !out) return GW_ERR_INVALID_ARG;
    if (n_prop > ctx->w.max_batch) return GW_ERR_INVALID_ARG;
    return GW_OK;
}

} // namespace

extern "C" {

int gw_abi_version(void) { return GW_ABI_VERSION; }

const char *gw_strerror(int code)
{
    switch (code) {
    case GW_OK:              return "ok";
    case GW_ERR_INVALID_ARG: return "invalid argument";
    case GW_ERR_ALLOC:       return "allocation failed";
    case GW_ERR_CUDA:        return "CUDA runtime error";
    case GW_ERR_ARCH:        return "device is not compute capability 10.x (sm_100a)";
    default:                 return "unknown error code";
    }
}

int gw_last_cuda_error(const gw_ctx *ctx) { return ctx ? ctx->last_cuda_error : 0; }

int gw_ctx_create(gw_ctx **out, int64_t n_bins, const double *freqs_hz, int n_det, const double *data_ri,
                  const double *psd, const gw_detector *dets, double gmst_rad, const gw_options *opt,
                  void *cuda_stream)
{
    if (!out) return GW_ERR_INVALID_ARG;
    *out = nullptr;
    if (!freqs_hz || !data_ri || !psd || !dets) return GW_ERR_INVALID_ARG;
    if (n_bins < 2 || n_bins > ((int64_t)1 << 30) || n_det < 1 || n_det > GW_MAX_DET) return GW_ERR_INVALID_ARG;
    if (!std::isfinite(gmst_rad)) return GW_ERR_INVALID_ARG;
    gw_options o = {1, 0, 4096, 0, 0};
    if (opt) o = *opt;
    if (o.spin_order < 0 || o.spin_order > 2 || o.isco_cut < 0 || o.isco_cut > 1 || o.max_batch < 1 ||
        o.phase_marginal < 0 || o.phase_marginal > 1 || o.tidal_order < 0 || o.tidal_order > 2)
        return GW_ERR_INVALID_ARG;

    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return GW_ERR_CUDA;
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess) return GW_ERR_CUDA;
    if (prop.major != 10) return GW_ERR_ARCH;

    // ---- host copies for validation (inputs may live on either side) ----
    const size_t nf = (size_t)n_bins, nd = (size_t)n_det * n_bins;
    std::vector<double> hf, hd, hp;
    try { hf.resize(nf); hd.resize(nd * 2); hp.resize(nd); } catch (const std::bad_alloc &) { return GW_ERR_ALLOC; }
    const cudaMemcpyKind kf = is_device_ptr(freqs_hz) ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost;
    const cudaMemcpyKind kd = is_device_ptr(data_ri) ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost;
    const cudaMemcpyKind kp = is_device_ptr(psd) ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost;
    if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return GW_ERR_CUDA;
    if ((e = cudaMemcpy(hf.data(), freqs_hz, nf * sizeof(double), kf)) != cudaSuccess) return GW_ERR_CUDA;
    if ((e = cudaMemcpy(hd.data(), data_ri, nd * 2 * sizeof(double), kd)) != cudaSuccess) return GW_ERR_CUDA;
    if ((e = cudaMemcpy(hp.data(), psd, nd * sizeof(double), kp)) != cudaSuccess) return GW_ERR_CUDA;

    const double f0 = hf[0];
    const double df = (hf[nf - 1] - hf[0]) / (double)(n_bins - 1);
    if (!finite_pos(f0) || !finite_pos(df)) return GW_ERR_INVALID_ARG;
    {
        // uniform to rounding: the time-shift recurrence assumes f_j = f_0 + j df
        const double tol = 1e-9 * df + 8.0 * std::ldexp(std::fabs(hf[nf - 1]), -52);
        for (size_t j = 0; j < nf; ++j) {
            if (!std::isfinite(hf[j]) || std::fabs(hf[j] - (f0 + (double)j * df)) > tol) return GW_ERR_INVALID_ARG;
        }
    }
    for (size_t k = 0; k < nd; ++k) if (!finite_pos(hp[k])) return GW_ERR_INVALID_ARG;
    for (size_t k = 0; k < nd * 2; ++k) if (!std::isfinite(hd[k])) return GW_ERR_INVALID_ARG;

    gw_ctx *ctx = new (std::nothrow) gw_ctx;
    if (!ctx) return GW_ERR_ALLOC;
    std::memset(ctx, 0, sizeof(*ctx));
    ctx->device = dev;
    ctx->n_sm = prop.multiProcessorCount;
    ctx->spin_order = o.spin_order;
    ctx->gmst = gmst_rad;
    for (int i = 0; i < n_det; ++i) {
        const gw_detector &d = dets[i];
        DetGeom &g = ctx->dets.d[i];
        g.kind = d.kind;
        if (d.kind == GW_DET_GEOMETRIC) {
            double nx = 0, ny = 0;
            for (int a = 0; a < 3; ++a) { nx += d.xarm[a] * d.xarm[a]; ny += d.yarm[a] * d.yarm[a]; }
            bool fin = true;
            for (int a = 0; a < 3; ++a) fin = fin && std::isfinite(d.vertex_m[a]);
            if (!fin || !(std::fabs(nx - 1.0) <= 2e-6) || !(std::fabs(ny - 1.0) <= 2e-6)) { delete ctx; return GW_ERR_INVALID_ARG; }
            const double *x = d.xarm, *y = d.yarm;
            g.D[0] = 0.5 * (x[0] * x[0] - y[0] * y[0]); g.D[1] = 0.5 * (x[0] * x[1] - y[0] * y[1]);
            g.D[2] = 0.5 * (x[0] * x[2] - y[0] * y[2]); g.D[3] = 0.5 * (x[1] * x[1] - y[1] * y[1]);
            g.D[4] = 0.5 * (x[1] * x[2] - y[1] * y[2]); g.D[5] = 0.5 * (x[2] * x[2] - y[2] * y[2]);
            for (int a = 0; a < 3; ++a) g.rc[a] = d.vertex_m[a] / 299792458.0;
        } else if (d.kind == GW_DET_FIXED) {
            if (!std::isfinite(d.fplus) || !std::isfinite(d.fcross) || !std::isfinite(d.dt_s)) { delete ctx; return GW_ERR_INVALID_ARG; }
            g.fplus = d.fplus; g.fcross = d.fcross; g.dt_s = d.dt_s;
        } else { delete ctx; return GW_ERR_INVALID_ARG; }
    }

    int rc = GW_OK;
    double *dfreq = nullptr, *ddata = nullptr, *dpsd = nullptr, *di7 = nullptr;
    Tables &t = ctx->t;
    t.n_bins = n_bins; t.n_pad = (n_bins + 31) / 32 * 32 + 32; t.n_det = n_det; t.f0 = f0; t.delta_f = df;
    t.isco_cut = o.isco_cut; t.phase_marginal = o.phase_marginal;
    t.tidal_order = o.tidal_order; t.n_param = o.tidal_order > 0 ? (int)GW_NPARAM_TIDAL : (int)GW_NPARAM;
    do {
        if ((e = configure_kernels(nullptr)) != cudaSuccess) { rc = cuda_fail(ctx, e); break; }
        ctx->ctas_per_sm = fused_ctas_per_sm(n_det);
        ctx->cluster_finish = fused_cluster_ok(n_det);
        bool ok = true;
        ok = ok && (e = cudaMalloc(&t.planes, sizeof(double) * 2 * (kBasisPlanes + n_det) * t.n_pad)) == cudaSuccess;
        if (t.isco_cut) ok = ok && (e = cudaMalloc(&t.i7cum, sizeof(double) * n_det * t.n_pad)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&dfreq, sizeof(double) * nf)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&ddata, sizeof(double) * nd * 2)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&dpsd, sizeof(double) * nd)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&di7, sizeof(double) * GW_MAX_DET)) == cudaSuccess;
        if (!ok) { rc = cuda_fail(ctx, e); break; }
        ok = ok && (e = cudaMemcpyAsync(dfreq, hf.data(), nf * sizeof(double), cudaMemcpyHostToDevice, s)) == cudaSuccess;
        ok = ok && (e = cudaMemcpyAsync(ddata, hd.data(), nd * 2 * sizeof(double), cudaMemcpyHostToDevice, s)) == cudaSuccess;
        ok = ok && (e = cudaMemcpyAsync(dpsd, hp.data(), nd * sizeof(double), cudaMemcpyHostToDevice, s)) == cudaSuccess;
        if (!ok) { rc = cuda_fail(ctx, e); break; }
        if ((e = launch_precompute(t, dfreq, ddata, dpsd, di7, s, &ctx->launches)) != cudaSuccess) { rc = cuda_fail(ctx, e); break; }
        if ((e = cudaMemcpyAsync(t.i7, di7, sizeof(double) * n_det, cudaMemcpyDeviceToHost, s)) != cudaSuccess) { rc = cuda_fail(ctx, e); break; }
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { rc = cuda_fail(ctx, e); break; }
        rc = reserve_impl(ctx, o.max_batch);
        if (rc != GW_OK) break;
        // pinned, mapped staging of the small-batch host path (fixed size: kHostGraphMax proposals)
        ctx->pin_cap = kHostGraphMax;
        ok = true;
        ok = ok && (e = cudaHostAlloc(&ctx->pin_theta, sizeof(double) * ctx->pin_cap * t.n_param, cudaHostAllocMapped)) == cudaSuccess;
        ok = ok && (e = cudaHostAlloc(&ctx->pin_lnl, sizeof(double) * ctx->pin_cap, cudaHostAllocMapped)) == cudaSuccess;
        ok = ok && (e = cudaHostAlloc(&ctx->pin_parts, sizeof(double) * ctx->pin_cap * n_det * 3, cudaHostAllocMapped)) == cudaSuccess;
        ok = ok && (e = cudaHostGetDevicePointer(&ctx->pin_theta_dev, ctx->pin_theta, 0)) == cudaSuccess;
        ok = ok && (e = cudaHostGetDevicePointer(&ctx->pin_lnl_dev, ctx->pin_lnl, 0)) == cudaSuccess;
        ok = ok && (e = cudaHostGetDevicePointer(&ctx->pin_parts_dev, ctx->pin_parts, 0)) == cudaSuccess;
        ok = ok && (e = cudaStreamCreateWithFlags(&ctx->capture_stream, cudaStreamNonBlocking)) == cudaSuccess;
        if (!ok) { rc = cuda_fail(ctx, e); break; }
        ctx->host_graph = 1;
        ctx->boundary_bins = kBoundaryBins;
    } while (0);
    cudaFree(dfreq); cudaFree(ddata); cudaFree(dpsd); cudaFree(di7);
    if (rc != GW_OK) {
        gw_ctx_destroy(ctx);
        cudaGetLastError();
        return rc;
    }
    *out = ctx;
    return GW_OK;
}

int gw_ctx_reserve(gw_ctx *ctx, int64_t max_batch)
{
    if (!ctx || max_batch < 1) return GW_ERR_INVALID_ARG;
    DeviceGuard guard(ctx);
    return reserve_impl(ctx, max_batch);
}

int gw_ctx_destroy(gw_ctx *ctx)
{
    if (!ctx) return GW_OK;
    DeviceGuard guard(ctx);
    cudaDeviceSynchronize();
    drop_host_graphs(ctx);
    if (ctx->capture_stream) cudaStreamDestroy(ctx->capture_stream);
    cudaFreeHost(ctx->pin_theta); cudaFreeHost(ctx->pin_lnl); cudaFreeHost(ctx->pin_parts);
    free_workspace(ctx->w);
    cudaFree(ctx->t.planes); cudaFree(ctx->t.i7cum);
    for (int i = 0; i < 3; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    delete ctx;
    cudaGetLastError();
    return GW_OK;
}

int gw_ctx_info(const gw_ctx *ctx, int64_t *n_bins, int *n_det, double *delta_f, int64_t *max_batch)
{
    if (!ctx) return GW_ERR_INVALID_ARG;
    if (n_bins) *n_bins = ctx->t.n_bins;
    if (n_det) *n_det = ctx->t.n_det;
    if (delta_f) *delta_f = ctx->t.delta_f;
    if (max_batch) *max_batch = ctx->w.max_batch;
    return GW_OK;
}

int gw_ctx_n_param(const gw_ctx *ctx) { return ctx ? ctx->t.n_param : -1; }

int gw_ctx_plan(const gw_ctx *ctx, int64_t n_prop, int *lanes_per_prop, int *props_per_cta, int *n_chunks,
                int64_t *n_ctas)
{
    if (!ctx || n_prop < 1) return GW_ERR_INVALID_ARG;
    const Plan p = make_plan(ctx, n_prop);
    if (lanes_per_prop) *lanes_per_prop = p.lpp;
    if (props_per_cta) *props_per_cta = p.props_per_cta;
    if (n_chunks) *n_chunks = p.max_seg;
    if (n_ctas) *n_ctas = p.n_cta;
    return GW_OK;
}

int gw_ctx_force_plan(gw_ctx *ctx, int lanes_per_prop, int n_chunks)
{
    if (!ctx || n_chunks < 0) return GW_ERR_INVALID_ARG;
    if (lanes_per_prop != 0 && (lanes_per_prop < 1 || lanes_per_prop > 32 || (lanes_per_prop & (lanes_per_prop - 1)) != 0))
        return GW_ERR_INVALID_ARG;
    ctx->force_lpp = lanes_per_prop;
    ctx->force_chunks = n_chunks;
    ctx->force_ctas = 0;
    for (int i = 0; i < 4; ++i) ctx->plan_n[i] = 0;          // cached plans were made for the previous pin
    drop_host_graphs(ctx);
    return GW_OK;
}

int gw_ctx_force_grid(gw_ctx *ctx, int lanes_per_prop, int64_t n_ctas)
{
    if (!ctx || n_ctas < 0 || n_ctas > 0x7fffffffLL) return GW_ERR_INVALID_ARG;
    if (lanes_per_prop != 0 && (lanes_per_prop < 1 || lanes_per_prop > 32 || (lanes_per_prop & (lanes_per_prop - 1)) != 0))
        return GW_ERR_INVALID_ARG;
    ctx->force_lpp = lanes_per_prop;
    ctx->force_chunks = 0;
    ctx->force_ctas = n_ctas;
    for (int i = 0; i < 4; ++i) ctx->plan_n[i] = 0;
    drop_host_graphs(ctx);
    return GW_OK;
}

int gw_ctx_cluster_finish(gw_ctx *ctx, int enable)
{
    if (!ctx) return GW_ERR_INVALID_ARG;
    ctx->cluster_finish = (enable && fused_cluster_ok(ctx->t.n_det)) ? 1 : 0;
    for (int i = 0; i < 4; ++i) ctx->plan_n[i] = 0;
    drop_host_graphs(ctx);
    return GW_OK;
}

int gw_ctx_host_graph(gw_ctx *ctx, int enable)
{
    if (!ctx) return GW_ERR_INVALID_ARG;
    ctx->host_graph = enable ? 1 : 0;
    return GW_OK;
}

int gw_plan_cta_segments(int64_t n_tiles, int64_t n_bins, int64_t boundary_bins, int64_t n_ctas, int64_t cta, int max_rows,
                         int64_t *rows6)
{
    if (n_tiles < 1 || n_bins < 1 || boundary_bins < 0 || n_ctas < 1 || cta < 0 || cta >= n_ctas || max_rows < 0 ||
        (max_rows > 0 && !rows6))
        return GW_ERR_INVALID_ARG;
    if ((double)n_tiles * ((double)n_bins + (double)boundary_bins) * (double)(n_ctas + 1) > 4.0e18) return GW_ERR_INVALID_ARG;
    const int64_t tile_len = n_bins + boundary_bins, work = flattened_work(n_tiles, n_bins, boundary_bins);
    const int64_t w_end = work_begin(cta + 1, work, n_ctas);
    int n = 0;
    for (int64_t w = work_begin(cta, work, n_ctas); w < w_end; ++n) {
        const Segment s = segment_at(w, w_end, cta, n_bins, tile_len, work, n_ctas);
        if (n < max_rows) {
            int64_t *r = rows6 + 6 * n;
            r[0] = s.tile; r[1] = s.j0; r[2] = s.j1; r[3] = s.index; r[4] = s.count; r[5] = s.slot;
        }
        w += s.len;
    }
    return n;
}

int gw_ctx_plan_boundary_bins(const gw_ctx *ctx, int64_t n_prop, int *boundary_bins)
{
    if (!ctx || n_prop < 1 || !boundary_bins) return GW_ERR_INVALID_ARG;
    *boundary_bins = make_plan(ctx, n_prop).vbins;
    return GW_OK;
}

int gw_ctx_boundary_bins(gw_ctx *ctx, int boundary_bins)
{
    if (!ctx || boundary_bins < 0 || boundary_bins > 4096) return GW_ERR_INVALID_ARG;
    ctx->boundary_bins = boundary_bins;
    for (int i = 0; i < 4; ++i) ctx->plan_n[i] = 0;
    drop_host_graphs(ctx);
    return GW_OK;
}

int gw_ctx_norms(const gw_ctx *ctx, double *i7_host)
{
    if (!ctx || !i7_host) return GW_ERR_INVALID_ARG;
    for (int i = 0; i < ctx->t.n_det; ++i) i7_host[i] = ctx->t.i7[i];
    return GW_OK;
}

int64_t gw_ctx_launch_count(const gw_ctx *ctx) { return ctx ? ctx->launches : 0; }

int gw_ctx_kernel_timing(gw_ctx *ctx, int enable)
{
    if (!ctx) return GW_ERR_INVALID_ARG;
    if (enable && !ctx->ev[0]) {
        for (int i = 0; i < 3; ++i) {
            cudaError_t e = cudaEventCreate(&ctx->ev[i]);
            if (e != cudaSuccess) return cuda_fail(ctx, e);
        }
    }
    ctx->timing = enable ? 1 : 0;
    return GW_OK;
}

int gw_ctx_last_kernel_ms(gw_ctx *ctx, double *setup_ms, double *main_ms)
{
    if (!ctx || !ctx->ev[0]) return GW_ERR_INVALID_ARG;
    cudaError_t e = cudaEventSynchronize(ctx->ev[2]);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    float a = 0.f, b = 0.f;
    if ((e = cudaEventElapsedTime(&a, ctx->ev[0], ctx->ev[1])) != cudaSuccess) return cuda_fail(ctx, e);
    if ((e = cudaEventElapsedTime(&b, ctx->ev[1], ctx->ev[2])) != cudaSuccess) return cuda_fail(ctx, e);
    if (setup_ms) *setup_ms = a;
    if (main_ms) *main_ms = b;
    return GW_OK;
}

// theta_in_host_memory: theta_dev is the device alias of a pinned host buffer (host variant, read in place)
static int lnl_batch_impl(gw_ctx *ctx, int64_t n_prop, const double *theta_dev, int theta_in_host_memory,
                          double *lnl_out_dev, double *parts_out_dev, void *cuda_stream)
{
    int rc = check_batch_args(ctx, n_prop, theta_dev, lnl_out_dev);
    if (rc != GW_OK || n_prop == 0) return rc;
    DeviceGuard guard(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const Plan p = cached_plan(ctx, n_prop);
    if (partial_need(ctx, p) > ctx->w.partial_doubles || p.n_tiles > ctx->w.n_tickets) return GW_ERR_INVALID_ARG;
    if (p.gmax > 1 && (p.n_tiles * p.gmax * (int64_t)(2 * ctx->t.n_det) * p.props_per_cta > ctx->w.gpartial_doubles ||
                       p.n_tiles * p.gmax > ctx->w.n_gtickets))
        return GW_ERR_INVALID_ARG;
    if ((double)p.n_tiles * (double)(ctx->t.n_bins + p.vbins) * (double)(p.n_cta + 1) > 4.0e18) return GW_ERR_INVALID_ARG;   // 64-bit range arithmetic
    if (ctx->timing) cudaEventRecord(ctx->ev[0], s);
    cudaError_t e = launch_setup(ctx->t, ctx->dets, ctx->gmst, ctx->spin_order, n_prop, theta_dev, ctx->w.rec,
                                 ctx->w.rec_stride, (double)p.lpp * ctx->t.delta_f, 1, theta_in_host_memory, s,
                                 &ctx->launches);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    if (ctx->timing) cudaEventRecord(ctx->ev[1], s);
    e = launch_fused(ctx->t, p, n_prop, ctx->w.rec, ctx->w.rec_stride, ctx->w.partial, ctx->w.tickets, ctx->w.gpartial, ctx->w.gtickets, lnl_out_dev,
                     parts_out_dev, s, &ctx->launches);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    if (ctx->timing) cudaEventRecord(ctx->ev[2], s);
    return GW_OK;
}

int gw_lnl_batch(gw_ctx *ctx, int64_t n_prop, const double *theta_dev, double *lnl_out_dev,
                 double *parts_out_dev, void *cuda_stream)
{
    return lnl_batch_impl(ctx, n_prop, theta_dev, 0, lnl_out_dev, parts_out_dev, cuda_stream);
}

int gw_waveform_batch(gw_ctx *ctx, int64_t n_prop, const double *theta_dev, double *h_out_dev, void *cuda_stream)
{
    int rc = check_batch_args(ctx, n_prop, theta_dev, h_out_dev);
    if (rc != GW_OK || n_prop == 0) return rc;
    if (((uintptr_t)h_out_dev & 15u) != 0) return GW_ERR_INVALID_ARG;
    DeviceGuard guard(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (ctx->timing) cudaEventRecord(ctx->ev[0], s);
    cudaError_t e = launch_setup(ctx->t, ctx->dets, ctx->gmst, ctx->spin_order, n_prop, theta_dev, ctx->w.rec,
                                 ctx->w.rec_stride, ctx->t.delta_f, 0, 0, s, &ctx->launches);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    if (ctx->timing) cudaEventRecord(ctx->ev[1], s);
    e = launch_waveform(ctx->t, n_prop, ctx->w.rec, ctx->w.rec_stride, h_out_dev, s, &ctx->launches);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    if (ctx->timing) cudaEventRecord(ctx->ev[2], s);
    return GW_OK;
}

int gw_lnl_batch_host(gw_ctx *ctx, int64_t n_prop, const double *theta_host, double *lnl_out_host,
                      double *parts_out_host, void *cuda_stream)
{
    int rc = check_batch_args(ctx, n_prop, theta_host, lnl_out_host);
    if (rc != GW_OK || n_prop == 0) return rc;
    DeviceGuard guard(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    Workspace &w = ctx->w;
    if (ctx->host_graph && !ctx->timing && n_prop <= ctx->pin_cap) {
        // Small batch: one graph launch (setup kernel reading theta in place from the pinned staging buffer, fused kernel
        // storing lnL and parts into pinned buffers) and one synchronise.  The graph of a batch size is captured once on
        // the library's own stream and kept (four sizes, with / without parts).
        const int want_parts = parts_out_host != nullptr;
        cudaGraphExec_t exec = nullptr;
        for (int i = 0; i < 4; ++i)
            if (ctx->graph_n[i] == n_prop && ctx->graph_parts[i] == want_parts) exec = ctx->graph_exec[i];
        cudaError_t e;
        if (!exec) {
            cudaGraph_t graph = nullptr;
            if ((e = cudaStreamBeginCapture(ctx->capture_stream, cudaStreamCaptureModeThreadLocal)) != cudaSuccess) return cuda_fail(ctx, e);
            rc = lnl_batch_impl(ctx, n_prop, ctx->pin_theta_dev, 1, ctx->pin_lnl_dev, want_parts ? ctx->pin_parts_dev : nullptr,
                                (void *)ctx->capture_stream);
            e = cudaStreamEndCapture(ctx->capture_stream, &graph);
            if (rc == GW_OK) ctx->launches -= 2;             // captured, not launched
            if (rc != GW_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) return cuda_fail(ctx, e);
            e = cudaGraphInstantiate(&exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) return cuda_fail(ctx, e);
            const int slot = ctx->graph_next;
            ctx->graph_next = (slot + 1) & 3;
            if (ctx->graph_exec[slot]) cudaGraphExecDestroy(ctx->graph_exec[slot]);
            ctx->graph_exec[slot] = exec; ctx->graph_n[slot] = n_prop; ctx->graph_parts[slot] = want_parts;
        }
        std::memcpy(ctx->pin_theta, theta_host, sizeof(double) * n_prop * ctx->t.n_param);
        if ((e = cudaGraphLaunch(exec, s)) != cudaSuccess) return cuda_fail(ctx, e);
        ctx->launches += 2;
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return cuda_fail(ctx, e);
        std::memcpy(lnl_out_host, ctx->pin_lnl, sizeof(double) * n_prop);
        if (want_parts) std::memcpy(parts_out_host, ctx->pin_parts, sizeof(double) * n_prop * ctx->t.n_det * 3);
        return GW_OK;
    }
    // A pinned theta buffer is read in place by the setup kernel (coalesced loads over the host link): one
    // copy-engine operation and its hand-over to the kernel less per call; pageable buffers and very large batches
    // (whose transfer the copy engine does faster) take the staged copy.
    const double *theta_src = nullptr;
    if (n_prop >= (int64_t)GW_ZERO_COPY_THETA_MIN && n_prop <= (int64_t)GW_ZERO_COPY_THETA_MAX)
        theta_src = mapped_alias(theta_host);
    const int in_place = theta_src != nullptr;
    cudaError_t e = cudaSuccess;
    if (!theta_src) {
        e = cudaMemcpyAsync(w.theta_stage, theta_host, sizeof(double) * n_prop * ctx->t.n_param,
                            cudaMemcpyHostToDevice, s);
        theta_src = w.theta_stage;
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    // lnL goes straight to a pinned output buffer (coalesced 8-byte stores of the finish stage over the host link):
    // one copy-engine round trip less per call; pageable buffers and `parts` take the staged copy
#if GW_ZERO_COPY_LNL
    double *direct = mapped_alias(lnl_out_host);
#else
    double *direct = nullptr;
#endif
    rc = lnl_batch_impl(ctx, n_prop, theta_src, in_place, direct ? direct : w.lnl_stage, parts_out_host ? w.parts_stage : nullptr,
                      cuda_stream);
    if (rc != GW_OK) return rc;
    if (!direct) e = cudaMemcpyAsync(lnl_out_host, w.lnl_stage, sizeof(double) * n_prop, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess && parts_out_host)
        e = cudaMemcpyAsync(parts_out_host, w.parts_stage, sizeof(double) * n_prop * ctx->t.n_det * 3,
                            cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    return GW_OK;
}

int gw_waveform_batch_host(gw_ctx *ctx, int64_t n_prop, const double *theta_host, double *h_out_host,
                           void *cuda_stream)
{
    int rc = check_batch_args(ctx, n_prop, theta_host, h_out_host);
    if (rc != GW_OK || n_prop == 0) return rc;
    DeviceGuard guard(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    Workspace &w = ctx->w;
    const int64_t per_prop = (int64_t)ctx->t.n_det * ctx->t.n_bins * 2;
    cudaError_t e;
    if (w.h_stage_doubles < per_prop) {                       // first use: allocate the slab (host variant only)
        int64_t want = per_prop * n_prop;
        if (want > kHStageMaxDoubles) want = (kHStageMaxDoubles / per_prop) * per_prop;
        if (want < per_prop) want = per_prop;
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return cuda_fail(ctx, e);
        cudaFree(w.h_stage); w.h_stage = nullptr; w.h_stage_doubles = 0;
        if ((e = cudaMalloc(&w.h_stage, sizeof(double) * want)) != cudaSuccess) { cudaGetLastError(); return cuda_fail(ctx, e); }
        w.h_stage_doubles = want;
    }
    const int64_t slab = w.h_stage_doubles / per_prop;
    e = cudaMemcpyAsync(w.theta_stage, theta_host, sizeof(double) * n_prop * ctx->t.n_param, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(ctx, e);
    for (int64_t b0 = 0; b0 < n_prop; b0 += slab) {
        const int64_t nb = (n_prop - b0 < slab) ? n_prop - b0 : slab;
        rc = gw_waveform_batch(ctx, nb, w.theta_stage + b0 * ctx->t.n_param, w.h_stage, cuda_stream);
        if (rc != GW_OK) return rc;
        e = cudaMemcpyAsync(h_out_host + b0 * per_prop, w.h_stage, sizeof(double) * nb * per_prop,
                            cudaMemcpyDeviceToHost, s);
        if (e != cudaSuccess) return cuda_fail(ctx, e);
    }
    if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return cuda_fail(ctx, e);
    return GW_OK;
}

} // extern "C"
