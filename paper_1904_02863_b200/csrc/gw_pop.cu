// gw_pop.cu -- population ("recycling") likelihood, Eq. 3 (data flow PAPER.md:109): kernels and
// C-ABI of include/gwpop.h.  sm_100a.  Shares nothing with oracle/.
//
//   lnL(Lambda) = sum_i ln [ sum_j p(theta_ij | Lambda) / p(theta_ij | 0) ]
//
//   P0 pop_precompute_kernel : per-sample planes, once per context (Lambda-independent logarithms and squares)
//   P1 pop_setup_kernel      : Lambda_b -> record of 16 doubles (normalisation constants; erf, lgamma, pow once per Lambda)
//   P2 pop_main_kernel<TL>   : the map-reduce: one CTA = one chunk of one event's samples x TL proposals; every sample
//                              plane value is read once per pass and used for TL weights; fixed-order block reduce
//   P3 pop_finish_kernel     : per Lambda: chunk sums in chunk order -> ln -> events in a fixed tree -> lnL
//
// Algebra (the oracle writes each density with pow / exp / erf in its natural form instead):
//   with lm = ln m1, lq = ln q, La = ln a1 + ln a2, Lb = ln(1-a1) + ln(1-a2), d_k = (c_k - 1)^2, lp = -ln prior,
//   e  = beta_q lq + (alpha_chi - 1) La + (beta_chi - 1) Lb + lp
//   A  = exp(r1 - alpha lm + e) + exp(r2 - (m1 - m_pp)^2 / (2 sig_pp^2) + e)          mass x ratio numerator x spins / prior
//   Qn = | 1 - exp((1 + beta_q)(ln m_min - lm)) |                                     ratio normalisation
//   T  = (1 - xi)/4 + xi C_1 C_2 exp(-d_1 / (2 sig_1^2) - d_2 / (2 sig_2^2))          tilts
//   w  = A T / Qn  inside the support (m_min < m1 <= m_max, lq >= ln m_min - lm), else 0
//   r1 = ln[(1 - lam) C_pl |1 + beta_q| / B(alpha_chi, beta_chi)^2],  r2 = ln[lam C_g |1 + beta_q| / B^2].
// Four exponentials and one division per (sample, Lambda); 64 bytes of planes per sample and pass.  (A hand-written exp --
// conversion-pipe range reduction, degree-11 Horner -- measured 15 % SLOWER than libdevice's exp here: DESIGN.md section 13.)
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/gwpop.h"

namespace gwpop {

constexpr int kThreads   = 256;
#ifndef GW_POP_PER_THREAD
#define GW_POP_PER_THREAD 4
#endif
#ifndef GW_POP_MIN_CTAS
#define GW_POP_MIN_CTAS 2
#endif
constexpr int kPerThread = GW_POP_PER_THREAD;       // samples per thread and chunk
constexpr int kChunk     = kThreads * kPerThread;   // samples per CTA
constexpr int kPlanes    = 8;
constexpr int kRec       = 16;                      // doubles per Lambda record
constexpr int kLamTile   = 4;                       // proposals per pass over the samples
constexpr int kFinThreads = 128;
constexpr double kPi = 3.14159265358979323846;

enum { R_NALPHA = 0, R_R1, R_R2, R_MU, R_HG, R_BETA, R_AC1, R_BC1, R_BP1, R_LNMMIN, R_MMIN, R_MMAX, R_T0, R_T1, R_H1, R_H2 };
enum { PL_LM = 0, PL_M1, PL_LQ, PL_LA, PL_LB, PL_D1, PL_D2, PL_LP };

__device__ __forceinline__ void pdl_wait()   { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- P0: per-sample planes ---------------------------------------------------------------------------------------
__global__ void pop_precompute_kernel(int64_t total, const double *__restrict__ samples, const double *__restrict__ prior,
                                      double *__restrict__ planes, int *__restrict__ bad)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    const double *th = samples + e * GW_POP_NTHETA;
    const double m1 = th[GW_POP_T_M1], q = th[GW_POP_T_Q], a1 = th[GW_POP_T_A1], a2 = th[GW_POP_T_A2];
    const double c1 = th[GW_POP_T_C1], c2 = th[GW_POP_T_C2], p0 = prior[e];
    const bool ok = isfinite(m1) && m1 > 0.0 && q > 0.0 && q <= 1.0 && a1 > 0.0 && a1 < 1.0 && a2 > 0.0 && a2 < 1.0 &&
                    fabs(c1) <= 1.0 && fabs(c2) <= 1.0 && isfinite(p0) && p0 > 0.0;
    if (!ok) atomicOr(bad, 1);
    planes[PL_LM * total + e] = log(m1);
    planes[PL_M1 * total + e] = m1;
    planes[PL_LQ * total + e] = log(q);
    planes[PL_LA * total + e] = log(a1) + log(a2);
    planes[PL_LB * total + e] = log1p(-a1) + log1p(-a2);
    planes[PL_D1 * total + e] = (c1 - 1.0) * (c1 - 1.0);
    planes[PL_D2 * total + e] = (c2 - 1.0) * (c2 - 1.0);
    planes[PL_LP * total + e] = -log(p0);
}

// ---- P1: per-Lambda record ---------------------------------------------------------------------------------------
__device__ __forceinline__ double normal_cdf(double z) { return 0.5 * erfc(-z * 0.70710678118654752440); }

__global__ void pop_setup_kernel(int64_t n_lambda, const double *__restrict__ lambda, double *__restrict__ rec)
{
    pdl_launch();
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_lambda) return;
    const double *L = lambda + b * GW_POP_NLAMBDA;
    double *r = rec + b * kRec;
    const double alpha = L[GW_POP_L_ALPHA], mmin = L[GW_POP_L_MMIN], mmax = L[GW_POP_L_MMAX], lam = L[GW_POP_L_LAM];
    const double mpp = L[GW_POP_L_MPP], sg = L[GW_POP_L_SIGPP], beta = L[GW_POP_L_BETAQ];
    const double ac = L[GW_POP_L_ALPHACHI], bc = L[GW_POP_L_BETACHI], xi = L[GW_POP_L_XI];
    const double s1 = L[GW_POP_L_SIG1], s2 = L[GW_POP_L_SIG2];
    bool ok = true;
    for (int k = 0; k < GW_POP_NLAMBDA; ++k) ok = ok && isfinite(L[k]);
    ok = ok && mmin > 0.0 && mmax > mmin && lam >= 0.0 && lam <= 1.0 && sg > 0.0 && ac > 0.0 && bc > 0.0 && xi >= 0.0 &&
         xi <= 1.0 && s1 > 0.0 && s2 > 0.0;
    // power law m^-alpha on [mmin, mmax]: 1 / integral
    const double oma = 1.0 - alpha;
    const double c_pl = fabs(oma) < 1e-12 ? 1.0 / log(mmax / mmin) : oma / (pow(mmax, oma) - pow(mmin, oma));
    // truncated normal peak
    const double c_g = 1.0 / (sg * sqrt(2.0 * kPi) * (normal_cdf((mmax - mpp) / sg) - normal_cdf((mmin - mpp) / sg)));
    // ratio: |1 + beta| q^beta / |1 - qlo^(1+beta)|; beta = -1: q^-1 / (ln m1 - ln mmin)
    const double bp1 = 1.0 + beta;
    const bool log_ratio = fabs(bp1) < 1e-12;
    const double ln_cb = log_ratio ? 0.0 : log(fabs(bp1));
    const double ln_beta_fn = lgamma(ac) + lgamma(bc) - lgamma(ac + bc);
    const double common = ln_cb - 2.0 * ln_beta_fn;
    // tilts: TN(c; 1, s, [-1, 1]) = exp(-(c-1)^2 / 2 s^2) / (s sqrt(2 pi) (Phi(0) - Phi(-2/s)))
    const double c_1 = 1.0 / (s1 * sqrt(2.0 * kPi) * (0.5 - normal_cdf(-2.0 / s1)));
    const double c_2 = 1.0 / (s2 * sqrt(2.0 * kPi) * (0.5 - normal_cdf(-2.0 / s2)));
    r[R_NALPHA] = -alpha;
    r[R_R1] = ok ? log((1.0 - lam) * c_pl) + common : __longlong_as_double(0x7ff8000000000000LL);   // NaN marks an invalid Lambda
    r[R_R2] = log(lam * c_g) + common;
    r[R_MU] = mpp;
    r[R_HG] = 0.5 / (sg * sg);
    r[R_BETA] = beta;
    r[R_AC1] = ac - 1.0;
    r[R_BC1] = bc - 1.0;
    r[R_BP1] = log_ratio ? 0.0 : bp1;               // 0 selects the logarithmic normalisation
    r[R_LNMMIN] = log(mmin);
    r[R_MMIN] = mmin;
    r[R_MMAX] = mmax;
    r[R_T0] = 0.25 * (1.0 - xi);
    r[R_T1] = xi * c_1 * c_2;
    r[R_H1] = 0.5 / (s1 * s1);
    r[R_H2] = 0.5 / (s2 * s2);
}

// ---- P2: map + first-stage reduce ------------------------------------------------------------------------------------
struct PopArgs {
    const double *planes, *rec;
    int64_t total;             // N * n: samples per plane
    int64_t n_samples, n_events, n_lambda;
    int     cpe;               // chunks per event
    double *partial;           // [n_lambda][n_events][cpe]
    double *lnl;
};

template <int TL>
__global__ void __launch_bounds__(kThreads, GW_POP_MIN_CTAS) pop_main_kernel(const PopArgs a)
{
    __shared__ double srec[TL][kRec];
    __shared__ double swarp[kThreads / 32][TL];
    pdl_launch();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t event = blockIdx.x / a.cpe;
    const int chunk = blockIdx.x % a.cpe;
    const int64_t lam0 = (int64_t)blockIdx.y * TL;
    const int nl = (int)((a.n_lambda - lam0 < TL) ? a.n_lambda - lam0 : TL);
    // the chunk's plane values do not depend on the setup kernel: load them before waiting for it
    const int64_t jbase = (int64_t)chunk * kChunk + tid;
    const double *pl = a.planes + event * a.n_samples;
    double v[kPerThread][kPlanes];
    bool live[kPerThread];
#pragma unroll
    for (int s = 0; s < kPerThread; ++s) {
        const int64_t j = jbase + (int64_t)s * kThreads;
        live[s] = j < a.n_samples;
        const int64_t jc = live[s] ? j : a.n_samples - 1;
#pragma unroll
        for (int p = 0; p < kPlanes; ++p) v[s][p] = __ldcs(pl + (int64_t)p * a.total + jc);
    }
    pdl_wait();
    for (int i = tid; i < TL * kRec; i += kThreads) {
        const int l = i / kRec;
        srec[l][i % kRec] = l < nl ? a.rec[(lam0 + l) * kRec + (i % kRec)] : 0.0;
    }
    __syncthreads();
    double acc[TL];
#pragma unroll
    for (int l = 0; l < TL; ++l) acc[l] = 0.0;
#pragma unroll
    for (int l = 0; l < TL; ++l) {
        if (l >= nl) break;
        const double *r = srec[l];                                   // warp-broadcast reads
        const double nalpha = r[R_NALPHA], r1 = r[R_R1], r2 = r[R_R2], mu = r[R_MU], hg = r[R_HG], beta = r[R_BETA];
        const double ac1 = r[R_AC1], bc1 = r[R_BC1], bp1 = r[R_BP1], lnmmin = r[R_LNMMIN], mmin = r[R_MMIN], mmax = r[R_MMAX];
        const double t0 = r[R_T0], t1 = r[R_T1], h1 = r[R_H1], h2 = r[R_H2];
        double sum = 0.0;
#pragma unroll
        for (int s = 0; s < kPerThread; ++s) {
            const double lm = v[s][PL_LM], m1 = v[s][PL_M1], lq = v[s][PL_LQ];
            const double e  = __fma_rn(beta, lq, __fma_rn(ac1, v[s][PL_LA], __fma_rn(bc1, v[s][PL_LB], v[s][PL_LP])));
            const double dm = m1 - mu;
            const double x1 = __fma_rn(nalpha, lm, r1 + e);
            const double x2 = __fma_rn(-(dm * dm), hg, r2 + e);
            const double A  = exp(x1) + exp(x2);
            const double dl = lnmmin - lm;
            const double Qn = bp1 != 0.0 ? fabs(1.0 - exp(bp1 * dl)) : -dl;
            const double T  = __fma_rn(t1, exp(-__fma_rn(v[s][PL_D1], h1, v[s][PL_D2] * h2)), t0);
            const bool in = live[s] && m1 > mmin && m1 <= mmax && lq >= dl;
            const double w = (A * T) / Qn;
            sum += in ? w : 0.0;                                     // ascending sample order within the thread
        }
        acc[l] = sum;
    }
    // fixed-order block reduce: xor-shuffle tree within the warp, then the warps in index order
#pragma unroll
    for (int l = 0; l < TL; ++l) {
        double x = acc[l];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if (lane == 0) swarp[warp][l] = x;
    }
    __syncthreads();
    if (tid < nl) {
        double x = 0.0;
#pragma unroll
        for (int w = 0; w < kThreads / 32; ++w) x += swarp[w][tid];
        a.partial[((lam0 + tid) * a.n_events + event) * a.cpe + chunk] = x;
    }
}

// ---- P3: chunks -> ln -> events ----------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kFinThreads) pop_finish_kernel(const PopArgs a)
{
    __shared__ double sh[kFinThreads];
    pdl_launch();
    pdl_wait();
    const int64_t b = blockIdx.x;
    const int tid = threadIdx.x;
    double s = 0.0;
    for (int64_t i = tid; i < a.n_events; i += kFinThreads) {        // this thread's events in ascending order
        const double *p = a.partial + (b * a.n_events + i) * a.cpe;
        double inner = 0.0;
        for (int c = 0; c < a.cpe; ++c) inner += __ldcg(p + c);      // chunk order
        s += log(inner);                                             // ln 0 = -inf: an event without support
    }
    sh[tid] = s;
    __syncthreads();
    for (int o = kFinThreads / 2; o > 0; o >>= 1) {
        if (tid < o) sh[tid] += sh[tid + o];
        __syncthreads();
    }
    if (tid == 0) {
        const double r1 = a.rec[b * kRec + R_R1];
        a.lnl[b] = (r1 != r1) ? r1 : sh[0];                          // an invalid Lambda is NaN whatever the sums say
    }
}

} // namespace gwpop

// =====================================================================================================================
// C-ABI (include/gwpop.h)
// =====================================================================================================================
using namespace gwpop;

struct gw_pop_ctx {
    int      device;
    int64_t  n_events, n_samples, total, max_batch;
    int      cpe;                  // chunks per event
    double  *planes;               // [kPlanes][total]
    double  *rec;                  // [max_batch][kRec]
    double  *partial;              // [max_batch][n_events][cpe]
    double  *lambda_stage, *lnl_stage;   // host-variant staging
    int64_t  launches;
    int      last_cuda_error;
    int      timing;
    cudaEvent_t ev[4];
};

namespace {

int pop_fail(gw_pop_ctx *ctx, cudaError_t e)
{
    if (ctx) ctx->last_cuda_error = (int)e;
    return e == cudaErrorMemoryAllocation ? GW_ERR_ALLOC : GW_ERR_CUDA;
}

bool pop_is_device_ptr(const void *p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

struct PopDeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit PopDeviceGuard(const gw_pop_ctx *ctx)
    {
        if (ctx && cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device)
            switched = cudaSetDevice(ctx->device) == cudaSuccess;
    }
    ~PopDeviceGuard() { if (switched) cudaSetDevice(prev); }
};

template <typename K, typename A>
cudaError_t launch_pdl(K kernel, dim3 grid, dim3 block, cudaStream_t s, const A &args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, args);
}

} // namespace

extern "C" {

int gw_pop_ctx_create(gw_pop_ctx **out, int64_t n_events, int64_t n_samples, const double *samples,
                      const double *prior, int64_t max_batch, void *cuda_stream)
{
    if (!out) return GW_ERR_INVALID_ARG;
    *out = nullptr;
    if (!samples || !prior || n_events < 1 || n_samples < 1 || max_batch < 1) return GW_ERR_INVALID_ARG;
    if ((double)n_events * (double)n_samples > 4.0e9 || max_batch > (1 << 24)) return GW_ERR_INVALID_ARG;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return GW_ERR_CUDA;
    if (prop.major != 10) return GW_ERR_ARCH;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    gw_pop_ctx *ctx = new (std::nothrow) gw_pop_ctx;
    if (!ctx) return GW_ERR_ALLOC;
    std::memset(ctx, 0, sizeof(*ctx));
    ctx->device = dev;
    ctx->n_events = n_events; ctx->n_samples = n_samples; ctx->total = n_events * n_samples; ctx->max_batch = max_batch;
    ctx->cpe = (int)((n_samples + kChunk - 1) / kChunk);
    const int64_t total = ctx->total;
    double *d_samples = nullptr, *d_prior = nullptr;
    int *d_bad = nullptr, h_bad = 0;
    int rc = GW_OK;
    cudaError_t e = cudaSuccess;
    do {
        bool ok = true;
        ok = ok && (e = cudaMalloc(&ctx->planes, sizeof(double) * kPlanes * total)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&ctx->rec, sizeof(double) * kRec * max_batch)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&ctx->partial, sizeof(double) * max_batch * n_events * ctx->cpe)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&ctx->lambda_stage, sizeof(double) * GW_POP_NLAMBDA * max_batch)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&ctx->lnl_stage, sizeof(double) * max_batch)) == cudaSuccess;
        ok = ok && (e = cudaMalloc(&d_bad, sizeof(int))) == cudaSuccess;
        if (!ok) { rc = pop_fail(ctx, e); break; }
        const double *src_s = samples, *src_p = prior;
        if (!pop_is_device_ptr(samples)) {
            if ((e = cudaMalloc(&d_samples, sizeof(double) * GW_POP_NTHETA * total)) != cudaSuccess) { rc = pop_fail(ctx, e); break; }
            if ((e = cudaMemcpyAsync(d_samples, samples, sizeof(double) * GW_POP_NTHETA * total, cudaMemcpyHostToDevice, s)) != cudaSuccess) { rc = pop_fail(ctx, e); break; }
            src_s = d_samples;
        }
        if (!pop_is_device_ptr(prior)) {
            if ((e = cudaMalloc(&d_prior, sizeof(double) * total)) != cudaSuccess) { rc = pop_fail(ctx, e); break; }
            if ((e = cudaMemcpyAsync(d_prior, prior, sizeof(double) * total, cudaMemcpyHostToDevice, s)) != cudaSuccess) { rc = pop_fail(ctx, e); break; }
            src_p = d_prior;
        }
        if ((e = cudaMemsetAsync(d_bad, 0, sizeof(int), s)) != cudaSuccess) { rc = pop_fail(ctx, e); break; }
        const unsigned blocks = (unsigned)((total + 255) / 256);
        pop_precompute_kernel<<<blocks, 256, 0, s>>>(total, src_s, src_p, ctx->planes, d_bad);
        ctx->launches += 1;
        if ((e = cudaGetLastError()) != cudaSuccess) { rc = pop_fail(ctx, e); break; }
        if ((e = cudaMemcpyAsync(&h_bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, s)) != cudaSuccess) { rc = pop_fail(ctx, e); break; }
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) { rc = pop_fail(ctx, e); break; }
        if (h_bad) rc = GW_ERR_INVALID_ARG;                  // a sample or a prior value outside the documented domain
    } while (0);
    cudaFree(d_samples); cudaFree(d_prior); cudaFree(d_bad);
    if (rc != GW_OK) { gw_pop_ctx_destroy(ctx); cudaGetLastError(); return rc; }
    *out = ctx;
    return GW_OK;
}

int gw_pop_ctx_destroy(gw_pop_ctx *ctx)
{
    if (!ctx) return GW_OK;
    PopDeviceGuard guard(ctx);
    cudaDeviceSynchronize();
    cudaFree(ctx->planes); cudaFree(ctx->rec); cudaFree(ctx->partial); cudaFree(ctx->lambda_stage); cudaFree(ctx->lnl_stage);
    for (int i = 0; i < 4; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    delete ctx;
    cudaGetLastError();
    return GW_OK;
}

int gw_pop_ctx_info(const gw_pop_ctx *ctx, int64_t *n_events, int64_t *n_samples, int64_t *max_batch, int *chunks_per_event)
{
    if (!ctx) return GW_ERR_INVALID_ARG;
    if (n_events) *n_events = ctx->n_events;
    if (n_samples) *n_samples = ctx->n_samples;
    if (max_batch) *max_batch = ctx->max_batch;
    if (chunks_per_event) *chunks_per_event = ctx->cpe;
    return GW_OK;
}

int64_t gw_pop_ctx_launch_count(const gw_pop_ctx *ctx) { return ctx ? ctx->launches : 0; }

int gw_pop_ctx_kernel_timing(gw_pop_ctx *ctx, int enable)
{
    if (!ctx) return GW_ERR_INVALID_ARG;
    if (enable && !ctx->ev[0])
        for (int i = 0; i < 4; ++i) {
            cudaError_t e = cudaEventCreate(&ctx->ev[i]);
            if (e != cudaSuccess) return pop_fail(ctx, e);
        }
    ctx->timing = enable ? 1 : 0;
    return GW_OK;
}

int gw_pop_ctx_last_kernel_ms(gw_pop_ctx *ctx, double *setup_ms, double *main_ms, double *finish_ms)
{
    if (!ctx || !ctx->ev[0]) return GW_ERR_INVALID_ARG;
    cudaError_t e = cudaEventSynchronize(ctx->ev[3]);
    if (e != cudaSuccess) return pop_fail(ctx, e);
    float t[3] = {0.f, 0.f, 0.f};
    for (int i = 0; i < 3; ++i)
        if ((e = cudaEventElapsedTime(&t[i], ctx->ev[i], ctx->ev[i + 1])) != cudaSuccess) return pop_fail(ctx, e);
    if (setup_ms) *setup_ms = t[0];
    if (main_ms) *main_ms = t[1];
    if (finish_ms) *finish_ms = t[2];
    return GW_OK;
}

int gw_pop_lnl_batch(gw_pop_ctx *ctx, int64_t n_lambda, const double *lambda_dev, double *lnl_out_dev, void *cuda_stream)
{
    if (!ctx || n_lambda < 0) return GW_ERR_INVALID_ARG;
    if (n_lambda == 0) return GW_OK;
    if (!lambda_dev || !lnl_out_dev || n_lambda > ctx->max_batch) return GW_ERR_INVALID_ARG;
    PopDeviceGuard guard(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    PopArgs a;
    a.planes = ctx->planes; a.rec = ctx->rec; a.total = ctx->total; a.n_samples = ctx->n_samples;
    a.n_events = ctx->n_events; a.n_lambda = n_lambda; a.cpe = ctx->cpe; a.partial = ctx->partial; a.lnl = lnl_out_dev;
    cudaError_t e;
    if (ctx->timing) cudaEventRecord(ctx->ev[0], s);
    pop_setup_kernel<<<(unsigned)((n_lambda + 63) / 64), 64, 0, s>>>(n_lambda, lambda_dev, ctx->rec);
    if ((e = cudaGetLastError()) != cudaSuccess) return pop_fail(ctx, e);
    if (ctx->timing) cudaEventRecord(ctx->ev[1], s);
    // one proposal per pass keeps the kernel on the HBM roofline; several per pass reuse every plane value read
    const int64_t grid_x = ctx->n_events * ctx->cpe;
    if (grid_x > 0x7fffffffLL) return GW_ERR_INVALID_ARG;
    if (n_lambda == 1)      e = launch_pdl(pop_main_kernel<1>, dim3((unsigned)grid_x, 1), dim3(kThreads), s, a);
    else if (n_lambda == 2) e = launch_pdl(pop_main_kernel<2>, dim3((unsigned)grid_x, 1), dim3(kThreads), s, a);
    else                    e = launch_pdl(pop_main_kernel<kLamTile>, dim3((unsigned)grid_x, (unsigned)((n_lambda + kLamTile - 1) / kLamTile)), dim3(kThreads), s, a);
    if (e != cudaSuccess) return pop_fail(ctx, e);
    if (ctx->timing) cudaEventRecord(ctx->ev[2], s);
    e = launch_pdl(pop_finish_kernel, dim3((unsigned)n_lambda), dim3(kFinThreads), s, a);
    if (e != cudaSuccess) return pop_fail(ctx, e);
    if (ctx->timing) cudaEventRecord(ctx->ev[3], s);
    ctx->launches += 3;
    return GW_OK;
}

int gw_pop_lnl_batch_host(gw_pop_ctx *ctx, int64_t n_lambda, const double *lambda_host, double *lnl_out_host, void *cuda_stream)
{
    if (!ctx || n_lambda < 0) return GW_ERR_INVALID_ARG;
    if (n_lambda == 0) return GW_OK;
    if (!lambda_host || !lnl_out_host || n_lambda > ctx->max_batch) return GW_ERR_INVALID_ARG;
    PopDeviceGuard guard(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemcpyAsync(ctx->lambda_stage, lambda_host, sizeof(double) * GW_POP_NLAMBDA * n_lambda, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return pop_fail(ctx, e);
    const int rc = gw_pop_lnl_batch(ctx, n_lambda, ctx->lambda_stage, ctx->lnl_stage, cuda_stream);
    if (rc != GW_OK) return rc;
    e = cudaMemcpyAsync(lnl_out_host, ctx->lnl_stage, sizeof(double) * n_lambda, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    return e == cudaSuccess ? GW_OK : pop_fail(ctx, e);
}

} // extern "C"

// =====================================================================================================================
// The no-allocation entry point (include/gwpop.h: gw_pop_lnl_static).  Same kernels, same grids and the same summation
// order as gw_pop_lnl_batch; every byte of scratch lives in the file-scope array below instead of a context's
// cudaMalloc'ed workspace.  This section calls no cudaMalloc / cudaFree / allocating routine and never synchronises.
// =====================================================================================================================

// Layout (doubles): [0, 32) flag block (word 0: the bad-sample flag, cleared by every call) | Lambda records
// [n_lambda][kRec] | partial sums [n_lambda][N][cpe] | planes [kPlanes][N n]; each part starts on a multiple of 32 doubles.
// Every GPU that loads the library holds these 16 MiB until the process exits; every call on a device shares them.
static __device__ __align__(256) double g_pop_static_scratch[GW_POP_STATIC_SCRATCH_DOUBLES];

namespace gwpop {

// a bad sample or prior value (flag set by pop_precompute_kernel) makes every lnL of the call NaN
__global__ void pop_static_poison_kernel(int64_t n_lambda, const int *__restrict__ bad, double *__restrict__ lnl)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n_lambda && *bad != 0) lnl[b] = __longlong_as_double(0x7ff8000000000000LL);
}

} // namespace gwpop

namespace {

constexpr int     kStaticFlagDoubles = 32;
constexpr int     kStaticMaxDevices  = 64;
constexpr int64_t kStaticCapacity    = GW_POP_STATIC_SCRATCH_DOUBLES;

// In host code `g_pop_static_scratch` is a host-side stand-in for the symbol, not a device address: the address the
// kernels may use comes from cudaGetSymbolAddress, looked up once per device with that device current.
std::mutex g_static_mutex;
double    *g_static_addr[kStaticMaxDevices];      // nullptr: this device has not been set up yet
int        g_static_last_cuda_error = 0;

int static_fail(cudaError_t e)
{
    g_static_last_cuda_error = (int)e;
    cudaGetLastError();
    return GW_ERR_CUDA;
}

int64_t round32(int64_t x) { return (x + 31) / 32 * 32; }

// `dev` is the current device
int static_scratch_address(int dev, double **addr)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        int major = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) return static_fail(e);
        if (major != 10) return GW_ERR_ARCH;
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_pop_static_scratch);
        if (e != cudaSuccess) return static_fail(e);
        if (!p) return static_fail(cudaErrorInvalidSymbol);
        g_static_addr[dev] = p;
    }
    *addr = g_static_addr[dev];
    return GW_OK;
}

// device memory (or managed memory) that belongs to device `dev`
bool device_ptr_of(const void *p, int dev)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return (at.type == cudaMemoryTypeDevice && at.device == dev) || at.type == cudaMemoryTypeManaged;
}

} // namespace

extern "C" {

int64_t gw_pop_static_need(int64_t n_events, int64_t n_samples, int64_t n_lambda)
{
    if (n_events < 1 || n_samples < 1 || n_lambda < 0 || n_lambda > (1 << 24)) return -1;
    if ((double)n_events * (double)n_samples > 4.0e9) return -1;
    const int64_t cpe = (n_samples + kChunk - 1) / kChunk;
    return kStaticFlagDoubles + round32(kRec * n_lambda) + round32(n_lambda * n_events * cpe) + kPlanes * n_events * n_samples;
}

int gw_pop_static_last_cuda_error(void) { return g_static_last_cuda_error; }

int gw_pop_lnl_static(int64_t n_events, int64_t n_samples, const double *samples_dev, const double *prior_dev,
                      int64_t n_lambda, const double *lambda_dev, double *lnl_out_dev, void *cuda_stream)
{
    const int64_t need = gw_pop_static_need(n_events, n_samples, n_lambda);
    if (need < 0) return GW_ERR_INVALID_ARG;
    if (n_lambda == 0) return GW_OK;
    if (!samples_dev || !prior_dev || !lambda_dev || !lnl_out_dev) return GW_ERR_INVALID_ARG;
    if (need > kStaticCapacity) return GW_POP_ERR_TOO_LARGE;
    const int64_t total = n_events * n_samples;
    const int     cpe = (int)((n_samples + kChunk - 1) / kChunk);
    const int64_t grid_x = n_events * cpe;
    if (grid_x > 0x7fffffffLL) return GW_ERR_INVALID_ARG;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(e);
    if (dev < 0 || dev >= kStaticMaxDevices) return GW_ERR_INVALID_ARG;
    if (!device_ptr_of(samples_dev, dev) || !device_ptr_of(prior_dev, dev) || !device_ptr_of(lambda_dev, dev) ||
        !device_ptr_of(lnl_out_dev, dev))
        return GW_ERR_INVALID_ARG;
    double *base = nullptr;
    const int rc = static_scratch_address(dev, &base);
    if (rc != GW_OK) return rc;
    int    *bad     = reinterpret_cast<int *>(base);
    double *rec     = base + kStaticFlagDoubles;
    double *partial = rec + round32(kRec * n_lambda);
    double *planes  = partial + round32(n_lambda * n_events * cpe);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    // the array keeps the last call's contents: the flag must start at zero; records, partial sums and planes are
    // written in full by this call's kernels before anything reads them
    if ((e = cudaMemsetAsync(base, 0, sizeof(double) * kStaticFlagDoubles, s)) != cudaSuccess) return static_fail(e);
    pop_precompute_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(total, samples_dev, prior_dev, planes, bad);
    if ((e = cudaGetLastError()) != cudaSuccess) return static_fail(e);
    // launched without the programmatic attribute: starts after the precompute kernel has finished, so the main
    // kernel (which may start as soon as the setup kernel runs, and loads planes before waiting for it) sees them
    pop_setup_kernel<<<(unsigned)((n_lambda + 63) / 64), 64, 0, s>>>(n_lambda, lambda_dev, rec);
    if ((e = cudaGetLastError()) != cudaSuccess) return static_fail(e);
    PopArgs a;
    a.planes = planes; a.rec = rec; a.total = total; a.n_samples = n_samples; a.n_events = n_events;
    a.n_lambda = n_lambda; a.cpe = cpe; a.partial = partial; a.lnl = lnl_out_dev;
    if (n_lambda == 1)      e = launch_pdl(pop_main_kernel<1>, dim3((unsigned)grid_x, 1), dim3(kThreads), s, a);
    else if (n_lambda == 2) e = launch_pdl(pop_main_kernel<2>, dim3((unsigned)grid_x, 1), dim3(kThreads), s, a);
    else                    e = launch_pdl(pop_main_kernel<kLamTile>, dim3((unsigned)grid_x, (unsigned)((n_lambda + kLamTile - 1) / kLamTile)), dim3(kThreads), s, a);
    if (e != cudaSuccess) return static_fail(e);
    if ((e = launch_pdl(pop_finish_kernel, dim3((unsigned)n_lambda), dim3(kFinThreads), s, a)) != cudaSuccess) return static_fail(e);
    pop_static_poison_kernel<<<(unsigned)((n_lambda + 127) / 128), 128, 0, s>>>(n_lambda, bad, lnl_out_dev);
    if ((e = cudaGetLastError()) != cudaSuccess) return static_fail(e);
    return GW_OK;
}

} // extern "C"
