// gw_math.cuh -- device-side fp64 helpers of the CUDA path: lean sin/cos in turns, complex helpers,
// mbarrier / bulk-copy (TMA) PTX wrappers.  sm_100a only.  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gw {

// ---- constants (from exactly defined values; DESIGN.md section 2 "Constants") -------------------------
constexpr double kPi      = 3.14159265358979323846;
constexpr double kTwoPi   = 6.28318530717958647692;
constexpr double kCSI     = 299792458.0;                 // m/s, exact
constexpr double kGMsun   = 1.3271244e20;                // m^3/s^2, IAU 2015 nominal
constexpr double kAU      = 149597870700.0;              // m, exact
constexpr double kEulerG  = 0.57721566490153286061;
constexpr double kLn4     = 1.38629436111989061883;
constexpr double kTsun    = kGMsun / (kCSI * kCSI * kCSI);                       // s
constexpr double kMpcSec  = 1.0e6 * (648000.0 / kPi) * kAU / kCSI;               // s

// ---- lean sincos of an angle given in TURNS ------------------------------------------------------------
// cis_turns(t) returns (cos 2 pi t, sin 2 pi t) for |t| < 2^49.
//   q = rint(4t) by the 1.5*2^52 trick (2 fp64 adds), r = t - q/4 in [-1/8, 1/8] (1 FMA, exact),
//   z = r^2, sin(2 pi r) = r*S(z) (degree 5), cos(2 pi r) = C(z) (degree 6), then the quadrant i^q is
//   applied with integer selects / sign-bit XORs (ALU pipe, not the fp64 pipe).
// 16 fp64-pipe instructions.  Coefficients from gen_sincos_coeffs.py (Chebyshev-node interpolation on
// z in [0, 1/64], 60 digits, rounded): max abs error 3.4e-15 (sin) and 1.0e-16 (cos), i.e. below one ulp
// of the phase itself whenever |phase| > 0.01 turn (the tolerance derivation is DESIGN.md section 8).
#define GW_SIN_S0 6.28318530717956
#define GW_SIN_S1 -41.34170224027578
#define GW_SIN_S2 81.60524918348393
#define GW_SIN_S3 -76.70583445845129
#define GW_SIN_S4 42.05556925594499
#define GW_SIN_S5 -14.916565118819118
#define GW_COS_C0 1.0
#define GW_COS_C1 -19.73920880217842
#define GW_COS_C2 64.93939402236538
#define GW_COS_C3 -85.45681709034115
#define GW_COS_C4 60.24462008593029
#define GW_COS_C5 -26.42425703488269
#define GW_COS_C6 7.810290968144191

__device__ __forceinline__ void cis_turns(double t, double &c_out, double &s_out)
{
    const double magic = 6755399441055744.0;              // 1.5 * 2^52
    const double tq = __fma_rn(t, 4.0, magic);            // low mantissa bits hold rint(4t)
    const int    q  = __double2loint(tq);
    const double n  = tq - magic;
    const double r  = __fma_rn(n, -0.25, t);              // exact
    const double z  = r * r;
    double ps = __fma_rn(GW_SIN_S5, z, GW_SIN_S4);
    double pc = __fma_rn(GW_COS_C6, z, GW_COS_C5);
    ps = __fma_rn(ps, z, GW_SIN_S3);
    pc = __fma_rn(pc, z, GW_COS_C4);
    ps = __fma_rn(ps, z, GW_SIN_S2);
    pc = __fma_rn(pc, z, GW_COS_C3);
    ps = __fma_rn(ps, z, GW_SIN_S1);
    pc = __fma_rn(pc, z, GW_COS_C2);
    ps = __fma_rn(ps, z, GW_SIN_S0);
    pc = __fma_rn(pc, z, GW_COS_C1);
    const double s = ps * r;
    const double c = __fma_rn(pc, z, GW_COS_C0);
    // multiply by i^q: q&3 = 0:(c,s) 1:(-s,c) 2:(-c,-s) 3:(s,-c)
    const bool   odd = (q & 1) != 0;
    const double re = odd ? s : c;
    const double im = odd ? c : s;
    const int neg_re = ((q + 1) & 2) << 30;               // quadrants 1,2
    const int neg_im = (q & 2) << 30;                     // quadrants 2,3
    c_out = __hiloint2double(__double2hiint(re) ^ neg_re, __double2loint(re));
    s_out = __hiloint2double(__double2hiint(im) ^ neg_im, __double2loint(im));
}

#ifndef GW_CIS_QUARTER
#define GW_CIS_QUARTER 1
#endif

// Variant with the range reduction on the conversion pipe (F2I.F64 / I2F.F64 run at 16/clk/SM beside the fp64
// pipe, measured): the argument is given in QUARTER turns, t4 = 4 t, |t4| < 2^31; q = rint(t4) is one conversion,
// r4 = t4 - q one fp64 add, and the polynomials are the same ones rescaled by exact powers of two.
// 14 fp64-pipe instructions instead of 16.
__device__ __forceinline__ void cis_quarter_turns(double t4, double &c_out, double &s_out)
{
    const int    q = __double2int_rn(t4);
    const double r = t4 - __int2double_rn(q);             // in [-1/2, 1/2] quarter turns, exact
    const double z = r * r;
    double ps = __fma_rn(GW_SIN_S5 / 4194304.0, z, GW_SIN_S4 / 262144.0);      // S_k / (4 * 16^k)
    double pc = __fma_rn(GW_COS_C6 / 16777216.0, z, GW_COS_C5 / 1048576.0);    // C_k / 16^k
    ps = __fma_rn(ps, z, GW_SIN_S3 / 16384.0);
    pc = __fma_rn(pc, z, GW_COS_C4 / 65536.0);
    ps = __fma_rn(ps, z, GW_SIN_S2 / 1024.0);
    pc = __fma_rn(pc, z, GW_COS_C3 / 4096.0);
    ps = __fma_rn(ps, z, GW_SIN_S1 / 64.0);
    pc = __fma_rn(pc, z, GW_COS_C2 / 256.0);
    ps = __fma_rn(ps, z, GW_SIN_S0 / 4.0);
    pc = __fma_rn(pc, z, GW_COS_C1 / 16.0);
    const double s = ps * r;
    const double c = __fma_rn(pc, z, GW_COS_C0);
    const bool   odd = (q & 1) != 0;
    const double re = odd ? s : c;
    const double im = odd ? c : s;
    const int neg_re = ((q + 1) & 2) << 30;
    const int neg_im = (q & 2) << 30;
    c_out = __hiloint2double(__double2hiint(re) ^ neg_re, __double2loint(re));
    s_out = __hiloint2double(__double2hiint(im) ^ neg_im, __double2loint(im));
}

// Trimmed variant for the fused likelihood kernel: sin of degree 4 and cos of degree 5 in z (gen_sincos_coeffs.py 4 5:
// max abs error 3.4e-12 and 5.6e-14), 12 fp64-pipe instructions.  The error is 300x below the 1e-9 waveform gate and
// enters lnL far below the 1e-8 gate; the waveform kernel, which is HBM-bound, keeps the
// full-degree polynomials.
#define GW_SINT_S0 6.2831853071524
#define GW_SINT_S1 -41.341702153394905
#define GW_SINT_S2 81.60520471104576
#define GW_SINT_S3 -76.6978663502028
#define GW_SINT_S4 41.47283323950919
#define GW_COST_C0 0.9999999999999444
#define GW_COST_C1 -19.739208801922548
#define GW_COST_C2 64.93939383134831
#define GW_COST_C3 -85.45676493719407
#define GW_COST_C4 60.23818359301454
#define GW_COST_C5 -26.058123753882793
__device__ __forceinline__ void cis_quarter_turns_trim(double t4, double &c_out, double &s_out)
{
    const int    q = __double2int_rn(t4);
    const double r = t4 - __int2double_rn(q);             // in [-1/2, 1/2] quarter turns, exact
    const double z = r * r;
    double ps = __fma_rn(GW_SINT_S4 / 262144.0, z, GW_SINT_S3 / 16384.0);      // S_k / (4 * 16^k)
    double pc = __fma_rn(GW_COST_C5 / 1048576.0, z, GW_COST_C4 / 65536.0);     // C_k / 16^k
    ps = __fma_rn(ps, z, GW_SINT_S2 / 1024.0);
    pc = __fma_rn(pc, z, GW_COST_C3 / 4096.0);
    ps = __fma_rn(ps, z, GW_SINT_S1 / 64.0);
    pc = __fma_rn(pc, z, GW_COST_C2 / 256.0);
    ps = __fma_rn(ps, z, GW_SINT_S0 / 4.0);
    pc = __fma_rn(pc, z, GW_COST_C1 / 16.0);
    const double s = ps * r;
    const double c = __fma_rn(pc, z, GW_COST_C0);
    const bool   odd = (q & 1) != 0;
    const double re = odd ? s : c;
    const double im = odd ? c : s;
    const int neg_re = ((q + 1) & 2) << 30;
    const int neg_im = (q & 2) << 30;
    c_out = __hiloint2double(__double2hiint(re) ^ neg_re, __double2loint(re));
    s_out = __hiloint2double(__double2hiint(im) ^ neg_im, __double2loint(im));
}

// The kernels carry the phase in units of 1/kPhaseScale turns and call cis_phase().
#if GW_CIS_QUARTER
constexpr double kPhaseScale = 4.0;
__device__ __forceinline__ void cis_phase(double t, double &c, double &s) { cis_quarter_turns(t, c, s); }
#ifndef GW_SINCOS_TRIM
#define GW_SINCOS_TRIM 1
#endif
#if GW_SINCOS_TRIM
__device__ __forceinline__ void cis_phase_lnl(double t, double &c, double &s) { cis_quarter_turns_trim(t, c, s); }
#else
__device__ __forceinline__ void cis_phase_lnl(double t, double &c, double &s) { cis_quarter_turns(t, c, s); }
#endif
#else
constexpr double kPhaseScale = 1.0;
__device__ __forceinline__ void cis_phase(double t, double &c, double &s) { cis_turns(t, c, s); }
__device__ __forceinline__ void cis_phase_lnl(double t, double &c, double &s) { cis_turns(t, c, s); }
#endif

// (cos, sin) of 2 pi * (a*b) with the product reduced mod 1 from its exact two-term expansion: used
// where the argument is a frequency times a delay (hundreds of turns) and is evaluated once per thread.
__device__ __forceinline__ void cis_turns_of_product(double a, double b, double &c_out, double &s_out)
{
    const double hi = a * b;
    const double lo = __fma_rn(a, b, -hi);
    const double fr = (hi - rint(hi)) + lo;               // |fr| <= 1/2 + tiny
    sincospi(2.0 * fr, &s_out, &c_out);
}

// ---- mbarrier + bulk async copy (TMA engine, SASS UBLKCP) ------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    const uint32_t addr = smem_u32(bar);
    do {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    } while (!done);
}
// global -> shared bulk copy; bytes % 16 == 0, both addresses 16-byte aligned; completes on `bar`.
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// thread-block cluster: barrier across the CTAs of the cluster, rank, and a load from another CTA's shared memory
// (distributed shared memory: mapa maps a local shared address to the same offset in CTA `rank` of the cluster)
__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ double ld_dsmem_f64(const void *local_smem, uint32_t rank)
{
    uint32_t remote;
    double v;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(local_smem)), "r"(rank));
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(remote) : "memory");
    return v;
}
// programmatic dependent launch
__device__ __forceinline__ void pdl_wait_primary()      { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

} // namespace gw
