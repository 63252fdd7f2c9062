// osc_math.cuh -- fp64 device primitives for the oscillation kernels (sm_100a).
//
// B200 has no fp64 special-function unit: division, sqrt, sincos and acos from the CUDA math library
// expand to long DFMA sequences with argument checks and slow paths.  The per-event closed form only
// needs a handful of primitives on well-conditioned, range-limited arguments, so they are written out
// here with exactly the work the method needs (op budget table):
//   rcp_pos / rsqrt_pos : MUFU seed (upper 32 bits) + one third-order correction
//   sincos_quarter      : argument already in units of pi/2 -> round, exact subtract, two degree-6
//                         polynomials in f^2 (coefficients: osc_coeffs.h), quadrant fix-up on the
//                         integer pipe
//   cos_third_acos      : largest root t of 8 t^3 - 6 t = U (U = 2 cos(3 phi) in [0, 2]) by an fp32
//                         polynomial seed and two chord-Newton steps -- replaces acos + cos.
#pragma once
#include <cuda_runtime.h>
#include "osc_coeffs.h"

namespace oscb {

__device__ __forceinline__ double mufu_rcp64(double a)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    return y;
}

__device__ __forceinline__ double mufu_rsqrt64(double a)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    return y;
}

// 1/a for normal, finite a > 0.  Seed error e0 <= ~2^-20; result error ~e0^3.
__device__ __forceinline__ double rcp_pos(double a)
{
    double y = mufu_rcp64(a);
    double e = fma(-a, y, 1.0);
    e = fma(e, e, e);
    return fma(y, e, y);
}

// 1/sqrt(a) for normal, finite a > 0.  y (1 + e/2 + 3 e^2/8), e = 1 - a y^2.
__device__ __forceinline__ double rsqrt_pos(double a)
{
    double y = mufu_rsqrt64(a);
    double ay = a * y;
    double e = fma(-ay, y, 1.0);
    double p = fma(0.375, e, 0.5);
    p = p * e;
    return fma(y, p, y);
}

__device__ __forceinline__ double flip_sign_if(double v, int cond_bit31)
{
    // cond_bit31: 0 or 0x80000000 -- XOR into the sign bit on the integer pipe
    return __hiloint2double(__double2hiint(v) ^ cond_bit31, __double2loint(v));
}

// sin and cos of (pi/2) * hq for |hq| < 2^31.
__device__ __forceinline__ void sincos_quarter(double hq, double& s, double& c)
{
    const double MAGIC = 6755399441055744.0; // 1.5 * 2^52: adding it rounds hq to the nearest integer
    double kd = hq + MAGIC;
    int k = __double2loint(kd);
    kd -= MAGIC;
    double f = hq - kd; // exact, |f| <= 1/2
    double z = f * f;
    double ps = fma(OSC_SINQ_6, z, OSC_SINQ_5);
    double pc = fma(OSC_COSQ_6, z, OSC_COSQ_5);
    ps = fma(ps, z, OSC_SINQ_4);
    pc = fma(pc, z, OSC_COSQ_4);
    ps = fma(ps, z, OSC_SINQ_3);
    pc = fma(pc, z, OSC_COSQ_3);
    ps = fma(ps, z, OSC_SINQ_2);
    pc = fma(pc, z, OSC_COSQ_2);
    ps = fma(ps, z, OSC_SINQ_1);
    pc = fma(pc, z, OSC_COSQ_1);
    ps = fma(ps, z, OSC_SINQ_0);
    pc = fma(pc, z, OSC_COSQ_0);
    ps = ps * f;
    // quadrant: k odd swaps; sin negative for k & 2; cos negative for (k + 1) & 2
    bool odd = (k & 1) != 0;
    double ss = odd ? pc : ps;
    double cc = odd ? ps : pc;
    s = flip_sign_if(ss, (k & 2) << 30);
    c = flip_sign_if(cc, ((k + 1) & 2) << 30);
}

// t = cos(acos(U/2)/3) in [sqrt(3)/2, 1] for U in [0, 2], i.e. the largest root of 8 t^3 - 6 t = U,
// and rh = 1 / (24 t^2 - 6) = 1 / (2 p'(t)) with p(t) = 4 t^3 - 3 t.
// The seed and the slope reciprocal come from the fp32 pipe; two chord steps (same slope) take the
// seed error (~1e-7) to ~1e-13 and ~1e-19; one third-order step makes rh fp64-accurate.
__device__ __forceinline__ void cos_third_acos(double U, double& t_out, double& rh_out)
{
    float v = __double2float_rn(U) - 1.0f;
    float tf = OSC_T0_9;
    tf = fmaf(tf, v, OSC_T0_8);
    tf = fmaf(tf, v, OSC_T0_7);
    tf = fmaf(tf, v, OSC_T0_6);
    tf = fmaf(tf, v, OSC_T0_5);
    tf = fmaf(tf, v, OSC_T0_4);
    tf = fmaf(tf, v, OSC_T0_3);
    tf = fmaf(tf, v, OSC_T0_2);
    tf = fmaf(tf, v, OSC_T0_1);
    tf = fmaf(tf, v, OSC_T0_0);
    float rf = __frcp_rn(fmaf(24.0f * tf, tf, -6.0f));
    double t = (double)tf;
    double rh = (double)rf;
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        double tt = t * t;
        double a = fma(8.0, tt, -6.0);
        double p2 = fma(a, t, -U);
        t = fma(-p2, rh, t);
    }
    double tt = t * t;
    double pp = fma(24.0, tt, -6.0);
    double d = fma(-pp, rh, 1.0);
    d = fma(d, d, d);
    rh_out = fma(rh, d, rh);
    t_out = t;
}

} // namespace oscb
