// osc_math.cuh -- fp64 device primitives for the oscillation kernels (sm_100a).
//
// B200 has no fp64 special-function unit: division, sqrt, sincos and acos from the CUDA math library
// expand to long DFMA sequences with argument checks and slow paths.  The per-event closed form only
// needs a handful of primitives on well-conditioned, range-limited arguments, so they are written out
// here with exactly the work the method needs (op budget table):
//   rcp_pos / rsqrt_pos : MUFU seed (upper 32 bits) + one third-order correction
//   sincos_quarter_mul  : sin, cos of (pi/2) a b -- the product is rounded to the nearest integer
//                         and subtracted inside fused multiply-adds (exact residual), then two
//                         polynomials in f^2 (degree 5 for the sine, 6 for the cosine) (coefficients: osc_coeffs.h) and a quadrant
//                         fix-up on the integer pipe
//   cos_third_acos      : largest root t of 8 t^3 - 6 t = U (U = 2 cos(3 phi) in [0, 2]) by an fp32
//                         polynomial seed and two chord-Newton steps -- replaces acos + cos.
//
// The fp64 pipe (16 lanes per SM sub-partition) is the resource that bounds the kernels, so everything
// that can run elsewhere does: selections, sign flips and guards use integer instructions, the seed of
// the cubic root runs on the fp32 pipe, and full-width fp64 constants live in __constant__ memory so
// that DFMA reads them as a constant-bank operand instead of materialising them with two moves each.
#pragma once
#include <cuda_runtime.h>
#include "osc_coeffs.h"

namespace oscb {

// [0..5] sin(pi/2 f)/f in z = f^2, [6..12] cos(pi/2 f) in z, [13] 1.5 * 2^52
__constant__ double kPoly[14] = {
    OSC_SINQ_0, OSC_SINQ_1, OSC_SINQ_2, OSC_SINQ_3, OSC_SINQ_4, OSC_SINQ_5,
    OSC_COSQ_0, OSC_COSQ_1, OSC_COSQ_2, OSC_COSQ_3, OSC_COSQ_4, OSC_COSQ_5, OSC_COSQ_6,
    6755399441055744.0};

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

__device__ __forceinline__ float mufu_rcp32(float a)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(a));
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

// v raised to at least 2^e by one integer max on the upper word (hi_floor = upper word of 2^e): zero, denormals,
// negatives and anything else below 2^e come out in [2^e, 2^(e+1)) -- the low word is kept, the result is only used
// where "some positive number of that size" is all that matters.  v must not be NaN.
__device__ __forceinline__ double floor_hi_word(double v, int hi_floor)
{
    return __hiloint2double(max(__double2hiint(v), hi_floor), __double2loint(v));
}

// The four coefficients that start the two polynomials: fma(c12, z, c11) and fma(c5, z, c4) have TWO constant
// operands, a DFMA takes one from a uniform register, so ptxas loads the other into a register with LDC -- inside the
// event loop, and the DFMA then waits for it on the short scoreboard.  A kernel whose loop has the registers keeps the
// four in registers (pin_loop_consts in osc_kernels.cuh); everyone else passes poly_top() and gets the code as before.
struct PolyTop {
    double c4, c5, c10, c11;
};
__device__ __forceinline__ PolyTop poly_top() { return PolyTop{kPoly[4], kPoly[5], kPoly[10], kPoly[11]}; }

// sin and cos of (pi/2) * a * b for |a b| < 2^31.
__device__ __forceinline__ void sincos_quarter_mul(double a, double b, double& s, double& c, const PolyTop& top)
{
    const double MAGIC = kPoly[13];          // adding 1.5 * 2^52 rounds to the nearest integer
    double kd = fma(a, b, MAGIC);
    const int k = __double2loint(kd);
    kd -= MAGIC;
    const double f = fma(a, b, -kd);         // exact product minus integer: |f| <= 1/2 (+ 1 ulp of a b)
    const double z = f * f;
    double pc = fma(kPoly[12], z, top.c11);
    double ps = fma(top.c5, z, top.c4);
    pc = fma(pc, z, top.c10);
    ps = fma(ps, z, kPoly[3]);
    pc = fma(pc, z, kPoly[9]);
    ps = fma(ps, z, kPoly[2]);
    pc = fma(pc, z, kPoly[8]);
    ps = fma(ps, z, kPoly[1]);
    pc = fma(pc, z, kPoly[7]);
    ps = fma(ps, z, kPoly[0]);
    pc = fma(pc, z, kPoly[6]);
    ps = ps * f;
    // quadrant: k odd swaps; sin negative for k & 2; cos negative for (k + 1) & 2
    const bool odd = (k & 1) != 0;
    const double ss = odd ? pc : ps;
    const double cc = odd ? ps : pc;
    s = flip_sign_if(ss, (k & 2) << 30);
    c = flip_sign_if(cc, ((k + 1) & 2) << 30);
}
__device__ __forceinline__ void sincos_quarter_mul(double a, double b, double& s, double& c)
{
    sincos_quarter_mul(a, b, s, c, poly_top());
}

// t = cos(acos(U/2)/3) in [sqrt(3)/2, 1] for U in [0, 2], i.e. the largest root of 8 t^3 - 6 t = U,
// and rh = 1 / (24 t^2 - 6) = 1 / (2 p'(t)) with p(t) = 4 t^3 - 3 t.
// The seed (degree-5 polynomial, |error| < 1e-6 including fp32 rounding) and the slope reciprocal come
// from the fp32 pipe; two chord steps with that fixed slope contract the error by ~3 e0 each
// (e0 -> ~3e-12 -> ~1e-17); one third-order step makes rh fp64-accurate for the final t.
__device__ __forceinline__ void cos_third_acos(double U, double& t_out, double& rh_out)
{
    const float v = __double2float_rn(U) - 1.0f;
    float tf = OSC_T5_5;
    tf = fmaf(tf, v, OSC_T5_4);
    tf = fmaf(tf, v, OSC_T5_3);
    tf = fmaf(tf, v, OSC_T5_2);
    tf = fmaf(tf, v, OSC_T5_1);
    tf = fmaf(tf, v, OSC_T5_0);
    const float rf = mufu_rcp32(fmaf(24.0f * tf, tf, -6.0f));
    double t = (double)tf;
    const double rh = (double)rf;
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const double tt = t * t;
        const double a = fma(8.0, tt, -6.0);
        const double p2 = fma(a, t, -U);
        t = fma(-p2, rh, t);
    }
    const double tt = t * t;
    const double pp = fma(24.0, tt, -6.0);
    double d = fma(-pp, rh, 1.0);
    d = fma(d, d, d);
    rh_out = fma(rh, d, rh);
    t_out = t;
}

} // namespace oscb
