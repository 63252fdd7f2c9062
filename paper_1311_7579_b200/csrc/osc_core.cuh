// osc_core.cuh -- the per-event closed form shared by all kernels (rows a2a-a2f of SURVEY.md 8(a)).
//
// Matter Hamiltonian in the flavour basis (eV^2): T = M + A e e^dagger, M = U diag(m^2) U^dagger,
// A = +-K_MATTER Y_E rho E (A3, A6).  With eigenvalues lam0 >= lam1 >= lam2 and
// the global phase exp(-i lam0 x) dropped (x = K_PHASE L / E),
//
//     S' = E1 I - a P0 + b P2,   E1 = exp(i g01 x),  a = E1 - 1,  b = exp(i g02 x) - E1,
//     P0 = (T - lam1)(T - lam2) / (g01 g02),          P2 = (T - lam0)(T - lam1) / (g02 g12),
//
// g_ij = lam_i - lam_j >= 0.  a/g01 and b/g12 are sinc-like and finite when a gap closes, so nothing
// here divides by a small gap.  Dropping one more common phase,
//
//     Z = delta e^{i h1} - i kap0 N0 + i kap2 e^{i h02} N2,     P(alpha -> beta) = |Z_{beta alpha}|^2,
//     h1 = g01 x / 2, h12 = g12 x / 2, h02 = h1 + h12,
//     kap0 = 2 sin(h1) / (g01 g02),  kap2 = 2 sin(h12) / (g12 g02),
//     N0 = T^2 - (lam1 + lam2) T + lam1 lam2 I,  N2 = T^2 - (lam0 + lam1) T + lam0 lam1 I.
//
// The eigenvalues come from the trigonometric solution of the characteristic cubic
// lam^3 - c2 lam^2 + c1 lam - c0 (BASELINE.json:north_star item 2): lam_k = c2/3 + (2/3) R tau_k with
// R^2 = c2^2 - 3 c1 and tau the roots of 4 tau^3 - 3 tau = u, u = (2 c2^3 - 9 c2 c1 + 27 c0)/(2 R^3).
// Only |u| is solved (largest root t, osc_math.cuh); for u < 0 the roots are negated, which is R -> -R.
#pragma once
#include "osc_math.cuh"
#include "osc_types.h"

namespace oscb {

struct OscEig {
    double c1h, s1h;       // cos, sin of h1
    double c02, s02;       // cos, sin of h02
    double kap0, kap2;
    double sum12, prod12;  // lam1 + lam2, lam1 lam2
    double sum01, prod01;  // lam0 + lam1, lam0 lam1
};

// Rows a2a-a2d: eigenvalues, gap phases and the two sinc-like factors for matter term A at 1/E.
__device__ __forceinline__ void eig_solve(const OscSet& ps, double A, double invE, OscEig& o, const PolyTop& top)
{
    const double SQ3 = 1.7320508075688772;
    const double HALF_SQ3 = 0.8660254037844386;

    // a2b characteristic polynomial
    double c2 = A + ps.tr;
    double c1 = fma(A, ps.k1, ps.dd);
    double c0_27 = A * ps.k0_27;
    double c1_3 = 3.0 * c1;
    double R2 = fma(c2, c2, -c1_3);             // (1/2) sum of squared gaps: > 0 for every valid parameter set
    R2 = floor_hi_word(R2, 0x03000000);         // (DESIGN.md "R2 > 0"); the floor 2^-975 only keeps NaN out
    double tq = fma(2.0, R2, -c1_3);            // 2 c2^2 - 9 c1
    double q = fma(c2, tq, c0_27);              // 2 c2^3 - 9 c2 c1 + 27 c0

    // a2c trigonometric cubic
    double rinv = rsqrt_pos(R2);
    double rinv2 = rinv * rinv;
    double U2 = (q * rinv) * rinv2;             // 2 u = 2 cos(3 phi)
    const int sgn = __double2hiint(U2) & 0x80000000; // sign of u: for u < 0 the roots of |u| are negated, i.e. R -> -R
    double t, rh;
    cos_third_acos(fabs(U2), t, rh);            // t = cos(phi'), rh = 1 / (24 t^2 - 6)
    double om = 1.0 - t;
    double w = fma(om, t, om);                  // 1 - t^2 = sin^2(phi')
    w = floor_hi_word(w, 0x39B00000);           // >= 2^-100: a closed gap stays finite (sinc form below)
    double y = rsqrt_pos(w);
    double s = w * y;                           // sin(phi')
    // roots of 4 tau^3 - 3 tau = |u|: t >= t - ga >= -m; gaps (in units of (2/3) R) ga >= gb >= 0
    double ga = fma(-HALF_SQ3, s, 1.5 * t);
    double gb = SQ3 * s;
    double m = fma(HALF_SQ3, s, 0.5 * t);

    // signed radius: eigenvalue "0" is c2/3 + Rs t, eigenvalue "2" is c2/3 - Rs m; for u < 0 that labelling runs
    // upwards instead of downwards, which the projector form does not care about (all gaps change sign together)
    double R = flip_sign_if(R2 * rinv, sgn);
    double Rs = R * (2.0 / 3.0);
    double c2_3 = c2 * (1.0 / 3.0);
    double lam0 = fma(Rs, t, c2_3);
    double lam2 = fma(-Rs, m, c2_3);
    o.sum12 = c2 - lam0;
    o.prod12 = fma(-lam0, o.sum12, c1);
    o.sum01 = c2 - lam2;
    o.prod01 = fma(-lam2, o.sum01, c1);

    // 2/(g01 g02) and 2/(g12 g02) (sign-free products of two gaps): ga (ga + gb) = 3 t^2 - 3/4 = (24 t^2 - 6) / 8
    double rr = rh * rinv2;
    double ka = 36.0 * rr;                                  // 2 / (Rs^2 ga gc)
    double kb = (rr * (36.0 / SQ3)) * (ga * y);             // 2 / (Rs^2 gb gc)

    // a2d gap phases in quarter turns: g R xq23 / E (signed with R)
    double RX = R * (ps.xq23 * invE);
    double s1, c1c, s12, c12;
    sincos_quarter_mul(ga, RX, s1, c1c, top);
    sincos_quarter_mul(gb, RX, s12, c12, top);
    o.s1h = s1;
    o.c1h = c1c;
    o.c02 = fma(c1c, c12, -(s1 * s12));
    o.s02 = fma(s1, c12, c1c * s12);
    o.kap0 = s1 * ka;
    o.kap2 = s12 * kb;
}

__device__ __forceinline__ void eig_solve(const OscSet& ps, double A, double invE, OscEig& o)
{
    eig_solve(ps, A, invE, o, poly_top());
}

// Rows a2e-a2f: |Z_{beta alpha}|^2 for one transition.
__device__ __forceinline__ double assemble(const OscEig& e, double A, const OscTrans& tr)
{
    double Tr = fma(A, tr.ee, tr.Tr0);
    double Ti = tr.Ti0;
    double T2r = fma(A, fma(A, tr.ee, tr.T2r1), tr.T2r0);
    double T2i = fma(A, tr.T2i1, tr.T2i0);
    double N0r = fma(e.prod12, tr.delta, fma(-e.sum12, Tr, T2r));
    double N0i = fma(-e.sum12, Ti, T2i);
    double N2r = fma(e.prod01, tr.delta, fma(-e.sum01, Tr, T2r));
    double N2i = fma(-e.sum01, Ti, T2i);
    double Wr = fma(e.c02, N2r, -(e.s02 * N2i));
    double Wi = fma(e.s02, N2r, e.c02 * N2i);
    double Zr = fma(tr.delta, e.c1h, fma(e.kap0, N0i, -(e.kap2 * Wi)));
    double Zi = fma(tr.delta, e.s1h, fma(e.kap2, Wr, -(e.kap0 * N0r)));
    return fma(Zr, Zr, Zi * Zi);
}

// The same for a diagonal element (alpha == beta): T and T^2 are Hermitian, so the imaginary parts of the entry
// vanish and delta = 1.  EE: the element is (e, e), the only one that carries the matter term.
template <bool EE>
__device__ __forceinline__ double assemble_diag(const OscEig& e, double A, const OscTrans& tr)
{
    const double Tr = EE ? A + tr.Tr0 : tr.Tr0;
    const double T2r = EE ? fma(A, A + tr.T2r1, tr.T2r0) : fma(A, tr.T2r1, tr.T2r0);
    const double N0r = e.prod12 + fma(-e.sum12, Tr, T2r);
    const double N2r = e.prod01 + fma(-e.sum01, Tr, T2r);
    const double kn = e.kap2 * N2r;
    const double Zr = fma(-kn, e.s02, e.c1h);
    const double Zi = fma(kn, e.c02, fma(-e.kap0, N0r, e.s1h));
    return fma(Zr, Zr, Zi * Zi);
}

// ... and for the off-diagonal pair (alpha, beta), (beta, alpha) with neither index on (e, e)'s matter term twice:
// delta = 0, ee = 0, and the two entries of T, T^2 are complex conjugates of each other, so N0, N2 of the second
// element are the conjugates of the first.  tr describes alpha -> beta; P_ab = P(alpha -> beta), P_ba the reverse.
__device__ __forceinline__ void assemble_offdiag_pair(const OscEig& e, double A, const OscTrans& tr, double& P_ab,
                                                      double& P_ba)
{
    const double T2r = fma(A, tr.T2r1, tr.T2r0);
    const double T2i = fma(A, tr.T2i1, tr.T2i0);
    const double N0r = fma(-e.sum12, tr.Tr0, T2r), N0i = fma(-e.sum12, tr.Ti0, T2i);
    const double N2r = fma(-e.sum01, tr.Tr0, T2r), N2i = fma(-e.sum01, tr.Ti0, T2i);
    const double cr = e.c02 * N2r, sr = e.s02 * N2r;
    const double Wr = fma(-e.s02, N2i, cr), Wi = fma(e.c02, N2i, sr);          // alpha -> beta
    const double Vr = fma(e.s02, N2i, cr), Vi = fma(-e.c02, N2i, sr);          // beta -> alpha (N2i -> -N2i)
    const double k0r = e.kap0 * N0r, k0i = e.kap0 * N0i;
    const double Zr = fma(-e.kap2, Wi, k0i), Zi = fma(e.kap2, Wr, -k0r);
    const double Yr = fma(-e.kap2, Vi, -k0i), Yi = fma(e.kap2, Vr, -k0r);
    P_ab = fma(Zr, Zr, Zi * Zi);
    P_ba = fma(Yr, Yr, Yi * Yi);
}

// One off-diagonal element alone (delta = 0, ee = 0).
__device__ __forceinline__ double assemble_offdiag(const OscEig& e, double A, const OscTrans& tr)
{
    const double T2r = fma(A, tr.T2r1, tr.T2r0);
    const double T2i = fma(A, tr.T2i1, tr.T2i0);
    const double N0r = fma(-e.sum12, tr.Tr0, T2r), N0i = fma(-e.sum12, tr.Ti0, T2i);
    const double N2r = fma(-e.sum01, tr.Tr0, T2r), N2i = fma(-e.sum01, tr.Ti0, T2i);
    const double Wr = fma(e.c02, N2r, -(e.s02 * N2i));
    const double Wi = fma(e.s02, N2r, e.c02 * N2i);
    const double Zr = fma(e.kap0, N0i, -(e.kap2 * Wi));
    const double Zi = fma(e.kap2, Wr, -(e.kap0 * N0r));
    return fma(Zr, Zr, Zi * Zi);
}

// KIND: 0 any element (run-time delta / ee), 1 diagonal (e, e), 2 diagonal (mu, mu) or (tau, tau), 3 off-diagonal.
template <int KIND>
__device__ __forceinline__ double assemble_kind(const OscEig& e, double A, const OscTrans& tr)
{
    if (KIND == 1) return assemble_diag<true>(e, A, tr);
    if (KIND == 2) return assemble_diag<false>(e, A, tr);
    if (KIND == 3) return assemble_offdiag(e, A, tr);
    return assemble(e, A, tr);
}

// A11: usable energy <=> finite and > 0 <=> 0 < bits < 0x7FF0000000000000 (integer pipe).
__device__ __forceinline__ bool energy_ok(double E)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(E);
    return (b - 1ull) < 0x7FEFFFFFFFFFFFFFull;
}

template <int KIND = 0>
__device__ __forceinline__ double prob_one(const OscSet& ps, const OscTrans& tr, double E)
{
    double invE = rcp_pos(E);
    double A = tr.sa * E;
    OscEig e;
    eig_solve(ps, A, invE, e);
    return assemble_kind<KIND>(e, A, tr);
}

} // namespace oscb
