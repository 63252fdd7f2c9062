// osc_precompute.h -- host-side per-parameter-set precompute.
//
// From the nine scalars of osc_set_params: the PMNS matrix U in the PDG parametrisation (A6),
// the mass-squared values m^2 = (0, dm2_21, dm2_31) (A5), the flavour-basis mass matrix
// M = U diag(m^2) U^dagger and its square, the energy-independent pieces of the characteristic cubic of
// T = M + A e e^dagger, and per transition the entries of M, M^2 that the kernels combine with A.
// Plain double arithmetic on the host; a few hundred flops per parameter set.
#pragma once
#include <cmath>
#include <complex>

#include "../../include/osc.h"
#include "osc_types.h"

namespace oscb {

struct HostSet {
    osc_params p;
    std::complex<double> M[3][3];  // U diag(m2) U^dagger          (neutrinos; antineutrinos use conj)
    std::complex<double> M2[3][3]; // M M
    double a = 0.0;                // K_MATTER Y_E rho             (A = +-a E)
    OscSet set;
};

inline bool finite_d(double v) { return std::isfinite(v); }

// Range checks of include/osc.h (osc_params field comments).  Returns nullptr if fine, else a message.
inline const char* check_params(const osc_params& p)
{
    const double v[8] = {p.sin2_th12, p.sin2_th23, p.sin2_th13, p.dm2_32, p.dm2_21, p.delta_cp, p.rho_g_cm3, p.L_km};
    for (double x : v)
        if (!finite_d(x)) return "non-finite oscillation parameter";
    if (p.sin2_th12 < 0.0 || p.sin2_th12 > 1.0) return "sin2_th12 outside [0, 1]";
    if (p.sin2_th23 < 0.0 || p.sin2_th23 > 1.0) return "sin2_th23 outside [0, 1]";
    if (p.sin2_th13 < 0.0 || p.sin2_th13 > 1.0) return "sin2_th13 outside [0, 1]";
    if (!(p.dm2_32 > 0.0)) return "dm2_32 must be > 0 (its sign comes from hierarchy)";
    if (p.dm2_21 < 0.0) return "dm2_21 must be >= 0";
    if (p.rho_g_cm3 < 0.0) return "rho_g_cm3 must be >= 0";
    if (p.L_km < 0.0) return "L_km must be >= 0";
    if (p.hierarchy != OSC_NORMAL && p.hierarchy != OSC_INVERTED) return "hierarchy must be +1 or -1";
    return nullptr;
}

inline void precompute(const osc_params& p, HostSet& h)
{
    typedef std::complex<double> cd;
    const double PI = 3.14159265358979323846;
    h.p = p;
    h.a = 0.0;
    const double s12 = std::sqrt(p.sin2_th12), c12 = std::sqrt(1.0 - p.sin2_th12);
    const double s23 = std::sqrt(p.sin2_th23), c23 = std::sqrt(1.0 - p.sin2_th23);
    const double s13 = std::sqrt(p.sin2_th13), c13 = std::sqrt(1.0 - p.sin2_th13);
    const cd ep(std::cos(p.delta_cp), std::sin(p.delta_cp)); // e^{+i delta}
    const cd em = std::conj(ep);

    cd U[3][3];
    U[0][0] = c12 * c13;
    U[0][1] = s12 * c13;
    U[0][2] = s13 * em;
    U[1][0] = -s12 * c23 - c12 * s23 * s13 * ep;
    U[1][1] = c12 * c23 - s12 * s23 * s13 * ep;
    U[1][2] = s23 * c13;
    U[2][0] = s12 * s23 - c12 * c23 * s13 * ep;
    U[2][1] = -c12 * s23 - s12 * c23 * s13 * ep;
    U[2][2] = c23 * c13;

    const double d21 = p.dm2_21;
    const double d31 = (p.hierarchy == OSC_INVERTED ? -p.dm2_32 : p.dm2_32) + p.dm2_21;
    const double m2[3] = {0.0, d21, d31};

    for (int b = 0; b < 3; ++b)
        for (int a = 0; a < 3; ++a) {
            cd s = 0.0;
            for (int i = 0; i < 3; ++i) s += U[b][i] * m2[i] * std::conj(U[a][i]);
            h.M[b][a] = s;
        }
    for (int b = 0; b < 3; ++b) h.M[b][b] = cd(h.M[b][b].real(), 0.0); // Hermitian: exact real diagonal
    for (int b = 0; b < 3; ++b)
        for (int a = 0; a < 3; ++a) {
            cd s = 0.0;
            for (int k = 0; k < 3; ++k) s += h.M[b][k] * h.M[k][a];
            h.M2[b][a] = s;
        }

    h.a = OSC_K_MATTER * OSC_Y_E * p.rho_g_cm3;

    // |U_ei|^2 straight from the angles (independent of delta and theta23)
    const double ue1 = (1.0 - p.sin2_th12) * (1.0 - p.sin2_th13);
    const double ue2 = p.sin2_th12 * (1.0 - p.sin2_th13);
    const double ue3 = p.sin2_th13;
    h.set.xq23 = (2.0 / 3.0) * OSC_K_PHASE * p.L_km / PI;
    h.set.tr = d21 + d31;
    h.set.dd = d21 * d31;
    h.set.k1 = d21 * (1.0 - ue2) + d31 * (1.0 - ue3);
    h.set.k0_27 = 27.0 * d21 * d31 * ue1;
}

// Entries for the transition alpha -> beta (P = |S_{beta alpha}|^2), neutrinos or antineutrinos.
inline OscTrans make_trans(const HostSet& h, int alpha, int beta, int antinu)
{
    typedef std::complex<double> cd;
    OscTrans t;
    const double sgn = antinu ? -1.0 : 1.0; // antineutrinos: M -> conj(M), A -> -A
    t.sa = sgn * h.a;
    t.delta = (alpha == beta) ? 1.0 : 0.0;
    t.ee = (alpha == 0 && beta == 0) ? 1.0 : 0.0;
    const cd m = h.M[beta][alpha], m2 = h.M2[beta][alpha];
    cd lin = 0.0; // coefficient of A in (T^2)_{beta alpha}: M_{beta e} d_{alpha e} + d_{beta e} M_{e alpha}
    if (alpha == 0) lin += h.M[beta][0];
    if (beta == 0) lin += h.M[0][alpha];
    t.Tr0 = m.real();
    t.Ti0 = sgn * m.imag();
    t.T2r0 = m2.real();
    t.T2i0 = sgn * m2.imag();
    t.T2r1 = lin.real();
    t.T2i1 = sgn * lin.imag();
    t.pad = 0.0;
    return t;
}

// Channel table of include/osc.h: (flavour_in, flavour_out, antinu).
inline void channel_def(int ch, int& fin, int& fout, int& anti)
{
    static const int IN[kChannels] = {1, 1, 1, 1};
    static const int OUT[kChannels] = {1, 0, 1, 0};
    static const int ANTI[kChannels] = {0, 0, 1, 1};
    fin = IN[ch];
    fout = OUT[ch];
    anti = ANTI[ch];
}

inline void make_bin_args(const HostSet& h, BinArgs& b)
{
    b.set = h.set;
    b.pad = 0.0;
    for (int c = 0; c < kChannels; ++c) {
        int fin, fout, anti;
        channel_def(c, fin, fout, anti);
        b.ch[c] = make_trans(h, fin, fout, anti);
    }
}

} // namespace oscb
