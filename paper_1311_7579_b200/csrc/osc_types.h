// osc_types.h -- plain-data parameter blocks handed from the host precompute (row a1) to the kernels.
// Everything here depends only on the oscillation parameters, never on the event energy
// ("components that are dependent only on the oscillation parameters ... are computed on
// the CPU and then copied to the GPU").  The blocks travel as __grid_constant__ kernel parameters, so
// every launch owns its copy in the constant bank (include/osc.h "Asynchrony").
#pragma once

namespace oscb {

constexpr int kChannels = 4;     // OSC_N_CHANNELS
constexpr int kTransDoubles = 10; // doubles per OscTrans (9 used + 1 pad: whole 16-byte words in shared memory)

// Energy-independent quantities of one parameter set that the eigenvalue solve needs.  The cubic's
// coefficients depend on U only through |U_ei|^2, so the block serves neutrinos and antineutrinos.
struct OscSet {
    double xq23;  // (2/3) K_PHASE L / pi : (2/3) R gap * xq23 / E is the half gap phase in units of pi/2
    double tr;    // dm2_21 + dm2_31                                   (c2 = A + tr)
    double dd;    // dm2_21 dm2_31                                     (c1 = A k1 + dd)
    double k1;    // dm2_21 (1 - |Ue2|^2) + dm2_31 (1 - |Ue3|^2)
    double k0_27; // 27 dm2_21 dm2_31 |Ue1|^2                          (27 c0 = A k0_27)
};

// One transition alpha -> beta for neutrinos or antineutrinos.
//   T_{beta alpha}     = (Tr0 + A ee) + i Ti0
//   (T^2)_{beta alpha} = (T2r0 + A T2r1 + A^2 ee) + i (T2i0 + A T2i1)
struct OscTrans {
    double sa;    // +-K_MATTER Y_E rho : A = sa * E
    double delta; // 1 if alpha == beta
    double ee;    // 1 if alpha == beta == e
    double Tr0, Ti0, T2r0, T2i0, T2r1, T2i1;
    double pad;
};

// osc_prob: one transition.
struct ProbArgs {
    OscSet set;
    OscTrans tr;
};

// osc_prob_all: the 2x2 block (alpha, beta in {e, mu}) is assembled, the other five probabilities
// follow from unitarity (rows and columns of |S|^2 sum to 1).
struct ProbAllArgs {
    OscSet set;
    OscTrans tr[4]; // index 2*beta + alpha, alpha, beta in {0, 1}
};

// osc_reweight_bin[_batch]: one parameter set with the four channels of include/osc.h.
// 46 doubles = 23 16-byte words (set padded to 6 doubles).
struct BinArgs {
    OscSet set;
    double pad;
    OscTrans ch[kChannels];
};
constexpr int kBinArgsDoubles = 6 + kChannels * kTransDoubles;
static_assert(sizeof(BinArgs) == sizeof(double) * kBinArgsDoubles, "BinArgs layout");

} // namespace oscb
