/*
 * osc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, CPU-only statement of what the hot path of arXiv:1311.7579 computes:
 * the three-flavour neutrino oscillation probability through matter of constant
 * density (section 1.1), followed by event-by-event reweighting and
 * histogram filling (section 1.1.1; section 2.2).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this file.  It shares no code, header, table or constant generator
 * with the CUDA path under paper_1311_7579_b200/csrc/, and it does NOT use the
 * closed-form cubic that the CUDA path uses: the matter Hamiltonian is diagonalised by
 * a generic cyclic Jacobi iteration in long double, and the evolution operator is the
 * plain definition S = V exp(-i diag(lambda) x) V^dagger.
 *
 * Steps follow SURVEY.md section 8(c), O1..O9 (readings A1..A16 are listed in DESIGN.md):
 *   O1 constants, O2 angles, O3 PMNS (PDG form), O4 masses, O5 Hamiltonian,
 *   O6 evolution, O7 probability, O8 reweight + bin, O9 batched.
 *
 * Pins (tests/test_oracle_pins.py): vacuum sum over mass states (eq. 1.1 as read in A1),
 * unitarity, two-flavour closed form, one-mass-scale MSW closed forms, T symmetry,
 * L = 0, CPT, independent RK4 integration of the Schroedinger equation, brute-force
 * binning.  No function in this file is "parity unpinned".
 *
 * Floating point: long double (x87 80-bit on x86-64) for everything except the
 * bin-index decision, which is taken in IEEE double exactly as the interface states
 * (one rounded multiply energy_scale * E_reco, then comparisons against the caller's
 * edges).  Build with -ffp-contract=off.
 */
#include <complex.h>
#include <float.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef long double real;
typedef long double complex cplx;

/* O1 constants (paper is silent, readings A2/A3). */
static const real K_PHASE = 2.5338653580781979L;    /* m^2[eV^2] L[km] / (2 E[GeV]) -> rad     */
static const real K_MATTER = 1.5264932449499478e-4L; /* 2 sqrt2 G_F N_A : eV^2 / (GeV g/cm^3)  */
static const real Y_E = 0.5L;                        /* electrons per nucleon                  */

/* Same fields and order as the C-ABI's osc_set_params (BASELINE.json north_star). */
typedef struct {
    double sin2_th12, sin2_th23, sin2_th13;
    double dm2_32, dm2_21, delta_cp;
    double rho_g_cm3, L_km;
    int hierarchy; /* +1 normal, -1 inverted */
} oracle_params;

/* O2 + O3: PMNS matrix in the PDG parametrisation, U[flavour][mass]. */
static void build_pmns(const oracle_params *p, cplx U[3][3])
{
    real s12 = sqrtl((real)p->sin2_th12), c12 = sqrtl(1.0L - (real)p->sin2_th12);
    real s23 = sqrtl((real)p->sin2_th23), c23 = sqrtl(1.0L - (real)p->sin2_th23);
    real s13 = sqrtl((real)p->sin2_th13), c13 = sqrtl(1.0L - (real)p->sin2_th13);
    real d = (real)p->delta_cp;
    cplx ep = cosl(d) + I * sinl(d); /* e^{+i delta} */
    cplx em = cosl(d) - I * sinl(d); /* e^{-i delta} */

    U[0][0] = c12 * c13;
    U[0][1] = s12 * c13;
    U[0][2] = s13 * em;
    U[1][0] = -s12 * c23 - c12 * s23 * s13 * ep;
    U[1][1] = c12 * c23 - s12 * s23 * s13 * ep;
    U[1][2] = s23 * c13;
    U[2][0] = s12 * s23 - c12 * c23 * s13 * ep;
    U[2][1] = -c12 * s23 - s12 * c23 * s13 * ep;
    U[2][2] = c23 * c13;
}

/* O4: mass-squared values (eV^2), m1^2 = 0. */
static void build_masses(const oracle_params *p, real m2[3])
{
    real h = (p->hierarchy >= 0) ? 1.0L : -1.0L;
    m2[0] = 0.0L;
    m2[1] = (real)p->dm2_21;
    m2[2] = h * fabsl((real)p->dm2_32) + (real)p->dm2_21; /* dm2_31 = h |dm2_32| + dm2_21 */
}

/* O5: flavour-basis Hamiltonian in eV^2 at energy E (GeV).
 * T = U' diag(m2) U'^dagger + diag(A,0,0); antineutrinos: U' = U*, A -> -A. */
static void build_hamiltonian(const oracle_params *p, real E, int antinu, cplx T[3][3])
{
    cplx U[3][3];
    real m2[3];
    build_pmns(p, U);
    build_masses(p, m2);
    if (antinu) {
        for (int a = 0; a < 3; ++a)
            for (int i = 0; i < 3; ++i) U[a][i] = conjl(U[a][i]);
    }
    for (int b = 0; b < 3; ++b)
        for (int a = 0; a < 3; ++a) {
            cplx s = 0.0L;
            for (int i = 0; i < 3; ++i) s += U[b][i] * m2[i] * conjl(U[a][i]);
            T[b][a] = s;
        }
    real A = K_MATTER * Y_E * (real)p->rho_g_cm3 * E;
    if (antinu) A = -A;
    T[0][0] += A;
}

static void matmul3(cplx C[3][3], cplx A[3][3], cplx B[3][3])
{
    cplx R[3][3];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            cplx s = 0.0L;
            for (int k = 0; k < 3; ++k) s += A[i][k] * B[k][j];
            R[i][j] = s;
        }
    memcpy(C, R, sizeof(R));
}

static void dagger3(cplx C[3][3], cplx A[3][3])
{
    cplx R[3][3];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) R[i][j] = conjl(A[j][i]);
    memcpy(C, R, sizeof(R));
}

static real offdiag_norm(cplx H[3][3])
{
    real s = 0.0L;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            if (i != j) s += creall(H[i][j] * conjl(H[i][j]));
    return sqrtl(s);
}

static real frob_norm(cplx H[3][3])
{
    real s = 0.0L;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) s += creall(H[i][j] * conjl(H[i][j]));
    return sqrtl(s);
}

/* Generic cyclic Jacobi eigen-decomposition of a 3x3 complex Hermitian matrix:
 * H = V diag(lam) V^dagger.  Each step zeroes one off-diagonal pair (p,q) with a plane
 * unitary J = D G: D = diag(.., 1, .., e^{-i phi}, ..) removes the phase of H_pq,
 * G is the real symmetric-Schur rotation (Golub & Van Loan, "symmetric Schur 2x2"). */
static void jacobi_hermitian3(cplx Hin[3][3], real lam[3], cplx V[3][3])
{
    cplx H[3][3];
    memcpy(H, Hin, sizeof(H));
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) V[i][j] = (i == j) ? 1.0L : 0.0L;

    real scale = frob_norm(H);
    if (scale == 0.0L) {
        lam[0] = lam[1] = lam[2] = 0.0L;
        return;
    }
    for (int sweep = 0; sweep < 64; ++sweep) {
        if (offdiag_norm(H) <= 1e-19L * scale) break;
        for (int p = 0; p < 2; ++p)
            for (int q = p + 1; q < 3; ++q) {
                real absb = cabsl(H[p][q]);
                if (absb == 0.0L) continue;
                cplx phase = H[p][q] / absb; /* e^{i phi} */
                real a = creall(H[p][p]), d = creall(H[q][q]);
                real tau = (d - a) / (2.0L * absb);
                real t = ((tau >= 0.0L) ? 1.0L : -1.0L) / (fabsl(tau) + sqrtl(1.0L + tau * tau));
                real c = 1.0L / sqrtl(1.0L + t * t);
                real s = t * c;
                cplx J[3][3], Jd[3][3];
                for (int i = 0; i < 3; ++i)
                    for (int j = 0; j < 3; ++j) J[i][j] = (i == j) ? 1.0L : 0.0L;
                /* J = D G in the (p,q) plane, D = diag(1, conj(phase)), G = [[c, s], [-s, c]] */
                J[p][p] = c;
                J[p][q] = s;
                J[q][p] = -s * conjl(phase);
                J[q][q] = c * conjl(phase);
                dagger3(Jd, J);
                matmul3(H, Jd, H);
                matmul3(H, H, J);
                matmul3(V, V, J);
                H[p][q] = 0.0L;
                H[q][p] = 0.0L;
            }
    }
    for (int i = 0; i < 3; ++i) lam[i] = creall(H[i][i]);
}

/* O6: S = exp(-i T x), x = K_PHASE L / E, from the Jacobi decomposition. */
static void evolution_matrix(const oracle_params *p, real E, int antinu, cplx S[3][3])
{
    cplx T[3][3], V[3][3];
    real lam[3];
    build_hamiltonian(p, E, antinu, T);
    jacobi_hermitian3(T, lam, V);
    real x = K_PHASE * (real)p->L_km / E;
    for (int b = 0; b < 3; ++b)
        for (int a = 0; a < 3; ++a) {
            cplx s = 0.0L;
            for (int k = 0; k < 3; ++k) {
                real ph = lam[k] * x;
                cplx e = cosl(ph) - I * sinl(ph);
                s += V[b][k] * e * conjl(V[a][k]);
            }
            S[b][a] = s;
        }
}

/* A11: an event energy is usable iff it is finite and > 0. */
static int energy_ok(double E) { return isfinite(E) && E > 0.0; }

/* O7: P(alpha -> beta) = |S_{beta alpha}|^2 for one energy. */
static real prob_one(const oracle_params *p, double E, int fl_in, int fl_out, int antinu)
{
    cplx S[3][3];
    evolution_matrix(p, (real)E, antinu, S);
    cplx z = S[fl_out][fl_in];
    return creall(z * conjl(z));
}

static int params_ok(const oracle_params *p)
{
    if (!p) return 0;
    if (p->hierarchy != 1 && p->hierarchy != -1) return 0;
    return 1;
}

/* ---------------------------------------------------------------------------------- */
/* Exported entry points (plain C, host pointers).                                    */
/* ---------------------------------------------------------------------------------- */

/* P_out[j] = P(fl_in -> fl_out) at E[j]; NaN where the energy is unusable (A11). */
int oracle_prob(const oracle_params *p, const double *E, size_t n, int fl_in, int fl_out, int antinu,
                double *P_out)
{
    if (!params_ok(p) || fl_in < 0 || fl_in > 2 || fl_out < 0 || fl_out > 2) return -1;
#pragma omp parallel for schedule(static)
    for (long long j = 0; j < (long long)n; ++j) {
        if (!energy_ok(E[j])) {
            P_out[j] = NAN;
            continue;
        }
        P_out[j] = (double)prob_one(p, E[j], fl_in, fl_out, antinu);
    }
    return 0;
}

/* P_out[(3*beta + alpha) * n + j] = P(alpha -> beta) at E[j]  (all nine transitions). */
int oracle_prob_all(const oracle_params *p, const double *E, size_t n, int antinu, double *P_out)
{
    if (!params_ok(p)) return -1;
#pragma omp parallel for schedule(static)
    for (long long j = 0; j < (long long)n; ++j) {
        if (!energy_ok(E[j])) {
            for (int k = 0; k < 9; ++k) P_out[(size_t)k * n + j] = NAN;
            continue;
        }
        cplx S[3][3];
        evolution_matrix(p, (real)E[j], antinu, S);
        for (int b = 0; b < 3; ++b)
            for (int a = 0; a < 3; ++a) {
                cplx z = S[b][a];
                P_out[(size_t)(3 * b + a) * n + j] = (double)creall(z * conjl(z));
            }
    }
    return 0;
}

/* Full complex S (row-major [beta][alpha], re/im interleaved, long double narrowed to double)
 * for one energy: lets the tests check unitarity of S itself. */
int oracle_evolution(const oracle_params *p, double E, int antinu, double *S_out /* 18 */)
{
    if (!params_ok(p) || !energy_ok(E)) return -1;
    cplx S[3][3];
    evolution_matrix(p, (real)E, antinu, S);
    for (int b = 0; b < 3; ++b)
        for (int a = 0; a < 3; ++a) {
            S_out[2 * (3 * b + a)] = (double)creall(S[b][a]);
            S_out[2 * (3 * b + a) + 1] = (double)cimagl(S[b][a]);
        }
    return 0;
}

/* Eigenvalues of the matter Hamiltonian (eV^2), ascending, for one energy (test hook). */
int oracle_eigenvalues(const oracle_params *p, double E, int antinu, double *lam_out /* 3 */)
{
    if (!params_ok(p) || !energy_ok(E)) return -1;
    cplx T[3][3], V[3][3];
    real lam[3];
    build_hamiltonian(p, (real)E, antinu, T);
    jacobi_hermitian3(T, lam, V);
    for (int i = 0; i < 3; ++i)
        for (int j = i + 1; j < 3; ++j)
            if (lam[j] < lam[i]) {
                real t = lam[i];
                lam[i] = lam[j];
                lam[j] = t;
            }
    for (int i = 0; i < 3; ++i) lam_out[i] = (double)lam[i];
    return 0;
}

/* Channel table (BASELINE.json configs[2]):
 * 0: numu->numu, 1: numu->nue, 2: numubar->numubar, 3: numubar->nuebar. */
#define ORACLE_N_CHANNELS 4
static const int CH_IN[ORACLE_N_CHANNELS] = {1, 1, 1, 1};
static const int CH_OUT[ORACLE_N_CHANNELS] = {1, 0, 1, 0};
static const int CH_ANTI[ORACLE_N_CHANNELS] = {0, 0, 1, 1};

/* O8 (bin index, readings A8/A9): x = fl64(energy_scale * E_reco); the bin is the unique i
 * with edges[i] <= x < edges[i+1] in IEEE double; -1 when there is none (under/overflow, NaN). */
static int bin_of(double energy_scale, double e_reco, const double *edges, int n_bins)
{
    volatile double x = energy_scale * e_reco; /* one rounded fp64 multiply */
    for (int i = 0; i < n_bins; ++i)
        if (edges[i] <= x && x < edges[i + 1]) return i;
    return -1;
}

/* bin_out[j] = bin index of event j, or -1 if the event is dropped (A8, A11). */
int oracle_bin_index(const double *E_true, const double *E_reco, const int8_t *channel, size_t n,
                     double energy_scale, const double *edges, int n_bins, int32_t *bin_out)
{
    for (size_t j = 0; j < n; ++j) {
        int ch = (int)channel[j];
        if (!energy_ok(E_true[j]) || ch < 0 || ch >= ORACLE_N_CHANNELS) {
            bin_out[j] = -1;
            continue;
        }
        bin_out[j] = bin_of(energy_scale, E_reco[j], edges, n_bins);
    }
    return 0;
}

/* O8: hist[ch][b] = sum over events of w0 * P_channel(E_true), events taken in index order,
 * accumulated in long double, rounded to double at the end.  hist_out is overwritten (A10).
 * The per-event weights are independent and are computed first; the binning
 * loop then runs serially in index order. */
int oracle_reweight_bin(const oracle_params *p, const double *E_true, const double *E_reco,
                        const double *w0, const int8_t *channel, size_t n, double energy_scale,
                        const double *edges, int n_bins, double *hist_out)
{
    if (!params_ok(p) || n_bins < 1) return -1;
    size_t nh = (size_t)ORACLE_N_CHANNELS * (size_t)n_bins;
    real *acc = (real *)calloc(nh, sizeof(real));
    real *w = (real *)malloc((n ? n : 1) * sizeof(real));
    int32_t *bin = (int32_t *)malloc((n ? n : 1) * sizeof(int32_t));
    if (!acc || !w || !bin) {
        free(acc);
        free(w);
        free(bin);
        return -2;
    }
    oracle_bin_index(E_true, E_reco, channel, n, energy_scale, edges, n_bins, bin);
#pragma omp parallel for schedule(static)
    for (long long j = 0; j < (long long)n; ++j) {
        if (bin[j] < 0) {
            w[j] = 0.0L;
            continue;
        }
        int ch = (int)channel[j];
        w[j] = (real)w0[j] * prob_one(p, E_true[j], CH_IN[ch], CH_OUT[ch], CH_ANTI[ch]);
    }
    for (size_t j = 0; j < n; ++j) {
        if (bin[j] < 0) continue;
        acc[(size_t)channel[j] * (size_t)n_bins + (size_t)bin[j]] += w[j];
    }
    for (size_t k = 0; k < nh; ++k) hist_out[k] = (double)acc[k];
    free(acc);
    free(w);
    free(bin);
    return 0;
}

/* O9: slice p of the batched output is O8 with parameter set p. */
int oracle_reweight_bin_batch(const oracle_params *points, int n_points, const double *E_true,
                              const double *E_reco, const double *w0, const int8_t *channel, size_t n,
                              double energy_scale, const double *edges, int n_bins, double *hist_out)
{
    if (n_points < 0) return -1;
    size_t nh = (size_t)ORACLE_N_CHANNELS * (size_t)n_bins;
    for (int k = 0; k < n_points; ++k) {
        int rc = oracle_reweight_bin(&points[k], E_true, E_reco, w0, channel, n, energy_scale, edges,
                                     n_bins, hist_out + (size_t)k * nh);
        if (rc) return rc;
    }
    return 0;
}

/* Binned Poisson likelihood ratio (eq. 2.1; reading R5 in DESIGN.md): for every point p
 *   out[p] = 2 sum_i [ mu - D_i + D_i ln(D_i / mu) ],  mu = norm * hist[p][i],
 * the term D_i ln(.) taken as 0 for D_i = 0; mu = 0 with D_i > 0 gives +inf, mu = 0 with D_i = 0 gives 0;
 * a negative or non-finite mu or D_i gives NaN.  Long double, bins in index order.
 * Pinned in tests/test_oracle_pins.py against scipy.stats.poisson.logpmf and closed forms. */
int oracle_neg2lnl(const double *hist, int n_points, int n_cells, const double *data, double norm, double *out)
{
    if (!hist || !data || !out || n_points < 0 || n_cells < 1 || !(norm > 0.0)) return -1;
    for (int p = 0; p < n_points; ++p) {
        real s = 0.0L;
        for (int i = 0; i < n_cells; ++i) {
            const real mu = (real)norm * (real)hist[(size_t)p * n_cells + i];
            const real D = (real)data[i];
            real term;
            if (!(mu >= 0.0L) || !(D >= 0.0L) || isinf(mu) || isinf(D)) term = NAN;
            else if (mu == 0.0L) term = (D == 0.0L) ? 0.0L : INFINITY;
            else if (D == 0.0L) term = mu;
            else term = mu - D + D * logl(D / mu);
            s += term;
        }
        out[p] = (double)(2.0L * s);
    }
    return 0;
}

/* Bin-centre reweighting beside event-by-event reweighting over TRUE-energy bins:
 *   hist_event[c][b]  = sum_j w0_j P_c(E_j)          over the events of channel c with edges[b] <= E_j < edges[b+1]
 *   hist_centre[c][b] = P_c((edges[b] + edges[b+1]) / 2) * sum_j w0_j   over the same events
 * Events in index order, long double sums; the bin decision in IEEE double as in oracle_reweight_bin. */
int oracle_bin_centre_compare(const oracle_params *p, const double *E_true, const double *w0, const int8_t *channel,
                              size_t n, const double *edges, int n_bins, double *hist_event, double *hist_centre)
{
    if (!params_ok(p) || n_bins < 1) return -1;
    const size_t nh = (size_t)ORACLE_N_CHANNELS * n_bins;
    real *ev = (real *)calloc(nh, sizeof(real)), *un = (real *)calloc(nh, sizeof(real));
    if (!ev || !un) { free(ev); free(un); return -2; }
    for (size_t j = 0; j < n; ++j) {
        const int c = channel[j];
        if (c < 0 || c >= ORACLE_N_CHANNELS || !energy_ok(E_true[j])) continue;
        const int b = bin_of(1.0, E_true[j], edges, n_bins);
        if (b < 0) continue;
        ev[(size_t)c * n_bins + b] += (real)w0[j] * prob_one(p, E_true[j], CH_IN[c], CH_OUT[c], CH_ANTI[c]);
        un[(size_t)c * n_bins + b] += (real)w0[j];
    }
    for (int c = 0; c < ORACLE_N_CHANNELS; ++c)
        for (int b = 0; b < n_bins; ++b) {
            const double centre = 0.5 * (edges[b] + edges[b + 1]);
            const size_t i = (size_t)c * n_bins + b;
            hist_event[i] = (double)ev[i];
            hist_centre[i] = energy_ok(centre) ? (double)(un[i] * prob_one(p, centre, CH_IN[c], CH_OUT[c], CH_ANTI[c])) : NAN;
        }
    free(ev);
    free(un);
    return 0;
}

int oracle_n_channels(void) { return ORACLE_N_CHANNELS; }

#ifdef _OPENMP
#include <omp.h>
int oracle_threads(void) { return omp_get_max_threads(); }
void oracle_set_threads(int n) { if (n > 0) omp_set_num_threads(n); }
#else
int oracle_threads(void) { return 1; }
void oracle_set_threads(int n) { (void)n; }
#endif
