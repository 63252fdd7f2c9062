/*
 * osc.h -- C ABI of libosc_b200: per-event three-flavour neutrino oscillation probability through
 * constant-density matter, event reweighting and binned-PDF filling on one NVIDIA B200 (sm_100a).
 *
 * The calls follow the paper's statement of the problem (arXiv:1311.7579; line numbers are those of
 * PAPER.md) and BASELINE.json:north_star:
 *   - the oscillation-parameter set of Table 1 goes in through osc_set_params;
 *     everything that depends only on the parameters is computed once on the host and handed to the
 *     kernels ("computed on the CPU and then copied to the GPU");
 *   - an array of true energies in, one oscillation weight per element out, double precision
 *     (Listing 1)                                                  -> osc_prob[_all];
 *   - each Monte Carlo event weighted by its oscillation probability and binned into a histogram, the
 *     PDF, with the energy-scale systematic applied by "simply scaling the ...
 *     reconstructed energy"                                          -> osc_reweight_bin;
 *   - one PDF rebuild per proposed parameter set                    -> osc_reweight_bin_batch.
 *
 * Conventions (DESIGN.md "Readings of the paper" A1..A16):
 *   - phase m^2 L / 2E = OSC_K_PHASE * m^2[eV^2] * L[km] / E[GeV];
 *     matter term A = OSC_K_MATTER * OSC_Y_E * rho[g/cm^3] * E[GeV] (eV^2), sign flipped for antineutrinos;
 *   - PMNS matrix in the PDG parametrisation, input angles as sin^2(theta_ij); antineutrinos use U*;
 *   - m^2 = (0, dm2_21, dm2_31), dm2_31 = hierarchy * |dm2_32| + dm2_21;
 *   - P(alpha -> beta) = |S_{beta alpha}|^2, S = exp(-i H L), flavour index 0 = e, 1 = mu, 2 = tau.
 *
 * Memory: every array argument marked DEVICE is caller-owned device memory on the current CUDA device
 * (for PyTorch: tensor.data_ptr()); the library neither frees nor keeps caller pointers beyond the work
 * it enqueues.  HOST arguments are read before the call returns.  fp64 arrays must be 8-byte aligned.
 *
 * Asynchrony: osc_prob*, osc_reweight_bin* enqueue work on `stream` (a cudaStream_t passed as void*;
 * NULL = the legacy default stream) and return without synchronising; results are valid once the caller
 * has synchronised the stream.  osc_set_params is host-synchronous and affects only calls made after it
 * returns: each launch carries its own copy of the parameter block (kernel-parameter constant bank), so
 * changing parameters never races with work already enqueued.
 *
 * Errors: every call returns an osc_status (0 = OK, negative = error) and never throws or aborts;
 * osc_last_error() gives the message of the calling thread's most recent failure.  Per-event data
 * faults cannot be reported synchronously and have defined data semantics instead (A11): an event whose
 * E_true is not finite or <= 0 yields NaN from osc_prob[_all] and is skipped by osc_reweight_bin*; so is
 * an event whose channel code is outside [0, n_channels).
 */
#ifndef OSC_B200_H
#define OSC_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OSC_K_PHASE 2.5338653580781979     /* rad per (eV^2 km / GeV): 1e3 / (2e9 hbar c [eV m])        */
#define OSC_K_MATTER 1.5264932449499478e-4 /* eV^2 per (GeV g/cm^3): 2 sqrt2 G_F (hbar c)^3 N_A 1e18    */
#define OSC_Y_E 0.5                        /* electrons per nucleon                                      */

typedef enum {
    OSC_OK = 0,
    OSC_ERR_INVALID_ARG = -1,    /* null pointer with n > 0, flavour/hierarchy/range violation, non-finite scalar */
    OSC_ERR_NOT_CONFIGURED = -2, /* osc_set_params has not been called successfully                               */
    OSC_ERR_CUDA = -3,           /* a CUDA runtime call failed (message in osc_last_error)                        */
    OSC_ERR_ALIGNMENT = -4       /* an fp64 array pointer is not 8-byte aligned                                   */
} osc_status;

enum { OSC_NU_E = 0, OSC_NU_MU = 1, OSC_NU_TAU = 2 }; /* flavour index */
enum { OSC_NORMAL = 1, OSC_INVERTED = -1 };           /* mass hierarchy */

/* Number of reweighting channels and their meaning (BASELINE.json configs[2]):
 * channel 0: nu_mu -> nu_mu, 1: nu_mu -> nu_e, 2: nubar_mu -> nubar_mu, 3: nubar_mu -> nubar_e. */
#define OSC_N_CHANNELS 4

/* One oscillation-parameter set; same fields and order as osc_set_params. */
typedef struct {
    double sin2_th12, sin2_th23, sin2_th13; /* sin^2(theta_ij), each in [0, 1]            */
    double dm2_32;                          /* |Delta m^2_32| in eV^2, > 0                 */
    double dm2_21;                          /* Delta m^2_21 in eV^2, >= 0                  */
    double delta_cp;                        /* radians                                     */
    double rho_g_cm3;                       /* matter density in g/cm^3, >= 0              */
    double L_km;                            /* baseline in km, >= 0                        */
    int hierarchy;                          /* OSC_NORMAL or OSC_INVERTED                  */
} osc_params;

/* Host-side per-parameter-set precompute.
 * Stores the parameter block that later calls hand to their kernels.  Thread-safe; host only.
 * Returns OSC_ERR_INVALID_ARG (state unchanged) if any value is outside the ranges listed above. */
int osc_set_params(double sin2_th12, double sin2_th23, double sin2_th13, double dm2_32, double dm2_21,
                   double delta_cp, double rho_g_cm3, double L_km, int hierarchy);

/* Per-event probability (rows a2a-a2f, kernel calculateOscProb of Listing 1).
 *   E_true  DEVICE [n]  true neutrino energies in GeV
 *   P_out   DEVICE [n]  P(flavour_in -> flavour_out) for (anti)neutrinos; NaN where E_true is unusable
 * n == 0 is a no-op returning OSC_OK. */
int osc_prob(const double *E_true, size_t n, int flavour_in, int flavour_out, int antinu, double *P_out,
             void *stream);

/* All nine transitions from one eigen-solve per event (BASELINE.json configs[1]).
 *   P_out   DEVICE [9][n] row-major; row 3*beta + alpha holds P(alpha -> beta). */
int osc_prob_all(const double *E_true, size_t n, int antinu, double *P_out, void *stream);

/* Fused reweight + histogram (rows a3a-a3c).  For every event j with usable
 * E_true[j] and channel[j] in [0, OSC_N_CHANNELS):
 *     x = fl64(energy_scale * E_reco[j])                      (one rounded fp64 multiply)
 *     b = the unique i with bin_edges[i] <= x < bin_edges[i+1] (fp64 compares); no such i -> event dropped
 *     hist_out[channel[j]][b] += w0[j] * P_channel(E_true[j])
 *   E_true, E_reco, w0  DEVICE [n] fp64;   channel  DEVICE [n] int8
 *   bin_edges           DEVICE [n_bins + 1] fp64, strictly increasing (not checked: device data)
 *   hist_out            DEVICE [OSC_N_CHANNELS][n_bins] fp64 row-major, OVERWRITTEN (zeroed when n == 0)
 * No per-event weight array is written to memory.  The result is bit-reproducible from run to run for
 * fixed inputs (fixed event -> thread map, fixed-order merges, no floating-point atomics).
 * The launch shape follows n_bins (one block per SM of 768, 512, 384 or 256 threads);
 * osc_set_k2_tuning overrides it for measurements and tests.  No environment variable is read. */
int osc_reweight_bin(const double *E_true, const double *E_reco, const double *w0, const int8_t *channel,
                     size_t n, double energy_scale, const double *bin_edges, int n_bins, double *hist_out,
                     void *stream);

/* osc_reweight_bin for several energy-scale values in one pass over the events: slice k
 * of hist_out equals osc_reweight_bin run with energy_scales[k] (to rounding: the order of the additions
 * differs; the result is bit-reproducible from run to run).  The oscillation weight does not depend on the
 * energy scale (it uses the unscaled E_true), so the closed form runs once per event instead of
 * once per event and scale.
 *   energy_scales  HOST [n_scales], 1 <= n_scales <= 4, each finite and > 0
 *   hist_out       DEVICE [n_scales][OSC_N_CHANNELS][n_bins] fp64, OVERWRITTEN
 * Binnings whose sub-histograms do not fit shared memory n_scales times fall back to one pass per scale. */
int osc_reweight_bin_scales(const double *E_true, const double *E_reco, const double *w0, const int8_t *channel,
                            size_t n, const double *energy_scales, int n_scales, const double *bin_edges,
                            int n_bins, double *hist_out, void *stream);

/* osc_reweight_bin for callers that cannot allocate (code under CUDA stream capture, tight serving loops, harnesses
 * that forbid cudaMalloc): same arguments, same result (to rounding; bit-identical where osc_reweight_bin picks the
 * same launch shape), but the kernel's scratch -- ticket counters, bin-table cache, per-block partial histograms -- is a
 * static device array inside the library instead of the per-stream buffer osc_reweight_bin allocates on first use.
 * This call and everything below it call no cudaMalloc / cudaMallocAsync / cudaFree and no allocating library routine.
 *   limit      n_bins <= 128 (OSC_ERR_INVALID_ARG above, state unchanged); any n as for osc_reweight_bin
 *   cost       the array is 1 130 496 bytes; every GPU that loads the library holds it until the process exits
 *   sharing    ALL calls on a device share the array, whatever their stream: calls that overlap on the GPU (different
 *              streams, or graphs replayed concurrently) RACE on it and give wrong histograms; calls on one stream are
 *              ordered and safe.  The array keeps the last call's contents; the call zeroes the counters it needs.
 * Inputs and outputs are the caller's, as for osc_reweight_bin; hist_out is OVERWRITTEN. */
int osc_reweight_bin_static(const double *E_true, const double *E_reco, const double *w0, const int8_t *channel,
                            size_t n, double energy_scale, const double *bin_edges, int n_bins, double *hist_out,
                            void *stream);

/* Batched parameter sets (row a4; BASELINE.json configs[3]): slice p of hist_out equals
 * osc_reweight_bin run with points[p] (to rounding: the order of the additions differs).  Independent of
 * the state set by osc_set_params.
 *   points    HOST [n_points]; validated and copied before the call returns
 *   hist_out  DEVICE [n_points][OSC_N_CHANNELS][n_bins] fp64, OVERWRITTEN
 * Three code paths, chosen per call from the point list (results agree to rounding, each is
 * bit-reproducible from run to run):
 *   - points that differ only in sin2_th23 and delta_cp share the matter eigen-problem.  When the list has
 *     at least 8 points per such group on average (a scan grid: "only theta23 and dm2_32
 *     float"), the events are sorted by histogram cell once and the eigen-solve is done once per (event,
 *     group); a point then costs 3 to 6 fused multiply-adds per event (k4, csrc/osc_scan.cuh: from 1e5 events
 *     on one launch per sub-group of 32 points with the point monomials in the kernel parameters, below that
 *     one launch with the event terms in shared memory);
 *   - otherwise every (event, point) pair gets the full closed form: from 4 points on (6 for more than
 *     2e6 events), on the events sorted by histogram cell, with the weights of a cell summed in registers
 *     (kernel k5); below that the sort does not pay and every point gets its own pass of
 *     osc_reweight_bin's kernel (k2).  Binnings up to the library's limit of 768 bins are taken by all paths.
 * osc_set_batch_path forces one path (tests use it to check the paths on the same inputs). */
int osc_reweight_bin_batch(const osc_params *points, int n_points, const double *E_true,
                           const double *E_reco, const double *w0, const int8_t *channel, size_t n,
                           double energy_scale, const double *bin_edges, int n_bins, double *hist_out,
                           void *stream);

/* Plans: the same histograms for callers that keep the event sample, the energy scale and the binning fixed
 * over many calls -- the Markov chain of the paper's toy fit proposes new oscillation parameters at every step
 * and rebuilds the PDF from the same simulated events.  osc_plan_create sorts the events by
 * histogram cell once (the sort of osc_reweight_bin_batch, kept on the device: 16 bytes per event); the
 * reweight calls then run the sorted-event kernels only: no bin search and no shared-memory histogram per
 * call, the weights of a cell are summed in registers.
 *   osc_plan_create              arguments as osc_reweight_bin; *plan_out receives the plan.  The caller's event
 *                                arrays are not needed once the work enqueued on `stream` has run.
 *   osc_plan_reweight_bin        hist_out DEVICE [OSC_N_CHANNELS][n_bins], OVERWRITTEN; parameters of osc_set_params;
 *                                equals osc_reweight_bin on the planned events to rounding (order of additions)
 *   osc_plan_reweight_bin_batch  hist_out DEVICE [n_points][OSC_N_CHANNELS][n_bins]; as osc_reweight_bin_batch
 *   osc_plan_destroy             frees the plan (synchronises with work that still reads it); NULL is a no-op
 * A plan belongs to the device that was current at creation.  Calls that use a plan must be ordered after its
 * creation (same stream, or a synchronisation in between).  Results are bit-reproducible from run to run. */
typedef struct osc_plan osc_plan;
int osc_plan_create(const double *E_true, const double *E_reco, const double *w0, const int8_t *channel, size_t n,
                    double energy_scale, const double *bin_edges, int n_bins, void *stream, osc_plan **plan_out);
int osc_plan_reweight_bin(const osc_plan *plan, double *hist_out, void *stream);
int osc_plan_reweight_bin_batch(const osc_plan *plan, const osc_params *points, int n_points, double *hist_out,
                                void *stream);
int osc_plan_destroy(osc_plan *plan);

/* Binned Poisson likelihood of rebuilt PDFs against a data histogram (PAPER.md:125-128,
 * eq. 2.1, read as a product of Poisson probabilities of the bin contents -- DESIGN.md R5):
 *     out[p] = -2 ln lambda_p = 2 sum_i [ mu - D_i + D_i ln(D_i / mu) ],   mu = norm * hist[p][i],
 * the likelihood ratio against the saturated model (D_i ln(...) := 0 for D_i = 0; mu = 0 with D_i > 0 gives
 * +inf; a negative or non-finite mu or D_i gives NaN).  Run after osc_reweight_bin_batch on the same stream,
 * it leaves n_points doubles to copy back per scan instead of n_points histograms.
 *   hist  DEVICE [n_points][n_cells] fp64 (n_cells = OSC_N_CHANNELS * n_bins for a full batched output)
 *   data  DEVICE [n_cells] fp64, >= 0;   norm  finite, > 0;   out  DEVICE [n_points] fp64, overwritten */
int osc_neg2lnl(const double *hist, int n_points, int n_cells, const double *data, double norm, double *out,
                void *stream);

/* Bin-centre reweighting against event-by-event reweighting ("calculate the
 * effect of the variation at the center of each bin and apply it to the whole bin" versus "retain all of the
 * simulated events", the comparison behind the paper's 2.6 % example).  Bins are in TRUE energy here:
 *     hist_event_out[c][b]  = sum over events j of channel c with bin_edges[b] <= E_true[j] < bin_edges[b+1]
 *                             of w0[j] * P_c(E_true[j])          (= osc_reweight_bin with E_reco := E_true, scale 1)
 *     hist_centre_out[c][b] = P_c((bin_edges[b] + bin_edges[b+1]) / 2) * sum over the same events of w0[j]
 * with the parameters of osc_set_params.  The binning bias of a cell is hist_centre / hist_event - 1.
 *   E_true, w0 DEVICE [n] fp64; channel DEVICE [n] int8; bin_edges DEVICE [n_bins + 1] fp64, strictly increasing
 *   hist_event_out, hist_centre_out  DEVICE [OSC_N_CHANNELS][n_bins] fp64, OVERWRITTEN
 * A bin centre that is not a usable energy (<= 0 or non-finite) gives NaN in hist_centre_out. */
int osc_bin_centre_compare(const double *E_true, const double *w0, const int8_t *channel, size_t n,
                           const double *bin_edges, int n_bins, double *hist_event_out, double *hist_centre_out,
                           void *stream);

/* Debug/verification export of the integer binning decision of osc_reweight_bin (row a3c):
 *   bin_out  DEVICE [n] int32: the bin index b of event j, or -1 if the event is dropped. */
int osc_bin_index(const double *E_true, const double *E_reco, const int8_t *channel, size_t n,
                  double energy_scale, const double *bin_edges, int n_bins, int32_t *bin_out, void *stream);

/* Same as the osc_prob / osc_reweight_bin pair but with HOST buffers: copies the inputs to the device,
 * runs the kernels, copies the result back and synchronises.  This is the flow of the paper's Listing 1
 * and what bench.py times as "e2e".  The reweight calls send more than 2^20 events in up to 8
 * chunks and run the kernel on one chunk while the next is on the bus; the per-chunk histograms are added in chunk
 * order, so the result is still a deterministic function of the inputs (equal to the device call to rounding).
 * Pinned host arrays make the copies asynchronous; pageable ones work, without the overlap. */
int osc_prob_host(const double *E_true_host, size_t n, int flavour_in, int flavour_out, int antinu,
                  double *P_out_host);
int osc_reweight_bin_host(const double *E_true_host, const double *E_reco_host, const double *w0_host,
                          const int8_t *channel_host, size_t n, double energy_scale,
                          const double *bin_edges_host, int n_bins, double *hist_out_host);
/* The same for several energy-scale values (osc_reweight_bin_scales): the events cross PCIe once for all scales.
 *   energy_scales  HOST [n_scales], 1 <= n_scales <= 4;   hist_out_host  HOST [n_scales][OSC_N_CHANNELS][n_bins] */
int osc_reweight_bin_scales_host(const double *E_true_host, const double *E_reco_host, const double *w0_host,
                                 const int8_t *channel_host, size_t n, const double *energy_scales, int n_scales,
                                 const double *bin_edges_host, int n_bins, double *hist_out_host);

/* Measurement and test overrides (process-wide, thread-safe; they affect calls enqueued afterwards).
 *   osc_set_batch_path  path = "auto" (default: the library chooses, see osc_reweight_bin_batch), "k2", "k4" or "k5":
 *                       the code path of osc_reweight_bin_batch / osc_plan_reweight_bin_batch ("k2" does not apply to plans);
 *                       "k4s" / "k4c": k4 with its shared-memory kernel / its kernel-parameter kernel whatever the size.
 *   osc_set_k2_tuning   launch shape of osc_reweight_bin's kernel; 0 leaves a field to the library.
 *                       threads in {128, 256, 384, 512, 768}, slots in {1, 2} (sub-histograms per warp: one, or one per
 *                       event of the lane), n_sub in {1, 2, 4} (sub-histograms per slot), blocks_per_sm <= 16.
 *                       A combination that does not fit in shared memory makes the call it would shape return
 *                       OSC_ERR_INVALID_ARG or OSC_ERR_CUDA, never a wrong histogram.
 * Both return OSC_ERR_INVALID_ARG (state unchanged) for any other value. */
int osc_set_batch_path(const char *path);
int osc_set_k2_tuning(int threads, int slots, int n_sub, int blocks_per_sm);

/* Message of the calling thread's most recent error ("" if none).  Never NULL. */
const char *osc_last_error(void);

/* Number of kernel launches this library has enqueued since it was loaded (for bench.py's gpu_launches). */
unsigned long long osc_launch_count(void);

/* Library version string, e.g. "osc_b200 0.2 (sm_100a)". */
const char *osc_version(void);

/* The library works on the calling thread's current CUDA device.  These two wrap cudaSetDevice /
 * cudaGetDevice of the library's own (statically linked) CUDA runtime so that a caller which picked its
 * device through another runtime instance (PyTorch) can check and align the two. */
int osc_set_device(int device);
int osc_get_device(int *device /* HOST, out */);

/* Measurement helper, not part of the hot path: enqueues one launch of a register-only chain of
 * independent fp64 fused multiply-adds on every SM (blocks_per_sm blocks of 256 threads each, 8 chains
 * per thread, `iters` DFMAs per chain) and reports in *flops_per_launch (HOST, out, may be NULL) the
 * floating-point operations of that launch (2 per DFMA).  bench.py times it with CUDA events to obtain
 * the measured fp64 peak that roofline fractions are quoted against. */
int osc_fp64_peak_probe(int iters, int blocks_per_sm, double *flops_per_launch, void *stream);

/* Measurement helper, not part of the hot path: one launch of a register-resident loop of ONE instruction pattern
 * (8 independent chains per thread, blocks_per_sm blocks of 256 threads on every SM), so that ncu's
 * smsp__inst_executed / sm__cycles_elapsed, or CUDA events and the SM clock, give the issue cost of the pattern in
 * cycles per warp instruction and SM sub-partition (profiles/r2_dfma_issue.md).
 *   kind 0: DFMA with three distinct register operands;  1: DFMA, two registers + immediate;  2: DFMA, one register;
 *        3: DMUL;  4: DADD;  5: kind 0 + two three-register FFMA per DFMA;  6: kind 0 + two IMAD per DFMA
 * *fp64_inst_per_launch (HOST, out, may be NULL) receives the fp64 thread instructions of the launch. */
int osc_fp64_issue_probe(int kind, int iters, int blocks_per_sm, double *fp64_inst_per_launch, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* OSC_B200_H */
