// osc_kernels.cuh -- sm_100a kernels of libosc_b200.
//
//   prob_kernel            k1   one transition per event                        (osc_prob)
//   prob_all_kernel        k1b  nine transitions from one eigen-solve           (osc_prob_all)
//   reweight_bin_kernel    k2   fused probability -> weight -> bin -> histogram  (osc_reweight_bin)
//   (the batched call, osc_reweight_bin_batch, lives in osc_scan.cuh: k4 and k5 on events sorted by histogram cell)
//   bin_index_kernel            the integer binning decision of k2, exported  (osc_bin_index)
//
// k1, k1b and k2 are persistent grid-stride kernels sized from the SM count; every thread carries two
// events per iteration (two independent fp64 dependency chains) and the parameter block arrives as a
// __grid_constant__ kernel parameter.  DESIGN.md "Kernels" has the per-event operation budget and
// the roofline that bounds each of them.
#pragma once
#include <cstdint>

#include "osc_bins.cuh"
#include "osc_core.cuh"
#include "osc_hist.cuh"

namespace oscb {

constexpr int kBlock = 256;          // threads per block of k1b and the small kernels (8 warps)
constexpr int kBlockProbAll = 640;   // k1b above ~4e5 events: one block of 20 warps per SM, 96 registers per thread (us per call of
                                     // 1e7 events: 384 threads 230, 512 150.7, 640 148.8, 768 154.4, 896 156.5, 1024 160.0;
                                     // two blocks of 512: 158.1, four of 256: 163.4)
constexpr int kProbAllAhead = 3;     // slots k1b loads its energies ahead of the arithmetic (us per call of 1e7 events:
                                     // 1 slot 148.8, 2 slots 143.7, 3 slots 138.8, 4 slots 148.9, 6 slots 146.7)
constexpr int kBlockProb = 768;      // k1 above ~5e5 events: ONE block of 24 warps per SM (as k2; 88.7 us against 95.0 us
                                     // per 1e7 events for four blocks of 256, whose warps finish at different times)

// Streaming loads/stores: every event byte is touched once (evict-first, no L1 allocation).
__device__ __forceinline__ double ld_stream(const double* p) { return __ldcs(p); }
__device__ __forceinline__ double2 ld_stream2(const double* p) { return __ldcs(reinterpret_cast<const double2*>(p)); }
__device__ __forceinline__ void st_stream(double* p, double v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream2(double* p, double a, double b)
{
    __stcs(reinterpret_cast<double2*>(p), make_double2(a, b));
}

// The same load as ld_stream, pinned where it is written: ptxas is free to sink an ordinary load of a __restrict__
// array down to its first use, which turns a prefetch issued at the top of a loop body into a load issued at its
// bottom (seen in k1b: the loop then waits a full memory latency at its head in every iteration).
__device__ __forceinline__ double ld_stream_pinned(const double* p)
{
    double v;
    asm volatile("ld.global.cs.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ double qnan() { return __longlong_as_double(0x7FF8000000000000LL); }

// Lanes of the warp below this one (%lanemask_lt): one special-register read where the compiler would otherwise
// rebuild (1 << lane) - 1 from the thread index in every iteration.
__device__ __forceinline__ unsigned lanemask_lt()
{
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// p[0 .. count) = 0.0 with 16-byte stores (p 16-byte aligned); called by all threads of the block.
__device__ __forceinline__ void zero_shared(double* p, int count)
{
    double2* q = reinterpret_cast<double2*>(p);
    for (int i = threadIdx.x; i < count / 2; i += blockDim.x) q[i] = make_double2(0.0, 0.0);
    if (threadIdx.x == 0 && (count & 1)) p[count - 1] = 0.0;
}

// ------------------------------------------------------------------------------------------------
// k1: P_out[j] = P(alpha -> beta)(E_true[j]).  VEC: pointers 16-byte aligned -> 128-bit accesses.
// KIND: which element of S is asked for (assemble_kind): the launch knows it, so the assembly is specialised.
// ------------------------------------------------------------------------------------------------
template <bool VEC, int KIND, int THREADS>
__global__ void __launch_bounds__(THREADS, THREADS >= 512 ? 1 : 4)
prob_kernel(const __grid_constant__ ProbArgs a, const double* __restrict__ E_true, size_t n,
            double* __restrict__ P_out)
{
    // VEC: slot i holds events (2i, 2i+1); otherwise tile i / THREADS holds events j0 and j0 + THREADS.
    // The energies of the thread's next slot are loaded before the arithmetic of the current one.
    const size_t nslots = VEC ? (n + 1) / 2 : ((n + 2 * THREADS - 1) / (2 * THREADS)) * THREADS;
    const size_t stride = (size_t)gridDim.x * THREADS;
    auto load = [&](size_t i, double& E0, double& E1) {
        const size_t j0 = VEC ? 2 * i : (i / THREADS) * (2 * THREADS) + (i % THREADS);
        const size_t j1 = VEC ? j0 + 1 : j0 + THREADS;
        if (VEC && j1 < n) {
            const double2 v = ld_stream2(E_true + j0);
            E0 = v.x;
            E1 = v.y;
        } else {
            E0 = (j0 < n) ? ld_stream(E_true + j0) : 1.0;
            E1 = (j1 < n) ? ld_stream(E_true + j1) : 1.0;
        }
    };
    size_t i = (size_t)blockIdx.x * THREADS + threadIdx.x;
    double N0 = 1.0, N1 = 1.0;
    if (i < nslots) load(i, N0, N1);
    while (i < nslots) {
        const size_t j0 = VEC ? 2 * i : (i / THREADS) * (2 * THREADS) + (i % THREADS);
        const size_t j1 = VEC ? j0 + 1 : j0 + THREADS;
        const bool has1 = j1 < n;
        const double E0 = N0, E1 = N1;
        i += stride;
        if (i < nslots) load(i, N0, N1);
        const bool ok0 = energy_ok(E0), ok1 = energy_ok(E1);
        double P0 = prob_one<KIND>(a.set, a.tr, ok0 ? E0 : 1.0);
        double P1 = prob_one<KIND>(a.set, a.tr, ok1 ? E1 : 1.0);
        P0 = ok0 ? P0 : qnan();
        P1 = ok1 ? P1 : qnan();
        if (VEC && has1) {
            st_stream2(P_out + j0, P0, P1);
        } else {
            if (j0 < n) st_stream(P_out + j0, P0);
            if (has1) st_stream(P_out + j1, P1);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// k1b: all nine transitions.  One eigen-solve, four assembled amplitudes (alpha, beta in {e, mu});
// the remaining five probabilities are the unitarity complements.  Row 3*beta + alpha of P_out.
// ------------------------------------------------------------------------------------------------
// max(x, 0) that lets NaN through (fmax would turn it into 0): the complements below are differences of numbers near
// 1 and may come out as -1e-17.  On the integer pipe: a negative number that is not NaN has its upper word in
// [0x80000000, 0xFFF00000) (the complements are never -inf), and is replaced by +0.0 with two selects.
__device__ __forceinline__ double clamp0_keep_nan(double x)
{
    const unsigned hi = (unsigned)__double2hiint(x);
    const bool neg = hi - 0x80000000u < 0x7FF00000u;
    return __hiloint2double(neg ? 0 : (int)hi, neg ? 0 : __double2loint(x));
}

__device__ __forceinline__ double2 ld_stream2_pinned(const double* p)
{
    double2 v;
    asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}

// A11: an unusable energy is replaced by NaN, which then propagates through the closed form into all nine outputs
// (two selects instead of nine).
__device__ __forceinline__ void prob_nine(const ProbAllArgs& a, double E, double P[9])
{
    const double Es = energy_ok(E) ? E : qnan();
    const double invE = rcp_pos(Es);
    const double A = a.tr[0].sa * Es;
    OscEig e;
    eig_solve(a.set, A, invE, e);
    const double p00 = assemble_diag<true>(e, A, a.tr[0]);  // e  -> e
    const double p11 = assemble_diag<false>(e, A, a.tr[3]); // mu -> mu
    double p01, p10;                                        // p01: mu -> e (beta = e, alpha = mu); p10: e -> mu
    assemble_offdiag_pair(e, A, a.tr[1], p01, p10);
    const double p20 = clamp0_keep_nan((1.0 - p00) - p10); // column alpha = e   sums to 1
    const double p21 = clamp0_keep_nan((1.0 - p11) - p01); // column alpha = mu
    const double p02 = clamp0_keep_nan((1.0 - p00) - p01); // row beta = e       sums to 1
    const double p12 = clamp0_keep_nan((1.0 - p11) - p10); // row beta = mu
    const double p22 = clamp0_keep_nan((1.0 - p20) - p21); // row beta = tau
    P[0] = p00;
    P[1] = p01;
    P[2] = p02;
    P[3] = p10;
    P[4] = p11;
    P[5] = p12;
    P[6] = p20;
    P[7] = p21;
    P[8] = p22;
}

// VEC (E_true and every row of P_out 16-byte aligned, i.e. n even): slot i holds the adjacent events (2i, 2i + 1), one
// 128-bit load and nine 128-bit streaming stores per slot; otherwise tile i / THREADS holds events j0 and j0 + THREADS
// with scalar accesses.  The energies are loaded (pinned, see ld_stream_pinned) kProbAllAhead slots ahead of the arithmetic.  THREADS = kBlockProbAll: one block per SM, as k1 and k2 (the warps of co-resident blocks
// finish at different times); 256: four blocks per SM for sizes that would leave SMs idle otherwise.
template <bool VEC, int THREADS>
__global__ void __launch_bounds__(THREADS, THREADS >= 512 ? 1 : 4)
prob_all_kernel(const __grid_constant__ ProbAllArgs a, const double* __restrict__ E_true, size_t n,
                double* __restrict__ P_out)
{
    pdl_launch_dependents();
    pdl_wait();
    const size_t nslots = VEC ? (n + 1) / 2 : ((n + 2 * THREADS - 1) / (2 * THREADS)) * THREADS;
    const size_t stride = (size_t)gridDim.x * THREADS;
    auto load = [&](size_t i, double& E0, double& E1) {
        const size_t j0 = VEC ? 2 * i : (i / THREADS) * (2 * THREADS) + (i % THREADS);
        const size_t j1 = VEC ? j0 + 1 : j0 + THREADS;
        if (VEC) {                                           // n is even: both events of a slot exist
            const double2 v = ld_stream2_pinned(E_true + j0);
            E0 = v.x;
            E1 = v.y;
        } else {
            E0 = (j0 < n) ? ld_stream_pinned(E_true + j0) : 1.0;
            E1 = (j1 < n) ? ld_stream_pinned(E_true + j1) : 1.0;
        }
    };
    // the energies are loaded kProbAllAhead slots ahead: the kernel runs at 0.8-0.9 of the HBM bandwidth, where a load
    // queues behind the stores of everybody's previous slots (ncu, one slot ahead: 30 % of all warp samples sat on the
    // first use of the prefetched energy, long scoreboard)
    size_t i = (size_t)blockIdx.x * THREADS + threadIdx.x;
    double Q[kProbAllAhead][2];
#pragma unroll
    for (int d = 0; d < kProbAllAhead; ++d) {
        Q[d][0] = 1.0;
        Q[d][1] = 1.0;
        if (i + d * stride < nslots) load(i + d * stride, Q[d][0], Q[d][1]);
    }
    while (i < nslots) {
        const size_t j0 = VEC ? 2 * i : (i / THREADS) * (2 * THREADS) + (i % THREADS);
        const size_t j1 = VEC ? j0 + 1 : j0 + THREADS;
        const double E0 = Q[0][0], E1 = Q[0][1];
#pragma unroll
        for (int d = 0; d + 1 < kProbAllAhead; ++d) {
            Q[d][0] = Q[d + 1][0];
            Q[d][1] = Q[d + 1][1];
        }
        i += stride;
        if (i + (kProbAllAhead - 1) * stride < nslots)
            load(i + (kProbAllAhead - 1) * stride, Q[kProbAllAhead - 1][0], Q[kProbAllAhead - 1][1]);
        double P0[9], P1[9];
        prob_nine(a, E0, P0);
        prob_nine(a, E1, P1);
        // one running pointer, advanced by the row stride: nine row bases would not fit the uniform registers next to
        // the constants of the closed form
        double* q = P_out + j0;
        if (VEC) {
            // nine row addresses in registers of their own: a store keeps its address register until the store unit has
            // taken it, and at 0.9 of the HBM bandwidth that is long enough for "q += n" to wait for the previous store
            // (ncu: 30 % of all warp samples on that one integer add, long scoreboard)
            double* qk[9];
#pragma unroll
            for (int k = 0; k < 9; ++k) qk[k] = q + (size_t)k * n;
#pragma unroll
            for (int k = 0; k < 9; ++k) st_stream2(qk[k], P0[k], P1[k]);
        } else {
            const bool in0 = j0 < n, in1 = j1 < n;
#pragma unroll
            for (int k = 0; k < 9; ++k) {
                if (in0) st_stream(q, P0[k]);
                if (in1) st_stream(q + THREADS, P1[k]);
                q += n;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Debug export of the binning decision (osc_bin_index): bin of every event, -1 if dropped (A8, A11).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlock)
bin_index_kernel(const double* __restrict__ E_true, const double* __restrict__ E_reco,
                 const int8_t* __restrict__ channel, size_t n, double energy_scale,
                 const double* __restrict__ edges, int nb, int32_t* __restrict__ bin_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    build_bin_table(smem_raw, edges, nb);
    const BinView bt = bin_view(smem_raw);
    const size_t stride = (size_t)gridDim.x * kBlock;
    for (size_t j = (size_t)blockIdx.x * kBlock + threadIdx.x; j < n; j += stride) {
        const double x = scaled_energy(energy_scale, E_reco[j]);
        const int ch = channel[j];
        const bool ok = energy_ok(E_true[j]) && (unsigned)ch < (unsigned)kChannels;
        const int b = find_bin<0>(bt, x);
        bin_out[j] = ok ? b : -1;
    }
}

// ------------------------------------------------------------------------------------------------
// Parameter block of one point in shared memory: kBinArgsDoubles doubles laid out as BinArgs.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ OscTrans load_trans(uint32_t pb, int c)
{
    const uint32_t q = pb + 8u * (6u + (unsigned)c * kTransDoubles);
    const double2 a = lds_f64x2(q), b = lds_f64x2(q + 16), d = lds_f64x2(q + 32), e = lds_f64x2(q + 48);
    OscTrans t;
    t.sa = a.x;
    t.delta = a.y;
    t.ee = b.x;
    t.Tr0 = b.y;
    t.Ti0 = d.x;
    t.T2r0 = d.y;
    t.T2i0 = e.x;
    t.T2r1 = e.y;
    t.T2i1 = lds_f64(q + 64);
    t.pad = 0.0;
    return t;
}

__device__ __forceinline__ OscSet load_set(const double* pb)
{
    const double2* q = reinterpret_cast<const double2*>(pb);
    const double2 a = q[0], b = q[1], d = q[2];
    OscSet s;
    s.xq23 = a.x;
    s.tr = a.y;
    s.dd = b.x;
    s.k1 = b.y;
    s.k0_27 = d.x;
    return s;
}

// Per-event part of k2 that does not need the probability: the histogram cell (channel * nb + bin, or -1 if the
// event is dropped, A8/A11), the channel whose transition block is to be used and the energy handed to the closed form.
// ch is the channel byte zero-extended: 0..3 are valid, every other code (negative int8 values, the 0xFF that
// load_pair puts in for events past the end) is not.
template <int STEPS>
__device__ __forceinline__ bool locate_one(const BinView& bt, double energy_scale, double Et, double Er, unsigned ch,
                                           int& cell, unsigned& c, double& Es)
{
    const double x = scaled_energy(energy_scale, Er);       // a3b: one rounded fp64 multiply
    int bin;
    const bool inside = find_bin_pred<STEPS>(bt, x, bin);   // a3c: bit-exact index
    const bool ok = energy_ok(Et) && ch < (unsigned)kChannels && inside;
    c = ok ? ch : 0u;
    Es = ok ? Et : 1.0;
    cell = (int)c * bt.nb + bin;                            // only used when ok
    return ok;
}

// Loop-invariant constants of the closed form that the event loops of k2 and k2s keep in registers.  ptxas does not keep
// them on its own: set.dd and set.k1 (c1 = fma(A, k1, dd): two constants in one DFMA) and the four leading polynomial
// coefficients (PolyTop, osc_math.cuh) are re-loaded with LDC.64 in every iteration, and the DFMAs that consume them
// wait on the short scoreboard -- 16 % of the warp-state samples of k2s.  Read through a volatile shared-memory load
// (the block's copy of BinArgs at `pb`; its pad word is 0.0) the values cannot be rematerialised from the constant
// bank, so they stay in registers.  Measured per 1e7 events: k2 124.6 -> 118.5 us (551 instead of 627 instructions per
// pair of events), k2s (three scales) 242 -> 198 us; only dd, k1: 121.5 / 213 us; only the coefficients: 123 us.
// k2 at 200 / 400 / 500 bins: 130.8 -> 121.0, 156.4 -> 139.3, 168.1 -> 165.2 us.  The one shape that loses is k2's
// 256 threads with one sub-histogram per warp (binnings above ~570 bins: 228 -> 238 us at 768 bins), which keeps the
// constants where ptxas puts them (PIN = false).
struct LoopConsts {
    OscSet set;
    PolyTop top;
};
template <bool PIN = true>
__device__ __forceinline__ LoopConsts pin_loop_consts(const BinArgs& a, uint32_t pb)
{
    LoopConsts c;
    c.set = a.set;
    c.top = poly_top();
    if (!PIN) return c;
    c.set.dd = lds_f64_volatile(pb + 8u * 2u);
    c.set.k1 = lds_f64_volatile(pb + 8u * 3u);
    const double zero = lds_f64_volatile(pb + 8u * 5u);
    c.top.c4 += zero;
    c.top.c5 += zero;
    c.top.c10 += zero;
    c.top.c11 += zero;
    return c;
}

// Two events of one thread as they come from global memory (VEC: events 2i, 2i+1 by 128-bit loads).  The two channel
// bytes stay packed (low byte: first event) until they are used, so that nothing waits on the load where it is issued.
struct EventPair {
    double Et0, Et1, Er0, Er1, wp0, wp1;
    unsigned chp;
};

template <bool VEC, int THREADS>
__device__ __forceinline__ EventPair load_pair(const double* __restrict__ E_true, const double* __restrict__ E_reco,
                                               const double* __restrict__ w0, const int8_t* __restrict__ channel,
                                               size_t n, unsigned tile)
{
    const size_t base = (size_t)tile * (2 * THREADS);
    const size_t j0 = VEC ? base + 2 * threadIdx.x : base + threadIdx.x;
    const size_t j1 = VEC ? j0 + 1 : j0 + THREADS;
    const bool in0 = j0 < n, in1 = j1 < n;
    EventPair e;
    if (VEC && in1) {
        const double2 vt = ld_stream2(E_true + j0), vr = ld_stream2(E_reco + j0), vw = ld_stream2(w0 + j0);
        e.chp = __ldcs(reinterpret_cast<const unsigned short*>(channel + j0));
        e.Et0 = vt.x; e.Et1 = vt.y;
        e.Er0 = vr.x; e.Er1 = vr.y;
        e.wp0 = vw.x; e.wp1 = vw.y;
    } else {
        e.Et0 = in0 ? ld_stream(E_true + j0) : 1.0;
        e.Et1 = in1 ? ld_stream(E_true + j1) : 1.0;
        e.Er0 = in0 ? ld_stream(E_reco + j0) : 0.0;
        e.Er1 = in1 ? ld_stream(E_reco + j1) : 0.0;
        e.wp0 = in0 ? ld_stream(w0 + j0) : 0.0;
        e.wp1 = in1 ? ld_stream(w0 + j1) : 0.0;
        const unsigned c0 = in0 ? (unsigned)(unsigned char)channel[j0] : 0xFFu;
        const unsigned c1 = in1 ? (unsigned)(unsigned char)channel[j1] : 0xFFu;
        e.chp = c0 | (c1 << 8);
    }
    return e;
}

// Event loop of k2 (STEPS as in find_bin): software-pipelined by hand, see the kernel's comment.
template <bool VEC, int THREADS, int STEPS, int SLOTS>
__device__ __forceinline__ void k2_loop(const BinArgs& a, const double* __restrict__ E_true,
                                        const double* __restrict__ E_reco, const double* __restrict__ w0,
                                        const int8_t* __restrict__ channel, size_t n, double energy_scale,
                                        const BinView& bt, uint32_t pb, const LaneHist& lh, unsigned lt_mask,
                                        unsigned ntiles, unsigned t, EventPair cur)
{
    const LoopConsts lc = pin_loop_consts<!(THREADS == 256 && SLOTS == 1)>(a, pb);
    // the tile stride: the 768-thread shape gets it through a uniform register; the others re-load gridDim.x with an LDC
    // in every iteration and wait for it (as k2s did), unless it is pinned in a register
    const unsigned stride = THREADS == 768 ? gridDim.x : pin_u32(gridDim.x);
    while (t < ntiles) {
        int cell0, cell1;
        unsigned c0, c1;
        double Es0, Es1;
        const bool ok0 = locate_one<STEPS>(bt, energy_scale, cur.Et0, cur.Er0, cur.chp & 0xFFu, cell0, c0, Es0);
        const bool ok1 = locate_one<STEPS>(bt, energy_scale, cur.Et1, cur.Er1, cur.chp >> 8, cell1, c1, Es1);
        HistPlan plan;
        warp_hist_match_pred(plan, lh, ok0, cell0, ok1, cell1);
        const double wp0 = cur.wp0, wp1 = cur.wp1;
        // prefetch: E_true, E_reco and channel of the current pair are dead from here on
        t += stride;
        if (t < ntiles) cur = load_pair<VEC, THREADS>(E_true, E_reco, w0, channel, n, t);
        const OscTrans tr0 = load_trans(pb, (int)c0);
        const OscTrans tr1 = load_trans(pb, (int)c1);
        const double A0 = tr0.sa * Es0, A1 = tr1.sa * Es1;  // a2a
        OscEig e0, e1;
        eig_solve(lc.set, A0, rcp_pos(Es0), e0, lc.top);    // a2b-a2d
        eig_solve(lc.set, A1, rcp_pos(Es1), e1, lc.top);
        int rmax1 = 0;
        if (SLOTS == 2) warp_hist_rank(plan, lt_mask);
        else warp_hist_rank_single(plan, lt_mask, rmax1);
        const double P0 = assemble(e0, A0, tr0);            // a2e-a2f
        const double P1 = assemble(e1, A1, tr1);
        if (SLOTS == 2) warp_hist_commit(plan, __dmul_rn(wp0, P0), __dmul_rn(wp1, P1));   // a3a, a3c
        else warp_hist_commit_single(plan, rmax1, __dmul_rn(wp0, P0), __dmul_rn(wp1, P1));
    }
}

// ------------------------------------------------------------------------------------------------
// k2: fused reweight + histogram, one parameter set.
// Shared memory per block:  param block | bin table | hist[warps][SLOTS][n_sub][4 * nb]
// The loop is software-pipelined by hand: the loads of the block's next tile are issued before the arithmetic
// of the current one (the kernel is bound by instruction issue around the fp64 pipe, so a warp that sits on a
// global load is an issue slot lost), and the histogram ranking (MATCH + first read) precedes the closed form.
// ------------------------------------------------------------------------------------------------
#ifndef OSC_K2_TPS
#define OSC_K2_TPS 768
#endif
// SLOTS = 1: one sub-histogram per warp instead of one per (warp, event of the lane), see lane_hist_single.
template <bool VEC, int THREADS, int SLOTS = kSlots>
__global__ void __launch_bounds__(THREADS, THREADS >= 384 ? 1 : OSC_K2_TPS / THREADS)
reweight_bin_kernel(const __grid_constant__ BinArgs a, const double* __restrict__ E_true,
                    const double* __restrict__ E_reco, const double* __restrict__ w0,
                    const int8_t* __restrict__ channel, size_t n, double energy_scale,
                    const double* __restrict__ edges, int nb, int n_sub, MergeScratch ms,
                    unsigned char* __restrict__ table_cache, double* __restrict__ hist_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int WARPS = THREADS / 32;
    const int nh = kChannels * nb;
    double* pbuf = reinterpret_cast<double*>(smem_raw);
    unsigned char* tab = smem_raw + sizeof(double) * kBinArgsDoubles;
    double* hist = reinterpret_cast<double*>(tab + bin_table_bytes(nb));
    __shared__ unsigned int s_ticket;
    __shared__ int s_cached;

    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = threadIdx.x >> 5;
    const int n_hist = WARPS * SLOTS * n_sub;

    // tiles are counted in 32 bits (the host rejects n >= 2^32 tiles).  Measured: handing ntiles over as a kernel
    // parameter removes the eleven uniform instructions with which the compiler re-derives it from n in every iteration
    // of the event loop -- and makes the loop 6 % SLOWER (1200 instead of 1132 us per 1e8 events: a different schedule
    // with more MIO-queue and short-scoreboard stalls), so it stays computed here
    const unsigned ntiles = pin_u32((unsigned)((n + 2 * THREADS - 1) / (2 * THREADS)));
    // before pdl_wait(): only kernel parameters and shared memory (the previous kernel on the stream may still run)
    pdl_launch_dependents();
    if (threadIdx.x < kBinArgsDoubles) pbuf[threadIdx.x] = reinterpret_cast<const double*>(&a)[threadIdx.x];
    const int keep = (nb + 2) & ~1;                           // the first nb + 1 words stage the edge keys below
    zero_shared(hist + keep, n_hist * nh - keep);
    pdl_wait();
    const unsigned t = blockIdx.x;
    EventPair cur = load_pair<VEC, THREADS>(E_true, E_reco, w0, channel, n, t);   // grid <= ntiles
    const bool cached = load_or_build_bin_table(tab, reinterpret_cast<long long*>(hist), table_cache, edges, nb);
    if (threadIdx.x == 0) s_cached = cached;
    for (int i = threadIdx.x; i < keep; i += THREADS) hist[i] = 0.0;
    __syncthreads();
    BinView bt = bin_view(tab);
    bt.ekey = pin_u32(bt.ekey);
    bt.lut = pin_u32(bt.lut);
    const uint32_t pb = pin_u32(smem_u32(pbuf));
    LaneHist lh = SLOTS == 2 ? lane_hist(hist, nh, n_sub, warp, lane) : lane_hist_single(hist, nh, warp);
    lh.h0 = pin_u32(lh.h0);
    lh.h1 = SLOTS == 2 ? pin_u32(lh.h1) : lh.h0;
    const unsigned lt_mask = lanemask_lt();

    if (bt.steps <= 1u)
        k2_loop<VEC, THREADS, 1, SLOTS>(a, E_true, E_reco, w0, channel, n, energy_scale, bt, pb, lh, lt_mask, ntiles, t, cur);
    else
        k2_loop<VEC, THREADS, 0, SLOTS>(a, E_true, E_reco, w0, channel, n, energy_scale, bt, pb, lh, lt_mask, ntiles, t, cur);
    const bool last = block_merge(hist, n_hist, nh, ms, hist_out, &s_ticket);
    if (last && !s_cached) store_bin_table(tab, table_cache, nb);      // every other block is past its read of the cache
}

// ------------------------------------------------------------------------------------------------
// k2s: k2 for several energy-scale values in one pass ("all-systematics call").  The
// oscillation weight does not depend on the energy scale (A9: it acts on E_reco only), so the closed form runs once
// per event and only the binning and the histogram update run once per scale.  The NS histograms are laid out as one
// histogram of NS * 4 * nb cells (scale-major), which is also the layout of hist_out, so the sub-histogram and merge
// machinery of k2 is used unchanged.
// ------------------------------------------------------------------------------------------------
constexpr int kMaxScales = 4;

struct ScaleArgs {
    double s[kMaxScales];
};

template <bool VEC, int THREADS, int NS, int STEPS>
__device__ __forceinline__ void k2s_loop(const BinArgs& a, const double* __restrict__ E_true,
                                         const double* __restrict__ E_reco, const double* __restrict__ w0,
                                         const int8_t* __restrict__ channel, size_t n, const ScaleArgs& sc,
                                         const BinView& bt, uint32_t pb, const LaneHist& lh, unsigned lt_mask,
                                         unsigned ntiles, unsigned t, EventPair cur)
{
    const int nh = kChannels * bt.nb;
    const LoopConsts lc = pin_loop_consts(a, pb);
    // gridDim.x in a register: ptxas otherwise re-loads it with LDC right before `t += gridDim.x`, and the add then waits
    // for it on the short scoreboard -- 11 % of the warp-state samples of this kernel (profiles/r2_k2s_full.md)
    const unsigned stride = pin_u32(gridDim.x);
    while (t < ntiles) {
        const unsigned ch0 = cur.chp & 0xFFu, ch1 = cur.chp >> 8;
        const bool ok0 = energy_ok(cur.Et0) && ch0 < (unsigned)kChannels;
        const bool ok1 = energy_ok(cur.Et1) && ch1 < (unsigned)kChannels;
        const unsigned c0 = ok0 ? ch0 : 0u, c1 = ok1 ? ch1 : 0u;
        const double Es0 = ok0 ? cur.Et0 : 1.0, Es1 = ok1 ? cur.Et1 : 1.0;
        HistPlan plan[NS];
#pragma unroll
        for (int k = 0; k < NS; ++k) {
            const int b0 = find_bin<STEPS>(bt, scaled_energy(sc.s[k], cur.Er0));     // a3b, a3c per scale
            const int b1 = find_bin<STEPS>(bt, scaled_energy(sc.s[k], cur.Er1));
            const int cell0 = (ok0 && b0 >= 0) ? k * nh + (int)c0 * bt.nb + b0 : -1;
            const int cell1 = (ok1 && b1 >= 0) ? k * nh + (int)c1 * bt.nb + b1 : -1;
            warp_hist_match(plan[k], lh, cell0, cell1);
        }
        const double wp0 = cur.wp0, wp1 = cur.wp1;
        t += stride;
        if (t < ntiles) cur = load_pair<VEC, THREADS>(E_true, E_reco, w0, channel, n, t);
        const OscTrans tr0 = load_trans(pb, (int)c0);
        const OscTrans tr1 = load_trans(pb, (int)c1);
        const double A0 = tr0.sa * Es0, A1 = tr1.sa * Es1;  // a2a
        OscEig e0, e1;
        eig_solve(lc.set, A0, rcp_pos(Es0), e0, lc.top);    // a2b-a2d
        eig_solve(lc.set, A1, rcp_pos(Es1), e1, lc.top);
#pragma unroll
        for (int k = 0; k < NS; ++k) warp_hist_rank(plan[k], lt_mask);
        const double w_0 = __dmul_rn(wp0, assemble(e0, A0, tr0));   // a2e-a2f, a3a
        const double w_1 = __dmul_rn(wp1, assemble(e1, A1, tr1));
#pragma unroll
        for (int k = 0; k < NS; ++k) warp_hist_commit(plan[k], w_0, w_1);
    }
}

// Shared memory per block:  param block | bin table | hist[warps][kSlots][n_sub][NS * 4 * nb]
template <bool VEC, int THREADS, int NS>
__global__ void __launch_bounds__(THREADS, 512 / THREADS)
reweight_bin_scales_kernel(const __grid_constant__ BinArgs a, const __grid_constant__ ScaleArgs sc,
                           const double* __restrict__ E_true, const double* __restrict__ E_reco,
                           const double* __restrict__ w0, const int8_t* __restrict__ channel, size_t n,
                           const double* __restrict__ edges, int nb, int n_sub, MergeScratch ms,
                           unsigned char* __restrict__ table_cache, double* __restrict__ hist_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int WARPS = THREADS / 32;
    const int nht = NS * kChannels * nb;
    double* pbuf = reinterpret_cast<double*>(smem_raw);
    unsigned char* tab = smem_raw + sizeof(double) * kBinArgsDoubles;
    double* hist = reinterpret_cast<double*>(tab + bin_table_bytes(nb));
    __shared__ unsigned int s_ticket;
    __shared__ int s_cached;

    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = threadIdx.x >> 5;
    const int n_hist = WARPS * kSlots * n_sub;
    const unsigned ntiles = pin_u32((unsigned)((n + 2 * THREADS - 1) / (2 * THREADS)));
    // before pdl_wait(): only kernel parameters and shared memory (the previous kernel on the stream may still run)
    pdl_launch_dependents();
    if (threadIdx.x < kBinArgsDoubles) pbuf[threadIdx.x] = reinterpret_cast<const double*>(&a)[threadIdx.x];
    const int keep = (nb + 2) & ~1;                           // the first nb + 1 words stage the edge keys below
    zero_shared(hist + keep, n_hist * nht - keep);
    pdl_wait();
    const unsigned t = blockIdx.x;
    EventPair cur = load_pair<VEC, THREADS>(E_true, E_reco, w0, channel, n, t);   // grid <= ntiles
    const bool cached = load_or_build_bin_table(tab, reinterpret_cast<long long*>(hist), table_cache, edges, nb);
    if (threadIdx.x == 0) s_cached = cached;
    for (int i = threadIdx.x; i < keep; i += THREADS) hist[i] = 0.0;
    __syncthreads();
    BinView bt = bin_view(tab);
    bt.ekey = pin_u32(bt.ekey);
    bt.lut = pin_u32(bt.lut);
    const uint32_t pb = pin_u32(smem_u32(pbuf));
    LaneHist lh = lane_hist(hist, nht, n_sub, warp, lane);
    lh.h0 = pin_u32(lh.h0);
    lh.h1 = pin_u32(lh.h1);
    const unsigned lt_mask = lanemask_lt();

    if (bt.steps <= 1u)
        k2s_loop<VEC, THREADS, NS, 1>(a, E_true, E_reco, w0, channel, n, sc, bt, pb, lh, lt_mask, ntiles, t, cur);
    else
        k2s_loop<VEC, THREADS, NS, 0>(a, E_true, E_reco, w0, channel, n, sc, bt, pb, lh, lt_mask, ntiles, t, cur);
    const bool last = block_merge(hist, n_hist, nht, ms, hist_out, &s_ticket);
    if (last && !s_cached) store_bin_table(tab, table_cache, nb);
}

// ------------------------------------------------------------------------------------------------
// Bin-centre comparator: the "quick" alternative the paper argues against
// multiplies the unoscillated content of a TRUE-energy bin by the probability at the bin centre.
// unit_hist_kernel fills hist[channel][bin] += w0 over true-energy bins (the machinery of k2 without the closed
// form); centre_weight_kernel multiplies each cell by P_channel(centre of the bin).
// ------------------------------------------------------------------------------------------------
// SLOTS = 2: a sub-histogram per (warp, event of the lane) as in k2; SLOTS = 1: one per warp (binnings above ~420 bins).
template <int SLOTS>
__global__ void __launch_bounds__(kBlock)
unit_hist_kernel(const double* __restrict__ E_true, const double* __restrict__ w0, const int8_t* __restrict__ channel,
                 size_t n, const double* __restrict__ edges, int nb, int n_sub, MergeScratch ms,
                 double* __restrict__ hist_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int WARPS = kBlock / 32;
    const int nh = kChannels * nb;
    double* hist = reinterpret_cast<double*>(smem_raw + bin_table_bytes(nb));
    __shared__ unsigned int s_ticket;
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int n_hist = WARPS * SLOTS * n_sub;
    for (int i = threadIdx.x; i < n_hist * nh; i += kBlock) hist[i] = 0.0;
    build_bin_table(smem_raw, edges, nb);
    const BinView bt = bin_view(smem_raw);
    const LaneHist lh = SLOTS == 2 ? lane_hist(hist, nh, n_sub, warp, lane) : lane_hist_single(hist, nh, warp);
    const size_t ntiles = (n + 2 * kBlock - 1) / (2 * kBlock);
    for (size_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const size_t j0 = t * (2 * kBlock) + threadIdx.x, j1 = j0 + kBlock;
        int cell[2];
        double w[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const size_t j = k ? j1 : j0;
            cell[k] = -1;
            w[k] = 0.0;
            if (j < n) {
                const double E = E_true[j];
                const unsigned ch = (unsigned)(unsigned char)channel[j];
                const int bin = find_bin<0>(bt, E);                      // true-energy bins: no energy scale
                if (energy_ok(E) && ch < (unsigned)kChannels && bin >= 0) {
                    cell[k] = (int)ch * nb + bin;
                    w[k] = w0[j];
                }
            }
        }
        if (SLOTS == 2) warp_hist_add2(lh, cell[0], w[0], cell[1], w[1], lt_mask);
        else warp_hist_add2_single(lh, cell[0], w[0], cell[1], w[1], lt_mask);
    }
    block_merge(hist, n_hist, nh, ms, hist_out, &s_ticket);
}

// hist[ch][b] *= P_ch((edges[b] + edges[b+1]) / 2); a centre that is not a usable energy gives NaN.
__global__ void __launch_bounds__(256)
centre_weight_kernel(const __grid_constant__ BinArgs a, const double* __restrict__ edges, int nb,
                     double* __restrict__ hist)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= kChannels * nb) return;
    const int ch = i / nb, b = i - ch * nb;
    const double c = 0.5 * (edges[b] + edges[b + 1]);
    const bool ok = energy_ok(c);
    const double P = prob_one(a.set, a.ch[ch], ok ? c : 1.0);
    hist[i] = ok ? hist[i] * P : qnan();
}

// Peak-rate probe for the roofline denominator: a chain-parallel DFMA loop, 8 independent chains per
// thread, 2 flops per DFMA.  Not part of the hot path.
__global__ void __launch_bounds__(kBlock) dfma_probe_kernel(double* out, int iters, double seed)
{
    double x0 = seed + threadIdx.x, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0;
    double x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0, x7 = x0 + 7.0;
    const double m = 0.999999, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, m, c); x1 = fma(x1, m, c); x2 = fma(x2, m, c); x3 = fma(x3, m, c);
        x4 = fma(x4, m, c); x5 = fma(x5, m, c); x6 = fma(x6, m, c); x7 = fma(x7, m, c);
    }
    const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456) out[0] = s; // keeps the loop alive, practically never stores
}

// Issue-rate probes behind DESIGN.md 5.1 ("what bounds these kernels"): register-resident loops of one instruction
// pattern, 8 independent chains per thread, so that ncu's smsp__inst_executed / sm__cycles_elapsed of a launch gives the
// issue cost of the pattern in cycles per warp instruction and sub-partition.  y, z come from memory (opaque to the
// compiler) and stay in registers.  KIND: 0 DFMA x = fma(y, z, x), three distinct register operands;
// 1 DFMA x = fma(x, y, c), two registers and an immediate; 2 DFMA x = fma(x, m, c), one register (dfma_probe_kernel's
// pattern); 3 DMUL x = x * y; 4 DADD x = x + y; 5 pattern 0 followed by two FFMA with three register operands each;
// 6 pattern 0 followed by two IMAD.  Not part of the hot path.
template <int KIND>
__global__ void __launch_bounds__(kBlock) issue_probe_kernel(const double* __restrict__ in, double* out, int iters)
{
    double x[8], y[8], z[8];
    float f[8], g[8];
    int q[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        // thread-dependent values: warp-uniform ones would be kept in uniform registers, which is the cheap operand kind
        x[k] = in[k] + threadIdx.x;
        y[k] = in[8 + k] - 1e-9 * threadIdx.x;
        z[k] = in[16 + k] + 1e-12 * threadIdx.x;
        f[k] = (float)in[k] + 1e-3f * threadIdx.x;
        g[k] = (float)in[8 + k] - 1e-6f * threadIdx.x;
        q[k] = (int)in[16 + k] + threadIdx.x;
    }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (KIND == 0 || KIND == 5 || KIND == 6) x[k] = fma(y[k], z[k], x[k]);
            if (KIND == 1) x[k] = fma(x[k], y[k], 0.5);
            if (KIND == 2) x[k] = fma(x[k], 0.999999, 1e-9);
            if (KIND == 3) x[k] = x[k] * y[k];
            if (KIND == 4) x[k] = x[k] + y[k];
            if (KIND == 5) {
                f[k] = fmaf(g[k], f[(k + 1) & 7], f[k]);
                g[k] = fmaf(f[k], g[(k + 3) & 7], g[k]);
            }
            if (KIND == 6) {
                q[k] = q[k] * q[(k + 1) & 7] + q[(k + 2) & 7];
                q[(k + 3) & 7] = q[k] * q[(k + 5) & 7] + q[(k + 3) & 7];
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += x[k] + (double)f[k] + (double)g[k] + (double)q[k];
    if (s == 123.456) out[0] = s; // keeps the loop alive, practically never stores
}

} // namespace oscb
