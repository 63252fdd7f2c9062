// osc_hist.cuh -- deterministic shared-memory histogram accumulation.
//
// sm_100a has no native fp64 shared-memory atomic add (atomicAdd(double*) on shared memory lowers to an
// ATOMS.CAST.SPIN loop whose order of additions is not defined).  Instead every warp owns private
// sub-histograms and resolves the collisions inside the warp itself:
//
//   * each lane carries two events (slot 0 and slot 1); slot s of the lanes with (lane mod n_sub) = u adds
//     into sub-histogram (s, u) of the warp, so the two slots never collide with each other and only
//     32 / n_sub lanes can collide at all (n_sub = 2 when shared memory allows, else 1);
//   * lanes that hit the same word are found with MATCH.ANY on the word's address; a lane's rank is the
//     number of lower lanes with the same address;
//   * phase r = 0, 1, ... lets exactly the lanes of rank r do a plain read-modify-write: inside a phase
//     all addresses are distinct, and for one address the additions happen in lane order.
//
// Block result = sub-histograms summed in (warp, slot, u) order; blocks are merged in two fixed-order
// levels by the last block to arrive (tickets), so every histogram is a deterministic function of the
// inputs.
#pragma once
#include <cuda_runtime.h>

#include "osc_smem.cuh"

namespace oscb {

constexpr int kSlots = 2; // events per lane per iteration

// Shared-window byte addresses of this lane's two sub-histograms (loop invariant).
struct LaneHist {
    uint32_t h0, h1;
};

__device__ __forceinline__ LaneHist lane_hist(const double* hist, int nh, int n_sub, unsigned warp, unsigned lane)
{
    const unsigned u = lane & (unsigned)(n_sub - 1);
    const uint32_t wbase = smem_u32(hist) + 8u * (warp * (unsigned)(kSlots * n_sub * nh));
    LaneHist lh;
    lh.h0 = wbase + 8u * (u * (unsigned)nh);
    lh.h1 = wbase + 8u * (((unsigned)n_sub + u) * (unsigned)nh);
    return lh;
}

// The accumulation of one warp iteration is split in two so that the latency of MATCH and of the first
// shared-memory read is hidden behind the probability arithmetic (the cell of an event is known before its
// weight): warp_hist_plan ranks the lanes and pre-reads the word of every rank-0 lane, warp_hist_commit adds
// the weights.  Nothing but this warp ever touches its sub-histograms, so the pre-read value is still current
// at commit time.  cell0 / cell1: histogram cell of the lane's slot-0 / slot-1 event, or -1 for a dropped event.
struct HistPlan {
    uint32_t a0, a1;   // shared-window byte address of the target word (all ones: dropped)
    unsigned m0, m1;   // lanes of the warp that target the same word (MATCH.ANY)
    int r0, r1;        // rank among those lanes (-1: dropped)
    int rmax;          // warp-uniform maximum rank
    double v0, v1;     // current content of the word, valid for rank 0
};

// Step 1 (as early as the cells are known): addresses and MATCH.
__device__ __forceinline__ void warp_hist_match(HistPlan& p, const LaneHist& lh, int cell0, int cell1)
{
    const unsigned FULL = 0xffffffffu;
    p.a0 = cell0 >= 0 ? lh.h0 + 8u * (unsigned)cell0 : 0xFFFFFFFFu;
    p.a1 = cell1 >= 0 ? lh.h1 + 8u * (unsigned)cell1 : 0xFFFFFFFFu;
    p.m0 = __match_any_sync(FULL, p.a0);
    p.m1 = __match_any_sync(FULL, p.a1);
}

// The same with the validity of each event as a predicate (cell may be anything for a dropped event).
__device__ __forceinline__ void warp_hist_match_pred(HistPlan& p, const LaneHist& lh, bool ok0, int cell0, bool ok1,
                                                     int cell1)
{
    const unsigned FULL = 0xffffffffu;
    p.a0 = ok0 ? lh.h0 + 8u * (unsigned)cell0 : 0xFFFFFFFFu;
    p.a1 = ok1 ? lh.h1 + 8u * (unsigned)cell1 : 0xFFFFFFFFu;
    p.m0 = __match_any_sync(FULL, p.a0);
    p.m1 = __match_any_sync(FULL, p.a1);
}

// Step 2 (once MATCH has had time to come back): ranks and the pre-read of the rank-0 lanes.
__device__ __forceinline__ void warp_hist_rank(HistPlan& p, unsigned lt_mask)
{
    const unsigned FULL = 0xffffffffu;
    p.r0 = p.a0 != 0xFFFFFFFFu ? __popc(p.m0 & lt_mask) : -1;
    p.r1 = p.a1 != 0xFFFFFFFFu ? __popc(p.m1 & lt_mask) : -1;
    p.rmax = __reduce_max_sync(FULL, max(p.r0, p.r1));
    p.v0 = 0.0;
    p.v1 = 0.0;
    if (p.r0 == 0) p.v0 = lds_f64_volatile(p.a0);
    if (p.r1 == 0) p.v1 = lds_f64_volatile(p.a1);
}

__device__ __forceinline__ HistPlan warp_hist_plan(const LaneHist& lh, int cell0, int cell1, unsigned lt_mask)
{
    HistPlan p;
    warp_hist_match(p, lh, cell0, cell1);
    warp_hist_rank(p, lt_mask);
    return p;
}

// Phase 0 stores the pre-read words plus the weights; phase r = 1, 2, ... lets exactly the lanes of rank r do a plain
// read-modify-write: inside a phase all addresses are distinct, and for one address the additions happen in lane order.
__device__ __forceinline__ void warp_hist_commit(const HistPlan& p, double w0, double w1)
{
    if (p.r0 == 0) sts_f64_volatile(p.a0, p.v0 + w0);
    if (p.r1 == 0) sts_f64_volatile(p.a1, p.v1 + w1);
    __syncwarp();
#pragma unroll 1
    for (int ph = 1; ph <= p.rmax; ++ph) {
        if (p.r0 == ph) sts_f64_volatile(p.a0, lds_f64_volatile(p.a0) + w0);
        if (p.r1 == ph) sts_f64_volatile(p.a1, lds_f64_volatile(p.a1) + w1);
        __syncwarp();
    }
}

// One sub-histogram per warp for both events of a lane (binnings whose two-slot layout leaves room for too few warps):
// slot 0 is committed completely before slot 1 reads anything, so the order of the additions to one word is
// slot 0 in lane order, then slot 1 in lane order.  Only slot 0 can be pre-read.
__device__ __forceinline__ LaneHist lane_hist_single(const double* hist, int nh, unsigned warp)
{
    LaneHist lh;
    lh.h0 = smem_u32(hist) + 8u * (warp * (unsigned)nh);
    lh.h1 = lh.h0;
    return lh;
}

__device__ __forceinline__ void warp_hist_rank_single(HistPlan& p, unsigned lt_mask, int& rmax1)
{
    const unsigned FULL = 0xffffffffu;
    p.r0 = p.a0 != 0xFFFFFFFFu ? __popc(p.m0 & lt_mask) : -1;
    p.r1 = p.a1 != 0xFFFFFFFFu ? __popc(p.m1 & lt_mask) : -1;
    p.rmax = __reduce_max_sync(FULL, p.r0);
    rmax1 = __reduce_max_sync(FULL, p.r1);
    p.v0 = 0.0;
    p.v1 = 0.0;
    if (p.r0 == 0) p.v0 = lds_f64_volatile(p.a0);
}

__device__ __forceinline__ void warp_hist_commit_single(const HistPlan& p, int rmax1, double w0, double w1)
{
    if (p.r0 == 0) sts_f64_volatile(p.a0, p.v0 + w0);
    __syncwarp();
#pragma unroll 1
    for (int ph = 1; ph <= p.rmax; ++ph) {
        if (p.r0 == ph) sts_f64_volatile(p.a0, lds_f64_volatile(p.a0) + w0);
        __syncwarp();
    }
#pragma unroll 1
    for (int ph = 0; ph <= rmax1; ++ph) {
        if (p.r1 == ph) sts_f64_volatile(p.a1, lds_f64_volatile(p.a1) + w1);
        __syncwarp();
    }
}

__device__ __forceinline__ void warp_hist_add2(const LaneHist& lh, int cell0, double w0, int cell1, double w1,
                                               unsigned lt_mask)
{
    const HistPlan p = warp_hist_plan(lh, cell0, cell1, lt_mask);
    warp_hist_commit(p, w0, w1);
}

// The same for the one-sub-histogram-per-warp layout (lane_hist_single).
__device__ __forceinline__ void warp_hist_add2_single(const LaneHist& lh, int cell0, double w0, int cell1, double w1,
                                                      unsigned lt_mask)
{
    HistPlan p;
    warp_hist_match(p, lh, cell0, cell1);
    int rmax1;
    warp_hist_rank_single(p, lt_mask, rmax1);
    warp_hist_commit_single(p, rmax1, w0, w1);
}

// Scratch of one call: counters[ngroups + 1] | partial[grid][nh] | gpartial[ngroups][nh].  It lives in a buffer the
// library keeps per (device, stream); calls on one stream are ordered, so they can share it.  The ticket counters are zero
// when a kernel starts and the blocks that consume them set them back to zero.  ngroups = 1: one-level merge.
struct MergeScratch {
    double* partial;
    double* gpartial;
    unsigned int* counters;
    int ngroups;
};

constexpr int kGroup = 16; // blocks per first-level group of the two-level merge

// src[0] + src[stride] + ... (count terms, added in that order), read through L2.  The loads of sixteen terms are
// issued together before they are added: the merge is a chain of dependent L2 round trips otherwise, and it sits on
// the critical path of every call (the last block does it alone).
__device__ __forceinline__ double ordered_sum_cg(const double* src, int count, int stride)
{
    double s = 0.0;
    int b = 0;
    for (; b + 16 <= count; b += 16) {
        double v[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = __ldcg(src + (size_t)(b + k) * stride);
#pragma unroll
        for (int k = 0; k < 16; ++k) s += v[k];
    }
    if (b + 8 <= count) {
        double v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = __ldcg(src + (size_t)(b + k) * stride);
#pragma unroll
        for (int k = 0; k < 8; ++k) s += v[k];
        b += 8;
    }
    for (; b < count; ++b) s += __ldcg(src + (size_t)b * stride);
    return s;
}

// The same for two adjacent cells at once (src 16-byte aligned, stride2 in units of double2), twelve terms per batch:
// with up to kMergeSegs threads per pair of cells the 148 block partials of a call arrive in two round trips.
constexpr int kMergeBatch = 12;
__device__ __forceinline__ double2 ordered_sum2_cg(const double2* src, int count, int stride2)
{
    double2 s = make_double2(0.0, 0.0);
    for (int b = 0; b < count; b += kMergeBatch) {
        double2 v[kMergeBatch];
#pragma unroll
        for (int k = 0; k < kMergeBatch; ++k)
            v[k] = b + k < count ? __ldcg(src + (size_t)(b + k) * stride2) : make_double2(0.0, 0.0);
#pragma unroll
        for (int k = 0; k < kMergeBatch; ++k) {
            if (b + k < count) {           // (a padding term would turn a -0.0 sum into +0.0; sums here are >= 0 anyway)
                s.x += v[k].x;
                s.y += v[k].y;
            }
        }
    }
    return s;
}

constexpr int kMergeSegs = 8; // at most this many threads share the partials of one pair of cells in a merge step

// dst[nh] = src[0][nh] + src[1][nh] + ... + src[count - 1][nh], added in that order per cell (src rows nh apart, read through
// L2; dst global).  A pair of cells is shared by up to kMergeSegs threads, each adds a contiguous range of rows with its
// loads in flight together; the ranges are then added in order.  scratch: shared memory for nh * kMergeSegs doubles
// (only used when a block has at least two threads per pair of cells).  Called by all threads of the block.
__device__ __forceinline__ void merge_rows(const double* src, int count, int nh, double* __restrict__ dst, double* scratch)
{
    const int npair = nh / 2;
    int nseg = (int)blockDim.x / npair;
    nseg = nseg < 1 ? 1 : (nseg > kMergeSegs ? kMergeSegs : nseg);
    if (nseg > count) nseg = count;
    if (nseg <= 1 || (reinterpret_cast<size_t>(dst) & 15)) {
        for (int i = threadIdx.x; i < nh; i += blockDim.x) __stcg(dst + i, ordered_sum_cg(src + i, count, nh));
        return;
    }
    const double2* src2 = reinterpret_cast<const double2*>(src);
    const int per = (count + nseg - 1) / nseg;
    const int t = (int)threadIdx.x;
    double2* seg_sum = reinterpret_cast<double2*>(scratch);
    if (t < nseg * npair) {
        const int seg = t / npair, i = t - seg * npair;
        const int b0 = seg * per, b1 = min(count, b0 + per);
        seg_sum[t] = b1 > b0 ? ordered_sum2_cg(src2 + (size_t)b0 * npair + i, b1 - b0, npair) : make_double2(0.0, 0.0);
    }
    __syncthreads();
    if (t < npair) {
        double2 s = seg_sum[t];
        for (int k = 1; k < nseg; ++k) {
            const double2 v = seg_sum[k * npair + t];
            s.x += v.x;
            s.y += v.y;
        }
        __stcg(reinterpret_cast<double2*>(dst) + t, s);
    }
}

// One thread takes a ticket with release-acquire semantics after a block barrier: the block's stores (ordered before by the
// barrier, cumulativity as in a grid-wide barrier) are visible to whoever sees the ticket, and the loads that follow see
// the stores of every block that took an earlier one.  Returns (block-uniform) whether this block took the last of `total`
// tickets; the counter is then set back to zero for the next kernel on the stream.
__device__ __forceinline__ bool take_ticket(unsigned int* counter, unsigned total, unsigned int* s_ticket)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned ticket;
        asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(ticket) : "l"(counter) : "memory");
        if (ticket == total - 1u) *counter = 0u;
        *s_ticket = ticket;
    }
    __syncthreads();
    return *s_ticket == total - 1u;
}

// hist: [n_sub][nh] sub-histograms of this block in shared memory (n_sub >= kMergeSegs, nh even, hist 16-byte aligned;
// the memory is reused as scratch by the merging blocks).  Every block writes its sum to ms.partial.
//   ms.ngroups == 1 (the host's choice while grid x nh partial sums are at most 512 kB): the block that arrives last
//     (ticket) adds the partials of all blocks in block order into out[nh].  The critical path after the slowest block is
//     one atomic and the loads of the partials -- 2.8 us for the 237 kB of 148 blocks x 200 cells through ONE SM; the
//     two-level scheme below was 1 us slower there (a second ticket and two more barriers);
//   otherwise: the last block of each group of kGroup adds the group's partials into ms.gpartial, and the last of those
//     adds the groups into out -- with 296 blocks x 600 cells (three energy scales) one SM would read 1.4 MB (16 us).
// One pass, no second launch.  Every sum has a fixed order (given the launch shape), so the result is a deterministic
// function of the inputs.  Must be called by all threads of the block; returns true in the block that wrote `out` (all
// threads), false elsewhere.
__device__ __forceinline__ bool block_merge(double* hist, int n_sub, int nh, const MergeScratch& ms,
                                            double* __restrict__ out, unsigned int* s_ticket)
{
    __syncthreads();
    double* my_partial = ms.partial + (size_t)blockIdx.x * nh;
    for (int i = threadIdx.x; i < nh; i += blockDim.x) {
        // four interleaved chains, combined at the end: a quarter of the dependent additions of a single chain
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
        int w = 0;
        for (; w + 4 <= n_sub; w += 4) {
            s0 += hist[(size_t)w * nh + i];
            s1 += hist[(size_t)(w + 1) * nh + i];
            s2 += hist[(size_t)(w + 2) * nh + i];
            s3 += hist[(size_t)(w + 3) * nh + i];
        }
        for (; w < n_sub; ++w) s0 += hist[(size_t)w * nh + i];
        __stcg(my_partial + i, (s0 + s1) + (s2 + s3));
    }
    if (ms.ngroups <= 1) {
        if (!take_ticket(ms.counters, gridDim.x, s_ticket)) return false;
        merge_rows(ms.partial, (int)gridDim.x, nh, out, hist);
        return true;
    }
    const int group = blockIdx.x / kGroup;
    const int gfirst = group * kGroup;
    const int gsize = min(kGroup, (int)gridDim.x - gfirst);
    if (!take_ticket(ms.counters + 1 + group, (unsigned)gsize, s_ticket)) return false;
    merge_rows(ms.partial + (size_t)gfirst * nh, gsize, nh, ms.gpartial + (size_t)group * nh, hist);
    if (!take_ticket(ms.counters, (unsigned)ms.ngroups, s_ticket)) return false;
    merge_rows(ms.gpartial, ms.ngroups, nh, out, hist);
    return true;
}

} // namespace oscb
