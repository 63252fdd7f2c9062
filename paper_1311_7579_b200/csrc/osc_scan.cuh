// osc_scan.cuh -- k4: the batched call for parameter scans.
//
// The paper's scan floats theta23 and dm2_32; BASELINE.json configs[3] is a 32 x 32 grid of the
// two with a delta_cp per point.  With U = R23 D R13 D^dagger R12, D = diag(1, 1, e^{i delta}) (PDG form,
// DESIGN.md A6), D^dagger commutes with R12 and with diag(m^2), and A e e^dagger commutes with W = R23 D, so
//
//     T = W T' W^dagger,   T' = R13 R12 diag(m^2) R12^T R13^T + A e e^T   (real symmetric, no theta23, no delta)
//     S = exp(-i T x) = W S' W^dagger,   S' = exp(-i T' x)                 (complex symmetric)
//     S_{beta alpha} = sum_{ij} W_{beta i} conj(W_{alpha j}) S'_{ij}        (antineutrinos: W -> conj(W), A -> -A)
//
// All points that share (theta12, theta13, dm2_21, dm2_32, rho, L, hierarchy) -- a "group" -- share S', which is
// where the eigen-solve and every transcendental sits; a point of the group costs a three-term complex
// combination of S' entries.  The rows of W are (1,0,0), (0,c23,s23 e^{i delta}), (0,-s23,c23 e^{i delta}), so a
// transition needs at most three distinct entries of S'.
//
// Work layout.  The histogram cell (channel, bin) of an event does not depend on the point either, so the events
// are first sorted by cell (stable counting sort: scan_count / scan_offsets / scan_scatter).  A sorted cell is
// cut into pieces of at most `piece` events; one warp takes a piece and, for every group, alternates
//     phase A  lane = event : S' entries z_k of 64 events; what goes into the warp's shared-memory slice are the
//              real numbers q_t = w0 |z_k|^2, w0 Re(z_k conj z_l), w0 Im(z_k conj z_l) that the points combine
//     phase B  lane = point : w0 |sum_k c_k z_k|^2 = sum_t q_t m_t with the lane's monomials m_t = |c_k|^2,
//              2 Re(c_k conj c_l), -2 Im(c_k conj c_l): every lane walks the slice (broadcast reads) and adds the
//              terms to ONE REGISTER, because every event of the piece falls into the same histogram cell.
//              Six fused multiply-adds per event and point for numu -> numu (real coefficients: the Im terms
//              drop out), four for numu -> nue.
// There is no histogram in shared memory, no atomic and no collision; partial[piece][point] is summed over the
// pieces of a cell in order by scan_merge, so the result is a deterministic function of the inputs.
#pragma once
#include <cstdint>

#include "osc_bins.cuh"
#include "osc_core.cuh"
#include "osc_types.h"

namespace oscb {

constexpr int kScanLanes = 32;        // points per sub-group (one per lane)
constexpr int kScanElems = 3;         // entries of S' per channel, at most
constexpr int kScanWarps = 4;         // warps per block of the event-ordered kernels
constexpr unsigned short kNoCell = 0xFFFFu;

// Entry (i, j) of T' and T'^2 as functions of the matter term A:  T'_ij = Tr0 + A ee,
// (T'^2)_ij = T2r0 + A T2r1 + A^2 ee;  delta = [i == j], ee = [i == j == e].
struct ScanElem {
    double delta, ee, Tr0, T2r0, T2r1;
};

constexpr int kScanTerms = 9;         // |z0|^2 |z1|^2 |z2|^2  Re01 Re02 Re12  Im01 Im02 Im12 (canonical order)

struct ScanChan {
    double sa;                 // +-K_MATTER Y_E rho (sign: antineutrino channel)
    int nk;                    // entries of S' used (1..3)
    int tmask;                 // bit t set: term t of the canonical list is used (its monomial is non-zero for some point)
    ScanElem el[kScanElems];
};

struct ScanGroup {
    OscSet set;
    double pad;
    ScanChan ch[kChannels];
};

// Monomials of one sub-group (at most 32 points of one group): mono[channel][t'][lane], t' counting the used
// terms of the channel in canonical order.
struct ScanSub {
    int group;
    int pt[kScanLanes];        // index of the lane's point in the caller's list, -1 for an unused lane
    int pad[3];
    double mono[kChannels][kScanTerms][kScanLanes];
};

// One sub-group as the parameter block of scan_const_kernel: it travels as a __grid_constant__ kernel parameter, so
// the monomials reach the fused multiply-adds of phase B through the constant bank.  A channel is of one of two kinds
// (osc_api.cu, make_const_args, for the algebra):
//   "three entries" (mm bit set; numu -> numu)  el[] = s, u, v;  w0 |s + a u + c v|^2 = w0 |s|^2 + sum_t q_t m_t with
//       q = w0 {|u|^2, |v|^2, Re(s u*), Re(s v*), Re(u v*)},  m = {a^2, c^2, 2a, 2c, 2ac}
//   "two entries" (numu -> nue)  el[] = z0, z1;  w0 |c0 z0 + c1 z1|^2 = w0 |z1|^2 + sum_t q_t m_t with
//       q = w0 {|z0|^2 - |z1|^2, Re(z0 z1*), Im(z0 z1*)},  m = {|c0|^2, 2 Re(c0 c1*), -2 Im(c0 c1*)}
// el[0] of a three-entry channel is a diagonal entry (delta = 1), every other el[] has delta = 0, and no entry is (e, e).
// mono[channel][t][lane]; bit t of ch[channel].tmask: some lane has a non-zero m_t.
constexpr int kConstTerms = 5;
struct ScanConstArgs {
    OscSet set;
    int mm;                    // bit c: channel c is of kind "three entries"
    int pad;
    ScanChan ch[kChannels];
    int pt[kScanLanes];
    double mono[kChannels][kConstTerms][kScanLanes];
};

struct ScanGeom {
    size_t range;              // events per warp range of the sort passes (multiple of 32)
    unsigned nranges;
    unsigned piece;            // events per piece (multiple of 32)
    unsigned max_units;        // upper bound on the number of pieces (grid size of the main kernel)
    int ncells;                // kChannels * nb
    int nsubs;
    int subs_per_slot;         // sub-groups one warp walks (blockIdx.y selects the slot)
};

} // namespace oscb

namespace oscb {

// ------------------------------------------------------------------------------------------------
// Sort pass 1: histogram cell of every event (kNoCell: dropped, A8/A11) and, per warp range, the number of
// events in every cell.  count is [ncells][nranges]: first sorted position of cell c plus the exclusive prefix over
// the ranges inside row c is the destination of the first event of (cell, range) in a stable sort by cell.
// Shared memory: bin table | wcnt[kScanWarps][ncells] (u32)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32 * kScanWarps)
scan_count_kernel(const double* __restrict__ E_true, const double* __restrict__ E_reco,
                  const int8_t* __restrict__ channel, size_t n, double energy_scale,
                  const double* __restrict__ edges, int nb, ScanGeom geo, unsigned short* __restrict__ cellid,
                  unsigned int* __restrict__ count)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    build_bin_table(smem_raw, edges, nb);
    const BinView bt = bin_view(smem_raw);
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned int* wcnt = reinterpret_cast<unsigned int*>(smem_raw + bin_table_bytes(nb)) + (size_t)warp * geo.ncells;
    // the grid is a few blocks per SM and every warp walks ranges r, r + warps of the grid, ...: the bin table is
    // built once per block, not once per 4 ranges (it was two thirds of this kernel's instructions)
    for (unsigned r = blockIdx.x * kScanWarps + warp; r < geo.nranges; r += gridDim.x * kScanWarps) {
        for (int c = lane; c < geo.ncells; c += 32) wcnt[c] = 0u;
        __syncwarp();
        const size_t begin = (size_t)r * geo.range, end = min(n, begin + geo.range);
        for (size_t j0 = begin; j0 < end; j0 += 32) {
            const size_t j = j0 + lane;
            unsigned cell = kNoCell;
            if (j < end) {
                const double x = scaled_energy(energy_scale, E_reco[j]);
                const int bin = find_bin<0>(bt, x);
                const unsigned ch = (unsigned)(unsigned char)channel[j];
                if (energy_ok(E_true[j]) && ch < (unsigned)kChannels && bin >= 0) cell = ch * (unsigned)nb + (unsigned)bin;
                cellid[j] = (unsigned short)cell;
            }
            const unsigned m = __match_any_sync(0xffffffffu, cell);
            if (cell != kNoCell && lane == 31u - (unsigned)__clz((int)m)) wcnt[cell] += (unsigned)__popc(m);
            __syncwarp();
        }
        for (int c = lane; c < geo.ncells; c += 32) count[(size_t)c * geo.nranges + r] = wcnt[c];
        __syncwarp();
    }
}

// Block-wide exclusive scan of one value per thread (1024 threads); returns the prefix, *total gets the sum.
__device__ __forceinline__ unsigned block_exclusive_scan_1024(unsigned v, unsigned* s_warp, unsigned* total)
{
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= (unsigned)d) inc += o;
    }
    __syncthreads();                       // s_warp may still be read from a previous call
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        unsigned w = s_warp[lane], winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned o = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= (unsigned)d) winc += o;
        }
        s_warp[lane] = winc - w;           // exclusive prefix of the warp sums
        if (lane == 31) s_warp[32] = winc;
    }
    __syncthreads();
    *total = s_warp[32];
    return s_warp[warp] + inc - v;
}

// Sort pass 2a (one block of 1024 threads per cell): count[cell][:] -> exclusive prefix within the cell, in place;
// cell_total[cell] = number of kept events of the cell.
__global__ void __launch_bounds__(1024)
scan_offsets_cell_kernel(unsigned int* __restrict__ count, ScanGeom geo, unsigned int* __restrict__ cell_total)
{
    __shared__ unsigned s_warp[33];
    unsigned int* row = count + (size_t)blockIdx.x * geo.nranges;
    unsigned carry = 0;
    for (unsigned base = 0; base < geo.nranges; base += 1024) {
        const unsigned i = base + threadIdx.x;
        const unsigned v = i < geo.nranges ? row[i] : 0u;
        unsigned total;
        const unsigned ex = block_exclusive_scan_1024(v, s_warp, &total);
        if (i < geo.nranges) row[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0) cell_total[blockIdx.x] = carry;
}

// Sort pass 2b (one block of 1024 threads): cell_begin[c] = first sorted position of cell c (cell_begin[ncells] =
// number of kept events; on entry cell_begin[c] holds the cell's total); unit_begin[c] = index of the first piece of
// cell c (unit_begin[ncells] = number of pieces), unit_cell[u] = cell of piece u.  At most 3 cells per thread
// (ncells <= 4 * 768).
__global__ void __launch_bounds__(1024)
scan_offsets_kernel(ScanGeom geo, unsigned int* __restrict__ cell_begin, unsigned int* __restrict__ unit_begin,
                    unsigned short* __restrict__ unit_cell)
{
    __shared__ unsigned s_warp[33];
    __shared__ unsigned s_ub[4 * 768 + 1];
    const int cper = (geo.ncells + 1023) / 1024;
    const int c0 = min(geo.ncells, (int)threadIdx.x * cper), c1 = min(geo.ncells, c0 + cper);
    unsigned len[3] = {0u, 0u, 0u};
    unsigned sum = 0, np = 0;
    for (int c = c0; c < c1; ++c) {
        len[c - c0] = cell_begin[c];
        sum += len[c - c0];
        np += (len[c - c0] + geo.piece - 1) / geo.piece;
    }
    unsigned total, utotal;
    unsigned run = block_exclusive_scan_1024(sum, s_warp, &total);
    unsigned urun = block_exclusive_scan_1024(np, s_warp, &utotal);
    for (int c = c0; c < c1; ++c) {
        cell_begin[c] = run;
        unit_begin[c] = urun;
        run += len[c - c0];
        urun += (len[c - c0] + geo.piece - 1) / geo.piece;
    }
    if (threadIdx.x == 0) {
        cell_begin[geo.ncells] = total;
        unit_begin[geo.ncells] = utotal;
    }
    // cell of every piece: a warp per cell, lanes over its pieces (a populated cell has thousands of pieces; one thread
    // per cell took 24 us at 1e7 events)
    __syncthreads();
    for (int c = threadIdx.x; c <= geo.ncells; c += 1024) s_ub[c] = unit_begin[c];
    __syncthreads();
    for (int c = threadIdx.x >> 5; c < geo.ncells; c += 32) {
        const unsigned u0 = s_ub[c], u1 = s_ub[c + 1];
        for (unsigned u = u0 + (threadIdx.x & 31u); u < u1; u += 32) unit_cell[u] = (unsigned short)c;
    }
}

// Sort pass 3: stable scatter of (E_true, w0) into cell order.  Same warp ranges as pass 1.
// Shared memory: wcnt[kScanWarps][ncells] (u32)
__global__ void __launch_bounds__(32 * kScanWarps)
scan_scatter_kernel(const double* __restrict__ E_true, const double* __restrict__ w0,
                    const unsigned short* __restrict__ cellid, size_t n, ScanGeom geo,
                    const unsigned int* __restrict__ offsets, const unsigned int* __restrict__ cell_begin,
                    double* __restrict__ sEt, double* __restrict__ sW)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    unsigned int* wcnt = reinterpret_cast<unsigned int*>(smem_raw) + (size_t)warp * geo.ncells;
    for (unsigned r = blockIdx.x * kScanWarps + warp; r < geo.nranges; r += gridDim.x * kScanWarps) {
        for (int c = lane; c < geo.ncells; c += 32) wcnt[c] = 0u;
        __syncwarp();
        const size_t begin = (size_t)r * geo.range, end = min(n, begin + geo.range);
        for (size_t j0 = begin; j0 < end; j0 += 32) {
            const size_t j = j0 + lane;
            const unsigned cell = j < end ? (unsigned)cellid[j] : (unsigned)kNoCell;
            const unsigned m = __match_any_sync(0xffffffffu, cell);
            unsigned before = 0;
            if (cell != kNoCell) before = wcnt[cell];
            __syncwarp();
            if (cell != kNoCell) {
                const size_t dst = (size_t)cell_begin[cell] + offsets[(size_t)cell * geo.nranges + r] + before +
                                   (unsigned)__popc(m & lt_mask);
                sEt[dst] = E_true[j];
                sW[dst] = w0[j];
                if (lane == 31u - (unsigned)__clz((int)m)) wcnt[cell] = before + (unsigned)__popc(m);
            }
            __syncwarp();
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Block-local sort (binnings of up to kSortMaxCells cells): the same stable sort by cell, with a block-wide chunk
// of geo.range events as the unit instead of a warp range.  The per-warp-range scatter above writes 8-byte words to
// ~200 destinations per warp (one sector per lane: 277 us per 1e7 events); here a block first sorts its chunk by cell
// in shared memory and then writes it out in sorted order, so that the events of a (chunk, cell) pair -- 4096 events
// over 200 cells: ~20 on average, hundreds in the populated cells -- leave as runs of whole sectors.
// The order inside a cell is chunk-major and, inside a chunk, the order of the caller's arrays: the sorted arrays are
// the ones the per-warp-range sort produces.
// ------------------------------------------------------------------------------------------------
constexpr int kSortThreads = 512;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortMaxCells = 1024;

// Pass 1: cell of every event, and count[cell][chunk].  Shared memory: bin table | cnt[ncells] (u32).
__global__ void __launch_bounds__(kSortThreads)
sort_count_kernel(const double* __restrict__ E_true, const double* __restrict__ E_reco,
                  const int8_t* __restrict__ channel, size_t n, double energy_scale,
                  const double* __restrict__ edges, int nb, ScanGeom geo, unsigned short* __restrict__ cellid,
                  unsigned int* __restrict__ count)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned int* cnt = reinterpret_cast<unsigned int*>(smem_raw + bin_table_bytes(nb));
    for (int c = threadIdx.x; c < geo.ncells; c += kSortThreads) cnt[c] = 0u;
    build_bin_table(smem_raw, edges, nb);                        // ends with a barrier
    const BinView bt = bin_view(smem_raw);
    for (unsigned r = blockIdx.x; r < geo.nranges; r += gridDim.x) {
        const size_t begin = (size_t)r * geo.range, end = min(n, begin + geo.range);
        for (size_t j = begin + threadIdx.x; j < end; j += kSortThreads) {
            const double x = scaled_energy(energy_scale, E_reco[j]);
            const int bin = find_bin<0>(bt, x);
            const unsigned ch = (unsigned)(unsigned char)channel[j];
            unsigned cell = kNoCell;
            if (energy_ok(E_true[j]) && ch < (unsigned)kChannels && bin >= 0) cell = ch * (unsigned)nb + (unsigned)bin;
            cellid[j] = (unsigned short)cell;
            if (cell != kNoCell) atomicAdd(cnt + cell, 1u);      // integer counts: the order does not matter
        }
        __syncthreads();
        for (int c = threadIdx.x; c < geo.ncells; c += kSortThreads) {
            count[(size_t)c * geo.nranges + r] = cnt[c];
            cnt[c] = 0u;
        }
        __syncthreads();
    }
}

// Pass 3: stable scatter of (E_true, w0) through a chunk sorted in shared memory.  A chunk is 32 * kSortWarps * STEPS
// events; a warp owns STEPS consecutive groups of 32 events and keeps their cells, match masks and payload in
// registers between the counting and the placing phase, so every global load of the chunk is issued up front.
// Shared memory: wcnt[kSortWarps][ncells] | cbase[ncells + 1] | gbase[ncells] (u32) | buf[range] (double2) | bcell[range] (u16)
template <int STEPS>
__global__ void __launch_bounds__(kSortThreads)
sort_scatter_kernel(const double* __restrict__ E_true, const double* __restrict__ w0,
                    const unsigned short* __restrict__ cellid, size_t n, ScanGeom geo,
                    const unsigned int* __restrict__ offsets, const unsigned int* __restrict__ cell_begin,
                    double* __restrict__ sEt, double* __restrict__ sW)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ unsigned s_warp[33];
    const int nc = geo.ncells;
    unsigned int* wcnt_all = reinterpret_cast<unsigned int*>(smem_raw);
    unsigned int* cbase = wcnt_all + (size_t)kSortWarps * nc;
    unsigned int* gbase = cbase + nc + 1;
    double2* buf = reinterpret_cast<double2*>(smem_raw + (((size_t)(kSortWarps + 2) * nc + 1) * 4 + 15) / 16 * 16);
    unsigned short* bcell = reinterpret_cast<unsigned short*>(buf + geo.range);
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    unsigned int* wcnt = wcnt_all + (size_t)warp * nc;
    constexpr unsigned per = 32u * STEPS;                        // events per warp; geo.range = per * kSortWarps

    for (unsigned r = blockIdx.x; r < geo.nranges; r += gridDim.x) {
        const size_t begin = (size_t)r * geo.range, end = min(n, begin + geo.range);
        const size_t wb = min(end, begin + (size_t)warp * per);
        unsigned cell[STEPS], m[STEPS];
        double ev[STEPS], wv[STEPS];
#pragma unroll
        for (int k = 0; k < STEPS; ++k) {
            const size_t j = wb + 32u * k + lane;
            const bool in = j < end;
            cell[k] = in ? (unsigned)__ldg(cellid + j) : (unsigned)kNoCell;
            ev[k] = in ? __ldcs(E_true + j) : 0.0;
            wv[k] = in ? __ldcs(w0 + j) : 0.0;
        }
        // phase A: events per (warp, cell)
        for (int c = lane; c < nc; c += 32) wcnt[c] = 0u;
        __syncwarp();
#pragma unroll
        for (int k = 0; k < STEPS; ++k) {
            m[k] = __match_any_sync(0xffffffffu, cell[k]);
            if (cell[k] != kNoCell && lane == 31u - (unsigned)__clz((int)m[k])) wcnt[cell[k]] += (unsigned)__popc(m[k]);
            __syncwarp();
        }
        __syncthreads();
        // per cell: exclusive prefix over the warps (in place), total into cbase
        for (int c = threadIdx.x; c < nc; c += kSortThreads) {
            unsigned run = 0;
#pragma unroll
            for (int w = 0; w < kSortWarps; ++w) {
                const unsigned v = wcnt_all[(size_t)w * nc + c];
                wcnt_all[(size_t)w * nc + c] = run;
                run += v;
            }
            cbase[c] = run;
        }
        __syncthreads();
        // exclusive scan of the cell totals (each thread a contiguous run of cells)
        {
            const int cper = (nc + kSortThreads - 1) / kSortThreads;
            const int c0 = min(nc, (int)threadIdx.x * cper), c1 = min(nc, c0 + cper);
            unsigned sum = 0;
            for (int c = c0; c < c1; ++c) sum += cbase[c];
            unsigned inc = sum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned o = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= (unsigned)d) inc += o;
            }
            if (lane == 31) s_warp[warp] = inc;
            __syncthreads();
            if (warp == 0) {
                const unsigned w = lane < (unsigned)kSortWarps ? s_warp[lane] : 0u;
                unsigned winc = w;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const unsigned o = __shfl_up_sync(0xffffffffu, winc, d);
                    if (lane >= (unsigned)d) winc += o;
                }
                s_warp[lane] = winc - w;
                if (lane == 31) s_warp[32] = winc;
            }
            __syncthreads();
            unsigned run = s_warp[warp] + inc - sum;
            for (int c = c0; c < c1; ++c) {
                const unsigned v = cbase[c];
                cbase[c] = run;
                gbase[c] = __ldg(cell_begin + c) + __ldg(offsets + (size_t)c * geo.nranges + r) - run;
                run += v;
            }
            if (threadIdx.x == 0) cbase[nc] = s_warp[32];
        }
        __syncthreads();
        // phase B: every event to its place in the sorted chunk
#pragma unroll
        for (int k = 0; k < STEPS; ++k) {
            if (cell[k] != kNoCell) {
                const unsigned pos = cbase[cell[k]] + wcnt[cell[k]] + (unsigned)__popc(m[k] & lt_mask);
                buf[pos] = make_double2(ev[k], wv[k]);
                bcell[pos] = (unsigned short)cell[k];
            }
            __syncwarp();
            if (cell[k] != kNoCell && lane == 31u - (unsigned)__clz((int)m[k])) wcnt[cell[k]] += (unsigned)__popc(m[k]);
            __syncwarp();
        }
        __syncthreads();
        // phase C: the sorted chunk leaves in order; neighbours in the chunk are neighbours in the sorted arrays
        const unsigned kept = cbase[nc];
        for (unsigned p = threadIdx.x; p < kept; p += kSortThreads) {
            const double2 v = buf[p];
            const unsigned dst = gbase[bcell[p]] + p;
            sEt[dst] = v.x;
            sW[dst] = v.y;
        }
        __syncthreads();
    }
}

} // namespace oscb

namespace oscb {

// Entry (i, j) of S' (common phase dropped, as in osc_core.cuh) for a real symmetric T': the imaginary parts of
// T'_ij and (T'^2)_ij vanish, which removes a third of assemble()'s arithmetic.
__device__ __forceinline__ void scan_amp(const OscEig& e, double A, const ScanElem& el, double& zr, double& zi)
{
    const double Tr = fma(A, el.ee, el.Tr0);
    const double T2r = fma(A, fma(A, el.ee, el.T2r1), el.T2r0);
    const double N0r = fma(e.prod12, el.delta, fma(-e.sum12, Tr, T2r));
    const double N2r = fma(e.prod01, el.delta, fma(-e.sum01, Tr, T2r));
    const double kn = e.kap2 * N2r;
    zr = fma(el.delta, e.c1h, -(kn * e.s02));
    zi = fma(el.delta, e.s1h, fma(kn, e.c02, -(e.kap0 * N0r)));
}

constexpr int kSliceEvents = 64;      // events per phase-A slice of a warp (two per lane)
constexpr int kSliceDoubles = 10;     // up to nine terms, padded to whole 16-byte words

__device__ __forceinline__ ScanElem ldg_elem(const ScanElem* p)
{
    ScanElem e;
    e.delta = __ldg(&p->delta);
    e.ee = __ldg(&p->ee);
    e.Tr0 = __ldg(&p->Tr0);
    e.T2r0 = __ldg(&p->T2r0);
    e.T2r1 = __ldg(&p->T2r1);
    return e;
}

// Phase A tail: the used terms of one event, times w0, compacted in canonical order into its slice row.
__device__ __forceinline__ void scan_store_terms(double* row, int tmask, double w, const double (&zr)[kScanElems],
                                                 const double (&zi)[kScanElems])
{
    int t = 0;
    if (tmask & 1) row[t++] = w * fma(zr[0], zr[0], zi[0] * zi[0]);
    if (tmask & 2) row[t++] = w * fma(zr[1], zr[1], zi[1] * zi[1]);
    if (tmask & 4) row[t++] = w * fma(zr[2], zr[2], zi[2] * zi[2]);
    if (tmask & 8) row[t++] = w * fma(zr[0], zr[1], zi[0] * zi[1]);
    if (tmask & 16) row[t++] = w * fma(zr[0], zr[2], zi[0] * zi[2]);
    if (tmask & 32) row[t++] = w * fma(zr[1], zr[2], zi[1] * zi[2]);
    if (tmask & 64) row[t++] = w * fma(zi[0], zr[1], -(zr[0] * zi[1]));
    if (tmask & 128) row[t++] = w * fma(zi[0], zr[2], -(zr[0] * zi[2]));
    if (tmask & 256) row[t++] = w * fma(zi[1], zr[2], -(zr[1] * zi[2]));
}

// Phase B: lane = point.  Every lane walks the `cnt` events of the slice (all lanes read the same words: one
// shared-memory wavefront per load) and accumulates sum_t q_t m_t.  Four events per step feed four independent
// accumulators, so that one warp alone covers the latency of the fp64 pipe; consecutive fused multiply-adds share
// the monomial operand.
template <int NT>
__device__ __forceinline__ void scan_phase_b(uint32_t slice, int cnt, const double (&m)[kScanTerms], double (&acc)[4])
{
    constexpr uint32_t ROW = 8u * kSliceDoubles;
    int j = 0;
    for (; j + 3 < cnt; j += 4) {
        const uint32_t a = slice + (uint32_t)j * ROW;
#pragma unroll
        for (int t = 0; t + 1 < NT; t += 2) {
            const double2 q0 = lds_f64x2(a + 8u * t), q1 = lds_f64x2(a + ROW + 8u * t);
            const double2 q2 = lds_f64x2(a + 2 * ROW + 8u * t), q3 = lds_f64x2(a + 3 * ROW + 8u * t);
            acc[0] = fma(q0.x, m[t], acc[0]);
            acc[1] = fma(q1.x, m[t], acc[1]);
            acc[2] = fma(q2.x, m[t], acc[2]);
            acc[3] = fma(q3.x, m[t], acc[3]);
            acc[0] = fma(q0.y, m[t + 1], acc[0]);
            acc[1] = fma(q1.y, m[t + 1], acc[1]);
            acc[2] = fma(q2.y, m[t + 1], acc[2]);
            acc[3] = fma(q3.y, m[t + 1], acc[3]);
        }
        if (NT & 1) {
            acc[0] = fma(lds_f64(a + 8u * (NT - 1)), m[NT - 1], acc[0]);
            acc[1] = fma(lds_f64(a + ROW + 8u * (NT - 1)), m[NT - 1], acc[1]);
            acc[2] = fma(lds_f64(a + 2 * ROW + 8u * (NT - 1)), m[NT - 1], acc[2]);
            acc[3] = fma(lds_f64(a + 3 * ROW + 8u * (NT - 1)), m[NT - 1], acc[3]);
        }
    }
    for (; j < cnt; ++j) {
        const uint32_t a = slice + (uint32_t)j * ROW;
#pragma unroll
        for (int t = 0; t < NT; ++t) acc[0] = fma(lds_f64(a + 8u * t), m[t], acc[0]);
    }
}

// ------------------------------------------------------------------------------------------------
// k4 main kernel.  Warp (blockIdx.x * kScanWarps + warp) owns one piece of one sorted cell; blockIdx.y selects the
// slot of sub-groups it walks.  partial[piece][point] is written once by exactly one lane.
// Shared memory: slice[kScanWarps][kSliceEvents][kSliceDoubles]
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32 * kScanWarps)
scan_main_kernel(const ScanGroup* __restrict__ groups, const ScanSub* __restrict__ subs,
                 const double* __restrict__ sEt, const double* __restrict__ sW,
                 const unsigned int* __restrict__ cell_begin, const unsigned int* __restrict__ unit_begin,
                 const unsigned short* __restrict__ unit_cell, ScanGeom geo, int nb, int npoints,
                 double* __restrict__ partial)
{
    __shared__ __align__(16) double s_slice[kScanWarps][kSliceEvents][kSliceDoubles];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned u = blockIdx.x * kScanWarps + warp;
    if (u >= __ldg(unit_begin + geo.ncells)) return;
    const int cell = (int)__ldg(unit_cell + u);
    const unsigned cb = __ldg(cell_begin + cell), ce = __ldg(cell_begin + cell + 1);
    const unsigned begin = cb + (u - __ldg(unit_begin + cell)) * geo.piece;
    const unsigned end = min(ce, begin + geo.piece);
    const int ch = cell / nb;

    double* my = &s_slice[warp][0][0];
    const uint32_t slice = smem_u32(my);
    const int s_begin = blockIdx.y * geo.subs_per_slot, s_end = min(geo.nsubs, s_begin + geo.subs_per_slot);
    for (int s = s_begin; s < s_end; ++s) {
        const ScanSub* sub = subs + s;
        const ScanGroup* g = groups + __ldg(&sub->group);
        OscSet set;
        set.xq23 = __ldg(&g->set.xq23);
        set.tr = __ldg(&g->set.tr);
        set.dd = __ldg(&g->set.dd);
        set.k1 = __ldg(&g->set.k1);
        set.k0_27 = __ldg(&g->set.k0_27);
        const ScanChan* gc = &g->ch[ch];
        const double sa = __ldg(&gc->sa);
        const int nk = __ldg(&gc->nk);
        const int tmask = __ldg(&gc->tmask);
        const int nt = __popc(tmask);
        const ScanElem el0 = ldg_elem(&gc->el[0]), el1 = ldg_elem(&gc->el[1]), el2 = ldg_elem(&gc->el[2]);
        double m[kScanTerms];
#pragma unroll
        for (int t = 0; t < kScanTerms; ++t) m[t] = t < nt ? __ldg(&sub->mono[ch][t][lane]) : 0.0;
        const int pt = __ldg(&sub->pt[lane]);
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        for (unsigned s0 = begin; s0 < end; s0 += kSliceEvents) {
            // ---- phase A: lane = event (two per lane): S' entries, then the terms into the slice ------------
            const unsigned e0 = s0 + lane, e1 = e0 + 32;
            const double E0 = e0 < end ? __ldg(sEt + e0) : 1.0, E1 = e1 < end ? __ldg(sEt + e1) : 1.0;
            const double w0v = e0 < end ? __ldg(sW + e0) : 0.0, w1v = e1 < end ? __ldg(sW + e1) : 0.0;
            const double A0 = sa * E0, A1 = sa * E1;
            OscEig g0, g1;
            eig_solve(set, A0, rcp_pos(E0), g0);
            eig_solve(set, A1, rcp_pos(E1), g1);
            double zr0[kScanElems] = {0.0, 0.0, 0.0}, zi0[kScanElems] = {0.0, 0.0, 0.0};
            double zr1[kScanElems] = {0.0, 0.0, 0.0}, zi1[kScanElems] = {0.0, 0.0, 0.0};
            scan_amp(g0, A0, el0, zr0[0], zi0[0]);
            scan_amp(g1, A1, el0, zr1[0], zi1[0]);
            if (nk > 1) {
                scan_amp(g0, A0, el1, zr0[1], zi0[1]);
                scan_amp(g1, A1, el1, zr1[1], zi1[1]);
            }
            if (nk > 2) {
                scan_amp(g0, A0, el2, zr0[2], zi0[2]);
                scan_amp(g1, A1, el2, zr1[2], zi1[2]);
            }
            scan_store_terms(my + (size_t)lane * kSliceDoubles, tmask, w0v, zr0, zi0);
            scan_store_terms(my + (size_t)(lane + 32) * kSliceDoubles, tmask, w1v, zr1, zi1);
            __syncwarp();
            // ---- phase B: lane = point ------------------------------------------------------------------
            const int cnt = (int)min((unsigned)kSliceEvents, end - s0);
            switch (nt) {
            case 1: scan_phase_b<1>(slice, cnt, m, acc); break;
            case 2: scan_phase_b<2>(slice, cnt, m, acc); break;
            case 3: scan_phase_b<3>(slice, cnt, m, acc); break;
            case 4: scan_phase_b<4>(slice, cnt, m, acc); break;
            case 5: scan_phase_b<5>(slice, cnt, m, acc); break;
            case 6: scan_phase_b<6>(slice, cnt, m, acc); break;
            case 7: scan_phase_b<7>(slice, cnt, m, acc); break;
            case 8: scan_phase_b<8>(slice, cnt, m, acc); break;
            case 9: scan_phase_b<9>(slice, cnt, m, acc); break;
            default: break;                                     // no term: every monomial of the group is zero
            }
            __syncwarp();
        }
        if (pt >= 0) partial[(size_t)u * npoints + pt] = (acc[0] + acc[1]) + (acc[2] + acc[3]);
    }
}

// ------------------------------------------------------------------------------------------------
// k4 main kernel, second form: ONE sub-group per launch, its tables in the kernel parameters (ScanConstArgs).
// Lane = event in both phases: phase A leaves the terms q_t of the lane's event in registers, phase B adds
// q_t m_t[point] to 32 accumulators (one per point of the sub-group) with the monomials as constant-bank operands.
// Why: a DFMA with three distinct register operands issues every 3 cycles on sm_100a, any other every 2
// (profiles/r2_dfma_issue.md); lane = point needs acc += q * m with q from a shared-memory broadcast load and m in a
// register (three registers plus a load per fused multiply-add), lane = event needs acc += q * c[bank][offset] (two
// registers, no load).  The 32 accumulators of a lane are transposed through shared memory once per piece: lane p
// sums the p-th accumulator of lanes 0..31 in that order, so partial[piece][point] is a deterministic function of
// the inputs.  The launches of the sub-groups of a call do not depend on one another: each triggers its successor at
// once (griddepcontrol.launch_dependents) and waits for its predecessor only before it exits, so the blocks of
// the next sub-group fill the SMs as the current one drains and the launches complete in order.
// Shared memory: red[kScanWarps][32][kRedStride]
// ------------------------------------------------------------------------------------------------
constexpr int kRedStride = 34;        // doubles per row of the transposition buffer: 16-byte rows, conflict-free

// Events per lane and step, blocks per SM (configs[3], 1e6 events x 1024 points, ms per call): 1 event, 4 blocks 0.852;
// 2 events, 4 blocks (128 registers, 250 bytes of spills) 0.747; 2 events, 3 blocks (168 registers) 0.807; 3 events,
// 3 blocks 0.883.  A pair of monomials loaded once (LDCU.128) serves kConstEv fused multiply-adds per point.
constexpr int kConstEv = 2;
constexpr int kConstBlocksPerSM = 4;

// Entry of S' with delta = 0, ee = 0 (an off-diagonal entry, or the difference of two diagonal ones), and with
// delta = 1, ee = 0: scan_amp with the flags folded in.
__device__ __forceinline__ void scan_amp_off(const OscEig& e, double A, const ScanElem& el, double& zr, double& zi)
{
    const double T2r = fma(A, el.T2r1, el.T2r0);
    const double N0r = fma(-e.sum12, el.Tr0, T2r);
    const double N2r = fma(-e.sum01, el.Tr0, T2r);
    const double kn = e.kap2 * N2r;
    zr = -(kn * e.s02);
    zi = fma(kn, e.c02, -(e.kap0 * N0r));
}
__device__ __forceinline__ void scan_amp_diag(const OscEig& e, double A, const ScanElem& el, double& zr, double& zi)
{
    const double T2r = fma(A, el.T2r1, el.T2r0);
    const double N0r = e.prod12 + fma(-e.sum12, el.Tr0, T2r);
    const double N2r = e.prod01 + fma(-e.sum01, el.Tr0, T2r);
    const double kn = e.kap2 * N2r;
    zr = fma(-kn, e.s02, e.c1h);
    zi = fma(kn, e.c02, fma(-e.kap0, N0r, e.s1h));
}

template <int CH, bool MM>
__device__ __forceinline__ void scan_const_piece(const ScanConstArgs& P, const double* __restrict__ sEt,
                                                 const double* __restrict__ sW, unsigned begin, unsigned end,
                                                 unsigned lane, double (&acc)[kScanLanes], double& cst)
{
    constexpr int NT = MM ? 5 : 3;
    const ScanChan& c = P.ch[CH];
    const int tm = c.tmask;
    unsigned e = begin + lane;
    double E[kConstEv], w[kConstEv];
#pragma unroll
    for (int k = 0; k < kConstEv; ++k) {
        E[k] = e + 32 * k < end ? __ldg(sEt + e + 32 * k) : 1.0;
        w[k] = e + 32 * k < end ? __ldg(sW + e + 32 * k) : 0.0;
    }
#pragma unroll 1
    for (unsigned s0 = begin; s0 < end; s0 += 32 * kConstEv) {
        e += 32 * kConstEv;
        double En[kConstEv], wn[kConstEv];
#pragma unroll
        for (int k = 0; k < kConstEv; ++k) {
            En[k] = e + 32 * k < end ? __ldg(sEt + e + 32 * k) : 1.0;
            wn[k] = e + 32 * k < end ? __ldg(sW + e + 32 * k) : 0.0;
        }
        // ---- phase A: S' entries of the lane's events, then the terms --------------------------------------
        double q[kConstEv][NT];
#pragma unroll
        for (int k = 0; k < kConstEv; ++k) {
            const double A = c.sa * E[k];
            OscEig g;
            eig_solve(P.set, A, rcp_pos(E[k]), g);
            if (MM) {
                double sr, si, ur, ui, vr, vi;
                scan_amp_diag(g, A, c.el[0], sr, si);
                scan_amp_off(g, A, c.el[1], ur, ui);
                scan_amp_off(g, A, c.el[2], vr, vi);
                cst = fma(w[k], fma(sr, sr, si * si), cst);
                q[k][0] = w[k] * fma(ur, ur, ui * ui);
                q[k][1] = w[k] * fma(vr, vr, vi * vi);
                q[k][2] = w[k] * fma(sr, ur, si * ui);
                q[k][3] = w[k] * fma(sr, vr, si * vi);
                q[k][4] = w[k] * fma(ur, vr, ui * vi);
            } else {
                double zr0, zi0, zr1, zi1;
                scan_amp_off(g, A, c.el[0], zr0, zi0);
                scan_amp_off(g, A, c.el[1], zr1, zi1);
                const double n1 = fma(zr1, zr1, zi1 * zi1);
                cst = fma(w[k], n1, cst);
                q[k][0] = w[k] * (fma(zr0, zr0, zi0 * zi0) - n1);
                q[k][1] = w[k] * fma(zr0, zr1, zi0 * zi1);
                q[k][2] = w[k] * fma(zi0, zr1, -(zr0 * zi1));
            }
        }
        // ---- phase B: 32 points, the monomials from the kernel parameters ----------------------------------
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            if (tm & (1 << t)) {
#pragma unroll
                for (int p = 0; p < kScanLanes; ++p) {
                    const double m = P.mono[CH][t][p];
#pragma unroll
                    for (int k = 0; k < kConstEv; ++k) acc[p] = fma(q[k][t], m, acc[p]);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < kConstEv; ++k) {
            E[k] = En[k];
            w[k] = wn[k];
        }
    }
}

__global__ void __launch_bounds__(32 * kScanWarps, kConstBlocksPerSM)
scan_const_kernel(const __grid_constant__ ScanConstArgs P, const double* __restrict__ sEt, const double* __restrict__ sW,
                  const unsigned int* __restrict__ cell_begin, const unsigned int* __restrict__ unit_begin,
                  const unsigned short* __restrict__ unit_cell, ScanGeom geo, int nb, int npoints,
                  double* __restrict__ partial)
{
    __shared__ __align__(16) double s_red[kScanWarps][kScanLanes * kRedStride];
    pdl_launch_dependents();
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned u = blockIdx.x * kScanWarps + warp;
    if (u < __ldg(unit_begin + geo.ncells)) {
        const int cell = (int)__ldg(unit_cell + u);
        const unsigned cb = __ldg(cell_begin + cell), ce = __ldg(cell_begin + cell + 1);
        const unsigned begin = cb + (u - __ldg(unit_begin + cell)) * geo.piece;
        const unsigned end = min(ce, begin + geo.piece);
        const int ch = cell / nb;
        double acc[kScanLanes];
#pragma unroll
        for (int p = 0; p < kScanLanes; ++p) acc[p] = 0.0;
        double cst = 0.0;                                       // the term every point shares
        const bool mm = (P.mm >> ch) & 1;
        switch (ch) {
        case 0: if (mm) scan_const_piece<0, true>(P, sEt, sW, begin, end, lane, acc, cst); else scan_const_piece<0, false>(P, sEt, sW, begin, end, lane, acc, cst); break;
        case 1: if (mm) scan_const_piece<1, true>(P, sEt, sW, begin, end, lane, acc, cst); else scan_const_piece<1, false>(P, sEt, sW, begin, end, lane, acc, cst); break;
        case 2: if (mm) scan_const_piece<2, true>(P, sEt, sW, begin, end, lane, acc, cst); else scan_const_piece<2, false>(P, sEt, sW, begin, end, lane, acc, cst); break;
        default: if (mm) scan_const_piece<3, true>(P, sEt, sW, begin, end, lane, acc, cst); else scan_const_piece<3, false>(P, sEt, sW, begin, end, lane, acc, cst); break;
        }
        // transposition: row = lane of the event, column = point; lane p then adds column p from the top
        double* r = s_red[warp];
#pragma unroll
        for (int p = 0; p < kScanLanes; p += 2)
            *reinterpret_cast<double2*>(r + lane * kRedStride + p) = make_double2(acc[p], acc[p + 1]);
        __syncwarp();
        double s[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int l = 0; l < kScanLanes; l += 4) {
#pragma unroll
            for (int k = 0; k < 4; ++k) s[k] += r[(l + k) * kRedStride + lane];
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) cst += __shfl_xor_sync(0xffffffffu, cst, off);
        const int pt = P.pt[lane];
        if (pt >= 0) partial[(size_t)u * npoints + pt] = ((s[0] + s[1]) + (s[2] + s[3])) + cst;
    }
    pdl_wait();
}

// ------------------------------------------------------------------------------------------------
// k5: the batched call for point lists WITHOUT scan structure (every point its own eigen-problem, e.g. a batch of
// Markov-chain proposals), on the sorted events of k4.  Warp (blockIdx.x * kScanWarps + warp) owns one piece of one
// sorted cell and stages its events (E_true, 1/E_true, w0) in shared memory once; blockIdx.y selects the slot of
// points it walks.  Lane = event throughout.  What the sort buys over one pass of k2 per point:
//   * every event of the piece has the same histogram cell: the weights are summed in a register and reduced over
//     the warp once per (piece, point) -- no bin search, no MATCH, no shared-memory histogram in the point loop;
//   * every event of the piece has the same channel: the transition block is loaded once per (piece, point) and the
//     amplitude assembly is the one specialised for the kind of element (assemble_kind), chosen by a uniform branch;
//   * 1/E is taken once per event, not once per event and point.
// partial[piece][point] and scan_merge are those of k4.  kinds[c] is the element kind of channel c (osc_core.cuh).
// Shared memory (dynamic): ev[kScanWarps][3][piece]
// ------------------------------------------------------------------------------------------------
struct ChannelKinds {
    int k[kChannels];
};

// Sum of w0 P over the events of the staged piece for one point; lane = event, kFullUnroll events per lane and step
// (independent dependency chains: the kernel runs few warps per SM, so the instruction-level parallelism has to come
// from inside the warp); padding slots carry E = 1, w0 = 0.  Fixed summation order: deterministic.
constexpr int kFullUnroll = 4;

// STAGED: the events come from the warp's shared-memory copy (E, 1/E, w0); otherwise straight from the sorted arrays
// in global memory with 1/E taken here -- for one or two points per piece the staging pass costs more than it saves.
template <int KIND, bool STAGED, int UNROLL = kFullUnroll>
__device__ __forceinline__ double full_piece_sum(const OscSet& set, const OscTrans& tr, const double* sE,
                                                 const double* sI, const double* sW, int len, unsigned lane)
{
    double acc[UNROLL];
#pragma unroll
    for (int k = 0; k < UNROLL; ++k) acc[k] = 0.0;
    // unstaged: the loads of the next step are issued before the arithmetic of the current one
    double nE[UNROLL], nW[UNROLL];
    if (!STAGED) {
#pragma unroll
        for (int k = 0; k < UNROLL; ++k) {
            const int j = (int)lane + 32 * k;
            nE[k] = j < len ? __ldg(sE + j) : 1.0;
            nW[k] = j < len ? __ldg(sW + j) : 0.0;
        }
    }
    for (int i = lane; i < len; i += 32 * UNROLL) {
        double E[UNROLL], I[UNROLL], w[UNROLL], A[UNROLL];
        OscEig e[UNROLL];
#pragma unroll
        for (int k = 0; k < UNROLL; ++k) {
            const int j = i + 32 * k;
            if (STAGED) {
                const bool has = j < len;
                E[k] = has ? sE[j] : 1.0;
                I[k] = has ? sI[j] : 1.0;
                w[k] = has ? sW[j] : 0.0;
            } else {
                E[k] = nE[k];
                w[k] = nW[k];
                const int jn = j + 32 * UNROLL;
                nE[k] = jn < len ? __ldg(sE + jn) : 1.0;
                nW[k] = jn < len ? __ldg(sW + jn) : 0.0;
            }
            A[k] = tr.sa * E[k];
        }
        if (!STAGED) {
#pragma unroll
            for (int k = 0; k < UNROLL; ++k) I[k] = rcp_pos(E[k]);
        }
#pragma unroll
        for (int k = 0; k < UNROLL; ++k) eig_solve(set, A[k], I[k], e[k]);
#pragma unroll
        for (int k = 0; k < UNROLL; ++k) acc[k] = fma(w[k], assemble_kind<KIND>(e[k], A[k], tr), acc[k]);
    }
    double s = acc[0];
#pragma unroll
    for (int k = 1; k < UNROLL; ++k) s += acc[k];
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    return s;
}

template <bool STAGED>
__global__ void __launch_bounds__(32 * kScanWarps, 3)
scan_full_kernel(const double* __restrict__ points, int npoints, int pts_per_slot, const ChannelKinds kinds,
                 const double* __restrict__ sEt, const double* __restrict__ sW,
                 const unsigned int* __restrict__ cell_begin, const unsigned int* __restrict__ unit_begin,
                 const unsigned short* __restrict__ unit_cell, ScanGeom geo, int nb, double* __restrict__ partial)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned u = blockIdx.x * kScanWarps + warp;
    if (u >= __ldg(unit_begin + geo.ncells)) return;
    const int cell = (int)__ldg(unit_cell + u);
    const unsigned cb = __ldg(cell_begin + cell), ce = __ldg(cell_begin + cell + 1);
    const unsigned begin = cb + (u - __ldg(unit_begin + cell)) * geo.piece;
    const int len = (int)(min(ce, begin + geo.piece) - begin);
    const int ch = cell / nb;

    const double* sE = sEt + begin;
    const double* sI = nullptr;
    const double* sWt = sW + begin;
    if (STAGED) {
        double* tE = reinterpret_cast<double*>(smem_raw) + (size_t)warp * 3 * geo.piece;
        double* tI = tE + geo.piece;
        double* tW = tI + geo.piece;
        for (int i = lane; i < len; i += 32) {
            const double E = __ldg(sEt + begin + i);
            tE[i] = E;
            tI[i] = rcp_pos(E);
            tW[i] = __ldg(sW + begin + i);
        }
        __syncwarp();
        sE = tE;
        sI = tI;
        sWt = tW;
    }

    const int p_begin = blockIdx.y * pts_per_slot, p_end = min(npoints, p_begin + pts_per_slot);
    const int kind = kinds.k[ch];
    for (int p = p_begin; p < p_end; ++p) {
        const double* pb = points + (size_t)p * kBinArgsDoubles;
        OscSet set;
        set.xq23 = __ldg(pb + 0);
        set.tr = __ldg(pb + 1);
        set.dd = __ldg(pb + 2);
        set.k1 = __ldg(pb + 3);
        set.k0_27 = __ldg(pb + 4);
        const double* tb = pb + 6 + ch * kTransDoubles;
        OscTrans tr;
        tr.sa = __ldg(tb + 0);
        tr.delta = __ldg(tb + 1);
        tr.ee = __ldg(tb + 2);
        tr.Tr0 = __ldg(tb + 3);
        tr.Ti0 = __ldg(tb + 4);
        tr.T2r0 = __ldg(tb + 5);
        tr.T2i0 = __ldg(tb + 6);
        tr.T2r1 = __ldg(tb + 7);
        tr.T2i1 = __ldg(tb + 8);
        tr.pad = 0.0;
        double s;
        if (kind == 2) s = full_piece_sum<2, STAGED>(set, tr, sE, sI, sWt, len, lane);
        else if (kind == 3) s = full_piece_sum<3, STAGED>(set, tr, sE, sI, sWt, len, lane);
        else if (kind == 1) s = full_piece_sum<1, STAGED>(set, tr, sE, sI, sWt, len, lane);
        else s = full_piece_sum<0, STAGED>(set, tr, sE, sI, sWt, len, lane);
        if (lane == 0) partial[(size_t)u * npoints + p] = s;
    }
}

constexpr int kOneUnroll = 4;

// k5 for ONE parameter set (osc_plan_reweight_bin): the parameter block travels as a kernel parameter, as in k2, so
// the call is two launches and nothing else on the stream (no table upload, no per-call allocation).
__global__ void __launch_bounds__(32 * kScanWarps, 3)
scan_full_one_kernel(const __grid_constant__ BinArgs a, const ChannelKinds kinds, const double* __restrict__ sEt,
                     const double* __restrict__ sW, const unsigned int* __restrict__ cell_begin,
                     const unsigned int* __restrict__ unit_begin, const unsigned short* __restrict__ unit_cell,
                     ScanGeom geo, int nb, double* __restrict__ partial)
{
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned u = blockIdx.x * kScanWarps + warp;
    if (u >= __ldg(unit_begin + geo.ncells)) return;
    const int cell = (int)__ldg(unit_cell + u);
    const unsigned cb = __ldg(cell_begin + cell), ce = __ldg(cell_begin + cell + 1);
    const unsigned begin = cb + (u - __ldg(unit_begin + cell)) * geo.piece;
    const int len = (int)(min(ce, begin + geo.piece) - begin);
    const int ch = cell / nb;
    const int kind = kinds.k[ch];
    // the channel is warp-uniform: copy its transition block out of the parameter space once
    OscTrans tr;
    const double* tb = reinterpret_cast<const double*>(&a.ch[0]) + ch * kTransDoubles;
    tr.sa = tb[0];
    tr.delta = tb[1];
    tr.ee = tb[2];
    tr.Tr0 = tb[3];
    tr.Ti0 = tb[4];
    tr.T2r0 = tb[5];
    tr.T2i0 = tb[6];
    tr.T2r1 = tb[7];
    tr.T2i1 = tb[8];
    tr.pad = 0.0;
    const double* sE = sEt + begin;
    const double* sWt = sW + begin;
    double s;
    if (kind == 2) s = full_piece_sum<2, false, kOneUnroll>(a.set, tr, sE, nullptr, sWt, len, lane);
    else if (kind == 3) s = full_piece_sum<3, false, kOneUnroll>(a.set, tr, sE, nullptr, sWt, len, lane);
    else if (kind == 1) s = full_piece_sum<1, false, kOneUnroll>(a.set, tr, sE, nullptr, sWt, len, lane);
    else s = full_piece_sum<0, false, kOneUnroll>(a.set, tr, sE, nullptr, sWt, len, lane);
    if (lane == 0) partial[u] = s;
}

// out[p][cell] = sum over the pieces of the cell, in order, of partial[piece][p]; 0 for an empty cell.
// grid (ncells, ceil(npoints / 256)); the loads of eight pieces are issued together before they are added.
__global__ void __launch_bounds__(256)
scan_merge_kernel(const double* __restrict__ partial, const unsigned int* __restrict__ unit_begin, int ncells,
                  int npoints, double* __restrict__ out)
{
    const int cell = blockIdx.x;
    const int p = blockIdx.y * blockDim.x + threadIdx.x;
    if (p >= npoints) return;
    const unsigned u0 = unit_begin[cell], u1 = unit_begin[cell + 1];
    const double* src = partial + (size_t)u0 * npoints + p;
    double s = 0.0;
    unsigned u = u0;
    for (; u + 8 <= u1; u += 8, src += (size_t)8 * npoints) {
        double v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = __ldg(src + (size_t)k * npoints);
#pragma unroll
        for (int k = 0; k < 8; ++k) s += v[k];
    }
    for (; u < u1; ++u, src += npoints) s += __ldg(src);
    out[(size_t)p * ncells + cell] = s;
}


// The same merge for a handful of points (one warp per (cell, point)): lane l adds the pieces u0 + l, u0 + l + 32, ...
// of the cell in order, then a fixed xor-tree over the lanes.  A different but equally fixed order of additions.
__global__ void __launch_bounds__(256)
scan_merge_few_kernel(const double* __restrict__ partial, const unsigned int* __restrict__ unit_begin, int ncells,
                      int npoints, double* __restrict__ out)
{
    const int cell = blockIdx.x;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned u0 = unit_begin[cell], u1 = unit_begin[cell + 1];
    for (int p = threadIdx.x >> 5; p < npoints; p += blockDim.x >> 5) {
        double s = 0.0;
        for (unsigned u = u0 + lane; u < u1; u += 32) s += __ldg(partial + (size_t)u * npoints + p);
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0) out[(size_t)p * ncells + cell] = s;
    }
}

} // namespace oscb
