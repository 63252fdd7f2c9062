// osc_bins.cuh -- the integer binning decision (readings A8, A9).
//
// The bin of x = fl64(energy_scale * E_reco) is the unique i with edges[i] <= x < edges[i+1] in IEEE
// double.  The comparisons are taken on order-preserving 64-bit integer images of the doubles ("keys"),
// so the decision is bit-identical to the fp64 comparisons and costs nothing on the fp64 pipe, which is
// the pipe that bounds the kernels.
//
// Every block of the event kernels builds a bin table in its shared memory (build_bin_table, a few
// thousand cycles, once per kernel):
//
//     head   : base, shift                        -- the key -> cell map
//     ekey[] : key(edges[0..nb]), then 3 sentinels (all ones)
//     lut[]  : kLutCells entries; lut[c] = largest i with ekey[i] <= first key of cell c (0 if none)
//
// A cell is a range of 2^shift consecutive values of the key's upper 32 bits, counted from `base` (the
// upper key word of edges[1], or of edges[0] when there is a single bin -- everything below edges[1] is
// bin 0 or underflow).  The upper key word of a positive double grows linearly inside a binade and by
// 2^20 per binade, so the cells resolve both linearly and logarithmically spaced edges; the look-up
// gives a lower bound of the bin, two branch-free forward steps finish the search for every sane
// binning, and a loop covers the rest (any strictly increasing edges are handled exactly).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "osc_smem.cuh"

namespace oscb {

constexpr int kLutCells = 2048;
constexpr int kKeySentinels = 3;
constexpr long long kKeyMax = 0x7FFFFFFFFFFFFFFFll;

struct BinHead {
    int base;            // upper key word where cell 0 starts
    unsigned int shift;  // cell = (upper key word - base) >> shift
    unsigned int nb;
    unsigned int steps;  // forward steps that finish the search from lut[cell], maximum over all cells
};

// Byte layout of the table in shared memory (all parts 16-byte aligned).
__host__ __device__ constexpr size_t bin_keys_offset() { return sizeof(BinHead); }
__host__ __device__ constexpr size_t bin_lut_offset(int nb)
{
    return (sizeof(BinHead) + sizeof(unsigned long long) * (size_t)(nb + 1 + kKeySentinels) + 15) / 16 * 16;
}
__host__ __device__ constexpr size_t bin_table_bytes(int nb)
{
    return bin_lut_offset(nb) + sizeof(unsigned short) * (size_t)kLutCells;
}

// Signed key: a < b as doubles  <=>  key(a) < key(b) for all non-NaN a, b.  Non-negative values keep their bit
// pattern; negative values have their 63 magnitude bits inverted (key = -1 - magnitude), three integer
// instructions on the two words.  That puts -0.0 at -1, just below +0.0 at 0, although the two compare equal as
// doubles; the table therefore stores an edge that is +-0.0 as -1 (edge_key), which makes
// "edge <= x" and "x < edge" come out as in IEEE for x = -0.0 and x = +0.0 alike.  Positive NaNs sort above
// +inf, negative NaNs below -inf: either way outside every bin.
__device__ __forceinline__ long long order_key(double v)
{
    const int hi = __double2hiint(v), lo = __double2loint(v);
    const int m = hi >> 31;                                  // all ones for a set sign bit
    return (long long)(((unsigned long long)(unsigned)(hi ^ (m & 0x7FFFFFFF)) << 32) | (unsigned)(lo ^ m));
}
__device__ __forceinline__ long long edge_key(double v)
{
    const long long k = order_key(v);
    return k == 0 ? -1ll : k;
}

// x = fl64(energy_scale * E_reco) (row a3b): one rounded fp64 multiply, never contracted into an fma.
__device__ __forceinline__ double scaled_energy(double energy_scale, double E_reco)
{
    return __dmul_rn(energy_scale, E_reco);
}

struct BinView {                       // 32-bit shared-window addresses into the shared-memory copy of the table
    uint32_t ekey;
    uint32_t lut;
    int base;
    unsigned int shift;
    int nb;
    unsigned int steps;                // forward steps that finish the search from lut[cell] (block-uniform)
    long long key0;                    // key(edges[0])
};

__device__ __forceinline__ BinView bin_view(const unsigned char* smem_table)
{
    const BinHead* h = reinterpret_cast<const BinHead*>(smem_table);
    BinView v;
    v.base = h->base;
    v.shift = h->shift;
    v.nb = (int)h->nb;
    v.steps = h->steps;
    v.ekey = smem_u32(smem_table + bin_keys_offset());
    v.lut = smem_u32(smem_table + bin_lut_offset(v.nb));
    v.key0 = *reinterpret_cast<const long long*>(smem_table + bin_keys_offset());
    return v;
}

// The unique i with edges[i] <= x < edges[i+1], or -1.  STEPS = 1: the caller has checked that t.steps <= 1 (one
// forward step finishes the search in every cell -- any sane binning); STEPS = 0: two branch-free steps and, if the
// table says that this is not enough, a loop.
template <int STEPS>
__device__ __forceinline__ int find_bin(const BinView& t, double x)
{
    const long long kx = order_key(x);
    const int khi = (int)(kx >> 32);
    const unsigned int rel = (unsigned int)max(khi, t.base) - (unsigned int)t.base;
    const unsigned int cell = min(rel >> t.shift, (unsigned int)(kLutCells - 1));
    int lo = (int)lds_u16(t.lut + 2u * cell);
    lo += ((long long)lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ? 1 : 0;       // sentinels keep these reads
    if (STEPS != 1) {                                                                 // inside the table
        lo += ((long long)lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ? 1 : 0;
        if (t.steps > 2u) {
            while (lo < t.nb && (long long)lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ++lo;
        }
    }
    return (lo < t.nb && t.key0 <= kx) ? lo : -1;
}

// The same search with the validity as a predicate instead of a -1 return value: `lo` is always a cell index that can
// be used in address arithmetic, the return value says whether x lies inside the binning.  Saves the select chain
// that the -1 convention forces on a caller which goes on to form an address.
template <int STEPS>
__device__ __forceinline__ bool find_bin_pred(const BinView& t, double x, int& lo_out)
{
    const long long kx = order_key(x);
    const int khi = (int)(kx >> 32);
    const unsigned int rel = (unsigned int)max(khi, t.base) - (unsigned int)t.base;
    const unsigned int cell = min(rel >> t.shift, (unsigned int)(kLutCells - 1));
    int lo = (int)lds_u16(t.lut + 2u * cell);
    lo += ((long long)lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ? 1 : 0;
    if (STEPS != 1) {
        lo += ((long long)lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ? 1 : 0;
        if (t.steps > 2u) {
            while (lo < t.nb && (long long)lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ++lo;
        }
    }
    lo_out = lo;
    return lo < t.nb && t.key0 <= kx;
}

// Builds the table for `edges` in shared memory.  Called by all threads of the block (it contains
// barriers); about 2 us per block, once per kernel.
__device__ __forceinline__ void build_bin_table(unsigned char* smem_table, const double* __restrict__ edges, int nb)
{
    long long* key = reinterpret_cast<long long*>(smem_table + bin_keys_offset());
    unsigned short* lut = reinterpret_cast<unsigned short*>(smem_table + bin_lut_offset(nb));
    BinHead* head = reinterpret_cast<BinHead*>(smem_table);

    for (int i = threadIdx.x; i < nb + 1 + kKeySentinels; i += blockDim.x)
        key[i] = (i <= nb) ? edge_key(__ldg(edges + i)) : kKeyMax;
    __syncthreads();
    if (threadIdx.x == 0) {
        const int lo = (int)(key[nb > 1 ? 1 : 0] >> 32);
        const int hi = (int)(key[nb] >> 32);
        const unsigned int span = hi > lo ? (unsigned int)hi - (unsigned int)lo : 0u;
        unsigned int shift = 0;
        while ((span >> shift) >= (unsigned int)kLutCells) ++shift;
        head->base = lo;
        head->shift = shift;
        head->nb = (unsigned int)nb;
        head->steps = 0u;
    }
    __syncthreads();
    const int base = head->base;
    const unsigned int shift = head->shift;
    for (int c = threadIdx.x; c < kLutCells; c += blockDim.x) {
        long long start_hi = (long long)base + ((long long)c << shift);                // first upper key word of cell c
        if (start_hi > 0x7FFFFFFFll) start_hi = 0x7FFFFFFFll;
        const long long start = start_hi * 4294967296ll;
        int lo = 0, hi = nb;                                   // largest i in [0, nb] with key[i] <= start, else 0
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (key[mid] <= start) lo = mid; else hi = mid - 1;
        }
        lut[c] = (unsigned short)(c == 0 ? 0 : lo);
    }
    __syncthreads();
    // forward steps needed from lut[c]: an x of cell c lies below the start of cell c + 1, so its bin is at
    // most lut[c + 1]; the last cell also takes everything above the last edge (walk ends at nb)
    unsigned int steps = 0;
    for (int c = threadIdx.x; c < kLutCells; c += blockDim.x) {
        const int nxt = (c + 1 < kLutCells) ? (int)lut[c + 1] : nb;
        steps = max(steps, (unsigned int)(nxt - (int)lut[c]));
    }
    steps = __reduce_max_sync(0xffffffffu, steps);
    if ((threadIdx.x & 31) == 0) atomicMax(&head->steps, steps);
    __syncthreads();
}

// The table of a call in shared memory, taken from a cache in global memory when that cache was built from the same
// edges.  `cache` is an image of a table (bin_table_bytes(nb) bytes, 16-byte aligned; all zero when nothing has been
// cached yet) that the library keeps per (device, stream): calls on a stream are ordered, the last block of a kernel
// that had to build the table writes it back (store_bin_table), and a fitter that rebuilds its PDF a million times with
// the same binning pays one L2 read and one comparison of the edge keys per block instead of the build.  The cache is
// validated against the caller's edges in every block -- same number of bins and bit-identical keys of all edges, which
// determine the rest of the table -- so a stale image is never used.  `fresh` is shared-memory scratch for nb + 1 keys
// (the caller's still unused histogram area).  Called by all threads of the block; ends with a barrier; returns
// (block-uniform) whether the cache was valid.
__device__ __forceinline__ bool load_or_build_bin_table(unsigned char* smem_table, long long* fresh,
                                                        const unsigned char* __restrict__ cache,
                                                        const double* __restrict__ edges, int nb)
{
    for (int i = threadIdx.x; i <= nb; i += blockDim.x) fresh[i] = edge_key(__ldg(edges + i));
    const int bytes = (int)bin_table_bytes(nb);
    for (int o = (int)threadIdx.x * 16; o < bytes; o += (int)blockDim.x * 16)
        *reinterpret_cast<int4*>(smem_table + o) = __ldcg(reinterpret_cast<const int4*>(cache + o));
    __syncthreads();
    const BinHead* h = reinterpret_cast<const BinHead*>(smem_table);
    const long long* key = reinterpret_cast<const long long*>(smem_table + bin_keys_offset());
    int ok = h->nb == (unsigned int)nb;
    if (ok)
        for (int i = threadIdx.x; i <= nb; i += blockDim.x) ok &= key[i] == fresh[i];
    ok = __syncthreads_and(ok);
    if (!ok) build_bin_table(smem_table, edges, nb);
    return ok != 0;
}

__device__ __forceinline__ void store_bin_table(const unsigned char* smem_table, unsigned char* __restrict__ cache, int nb)
{
    const int bytes = (int)bin_table_bytes(nb);
    for (int o = (int)threadIdx.x * 16; o < bytes; o += (int)blockDim.x * 16)
        *reinterpret_cast<int4*>(cache + o) = *reinterpret_cast<const int4*>(smem_table + o);
}

} // namespace oscb
