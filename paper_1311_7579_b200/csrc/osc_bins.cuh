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
constexpr unsigned long long kKeyMax = 0xFFFFFFFFFFFFFFFFull;

struct BinHead {
    unsigned int base;   // upper key word where cell 0 starts
    unsigned int shift;  // cell = (upper key word - base) >> shift
    unsigned int nb;
    unsigned int steps;  // forward steps that finish the search from lut[cell], maximum over all cells
};

// Byte layout of the table in shared memory (all parts 16-byte aligned).
__host__ __device__ inline size_t bin_keys_offset() { return sizeof(BinHead); }
__host__ __device__ inline size_t bin_lut_offset(int nb)
{
    return (sizeof(BinHead) + sizeof(unsigned long long) * (size_t)(nb + 1 + kKeySentinels) + 15) / 16 * 16;
}
__host__ __device__ inline size_t bin_table_bytes(int nb)
{
    return bin_lut_offset(nb) + sizeof(unsigned short) * (size_t)kLutCells;
}

// Unsigned key: a < b as doubles  <=>  key(a) < key(b) for all non-NaN a, b, and key(-0.0) == key(+0.0).
// Non-negative values keep their bit pattern with the top bit set; negative values map to the two's
// complement of their bit pattern (2^63 - magnitude).  Positive NaNs sort above +inf, negative NaNs
// below -inf: either way outside every bin.
__device__ __forceinline__ unsigned long long order_key(double v)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return ((long long)b < 0) ? (0ull - b) : (b | 0x8000000000000000ull);
}

// x = fl64(energy_scale * E_reco) (row a3b): one rounded fp64 multiply, never contracted into an fma.
__device__ __forceinline__ double scaled_energy(double energy_scale, double E_reco)
{
    return __dmul_rn(energy_scale, E_reco);
}

struct BinView {                       // 32-bit shared-window addresses into the shared-memory copy of the table
    uint32_t ekey;
    uint32_t lut;
    unsigned int base, shift;
    int nb;
    bool two_steps;                    // two forward steps are enough for every cell
    unsigned long long key0;           // key(edges[0])
};

__device__ __forceinline__ BinView bin_view(const unsigned char* smem_table)
{
    const BinHead* h = reinterpret_cast<const BinHead*>(smem_table);
    BinView v;
    v.base = h->base;
    v.shift = h->shift;
    v.nb = (int)h->nb;
    v.two_steps = h->steps <= 2u;
    v.ekey = smem_u32(smem_table + bin_keys_offset());
    v.lut = smem_u32(smem_table + bin_lut_offset(v.nb));
    v.key0 = *reinterpret_cast<const unsigned long long*>(smem_table + bin_keys_offset());
    return v;
}

// The unique i with edges[i] <= x < edges[i+1], or -1.
__device__ __forceinline__ int find_bin(const BinView& t, double x)
{
    const unsigned long long kx = order_key(x);
    const unsigned int khi = (unsigned int)(kx >> 32);
    const unsigned int rel = max(khi, t.base) - t.base;
    const unsigned int cell = min(rel >> t.shift, (unsigned int)(kLutCells - 1));
    int lo = (int)lds_u16(t.lut + 2u * cell);
    lo += (lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ? 1 : 0;   // sentinels keep these reads inside the table
    lo += (lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ? 1 : 0;
    if (!t.two_steps) {                                               // uniform; not taken for sane binnings
        while (lo < t.nb && lds_u64(t.ekey + 8u * (unsigned)(lo + 1)) <= kx) ++lo;
    }
    return (lo < t.nb && t.key0 <= kx) ? lo : -1;
}

// Builds the table for `edges` in shared memory.  Called by all threads of the block (it contains
// barriers); about 2 us per block, once per kernel.
__device__ __forceinline__ void build_bin_table(unsigned char* smem_table, const double* __restrict__ edges, int nb)
{
    unsigned long long* key = reinterpret_cast<unsigned long long*>(smem_table + bin_keys_offset());
    unsigned short* lut = reinterpret_cast<unsigned short*>(smem_table + bin_lut_offset(nb));
    BinHead* head = reinterpret_cast<BinHead*>(smem_table);

    for (int i = threadIdx.x; i < nb + 1 + kKeySentinels; i += blockDim.x)
        key[i] = (i <= nb) ? order_key(__ldg(edges + i)) : kKeyMax;
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int lo = (unsigned int)(key[nb > 1 ? 1 : 0] >> 32);
        const unsigned int hi = (unsigned int)(key[nb] >> 32);
        const unsigned int span = hi > lo ? hi - lo : 0u;
        unsigned int shift = 0;
        while ((span >> shift) >= (unsigned int)kLutCells) ++shift;
        head->base = lo;
        head->shift = shift;
        head->nb = (unsigned int)nb;
        head->steps = 0u;
    }
    __syncthreads();
    const unsigned int base = head->base, shift = head->shift;
    for (int c = threadIdx.x; c < kLutCells; c += blockDim.x) {
        unsigned long long start_hi = (unsigned long long)base + ((unsigned long long)c << shift);
        if (start_hi > 0xFFFFFFFFull) start_hi = 0xFFFFFFFFull;
        const unsigned long long start = start_hi << 32;
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

} // namespace oscb
