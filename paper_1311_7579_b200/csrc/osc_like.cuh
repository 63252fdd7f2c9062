// osc_like.cuh -- binned Poisson likelihood of the rebuilt PDFs against a data histogram.
//
// PAPER.md:125-128, eq. 2.1: L(o, f | D) = prod_i p(D_i | o, f) with p "the probability mass function" of the
// dataset; the toy fit compares the rebuilt PDF with a binned spectrum at every step of the Markov chain
// (PAPER.md:132).  Reading R5: p is the Poisson distribution of the bin content with mean
// mu_i = norm * hist_i, and what is returned is the likelihood ratio against the saturated model,
//
//     -2 ln lambda = 2 sum_i [ mu_i - D_i + D_i ln(D_i / mu_i) ]        (D_i ln(...) := 0 for D_i = 0),
//
// which differs from -2 ln L by a constant that does not depend on the oscillation parameters.  A bin with
// mu_i = 0 and D_i > 0 gives +inf; mu_i = 0 and D_i = 0 contributes 0.  Non-finite or negative inputs give NaN.
// With this call after osc_reweight_bin_batch only n_points doubles leave the device per scan.
#pragma once
#include <cuda_runtime.h>

namespace oscb {

__device__ __forceinline__ double poisson_term(double mu, double D)
{
    if (!(mu >= 0.0) || !(D >= 0.0) || isinf(mu) || isinf(D)) return __longlong_as_double(0x7FF8000000000000LL);
    if (mu == 0.0) return D == 0.0 ? 0.0 : __longlong_as_double(0x7FF0000000000000LL);
    if (D == 0.0) return mu;
    // D ln(D / mu) - (D - mu), with the logarithm taken of a ratio near 1 as log1p when the bin is close to its
    // expectation (no cancellation in the common case of a good fit)
    const double r = (D - mu) / mu;
    const double lg = fabs(r) < 0.5 ? log1p(r) : log(D / mu);
    return fma(D, lg, mu - D);
}

// One warp per point: lane l sums cells l, l + 32, ... in order, then a fixed xor-tree over the lanes.
__global__ void __launch_bounds__(256)
neg2lnl_kernel(const double* __restrict__ hist, int n_points, int n_cells, const double* __restrict__ data, double norm,
               double* __restrict__ out)
{
    const int p = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (p >= n_points) return;
    const unsigned lane = threadIdx.x & 31u;
    const double* h = hist + (size_t)p * n_cells;
    double s = 0.0;
    for (int i = lane; i < n_cells; i += 32) s += poisson_term(norm * h[i], data[i]);
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if (lane == 0) out[p] = 2.0 * s;
}

} // namespace oscb
