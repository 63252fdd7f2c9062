// osc_host.cuh -- device side of the *_host entry points (include/osc.h): the events of a host call cross PCIe in
// chunks and the fused kernel runs on chunk c while chunk c + 1 is still on the bus; every chunk leaves its own set of
// histograms, which this kernel adds in chunk order (a fixed order: the result is a deterministic function of the inputs).
#pragma once
#include <cuda_runtime.h>

namespace oscb {

// out[i] = chunk[0][i] + chunk[1][i] + ... (n_chunks sets of `count` values, contiguous)
__global__ void __launch_bounds__(256)
chunk_sum_kernel(const double* __restrict__ chunks, int n_chunks, size_t count, double* __restrict__ out)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    double s = chunks[i];
    for (int c = 1; c < n_chunks; ++c) s += chunks[(size_t)c * count + i];
    out[i] = s;
}

} // namespace oscb
