// Deterministic grid reductions shared by the Lanczos and PCG vector kernels: per-CTA partial sums in a
// fixed order, re-summed in the same fixed order by every CTA of the consuming kernel (no atomics, no
// separate finalize launch, bitwise reproducible run to run).
#pragma once

#include <stdint.h>

namespace bj {

// fixed-order block reduction: shuffle tree inside each warp, then warp 0 adds the warp sums in order
__device__ __forceinline__ double block_sum(double v, double* sh)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int q = 0; q < (int)(blockDim.x >> 5); ++q) s += sh[q];
    return s;  // valid on thread 0
}

struct Chunk {
    int64_t lo, hi;
};
__device__ __forceinline__ Chunk my_chunk(int64_t n)
{
    const int64_t per = (n + gridDim.x - 1) / gridDim.x;
    Chunk c;
    c.lo = (int64_t)blockIdx.x * per;
    c.hi = c.lo + per < n ? c.lo + per : n;
    if (c.lo > n) c.lo = n;
    return c;
}

// Every CTA of a consumer kernel re-sums the producer's per-CTA partials in the same fixed order, so all
// CTAs hold the identical scalar without a separate finalize launch (deterministic, no atomics).
__device__ __forceinline__ double reduce_partials(const double* __restrict__ part, int nparts, double* sh)
{
    double s = 0.0;
    for (int p = threadIdx.x; p < nparts; p += blockDim.x) s += part[p];
    s = block_sum(s, sh);
    __syncthreads();
    if (threadIdx.x == 0) sh[0] = s;
    __syncthreads();
    return sh[0];
}

}  // namespace bj
