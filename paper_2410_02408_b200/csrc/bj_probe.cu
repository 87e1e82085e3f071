// Machine probe behind the roofline of the SpMV on matrices with RANDOM column structure (config 3):
// that kernel is not HBM-bound.  Every entry costs one 8-byte gather from the (L2-resident) vector, an L1
// wavefront of its own, while the matrix itself streams in through the TMA engine; the two share the
// SM <-> L2 path.  bj_probe_gather_stream measures, on the device it runs on, the time of
//   (a) `gathers` random 8-byte loads from a vector of `vec_len` doubles, all SMs, 8 loads in flight per lane,
//   (b) `stream_bytes` moved HBM -> shared memory by 1-D bulk async copies (nobody reads the data),
//   (c) both at once in the same kernel (gather warps + one producer thread per CTA),
// so that the SpMV's duration can be put against (c) -- the envelope of the hardware for that mix -- rather than
// against an HBM peak it cannot reach.  Diagnostic only: nothing on the operator path calls it.
#include <stdint.h>

#include <algorithm>

#include "bj_device.cuh"
#include "bj_internal.cuh"

namespace bj {
namespace {

constexpr int kProbeStages = 4;
constexpr int kProbeChunk = 16384;
constexpr int kProbeGatherWarps = 16;
constexpr int kProbeUnroll = 8;

__device__ __forceinline__ uint32_t probe_hash(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}

__global__ void __launch_bounds__((kProbeGatherWarps + 1) * 32)
probe_mix_kernel(const double* __restrict__ x, uint32_t vec_len, int gather_iters, const unsigned char* __restrict__ big,
                 size_t bytes_per_cta, double* sink)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kProbeStages; ++s) mbar_init(&bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    double acc = 0.0;
    if (warp < kProbeGatherWarps) {
        uint32_t s = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
        for (int it = 0; it < gather_iters; ++it) {
            uint32_t idx[kProbeUnroll];
            double v[kProbeUnroll];
#pragma unroll
            for (int k = 0; k < kProbeUnroll; ++k) { s = probe_hash(s + k + 1); idx[k] = __umulhi(s, vec_len); }
#pragma unroll
            for (int k = 0; k < kProbeUnroll; ++k) v[k] = __ldg(x + idx[k]);
#pragma unroll
            for (int k = 0; k < kProbeUnroll; ++k) acc += v[k];
        }
    } else if (lane == 0) {
        const unsigned char* src = big + (size_t)blockIdx.x * bytes_per_cta;
        const size_t nchunks = bytes_per_cta / kProbeChunk;
        const uint64_t pol = policy_evict_first();
        for (size_t c = 0; c < nchunks; ++c) {
            const int s = (int)(c % kProbeStages);
            if (c >= (size_t)kProbeStages) mbar_wait(&bar[s], (uint32_t)(((c / kProbeStages) - 1) & 1));
            mbar_expect_tx(&bar[s], kProbeChunk);
            bulk_g2s(smem + 128 + (size_t)s * kProbeChunk, src + c * kProbeChunk, kProbeChunk, &bar[s], pol);
        }
        for (size_t c = nchunks > (size_t)kProbeStages ? nchunks - kProbeStages : 0; c < nchunks; ++c)
            mbar_wait(&bar[c % kProbeStages], (uint32_t)((c / kProbeStages) & 1));  // copies must land before exit
    }
    if (acc == 1.2345) sink[0] = acc;
}

}  // namespace
}  // namespace bj

using namespace bj;

extern "C" int bj_probe_gather_stream(int64_t vec_len, int64_t gathers, int64_t stream_bytes, double* us_gather_host,
                                      double* us_stream_host, double* us_both_host)
{
    if (vec_len < 1 || vec_len >= (1ll << 31) || gathers < 0 || stream_bytes < 0 || !us_gather_host || !us_stream_host || !us_both_host)
        return BJ_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    BJ_CUDA(cudaGetDevice(&dev));
    BJ_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t per_cta = ((size_t)stream_bytes / sms / kProbeChunk) * kProbeChunk;
    const int iters = (int)std::min<int64_t>(1 << 30, gathers / ((int64_t)sms * kProbeGatherWarps * 32 * kProbeUnroll));
    double* x = nullptr;
    unsigned char* big = nullptr;
    double* sink = nullptr;
    const size_t big_bytes = std::max<size_t>(per_cta * sms, 16);
    if (cudaMalloc((void**)&x, (size_t)vec_len * 8) != cudaSuccess || cudaMalloc((void**)&big, big_bytes) != cudaSuccess ||
        cudaMalloc((void**)&sink, 8) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(x); cudaFree(big); cudaFree(sink);
        return BJ_ERR_ALLOC;
    }
    cudaMemset(x, 0, (size_t)vec_len * 8);
    cudaMemset(big, 0, big_bytes);
    const size_t smem = 128 + (size_t)kProbeStages * kProbeChunk;
    cudaFuncSetAttribute(probe_mix_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double* outs[3] = {us_gather_host, us_stream_host, us_both_host};
    int rc = BJ_OK;
    for (int combo = 0; combo < 3 && rc == BJ_OK; ++combo) {
        const int gi = combo == 1 ? 0 : iters;
        const size_t sb = combo == 0 ? 0 : per_cta;
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {  // first repetition warms up
            cudaEventRecord(e0);
            probe_mix_kernel<<<sms, (kProbeGatherWarps + 1) * 32, smem>>>(x, (uint32_t)vec_len, gi, big, sb, sink);
            cudaEventRecord(e1);
            cudaError_t e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) { set_cuda_error(e, "probe_mix_kernel"); rc = BJ_ERR_CUDA; break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0) best = std::min(best, ms);
        }
        *outs[combo] = 1e3 * (double)best;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(x); cudaFree(big); cudaFree(sink);
    return rc;
}
