// CSR SpMV  u = A t  (a6), the dominant byte stream of the preconditioned operator (a7).
//
// Kernel 0  (spmv_vector_kernel): one sub-warp of LPR lanes per row; column/value loads of
//   consecutive rows are contiguous, so a warp's loads coalesce; partial sums are combined with
//   warp shuffles.  It needs no plan and no alignment, handles any row length, and is the
//   fall-back for matrices the streamed kernel cannot take.
// Kernel 1  (spmv_stream_kernel, below): persistent CTAs; a producer thread streams each tile's
//   contiguous col/val (and factor) ranges into a shared-memory ring with 1-D bulk async copies
//   (cp.async.bulk + mbarrier, i.e. the TMA engine: no registers staged, deep memory-level
//   parallelism), consumer warps reduce rows out of shared memory, gather t through L1/L2, and can
//   run the forward block solve y = L^-1 u on the tile before y is written (fuses a7's last factor).
#include "bj_internal.cuh"

namespace bj {

__device__ __forceinline__ double ldg_stream_f64(const double* p)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ int ldg_stream_s32(const int* p)
{
    int v;
    asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}

// ------------------------------------------------------------------------------------------------
// Kernel 0: LPR lanes per row
// ------------------------------------------------------------------------------------------------
template <int LPR>
__global__ void __launch_bounds__(256)
spmv_vector_kernel(int64_t n, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci,
                   const double* __restrict__ val, const double* __restrict__ x, double* __restrict__ y)
{
    const int64_t gtid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t row = gtid / LPR;
    const int lane = threadIdx.x & (LPR - 1);
    double acc = 0.0;
    if (row < n) {
        const int s = rp[row], e = rp[row + 1];
        for (int p = s + lane; p < e; p += LPR) {
            const int c = ldg_stream_s32(ci + p);
            const double v = ldg_stream_f64(val + p);
            acc = fma(v, __ldg(x + c), acc);
        }
    }
#pragma unroll
    for (int off = LPR / 2; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off, LPR);
    if (row < n && lane == 0) y[row] = acc;
}

int launch_spmv_vector(bj_handle_s* h, const double* x, double* y)
{
    const int threads = 256;
    const int lpr = h->spmv_lanes;
    const unsigned blocks = (unsigned)((h->n * lpr + threads - 1) / threads);
    KernelScope scope(h, BJ_K_SPMV);
#define BJ_CASE(L)                                                                                              \
    case L:                                                                                                     \
        spmv_vector_kernel<L><<<blocks, threads, 0, h->stream>>>(h->n, h->row_ptr, h->col_idx, h->val, x, y);  \
        break;
    switch (lpr) {
        BJ_CASE(1) BJ_CASE(2) BJ_CASE(4) BJ_CASE(8) BJ_CASE(16) BJ_CASE(32)
        default: return BJ_ERR_INVALID_ARG;
    }
#undef BJ_CASE
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

// ------------------------------------------------------------------------------------------------
// Kernel 1: placeholder until the streamed kernel lands (never selected while stream_ok is false)
// ------------------------------------------------------------------------------------------------
int spmv_stream_configure(bj_handle_s* h)
{
    h->stream_ok = false;
    h->fuse_ok = false;
    h->ntiles = 0;
    return BJ_OK;
}

int launch_spmv_stream(bj_handle_s*, const double*, double*, bool) { return BJ_ERR_INVALID_ARG; }

}  // namespace bj
