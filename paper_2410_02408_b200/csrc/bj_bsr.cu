// 3x3-blocked storage of the matrix (opt-in with bj_setup_opts_t.bsr).
//
// A system with three unknowns per node (config 5: 3 dofs per node, 27-point node stencil) has a CSR whose rows come in
// triples with identical column patterns made of dense 3-column groups.  Stored as BSR(3) a block costs 72 bytes of
// values + ONE 4-byte block column instead of nine (value, column) pairs: 8.44 bytes per entry instead of 12.  This
// moves FEWER bytes than the CSR count of SURVEY.md 8(d) and carries its own byte accounting:
//   SpMV = 8 nnz + 4 nnz/9 + 4 (N/3 + 1) + 16 N     instead of     12 nnz + 4 (N+1) + 16 N.
// The handle owns the BSR copy (the caller's CSR stays the reference for setup); products are summed per row in
// block order by a shuffle tree, i.e. in a different order from the oracle's left-to-right row sum (rounding level).
#include <stdint.h>

#include <algorithm>

#include "bj_device.cuh"
#include "bj_internal.cuh"

namespace bj {

namespace {

// flag[0] |= 1 if block row I is not made of dense 3x3 blocks with a common pattern; warp per block row
__global__ void __launch_bounds__(256)
bsr_check_kernel(int64_t nbrows, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci, int* __restrict__ flag)
{
    const int64_t I = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (I >= nbrows) return;
    const int s0 = rp[3 * I], s1 = rp[3 * I + 1], s2 = rp[3 * I + 2], s3 = rp[3 * I + 3];
    const int len = s1 - s0;
    bool bad = (s2 - s1 != len) || (s3 - s2 != len) || (len % 3 != 0) || (s0 % 9 != 0);
    if (!bad) {
        for (int p = lane; p < len; p += 32) {
            const int c0 = ci[s0 + p];
            const int q = p / 3, c = p - 3 * q;
            const int head = ci[s0 + 3 * q];
            if (ci[s1 + p] != c0 || ci[s2 + p] != c0 || head % 3 != 0 || c0 != head + c) bad = true;
        }
    }
    if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(flag, 1);
}

// CSR -> BSR(3): brp[I] = rp[3I] / 9, bcol[brp[I] + q] = ci[rp[3I] + 3q] / 3, bval[(brp[I] + q) 9 + 3 r + c] = val[rp[3I + r] + 3q + c]
// (each block's nine values contiguous, row-major).  Warp per scalar row
__global__ void __launch_bounds__(256)
bsr_convert_kernel(int64_t n, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci, const double* __restrict__ val,
                   int32_t* __restrict__ brp, int32_t* __restrict__ bcol, double* __restrict__ bval)
{
    const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (i >= n) return;
    const int64_t I = i / 3;
    const int r = (int)(i - 3 * I);
    const int s = rp[i], len = rp[i + 1] - s;
    const int64_t b0 = rp[3 * I] / 9;
    if (r == 0 && lane == 0) {
        brp[I] = (int32_t)b0;
        if (i + 3 == n) brp[I + 1] = rp[n] / 9;
    }
    for (int p = lane; p < len; p += 32) {
        const int q = p / 3, c = p - 3 * q;
        bval[(b0 + q) * 9 + 3 * r + c] = val[s + p];
        if (r == 0 && c == 0) bcol[b0 + q] = ci[s + p] / 3;
    }
}

// y = A x from the BSR(3) copy: the persistent, TMA-streamed design of spmv_stream_kernel (bj_spmv_kernels.cu) with a
// block as the unit.  A tile is R consecutive block rows; its values (72 bytes per block), block columns and block-row
// pointers are each ONE contiguous byte range, moved by an elected producer thread with 1-D bulk async copies into a
// shared-memory ring (mbarrier transaction counts; ranges widened to whole quads of blocks, the <= 3 trailing blocks of
// the arrays copied by hand).  Each consumer warp takes block rows of the tile round-robin: lane = (block q, column c) for
// ten blocks at a time reads x[3 J_q + c] once (the three lanes of a block read consecutive addresses: one L1 wavefront
// per block) and the three values of column c of its block out of shared memory; no integer divisions, no selects; the
// three row sums are reduced over the warp.
struct BsrParams {
    int64_t nbrows, nblk, ntiles;
    const int32_t* brp;
    const int32_t* bcol;
    const double* bval;
    const double* x;
    double* y;
    int R, cap, stages, stage_bytes;
};

constexpr int kBsrConsumerWarps = 8;

__global__ void __launch_bounds__(32 + 32 * kBsrConsumerWarps)
spmv_bsr3_kernel(const BsrParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);
    uint64_t* empty = full + p.stages;
    unsigned char* stage0 = smem_raw + 128;
    // per stage: val[cap * 9] | col[cap] | rp[R + 4]
    auto s_val = [&](int s) { return reinterpret_cast<double*>(stage0 + (size_t)s * p.stage_bytes); };
    auto s_col = [&](int s) { return reinterpret_cast<int*>(stage0 + (size_t)s * p.stage_bytes + (size_t)p.cap * 72); };
    auto s_rp = [&](int s) { return reinterpret_cast<int*>(stage0 + (size_t)s * p.stage_bytes + (size_t)p.cap * 76); };
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < p.stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kBsrConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int R = p.R;
    if (warp == 0) {
        if (lane == 0) {
            const uint64_t pol = policy_evict_first();
            const int nblk4 = (int)(p.nblk & ~3ll);
            int it = 0;
            for (int64_t tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x, ++it) {
                const int s = it % p.stages;
                const uint32_t ph = (uint32_t)((it / p.stages) & 1);
                mbar_wait(&empty[s], ph ^ 1u);
                const int64_t r0 = tile * R;
                const int rows = (int)(r0 + R <= p.nbrows ? R : p.nbrows - r0);
                const int p0 = __ldg(p.brp + r0), p1 = __ldg(p.brp + r0 + rows);
                const int a0 = p0 & ~3;
                int a1 = (p1 + 3) & ~3;
                if (a1 > nblk4) a1 = nblk4;
                if (a1 < a0) a1 = a0;
                double* dv = s_val(s);
                int* dc = s_col(s);
                int* dr = s_rp(s);
                for (int q = (a1 > p0 ? a1 : p0); q < p1; ++q) {  // blocks past the last whole quad of the arrays
                    for (int e = 0; e < 9; ++e) dv[(q - a0) * 9 + e] = p.bval[(int64_t)q * 9 + e];
                    dc[q - a0] = p.bcol[q];
                }
                const int64_t np1 = p.nbrows + 1;
                const int want = rows + 1;
                int rq = (want + 3) & ~3;
                if (r0 + rq > np1) rq = (int)((np1 - r0) & ~3ll);
                for (int q = rq; q < want; ++q) dr[q] = p.brp[r0 + q];
                const uint32_t bytes = (uint32_t)(a1 - a0) * 76u + (uint32_t)rq * 4u;
                mbar_expect_tx(&full[s], bytes);
                if (a1 > a0) {
                    bulk_g2s(dv, p.bval + (int64_t)a0 * 9, (uint32_t)(a1 - a0) * 72u, &full[s], pol);
                    bulk_g2s(dc, p.bcol + a0, (uint32_t)(a1 - a0) * 4u, &full[s], pol);
                }
                if (rq > 0) bulk_g2s(dr, p.brp + r0, (uint32_t)rq * 4u, &full[s], pol);
            }
        }
    } else {
        const int cw = warp - 1;
        const int q0 = lane / 3, c = lane - 3 * q0;
        const bool lane_ok = lane < 30;
        pdl_wait();  // x may come from the previous kernel; the producer streams only setup-time constants
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x, ++it) {
            const int s = it % p.stages;
            const uint32_t ph = (uint32_t)((it / p.stages) & 1);
            const int64_t r0 = tile * R;
            const int rows = (int)(r0 + R <= p.nbrows ? R : p.nbrows - r0);
            mbar_wait(&full[s], ph);
            const double* sv = s_val(s);
            const int* sc = s_col(s);
            const int* sr = s_rp(s);
            const int a0 = sr[0] & ~3;
            for (int i = cw; i < rows; i += kBsrConsumerWarps) {
                const int b0 = sr[i] - a0, nb = sr[i + 1] - sr[i];
                double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0;
                for (int qb = 0; qb < nb; qb += 30) {  // three groups of ten blocks: their gathers are in flight together
                    double xv[3];
                    int qq[3];
#pragma unroll
                    for (int u = 0; u < 3; ++u) {
                        const int q = qb + 10 * u + q0;
                        const bool live = lane_ok && q < nb;
                        qq[u] = live ? b0 + q : -1;
                        xv[u] = live ? __ldg(p.x + 3 * (int64_t)sc[b0 + q] + c) : 0.0;
                    }
#pragma unroll
                    for (int u = 0; u < 3; ++u) {
                        if (qq[u] >= 0) {
                            const double* blk = sv + qq[u] * 9 + c;
                            acc0 = fma(blk[0], xv[u], acc0);
                            acc1 = fma(blk[3], xv[u], acc1);
                            acc2 = fma(blk[6], xv[u], acc2);
                        }
                    }
                }
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) {
                    acc0 += __shfl_down_sync(0xffffffffu, acc0, off);
                    acc1 += __shfl_down_sync(0xffffffffu, acc1, off);
                    acc2 += __shfl_down_sync(0xffffffffu, acc2, off);
                }
                if (lane == 0) {
                    double* yy = p.y + 3 * (r0 + i);
                    yy[0] = acc0; yy[1] = acc1; yy[2] = acc2;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }
    }
}

}  // namespace

void bsr_free(bj_handle_s* h)
{
    if (h->bsr_val) h->workspace_bytes -= h->bsr_bytes;
    cudaFree(h->bsr_val);
    cudaFree(h->bsr_col);
    cudaFree(h->bsr_rp);
    h->bsr_val = nullptr; h->bsr_col = nullptr; h->bsr_rp = nullptr;
    h->bsr_ok = false;
    h->bsr_bytes = 0;
}

// Called by bj_setup when opts.bsr is set: checks the structure, builds the copy.  Leaves bsr_ok false (no error) when the
// matrix is not 3x3-blocked.  Synchronises once.
int bsr_build(bj_handle_s* h)
{
    h->bsr_ok = false;
    if (h->n % 3 != 0 || h->nnz % 9 != 0 || h->nnz == 0) return BJ_OK;
    const int64_t nbrows = h->n / 3, nblocks = h->nnz / 9;
    int* flag = &h->status->pad;  // a spare int of the device status word
    BJ_CUDA(cudaMemsetAsync(flag, 0, sizeof(int), h->stream));
    const unsigned gb = (unsigned)((nbrows * 32 + 255) / 256);
    bsr_check_kernel<<<gb, 256, 0, h->stream>>>(nbrows, h->row_ptr, h->col_idx, flag);
    h->launches++;
    int bad = 1;
    BJ_CUDA(cudaMemcpyAsync(&bad, flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    BJ_CUDA(cudaStreamSynchronize(h->stream));
    if (bad) return BJ_OK;
    if (cudaMalloc((void**)&h->bsr_val, (size_t)h->nnz * sizeof(double)) != cudaSuccess ||
        cudaMalloc((void**)&h->bsr_col, (size_t)nblocks * sizeof(int32_t)) != cudaSuccess ||
        cudaMalloc((void**)&h->bsr_rp, (size_t)(nbrows + 1) * sizeof(int32_t)) != cudaSuccess) {
        cudaGetLastError();
        bsr_free(h);
        return BJ_ERR_ALLOC;
    }
    h->bsr_bytes = (int64_t)h->nnz * 8 + nblocks * 4 + (nbrows + 1) * 4;
    h->workspace_bytes += h->bsr_bytes;
    const unsigned gr = (unsigned)((h->n * 32 + 255) / 256);
    bsr_convert_kernel<<<gr, 256, 0, h->stream>>>(h->n, h->row_ptr, h->col_idx, h->val, h->bsr_rp, h->bsr_col, h->bsr_val);
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    // tile geometry of the streamed kernel: about 512 blocks (38 KB) per stage (measured best on config 5), bounded by the longest block row
    const int max_nb = std::max(1, h->bsr_max_row_nnz / 3);
    int R = std::max(1, std::min(64, env_int("BJ_BSR_TILE_BLOCKS", 512) / max_nb));
    R = std::max(4, R & ~3);  // tile starts must be multiples of four block rows: 16-byte aligned row-pointer copies
    h->bsr_tile_rows = R;
    h->bsr_tile_cap = ((R * max_nb + 8) + 3) & ~3;
    if (128 + 2 * ((size_t)h->bsr_tile_cap * 76 + (R + 4) * 4 + 16) > 220 * 1024) { bsr_free(h); return BJ_OK; }  // rows too long to stage
    h->bsr_ok = true;
    return BJ_OK;
}

int launch_spmv_bsr(bj_handle_s* h, const double* x, double* y)
{
    if (!h->bsr_ok) return BJ_ERR_INVALID_ARG;
    BsrParams p;
    p.nbrows = h->n / 3; p.nblk = h->nnz / 9;
    p.brp = h->bsr_rp; p.bcol = h->bsr_col; p.bval = h->bsr_val; p.x = x; p.y = y;
    p.R = h->bsr_tile_rows; p.cap = h->bsr_tile_cap; p.stages = 2;
    p.ntiles = (p.nbrows + p.R - 1) / p.R;
    p.stage_bytes = (p.cap * 76 + (p.R + 4) * 4 + 15) & ~15;
    const size_t smem = 128 + (size_t)p.stages * p.stage_bytes;
    const int threads = 32 + 32 * kBsrConsumerWarps;
    static std::atomic<bool> configured[64];
    {
        cudaError_t e = ensure_big_smem(spmv_bsr3_kernel, configured);
        if (e != cudaSuccess) { set_cuda_error(e, "cudaFuncSetAttribute(spmv_bsr3_kernel)"); return BJ_ERR_CUDA; }
    }
    int occ = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, spmv_bsr3_kernel, threads, smem);
    const int per_sm = std::max(1, std::min(occ, h->tune.ctas_per_sm));
    const int grid = (int)std::min<int64_t>(p.ntiles, (int64_t)h->num_sms * per_sm);
    KernelScope scope(h, BJ_K_SPMV);
    cudaError_t e = launch_kernel(spmv_bsr3_kernel, grid, threads, smem, h->stream, h->pdl && !h->prof_on, p);
    if (e != cudaSuccess) { set_cuda_error(e, "spmv_bsr3_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}

}  // namespace bj
