// Setup kernels: CSR validation (a1), diagonal-block extraction (a2, PAPER.md:76-82 and the
// listing at 191-197) and batched Cholesky (a3; b = 1 is the paper's kernel at PAPER.md:214-235
// in split form).  One warp owns one block: the block's CSR range is contiguous, so the warp
// streams its column indices with coalesced loads, drops in-block entries into a dense tile in
// shared memory, factors it there and writes the layouts the solve kernels want.
#include "bj_internal.cuh"

namespace bj {

// ------------------------------------------------------------------------------------------------
// a1: one thread per row.  Also records the longest row (for the SpMV plan).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
validate_kernel(int64_t n, int64_t nnz, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci,
                Status* st)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int flags = 0;
    int len = 0;
    unsigned coh = 0, cmp = 0;
    if (i < n) {
        int64_t s = rp[i], e = rp[i + 1];
        if (s > e || s < 0 || e > nnz || (i == 0 && s != 0) || (i == n - 1 && e != nnz)) {
            flags |= ST_BAD_ROWPTR;
        } else {
            len = (int)(e - s);
            // next row, only if its pointers are sane (it validates itself): used for the coherence statistic
            int64_t s2 = 0, e2 = 0;
            if (i + 1 < n) { s2 = e; e2 = rp[i + 2]; if (e2 < s2 || e2 > nnz) e2 = s2; }
            int prev = -1;
            for (int64_t p = s; p < e; ++p) {
                int c = ci[p];
                if (c < 0 || c >= n) flags |= ST_BAD_COL;
                if (c <= prev) flags |= ST_UNSORTED;
                prev = c;
                if (s2 + (p - s) < e2) { ++cmp; const int d = ci[s2 + (p - s)] - c; coh += (d >= -16 && d <= 16); }
            }
        }
    }
    flags = __reduce_or_sync(0xffffffffu, flags);
    len = __reduce_max_sync(0xffffffffu, len);
    coh = __reduce_add_sync(0xffffffffu, coh);
    cmp = __reduce_add_sync(0xffffffffu, cmp);
    if ((threadIdx.x & 31) == 0) {
        if (flags) atomicOr(&st->flags, flags);
        atomicMax(&st->max_row_nnz, len);
        atomicAdd(&st->coherent, (unsigned long long)coh);
        atomicAdd(&st->compared, (unsigned long long)cmp);
    }
}

int launch_validate(bj_handle_s* h)
{
    int64_t blocks = (h->n + 255) / 256;
    validate_kernel<<<(unsigned)blocks, 256, 0, h->stream>>>(h->n, h->nnz, h->row_ptr, h->col_idx, h->status);
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

// ------------------------------------------------------------------------------------------------
// SpMV plan: nnz of the fullest tile of `tile_rows` consecutive rows
// ------------------------------------------------------------------------------------------------
__global__ void tile_nnz_kernel(int64_t n, int tile_rows, int64_t ntiles, const int32_t* __restrict__ rp, Status* st)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int v = 0;
    if (t < ntiles) {
        int64_t r0 = t * tile_rows, r1 = r0 + tile_rows < n ? r0 + tile_rows : n;
        v = rp[r1] - rp[r0];
    }
    v = __reduce_max_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0) atomicMax(&st->max_tile_nnz, v);
}

int launch_spmv_plan(bj_handle_s* h)
{
    if (h->ntiles <= 0) return BJ_OK;
    int64_t blocks = (h->ntiles + 255) / 256;
    tile_nnz_kernel<<<(unsigned)blocks, 256, 0, h->stream>>>(h->n, h->tile_rows, h->ntiles, h->row_ptr, h->status);
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

// ------------------------------------------------------------------------------------------------
// a2 + a3: one warp per diagonal block.
//   D  : dense b x b tile, leading dimension b+1, warp-private shared memory
//   rpl: the block's row pointers
// Left-looking Cholesky in the textbook order: for each column j, s_i = d_ij - sum_{p<j} l_ip l_jp
// for i >= j, l_jj = sqrt(s_j), l_ij = s_i / l_jj.  Only the lower triangle is read.
// Rows past the end of a ragged last block are treated as identity rows.
// Output layouts (diagonal entries stored as RECIPROCALS so the solves multiply instead of divide):
//   KIND 1 (b <= 8)  fac_small[(k/32) * P * 32 + e * 32 + k % 32],  e = i(i+1)/2 + j  (row-major packed)
//   KIND 2 (b  > 8)  fac_fwd[k * P + j*b - j(j-1)/2 + (i-j)] = l_ij / l_ii  (column-major packed lower, forward)
//                    fac_bwd[k * P + i(i+1)/2 + j]           = l_ij / l_jj  (row-major packed lower, backward)
// ------------------------------------------------------------------------------------------------
constexpr int kSetupWarps = 4;

template <int KIND>
__global__ void __launch_bounds__(kSetupWarps * 32)
extract_factor_kernel(int64_t n, int b, int64_t nblocks, const int32_t* __restrict__ rp,
                      const int32_t* __restrict__ ci, const double* __restrict__ val,
                      double* __restrict__ out0, double* __restrict__ out1, Status* st)
{
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int ld = b + 1;
    const int per_warp = b * ld + ((b + 2 + 1) / 2);  // D + rpl (ints packed into doubles)
    double* D = smem + (size_t)warp * per_warp;
    int* rpl = reinterpret_cast<int*>(D + b * ld);

    const int64_t k = (int64_t)blockIdx.x * kSetupWarps + warp;
    if (k >= nblocks) return;
    const int64_t lo = k * b;
    const int64_t hi = lo + b < n ? lo + b : n;
    const int nb = (int)(hi - lo);

    for (int e = lane; e < b * ld; e += 32) D[e] = 0.0;
    for (int i = lane; i <= nb; i += 32) rpl[i] = rp[lo + i];
    __syncwarp();
    for (int i = nb + lane; i < b; i += 32) D[i * ld + i] = 1.0;
    const int s = rpl[0], e_ = rpl[nb];
    for (int p = s + lane; p < e_; p += 32) {
        const int64_t c = ci[p];
        if (c >= lo && c < hi) {
            int i = 0;
            while (i + 1 < nb && rpl[i + 1] <= p) ++i;
            const int j = (int)(c - lo);
            if (j <= i) D[i * ld + j] = val[p];
        }
    }
    __syncwarp();

    bool bad = false;
    for (int j = 0; j < b; ++j) {
        for (int i = j + lane; i < b; i += 32) {
            double acc = D[i * ld + j];
            for (int p = 0; p < j; ++p) acc -= D[i * ld + p] * D[j * ld + p];
            D[i * ld + j] = acc;
        }
        __syncwarp();
        double sjj = D[j * ld + j];
        if (!(sjj > 0.0) || isinf(sjj)) { bad = true; sjj = 1.0; }
        const double ljj = sqrt(sjj);
        __syncwarp();
        for (int i = j + 1 + lane; i < b; i += 32) D[i * ld + j] = D[i * ld + j] / ljj;
        if (lane == 0) D[j * ld + j] = ljj;
        __syncwarp();
    }
    if (bad && lane == 0) {
        atomicOr(&st->flags, ST_NOT_SPD);
        atomicMin(&st->bad_block, (long long)k);
    }

    const int P = b * (b + 1) / 2;
    for (int idx = lane; idx < b * b; idx += 32) {
        const int i = idx / b, j = idx - i * b;
        if (j > i) continue;
        const double v = D[i * ld + j];
        if (KIND == 1) {
            out0[(k >> 5) * (int64_t)P * kInterleave + (int64_t)(i * (i + 1) / 2 + j) * kInterleave + (k & 31)] =
                (i == j) ? 1.0 / v : v;
        } else {
            // forward copy: row i scaled by 1/l_ii; backward copy: column j scaled by 1/l_jj
            out0[k * P + (j * b - j * (j - 1) / 2 + (i - j))] = (i == j) ? 1.0 / v : v / D[i * ld + i];
            out1[k * P + (i * (i + 1) / 2 + j)] = (i == j) ? 1.0 / v : v / D[j * ld + j];
        }
    }
}

int launch_extract_factor(bj_handle_s* h)
{
    const int b = h->b;
    const int per_warp = b * (b + 1) + ((b + 2 + 1) / 2);
    const size_t smem = (size_t)kSetupWarps * per_warp * sizeof(double);
    const int64_t blocks = (h->nblocks + kSetupWarps - 1) / kSetupWarps;
    if (h->solve_kind == 1) {
        extract_factor_kernel<1><<<(unsigned)blocks, kSetupWarps * 32, smem, h->stream>>>(
            h->n, b, h->nblocks, h->row_ptr, h->col_idx, h->val, h->fac_small, nullptr, h->status);
    } else {
        extract_factor_kernel<2><<<(unsigned)blocks, kSetupWarps * 32, smem, h->stream>>>(
            h->n, b, h->nblocks, h->row_ptr, h->col_idx, h->val, h->fac_fwd, h->fac_bwd, h->status);
    }
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

}  // namespace bj
