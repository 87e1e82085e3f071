// Setup kernels: CSR validation (a1), diagonal-block extraction (a2, PAPER.md:76-82 and the
// listing at 191-197) and batched Cholesky (a3; b = 1 is the paper's kernel at PAPER.md:214-235
// in split form).  One warp owns one block: the block's CSR range is contiguous, so the warp
// streams its column indices with coalesced loads, drops in-block entries into a dense tile in
// shared memory, factors it there and writes the layouts the solve kernels want.
#include <algorithm>

#include "bj_device.cuh"
#include "bj_internal.cuh"

namespace bj {

// ------------------------------------------------------------------------------------------------
// a1, two coalesced passes, no per-entry search and almost no atomics.
//   entries pass : grid-stride over the entries -- 0 <= col < n; counts the DESCENTS col[p] <= col[p-1].
//   rows pass    : one thread per row -- row_ptr monotone, starts at 0, ends at nnz; longest row; counts the
//                  descents that sit at the start of a non-empty row (the only legal ones).
//   Columns are strictly increasing inside every row  <=>  both counts agree (checked on the host).
//   Every 8th CTA of the rows pass also gathers the column-coherence statistic that steers the SpMV shape.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
validate_rows_kernel(int64_t n, int64_t nnz, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci,
                     Status* st)
{
    __shared__ unsigned sh[3][8];
    int flags = 0, len = 0;
    unsigned coh = 0, cmp = 0, legal = 0;
    // grid-stride over chunks of 256 rows: a few CTAs per SM, so that the same-address atomics at the end (which serialise
    // in L2) number a few thousand, not one set per 256 rows
    for (int64_t base = (int64_t)blockIdx.x * blockDim.x; base < n; base += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = base + threadIdx.x;
        if (i >= n) continue;
        const int64_t s = rp[i], e = rp[i + 1];
        if (s > e || s < 0 || e > nnz || (i == 0 && s != 0) || (i == n - 1 && e != nnz)) {
            flags |= ST_BAD_ROWPTR;
        } else {
            const int l = (int)(e - s);
            len = l > len ? l : len;
            if (l > 0 && s > 0) legal += ci[s] <= ci[s - 1];
            if (((base >> 8) & 7) == 0 && i + 1 < n) {  // every eighth chunk also gathers the column-coherence statistic
                const int64_t e2 = rp[i + 2];
                if (e2 >= e && e2 <= nnz) {
                    int64_t m = (e2 - e) < (e - s) ? (e2 - e) : (e - s);
                    if (m > 8) m = 8;  // a sample: the first entries of the two rows
                    for (int64_t q = 0; q < m; ++q) {
                        const int d = ci[e + q] - ci[s + q];
                        ++cmp;
                        coh += (d >= -16 && d <= 16);
                    }
                }
            }
        }
    }
    flags = __reduce_or_sync(0xffffffffu, flags);
    len = __reduce_max_sync(0xffffffffu, len);
    coh = __reduce_add_sync(0xffffffffu, coh);
    cmp = __reduce_add_sync(0xffffffffu, cmp);
    legal = __reduce_add_sync(0xffffffffu, legal);
    const int warp = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) {
        if (flags) atomicOr(&st->flags, flags);
        if (len > *(volatile int*)&st->max_row_nnz) atomicMax(&st->max_row_nnz, len);
        sh[0][warp] = coh; sh[1][warp] = cmp; sh[2][warp] = legal;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned a = 0, c = 0, l = 0;
        for (int w = 0; w < 8; ++w) { a += sh[0][w]; c += sh[1][w]; l += sh[2][w]; }
        if (c) { atomicAdd(&st->coherent, (unsigned long long)a); atomicAdd(&st->compared, (unsigned long long)c); }
        if (l) atomicAdd(&st->legal_descents, (unsigned long long)l);
    }
}

__global__ void __launch_bounds__(256)
validate_entries_kernel(int64_t n, int64_t nnz, const int32_t* __restrict__ ci, Status* st)
{
    __shared__ unsigned sh[8];
    int flags = 0;
    unsigned desc = 0;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < nnz; p += (int64_t)gridDim.x * blockDim.x) {
        const int c = ci[p];
        if (c < 0 || c >= n) flags |= ST_BAD_COL;
        if (p > 0) desc += (c <= ci[p - 1]);
    }
    flags = __reduce_or_sync(0xffffffffu, flags);
    desc = __reduce_add_sync(0xffffffffu, desc);
    if ((threadIdx.x & 31) == 0) {
        if (flags) atomicOr(&st->flags, flags);
        sh[threadIdx.x >> 5] = desc;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned d = 0;
        for (int w = 0; w < 8; ++w) d += sh[w];
        if (d) atomicAdd(&st->descents, (unsigned long long)d);
    }
}

int launch_validate(bj_handle_s* h)
{
    const int64_t blocks = std::min<int64_t>((h->n + 255) / 256, (int64_t)h->num_sms * 8);
    { SetupSpan span(h); validate_rows_kernel<<<(unsigned)blocks, 256, 0, h->stream>>>(h->n, h->nnz, h->row_ptr, h->col_idx, h->status); }
    h->launches++;
    if (h->nnz > 0) {
        const int64_t want = (h->nnz + 256 * 8 - 1) / (256 * 8);
        const unsigned eb = (unsigned)std::max<int64_t>(1, std::min<int64_t>(want, (int64_t)h->num_sms * 8));
        { SetupSpan span(h); validate_entries_kernel<<<eb, 256, 0, h->stream>>>(h->n, h->nnz, h->col_idx, h->status); }
        h->launches++;
    }
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

// ------------------------------------------------------------------------------------------------
// SpMV plan: nnz of the fullest tile of `tile_rows` consecutive rows
// ------------------------------------------------------------------------------------------------
__global__ void tile_nnz_kernel(int64_t n, int tile_rows, int64_t ntiles, const int32_t* __restrict__ rp, int* __restrict__ out)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int v = 0;
    if (t < ntiles) {
        int64_t r0 = t * tile_rows, r1 = r0 + tile_rows < n ? r0 + tile_rows : n;
        v = rp[r1] - rp[r0];
    }
    v = __reduce_max_sync(0xffffffffu, v);
    if ((threadIdx.x & 31) == 0) atomicMax(out, v);
}

int launch_spmv_plan(bj_handle_s* h, int tile_rows)
{
    if (tile_rows <= 0) return BJ_OK;
    const int64_t ntiles = (h->n + tile_rows - 1) / tile_rows;
    int64_t blocks = (ntiles + 255) / 256;
    SetupSpan span(h);
    tile_nnz_kernel<<<(unsigned)blocks, 256, 0, h->stream>>>(h->n, tile_rows, ntiles, h->row_ptr,
                                                              &h->status->max_tile_nnz);
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

// Output layouts of a2 + a3 (diagonal entries stored as RECIPROCALS so the solves multiply instead of divide):
//   b <= 8  fac_small[(k/32) * P * 32 + e * 32 + k % 32],  e = i(i+1)/2 + j  (row-major packed, 32 blocks interleaved)
//   b  > 8  fac_fwd[k * P + j*b - j(j-1)/2 + (i-j)] = l_ij / l_ii  (column-major packed lower, forward copy)
//           fac_bwd[k * P + i(i+1)/2 + j]           = l_ij / l_jj  (row-major packed lower; not kept for b = 16, 24, 32)
// Left-looking Cholesky in the textbook order; only the lower triangle is read; rows past the end of a ragged last
// block are identity rows.
// ------------------------------------------------------------------------------------------------
// a2 + a3 for b <= 8: one THREAD per diagonal block, the block in registers (compile-time B).
// A warp covers 32 consecutive blocks = 32 B consecutive rows, so its CSR reads stay inside one
// contiguous range (L1 absorbs the per-thread strides) and its interleaved factor writes are whole
// 256-byte lines.  Same left-looking Cholesky order as above.
// ------------------------------------------------------------------------------------------------
template <int B>
__global__ void __launch_bounds__(128)
extract_factor_small_kernel(int64_t n, int64_t nblocks, const int32_t* __restrict__ rp,
                            const int32_t* __restrict__ ci, const double* __restrict__ val,
                            double* __restrict__ fac, Status* st, int tri,
                            const int32_t* __restrict__ perm, const int32_t* __restrict__ pinv)  // both null: no permutation
{
    constexpr int P = B * (B + 1) / 2;
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nblocks) return;
    const int64_t lo = k * B;
    double d[P];  // packed lower triangle, e = i(i+1)/2 + j
#pragma unroll
    for (int e = 0; e < P; ++e) d[e] = 0.0;
    if (perm) {
        // permuted handle (reading 23): row lo + i of P A P^T is row perm[lo + i] of A, a column c sits at permuted
        // position pinv[c]; positions are not sorted along the row, so the whole row is scanned
#pragma unroll
        for (int i = 0; i < B; ++i) {
            if (lo + i < n) {
                const int row = perm[lo + i];
                const int e_ = rp[row + 1];
                for (int p = rp[row]; p < e_; ++p) {
                    const int64_t cp = pinv[ci[p]];
                    if (cp >= lo && cp <= lo + i) {
                        const double v = val[p];
                        const int j = (int)(cp - lo);
#pragma unroll
                        for (int jj = 0; jj < B; ++jj)
                            if (jj <= i && jj == j) d[i * (i + 1) / 2 + jj] = v;
                    }
                }
            } else {
                d[i * (i + 1) / 2 + i] = 1.0;
            }
        }
    } else {
#pragma unroll
    for (int i = 0; i < B; ++i) {
        const int64_t row = lo + i;
        if (row < n) {
            int s = rp[row];
            const int e_ = rp[row + 1];
            if (e_ - s > 16) {                 // long row: binary search for the first column >= lo
                int hi = e_;
                while (s < hi) {
                    const int mid = (s + hi) >> 1;
                    if (ci[mid] < lo) s = mid + 1; else hi = mid;
                }
            }
            for (int p = s; p < e_; ++p) {
                const int64_t c = ci[p];
                if (c > row) break;            // columns ascend: nothing of the lower triangle is left
                if (c >= lo) {
                    const double v = val[p];
                    const int j = (int)(c - lo);
#pragma unroll
                    for (int jj = 0; jj < B; ++jj)
                        if (jj <= i && jj == j) d[i * (i + 1) / 2 + jj] = v;
                }
            }
        } else {
            d[i * (i + 1) / 2 + i] = 1.0;      // identity rows pad a ragged last block
        }
    }
    }
    bool bad = false;
    double rinv[B];
    // every loop has the constant trip count B (triangular bounds as predicates): all of them unroll, d[] stays in registers
#pragma unroll
    for (int j = 0; j < B; ++j) {
        double sjj = d[j * (j + 1) / 2 + j];
#pragma unroll
        for (int p = 0; p < B; ++p)
            if (p < j) sjj -= d[j * (j + 1) / 2 + p] * d[j * (j + 1) / 2 + p];
        if (!(sjj > 0.0) || isinf(sjj)) { bad = true; sjj = 1.0; }
        const double ljj = sqrt(sjj);
        const double rjj = __drcp_rn(ljj);  // also the stored diagonal slot 1 / l_jj
        rinv[j] = rjj;
        d[j * (j + 1) / 2 + j] = ljj;
#pragma unroll
        for (int i = 0; i < B; ++i) {
            if (i > j) {
                double t = d[i * (i + 1) / 2 + j];
#pragma unroll
                for (int p = 0; p < B; ++p)
                    if (p < j) t -= d[i * (i + 1) / 2 + p] * d[j * (j + 1) / 2 + p];
                d[i * (i + 1) / 2 + j] = div_by(t, ljj, rjj);  // (the library division: ~55 instructions whenever a lane's t is 0)
            }
        }
    }
    if (bad) {
        atomicOr(&st->flags, ST_NOT_SPD);
        atomicMin(&st->bad_block, (long long)k);
    }
    if (tri) {
        // tridiagonal blocks (opts.band): the factor is bidiagonal, only the 2B - 1 elements (i, i-1), (i, i) are kept,
        // element (i, j) at slot i + j
        double* f = fac + (k >> 5) * (int64_t)((2 * B - 1) * kInterleave) + (k & 31);
#pragma unroll
        for (int i = 0; i < B; ++i) {
            if (i > 0) f[(2 * i - 1) * kInterleave] = d[i * (i + 1) / 2 + i - 1];
            f[(2 * i) * kInterleave] = rinv[i];
        }
        return;
    }
    double* f = fac + (k >> 5) * (int64_t)(P * kInterleave) + (k & 31);
#pragma unroll
    for (int i = 0; i < B; ++i)
#pragma unroll
        for (int j = 0; j <= i; ++j) {
            const double v = d[i * (i + 1) / 2 + j];
            f[(i * (i + 1) / 2 + j) * kInterleave] = (i == j) ? rinv[i] : v;
        }
}

// ------------------------------------------------------------------------------------------------
// a2 + a3 for b > 8: one SUB-WARP of W lanes per diagonal block, lane i owns row i IN REGISTERS.
//   extraction : each lane binary-searches its (sorted) row for the first column >= kb and copies the
//                entries up to the diagonal into its row of a small shared-memory tile;
//   Cholesky   : right-looking in registers -- column j: l_jj = sqrt(a_jj) (broadcast from lane j),
//                l_ij = a_ij / l_jj, then a_ik -= l_ij l_kj for k in (j, i] with column j passed between the
//                lanes through shared memory (broadcast loads).  Updates hit a_ik in the order j = 0, 1, ..:
//                the same subtraction order as the oracle's left-looking sum.
//   output     : both scaled packed copies, written with consecutive lanes on consecutive addresses.
// ------------------------------------------------------------------------------------------------
// BM: compile-time bound on the block size (b <= BM <= W): the unrolled loops of the factorisation run to BM with no
// runtime guard -- rows and columns b .. BM-1 are identity padding (l = 1, zeros), whose arithmetic is harmless.
// The factorisation is a dependent chain per column (shuffle, sqrt, reciprocal, store, barrier, loads, FMAs): resident warps
// hide it, so registers are capped for 4 / 5 / 6 CTAs per SM (measured best per variant; a few spilled bytes cost less).
template <int W, int BM>
__global__ void __launch_bounds__(128, BM == 32 ? 4 : (BM == 24 ? 5 : 6))
extract_factor_subwarp_kernel(int64_t n, int b, int64_t nblocks, const int32_t* __restrict__ rp,
                              const int32_t* __restrict__ ci, const double* __restrict__ val,
                              double* __restrict__ out0, double* __restrict__ out1, Status* st,
                              const int32_t* __restrict__ perm, const int32_t* __restrict__ pinv)  // both null: no permutation
{
    extern __shared__ __align__(16) double smem[];
    constexpr int LD = BM + 1;
    const int nsub = blockDim.x / W;
    const int sub = threadIdx.x / W;
    const int i = threadIdx.x & (W - 1);
    double* D = smem + (size_t)sub * (W * LD);
    int64_t k = (int64_t)blockIdx.x * nsub + sub;
    const bool act = k < nblocks;
    if (!act) k = nblocks - 1;  // redundant work, nothing written: the shuffles below need every lane
    const int64_t lo = k * b;
    const int64_t row = lo + i;
    const bool rowlive = i < b && row < n;

#pragma unroll
    for (int c = 0; c < BM; ++c) D[i * LD + c] = 0.0;
    if (!rowlive && i < BM) D[i * LD + i] = 1.0;  // identity rows pad ragged blocks and idle lanes
    if (rowlive && perm) {
        // permuted handle: row lo + i of P A P^T is row perm[lo + i] of A; the whole row is scanned, columns through pinv
        const int ro = perm[row];
        const int e = rp[ro + 1];
        for (int p = rp[ro]; p < e; ++p) {
            const int64_t cp = pinv[ci[p]];
            if (cp >= lo && cp <= row) D[i * LD + (int)(cp - lo)] = val[p];
        }
    } else if (rowlive) {
        int s = rp[row];
        const int e = rp[row + 1];
        int hi = e;
        while (s < hi) {  // first entry with column >= lo
            const int mid = (s + hi) >> 1;
            if (ci[mid] < lo) s = mid + 1; else hi = mid;
        }
        // entries up to the diagonal, eight loads in flight at a time
        for (int p = s; p < e; p += 8) {
            int cc[8];
            double vv[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) cc[q] = (p + q < e) ? ci[p + q] : 0x7fffffff;
#pragma unroll
            for (int q = 0; q < 8; ++q) vv[q] = (p + q < e && cc[q] <= row) ? val[p + q] : 0.0;
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (cc[q] <= row) D[i * LD + (int)(cc[q] - lo)] = vv[q];
            if (cc[7] > row) break;  // columns ascend: the lower triangle is done
        }
    }
    __syncwarp();
    double a[BM];
#pragma unroll
    for (int c = 0; c < BM; ++c) a[c] = D[i * LD + c];

    // Column j of L goes from the lanes to the lanes through shared memory (the tile D is free while the rows sit in
    // registers): every lane stores its l_ij, then all lanes read l_kj for k > j as BROADCAST 128-bit loads, two k per
    // instruction.  A shuffle per (j, k) pair -- b^2 / 2 64-bit shuffles = 1024 SHFL per 32 x 32 block -- made the kernel
    // shuffle-bound.  Two column buffers alternate: one __syncwarp per column.  The update a_ik -= l_ij l_kj runs on every
    // lane for every k > j: entries above the diagonal (k > i) collect garbage that nothing reads.
    __syncwarp();  // every lane has its row of D in registers
    const double2* Lc2 = reinterpret_cast<const double2*>(D);  // [2][W / 2]
    bool bad = false;
    double inv = 1.0;  // 1 / l_ii of this lane's row
#pragma unroll
    for (int j = 0; j < BM; ++j) {
        double ajj = __shfl_sync(0xffffffffu, a[j], j, W);
        if (!(ajj > 0.0) || isinf(ajj)) { bad = true; ajj = 1.0; }
        const double ljj = sqrt(ajj);
        const double rjj = __drcp_rn(ljj);
        const double lij = (i > j) ? div_by(a[j], ljj, rjj) : (i == j ? ljj : 0.0);
        if (i == j) inv = rjj;
        a[j] = lij;
        if (j + 1 < BM) {
            D[(j & 1) * W + i] = lij;
            __syncwarp();
#pragma unroll
            for (int pp = (j + 1) / 2; pp < BM / 2; ++pp) {
                const double2 t = Lc2[(j & 1) * (W / 2) + pp];
                if (2 * pp > j) a[2 * pp] = fma(-lij, t.x, a[2 * pp]);
                a[2 * pp + 1] = fma(-lij, t.y, a[2 * pp + 1]);
            }
        }
    }
    if (bad && act && i == 0) {
        atomicOr(&st->flags, ST_NOT_SPD);
        atomicMin(&st->bad_block, (long long)k);
    }
    const int P = b * (b + 1) / 2;
    // forward copy straight from the registers: column-major packed, row i scaled by 1 / l_ii, consecutive lanes on
    // consecutive addresses
    if (act && i < b) {
        double* o = out0 + k * P;
#pragma unroll
        for (int j = 0; j < BM; ++j)
            if (j < b && i >= j) o[(j * b - j * (j - 1) / 2) + (i - j)] = (i == j) ? inv : a[j] * inv;
    }
    // backward copy: row-major packed, column i scaled by 1 / l_ii (not kept when the solves use the forward copy for both):
    // through the tile, read transposed
    if (out1) {
        __syncwarp();  // the column buffers in D are dead
#pragma unroll
        for (int c = 0; c < BM; ++c) D[i * LD + c] = a[c];
        __syncwarp();
        if (act)
            for (int r = 0; r < b; ++r)
                if (i <= r) out1[k * P + r * (r + 1) / 2 + i] = (i == r) ? inv : D[r * LD + i] * inv;
    }
}

// ------------------------------------------------------------------------------------------------
// 16-bit column deltas (opt-in: bj_setup_opts_t.col16): col - row fits int16 for stencil matrices whose bandwidth
// is below 32768 (configs 2 and 4); the handle then owns a 2-byte-per-entry copy of the column stream.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
col16_check_kernel(int64_t n, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci, int* __restrict__ flag)
{
    const int64_t row = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 3;  // eight lanes per row
    const int sub = threadIdx.x & 7;
    bool bad = false;
    if (row < n) {
        const int e = rp[row + 1];
        for (int p = rp[row] + sub; p < e; p += 8) {
            const int64_t d = (int64_t)ci[p] - row;
            if (d < -32768 || d > 32767) bad = true;
        }
    }
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(flag, 1);
}

__global__ void __launch_bounds__(256)
col16_build_kernel(int64_t n, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci, int16_t* __restrict__ out)
{
    const int64_t row = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 3;
    const int sub = threadIdx.x & 7;
    if (row >= n) return;
    const int e = rp[row + 1];
    for (int p = rp[row] + sub; p < e; p += 8) out[p] = (int16_t)((int64_t)ci[p] - row);
}

void col16_free(bj_handle_s* h)
{
    if (h->col16) h->workspace_bytes -= (int64_t)h->nnz * 2;
    cudaFree(h->col16);
    h->col16 = nullptr;
}

// checks the bandwidth, builds the copy; leaves col16 null (no error) when a delta does not fit.  Synchronises once.
int col16_build(bj_handle_s* h)
{
    if (h->nnz == 0) return BJ_OK;
    int* flag = &h->status->pad;
    BJ_CUDA(cudaMemsetAsync(flag, 0, sizeof(int), h->stream));
    const unsigned grid = (unsigned)((h->n * 8 + 255) / 256);
    col16_check_kernel<<<grid, 256, 0, h->stream>>>(h->n, h->row_ptr, h->col_idx, flag);
    h->launches++;
    int bad = 1;
    BJ_CUDA(cudaMemcpyAsync(&bad, flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    BJ_CUDA(cudaStreamSynchronize(h->stream));
    if (bad) return BJ_OK;
    if (cudaMalloc((void**)&h->col16, (size_t)h->nnz * 2 + 16) != cudaSuccess) { cudaGetLastError(); h->col16 = nullptr; return BJ_ERR_ALLOC; }
    h->workspace_bytes += (int64_t)h->nnz * 2;
    col16_build_kernel<<<grid, 256, 0, h->stream>>>(h->n, h->row_ptr, h->col_idx, h->col16);
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

int launch_extract_factor(bj_handle_s* h)
{
    const int b = h->b;
    SetupSpan span(h);
    if (h->solve_kind == 1) {
        const unsigned tb = (unsigned)((h->nblocks + 127) / 128);
#define BJ_CASE(B)                                                                                          \
    case B:                                                                                                 \
        extract_factor_small_kernel<B><<<tb, 128, 0, h->stream>>>(h->n, h->nblocks, h->row_ptr, h->col_idx,  \
                                                                  h->val, h->fac_small, h->status,          \
                                                                  h->tri ? 1 : 0, h->var_perm, h->var_pinv); \
        break;
        switch (b) {
            BJ_CASE(1) BJ_CASE(2) BJ_CASE(3) BJ_CASE(4) BJ_CASE(5) BJ_CASE(6) BJ_CASE(7) BJ_CASE(8)
            default: return BJ_ERR_INVALID_ARG;
        }
#undef BJ_CASE
    } else {
        const int W = h->lanes;
        const int BM = W == 16 ? 16 : (b <= 24 ? 24 : 32);  // compile-time loop bound of the factorisation
        const int nsub = 128 / W;
        const size_t sm = (size_t)nsub * W * (BM + 1) * sizeof(double);
        const unsigned sb = (unsigned)((h->nblocks + nsub - 1) / nsub);
#define BJ_SUBWARP(WW, BB)                                                                                             \
    extract_factor_subwarp_kernel<WW, BB><<<sb, 128, sm, h->stream>>>(h->n, b, h->nblocks, h->row_ptr, h->col_idx, h->val, \
                                                                      h->fac_fwd, h->fac_bwd, h->status, h->var_perm, h->var_pinv)
        if (BM == 16) BJ_SUBWARP(16, 16);
        else if (BM == 24) BJ_SUBWARP(32, 24);
        else BJ_SUBWARP(32, 32);
#undef BJ_SUBWARP
    }
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

}  // namespace bj
