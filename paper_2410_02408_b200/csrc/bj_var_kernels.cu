// Variable-size Jacobi blocks ("variable-size / supervariable blocks").
// block_ptr[0..nblocks] delimits contiguous index ranges of 1..32 rows; block k is the dense diagonal slice
// D_k = A[p_k:p_{k+1}, p_k:p_{k+1}] (the listing of PAPER.md:191-197 with a per-block size), D_k = L_k L_k^T.
// Optional symmetric PERMUTATION ("a permutation argument (RCM or strong-coupling lines)"):
// perm[i] = original index of the unknown at permuted position i; the blocks are those of P A P^T,
// (P A P^T)[i, j] = A[perm[i], perm[j]], i.e. M = P^T blockdiag(D_k) P, and every vector stays in the ORIGINAL ordering:
// the extraction looks columns up through the inverse permutation, the solves gather their right-hand side through perm
// and scatter the result back through it.  No permuted copy of A is made; the SpMV runs on A as it is.
// Storage: the lower triangles, column-major packed, back to back: block k starts at foff[k] = sum_{q<k} s_q (s_q+1)/2,
// element (i, j), i >= j, at j s - j (j-1)/2 + (i - j); the diagonal slot holds 1 / l_jj.
// One warp per block in both kernels (lane = row): the block sizes differ, so neither the 32-block interleave of the
// b <= 8 kernels nor the fixed tile geometry of the group kernel applies; the packed factor of a block is one
// contiguous range that the warp copies to shared memory with coalesced loads before the substitutions.
#include <algorithm>
#include <vector>

#include "bj_device.cuh"
#include "bj_internal.cuh"

namespace bj {

namespace {

constexpr int kVarWarps = 4;
constexpr int kVarMax = 32;
constexpr int kVarPacked = kVarMax * (kVarMax + 1) / 2;  // 528

__device__ __forceinline__ int var_col_start(int j, int s) { return j * s - (j * (j - 1)) / 2; }

// a2-a4 for one block per warp: dense lower triangle out of the CSR rows, Cholesky (left-looking, column by column,
// each sum in increasing k like the oracle's chol_block), packed store.  A non-positive or non-finite pivot flags
// ST_NOT_SPD and records the smallest such block.
__global__ void __launch_bounds__(kVarWarps * 32)
extract_factor_var_kernel(int64_t nblocks, const int32_t* __restrict__ bptr, const int64_t* __restrict__ foff,
                          const int32_t* __restrict__ rp, const int32_t* __restrict__ ci, const double* __restrict__ val,
                          double* __restrict__ fac, Status* __restrict__ status,
                          const int32_t* __restrict__ perm, const int32_t* __restrict__ pinv)  // both null: no permutation
{
    __shared__ double Dsh[kVarWarps][kVarMax * (kVarMax + 1)];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t k = (int64_t)blockIdx.x * kVarWarps + warp;
    if (k >= nblocks) return;
    const int lo = bptr[k], s = bptr[k + 1] - lo;
    double* D = Dsh[warp];  // row i at D + i * 33
    if (lane < s) {
        for (int j = 0; j < s; ++j) D[lane * (kVarMax + 1) + j] = 0.0;
        const int row = perm ? perm[lo + lane] : lo + lane;
        for (int e = rp[row]; e < rp[row + 1]; ++e) {
            const int c = (pinv ? pinv[ci[e]] : ci[e]) - lo;  // position of the column in the permuted ordering
            if (c >= 0 && c <= lane) D[lane * (kVarMax + 1) + c] = val[e];  // lower triangle only
        }
    }
    __syncwarp();
    bool bad = false;
    for (int j = 0; j < s; ++j) {
        double sum = 0.0;
        if (lane >= j && lane < s) {
            sum = D[lane * (kVarMax + 1) + j];
            for (int q = 0; q < j; ++q) sum -= D[lane * (kVarMax + 1) + q] * D[j * (kVarMax + 1) + q];
        }
        const double piv = __shfl_sync(0xffffffffu, sum, j);
        if (!(piv > 0.0) || !isfinite(piv)) { bad = true; break; }  // uniform over the warp
        const double d = sqrt(piv);
        const double rd = __drcp_rn(d);  // sum / d below = one multiplication + a residual correction (div_by): the library
                                         // division takes its slow path for the whole warp whenever one lane's sum is 0
        __syncwarp();
        if (lane == j) D[lane * (kVarMax + 1) + j] = d;
        else if (lane > j && lane < s) D[lane * (kVarMax + 1) + j] = div_by(sum, d, rd);
        __syncwarp();
    }
    if (bad) {
        if (lane == 0) {
            atomicOr(&status->flags, ST_NOT_SPD);
            atomicMin(&status->bad_block, (long long)k);
        }
        return;
    }
    double* f = fac + foff[k];
    const int P = s * (s + 1) / 2;
    // packed index e -> (i, j): walk the columns; each lane converts its own indices
    for (int e = lane; e < P; e += 32) {
        int j = 0, start = 0;
        while (start + (s - j) <= e) { start += s - j; ++j; }
        const int i = j + (e - start);
        const double v = D[i * (kVarMax + 1) + j];
        f[e] = (i == j) ? 1.0 / v : v;
    }
}

// The substitutions of one block by one warp (lane = row, all 32 lanes call): F = packed factor in shared memory.
// The loops keep the packed index of this lane's entry as a running value (one add per step) and the lane's own
// reciprocal diagonal in a register.
template <int DIR>
__device__ __forceinline__ double var_block_solve(const double* F, int s, int lane, double v)
{
    const bool act = lane < s;
    const int csl = var_col_start(act ? lane : 0, s);
    const double dinv = F[csl];
    if (DIR == 0 || DIR == 2) {
        int idx = lane, stride = s - 1;                  // l_{lane,j} at cs(j) + lane - j; cs(j + 1) - cs(j) = s - j
#pragma unroll 4
        for (int j = 0; j < s; ++j) {
            if (lane == j) v *= dinv;
            const double yj = __shfl_sync(0xffffffffu, v, j);
            if (act && lane > j) v -= F[idx] * yj;
            idx += stride;
            --stride;
        }
    }
    if (DIR == 1 || DIR == 2) {
        int idb = csl + (s - 1 - lane);                  // l_{j,lane} at cs(lane) + j - lane, j = s - 1 first
#pragma unroll 4
        for (int j = s - 1; j >= 0; --j) {
            if (lane == j) v *= dinv;
            const double xj = __shfl_sync(0xffffffffu, v, j);
            if (lane < j) v -= F[idb] * xj;
            --idb;
        }
    }
    return v;
}

// DIR 0: y = L^-1 r, 1: x = L^-T y, 2: z = L^-T L^-1 r.  One warp per block, lane = row, factor in shared memory.
template <int DIR>
__global__ void __launch_bounds__(kVarWarps * 32)
solve_var_kernel(int64_t nblocks, const int32_t* __restrict__ bptr, const int64_t* __restrict__ foff,
                 const double* __restrict__ fac, const double* in, double* out, const int32_t* __restrict__ perm)
{
    __shared__ double Fsh[kVarWarps][kVarPacked];
    pdl_trigger();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t k = (int64_t)blockIdx.x * kVarWarps + warp;
    if (k >= nblocks) return;
    const int lo = bptr[k], s = bptr[k + 1] - lo;
    const double* f = fac + foff[k];
    double* F = Fsh[warp];
    const int P = s * (s + 1) / 2;
    for (int e = lane; e < P; e += 32) F[e] = ld_stream(f + e);  // factors never change after setup
    pdl_wait();                                                  // `in` may come from the previous kernel
    // row of this lane in the caller's (original) ordering: in == out stays safe, a lane reads and writes one index
    const int row = lane < s ? (perm ? perm[lo + lane] : lo + lane) : 0;
    double v = lane < s ? in[row] : 0.0;
    __syncwarp();
    v = var_block_solve<DIR>(F, s, lane, v);
    if (lane < s) out[row] = v;
}

// pinv[perm[i]] = i; flag[0] |= 1 when an entry is out of range or occurs twice (pinv is preset to -1)
__global__ void __launch_bounds__(256)
perm_invert_kernel(int64_t n, const int32_t* __restrict__ perm, int32_t* __restrict__ pinv, int* __restrict__ flag)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int p = perm[i];
    if (p < 0 || p >= n) { atomicOr(flag, 1); return; }
    if (atomicExch(&pinv[p], (int)i) != -1) atomicOr(flag, 1);
}

}  // namespace

void perm_free(bj_handle_s* h)
{
    cudaFree(h->var_perm);
    cudaFree(h->var_pinv);
    h->var_perm = nullptr;
    h->var_pinv = nullptr;
}

void var_free(bj_handle_s* h)
{
    if (h->var_fac) h->factor_bytes = 0;
    perm_free(h);
    cudaFree(h->var_bptr);
    cudaFree(h->var_foff);
    cudaFree(h->var_fac);
    h->var_bptr = nullptr;
    h->var_foff = nullptr;
    h->var_fac = nullptr;
}

// Turns a b = 0 handle (validated matrix, SpMV plan) into a variable-block handle: uploads the block layout, extracts
// and factors every block.  ptr_host was validated by the caller.
// The handle's own copy of a permutation and of its inverse (bj_setup_perm, bj_setup_blocks_perm).  A sequence that is not
// a permutation of 0..n-1 is BJ_ERR_INVALID_ARG.  Synchronises.
int perm_install(bj_handle_s* h, const int32_t* perm_dev)
{
    cudaStream_t st = h->stream;
    const size_t pb = sizeof(int32_t) * (size_t)h->n;
    if (cudaMalloc((void**)&h->var_perm, pb) != cudaSuccess || cudaMalloc((void**)&h->var_pinv, pb) != cudaSuccess) {
        cudaGetLastError();
        perm_free(h);
        return BJ_ERR_ALLOC;
    }
    int* flag = &h->status->pad;
    BJ_CUDA(cudaMemcpyAsync(h->var_perm, perm_dev, pb, cudaMemcpyDeviceToDevice, st));
    BJ_CUDA(cudaMemsetAsync(h->var_pinv, 0xff, pb, st));
    BJ_CUDA(cudaMemsetAsync(flag, 0, sizeof(int), st));
    perm_invert_kernel<<<(unsigned)((h->n + 255) / 256), 256, 0, st>>>(h->n, h->var_perm, h->var_pinv, flag);
    h->launches++;
    int bad = 1;
    BJ_CUDA(cudaMemcpyAsync(&bad, flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaStreamSynchronize(st));
    if (bad) { perm_free(h); return BJ_ERR_INVALID_ARG; }
    h->workspace_bytes += 2 * (int64_t)pb;
    return BJ_OK;
}

int var_setup(bj_handle_s* h, const int64_t* ptr_host, int64_t nblocks, const int32_t* perm_dev)
{
    cudaStream_t st = h->stream;
    if (perm_dev) {
        const int prc = perm_install(h, perm_dev);
        if (prc != BJ_OK) return prc;
    }
    std::vector<int32_t> bp((size_t)nblocks + 1);
    std::vector<int64_t> fo((size_t)nblocks + 1);
    int64_t off = 0;
    int smax = 0;
    for (int64_t k = 0; k < nblocks; ++k) {
        const int64_t s = ptr_host[k + 1] - ptr_host[k];
        bp[k] = (int32_t)ptr_host[k];
        fo[k] = off;
        off += s * (s + 1) / 2;
        smax = std::max<int>(smax, (int)s);
    }
    bp[nblocks] = (int32_t)ptr_host[nblocks];
    fo[nblocks] = off;
    if (cudaMalloc((void**)&h->var_bptr, sizeof(int32_t) * bp.size()) != cudaSuccess ||
        cudaMalloc((void**)&h->var_foff, sizeof(int64_t) * fo.size()) != cudaSuccess ||
        cudaMalloc((void**)&h->var_fac, sizeof(double) * (size_t)off) != cudaSuccess) {
        cudaGetLastError();
        var_free(h);
        return BJ_ERR_ALLOC;
    }
    BJ_CUDA(cudaMemcpyAsync(h->var_bptr, bp.data(), sizeof(int32_t) * bp.size(), cudaMemcpyHostToDevice, st));
    BJ_CUDA(cudaMemcpyAsync(h->var_foff, fo.data(), sizeof(int64_t) * fo.size(), cudaMemcpyHostToDevice, st));
    h->nblocks = nblocks;
    h->var_smax = smax;
    h->solve_kind = 4;
    h->factor_bytes = (int64_t)sizeof(double) * off + (int64_t)(sizeof(int32_t) * bp.size() + sizeof(int64_t) * fo.size());
    const unsigned grid = (unsigned)((nblocks + kVarWarps - 1) / kVarWarps);
    extract_factor_var_kernel<<<grid, kVarWarps * 32, 0, st>>>(nblocks, h->var_bptr, h->var_foff, h->row_ptr, h->col_idx, h->val,
                                                               h->var_fac, h->status, h->var_perm, h->var_pinv);
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    Status stt;
    BJ_CUDA(cudaMemcpyAsync(&stt, h->status, sizeof(stt), cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaStreamSynchronize(st));  // also keeps bp / fo alive until the copies are done
    if (stt.flags & ST_NOT_SPD) {
        h->failed = true;
        h->bad_block = (int64_t)stt.bad_block;
        return BJ_ERR_NOT_SPD;
    }
    return BJ_OK;
}

int launch_solve_var(bj_handle_s* h, int dir, const double* in, double* out)
{
    const unsigned grid = (unsigned)((h->nblocks + kVarWarps - 1) / kVarWarps);
    const bool pdl = h->pdl && !h->prof_on;
    cudaError_t e;
    if (dir == 0)
        e = launch_kernel(solve_var_kernel<0>, dim3(grid), dim3(kVarWarps * 32), 0, h->stream, pdl, h->nblocks,
                          (const int32_t*)h->var_bptr, (const int64_t*)h->var_foff, (const double*)h->var_fac, in, out,
                          (const int32_t*)h->var_perm);
    else if (dir == 1)
        e = launch_kernel(solve_var_kernel<1>, dim3(grid), dim3(kVarWarps * 32), 0, h->stream, pdl, h->nblocks,
                          (const int32_t*)h->var_bptr, (const int64_t*)h->var_foff, (const double*)h->var_fac, in, out,
                          (const int32_t*)h->var_perm);
    else
        e = launch_kernel(solve_var_kernel<2>, dim3(grid), dim3(kVarWarps * 32), 0, h->stream, pdl, h->nblocks,
                          (const int32_t*)h->var_bptr, (const int64_t*)h->var_foff, (const double*)h->var_fac, in, out,
                          (const int32_t*)h->var_perm);
    if (e != cudaSuccess) { set_cuda_error(e, "solve_var_kernel"); return BJ_ERR_CUDA; }
    h->launches++;
    return BJ_OK;
}

}  // namespace bj
