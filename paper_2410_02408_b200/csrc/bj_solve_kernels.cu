// Batched block triangular solves (a5 and the two outer factors of a7):
//   forward  y = L^-1 r,   backward  x = L^-T y,   both  z = L^-T L^-1 r  (= M^-1 r).
// Diagonals are stored as reciprocals by the setup kernel.
//
// Two layouts, both HBM-bound by design (0.25 flop per byte):
//   b <= 8 : one THREAD per block.  The packed factor of 32 consecutive blocks is interleaved so that
//            element e of blocks 32g..32g+31 is one 256-byte line: every load of the warp is fully
//            coalesced and all P = b(b+1)/2 loads of a thread are independent (deep MLP).
//   b  > 8 : one SUB-WARP (16 or 32 lanes) per block, lane i owns row i.  Forward substitution is
//            column oriented: at step j lane j finalises y_j, broadcasts it by shuffle, lanes i > j
//            subtract L_ij y_j.  Column j of L is contiguous in the column-major packed copy, so the
//            lanes' loads coalesce; the backward solve reads the row-major packed copy the same way.
//            All b column loads of a lane are issued before the dependent chain starts.
#include "bj_device.cuh"
#include "bj_internal.cuh"

namespace bj {

// ------------------------------------------------------------------------------------------------
// thread per block, compile-time B.  DIR: 0 forward, 1 backward, 2 both.
// ------------------------------------------------------------------------------------------------
template <int B, int DIR, bool VEC>
__global__ void __launch_bounds__(128)
solve_small_kernel(int64_t n, int64_t nblocks, const double* __restrict__ fac,
                   const double* in, double* out)  // in == out allowed: a thread touches only its own block
{
    constexpr int P = B * (B + 1) / 2;
    pdl_trigger();
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nblocks) return;
    const double* f = fac + (k >> 5) * (int64_t)(P * kInterleave) + (k & 31);
    double l[P];
#pragma unroll
    for (int e = 0; e < P; ++e) l[e] = ld_stream(f + e * kInterleave);   // factors never change after setup
    pdl_wait();                                                          // `in` may come from the previous kernel
    const int64_t lo = k * B;
    double v[B];
    const bool whole = lo + B <= n;
    if (whole) {
        if constexpr (VEC && B % 4 == 0) {
#pragma unroll
            for (int i = 0; i < B; i += 4) ld_v4(in + lo + i, v + i);
        } else if constexpr (VEC && B % 2 == 0) {
#pragma unroll
            for (int i = 0; i < B; i += 2) ld_v2(in + lo + i, v + i);
        } else {
#pragma unroll
            for (int i = 0; i < B; ++i) v[i] = in[lo + i];
        }
    } else {
#pragma unroll
        for (int i = 0; i < B; ++i) v[i] = (lo + i < n) ? in[lo + i] : 0.0;
    }
    if (DIR == 0 || DIR == 2) {
#pragma unroll
        for (int i = 0; i < B; ++i) {
            double s = v[i];
#pragma unroll
            for (int j = 0; j < i; ++j) s -= l[i * (i + 1) / 2 + j] * v[j];
            v[i] = s * l[i * (i + 1) / 2 + i];
        }
    }
    if (DIR == 1 || DIR == 2) {
#pragma unroll
        for (int i = B - 1; i >= 0; --i) {
            double s = v[i];
#pragma unroll
            for (int j = i + 1; j < B; ++j) s -= l[j * (j + 1) / 2 + i] * v[j];
            v[i] = s * l[i * (i + 1) / 2 + i];
        }
    }
    if (whole) {
        if constexpr (VEC && B % 4 == 0) {
#pragma unroll
            for (int i = 0; i < B; i += 4) st_v4(out + lo + i, v + i);
        } else if constexpr (VEC && B % 2 == 0) {
#pragma unroll
            for (int i = 0; i < B; i += 2) st_v2(out + lo + i, v + i);
        } else {
#pragma unroll
            for (int i = 0; i < B; ++i) out[lo + i] = v[i];
        }
    } else {
#pragma unroll
        for (int i = 0; i < B; ++i)
            if (lo + i < n) out[lo + i] = v[i];
    }
}

// ------------------------------------------------------------------------------------------------
// sub-warp per block, W lanes (b <= W), lane i owns row i.
// ------------------------------------------------------------------------------------------------
template <int W, int DIR>
__global__ void __launch_bounds__(256)
solve_warp_kernel(int64_t n, int b, int64_t nblocks, const double* __restrict__ fwd,
                  const double* __restrict__ bwd, const double* in, double* out)  // in == out allowed
{
    pdl_trigger();
    const int i = threadIdx.x & (W - 1);
    int64_t k = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / W;
    const bool act = k < nblocks;  // no early return: the full-mask shuffles below need every lane
    if (!act) k = 0;
    const unsigned full = 0xffffffffu;
    const int P = b * (b + 1) / 2;
    const int64_t row = k * b + i;
    const bool live = act && (i < b) && (row < n);
    double r = 0.0;
    double l[W];

    if (DIR == 0 || DIR == 2) {
        const double* f = fwd + k * (int64_t)P;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            // column j: rows j..b-1 at offset j*b - j(j-1)/2
            l[j] = (act && j < b && i >= j && i < b) ? ld_stream(f + (j * b - j * (j - 1) / 2) + (i - j)) : 0.0;
        }
        pdl_wait();
        r = live ? in[row] : 0.0;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            if (j < b) {
                const double cand = r * l[j];                      // lane j: y_j = r_j / l_jj
                const double yj = __shfl_sync(full, cand, j, W);
                r = (i == j) ? yj : fma(-l[j], yj, r);             // lanes i < j hold l[j] = 0
            }
        }
    }
    if (DIR == 1 || DIR == 2) {
        const double* f = bwd + k * (int64_t)P;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            // row j: columns 0..j at offset j(j+1)/2
            l[j] = (act && j < b && i <= j) ? ld_stream(f + j * (j + 1) / 2 + i) : 0.0;
        }
        if (DIR == 1) {
            pdl_wait();
            r = live ? in[row] : 0.0;
        }
#pragma unroll
        for (int jj = 0; jj < W; ++jj) {
            const int j = W - 1 - jj;
            if (j < b) {
                const double cand = r * l[j];                      // lane j: x_j = r_j / l_jj
                const double xj = __shfl_sync(full, cand, j, W);
                r = (i == j) ? xj : fma(-l[j], xj, r);             // lanes i > j hold l[j] = 0
            }
        }
    }
    if (live) out[row] = r;
}

// b == 1 fast path is just the B = 1 instance of solve_small_kernel.

template <int DIR>
static int launch_small(bj_handle_s* h, const double* in, double* out)
{
    const int threads = 128;
    const unsigned blocks = (unsigned)((h->nblocks + threads - 1) / threads);
    const bool vec = ((((uintptr_t)in) | ((uintptr_t)out)) & 31) == 0;
    const bool pdl = h->pdl && !h->prof_on;
    cudaError_t e = cudaSuccess;
#define BJ_CASE(B)                                                                                                   \
    case B:                                                                                                          \
        e = vec ? launch_kernel(solve_small_kernel<B, DIR, true>, blocks, threads, 0, h->stream, pdl, h->n, h->nblocks,  \
                                (const double*)h->fac_small, in, out)                                                \
                : launch_kernel(solve_small_kernel<B, DIR, false>, blocks, threads, 0, h->stream, pdl, h->n, h->nblocks, \
                                (const double*)h->fac_small, in, out);                                               \
        break;
    switch (h->b) {
        BJ_CASE(1) BJ_CASE(2) BJ_CASE(3) BJ_CASE(4) BJ_CASE(5) BJ_CASE(6) BJ_CASE(7) BJ_CASE(8)
        default: return BJ_ERR_INVALID_ARG;
    }
#undef BJ_CASE
    if (e != cudaSuccess) { set_cuda_error(e, "solve_small_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}

template <int DIR>
static int launch_warp(bj_handle_s* h, const double* in, double* out)
{
    const int threads = 256;
    const bool pdl = h->pdl && !h->prof_on;
    cudaError_t e;
    if (h->lanes == 16) {
        const unsigned blocks = (unsigned)((h->nblocks * 16 + threads - 1) / threads);
        e = launch_kernel(solve_warp_kernel<16, DIR>, blocks, threads, 0, h->stream, pdl, h->n, h->b, h->nblocks,
                          (const double*)h->fac_fwd, (const double*)h->fac_bwd, in, out);
    } else {
        const unsigned blocks = (unsigned)((h->nblocks * 32 + threads - 1) / threads);
        e = launch_kernel(solve_warp_kernel<32, DIR>, blocks, threads, 0, h->stream, pdl, h->n, h->b, h->nblocks,
                          (const double*)h->fac_fwd, (const double*)h->fac_bwd, in, out);
    }
    if (e != cudaSuccess) { set_cuda_error(e, "solve_warp_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}

int launch_solve(bj_handle_s* h, int dir, const double* in, double* out)
{
    int rc = BJ_OK;
    if (h->solve_kind == 0) {
        if (in != out) BJ_CUDA(cudaMemcpyAsync(out, in, (size_t)h->n * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
        return BJ_OK;
    }
    const int kind = dir == 0 ? BJ_K_SOLVE_L : (dir == 1 ? BJ_K_SOLVE_LT : BJ_K_APPLY);
    {
        KernelScope scope(h, kind);
        if (h->solve_kind == 1) {
            rc = dir == 0 ? launch_small<0>(h, in, out) : dir == 1 ? launch_small<1>(h, in, out) : launch_small<2>(h, in, out);
        } else {
            rc = dir == 0 ? launch_warp<0>(h, in, out) : dir == 1 ? launch_warp<1>(h, in, out) : launch_warp<2>(h, in, out);
        }
    }
    if (rc != BJ_OK) return rc;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

}  // namespace bj
