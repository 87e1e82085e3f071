// Launch-bound sizes (config 1: N = 1024, the paper's smallest size): the WHOLE m-step Lanczos run of
// bj_lanczos.cu -- operator applies, alpha / beta, full reorthogonalisation (twice), breakdown test -- as ONE kernel of one
// CTA.  An iteration of the multi-launch path is about ten launches of ~5 us each for 0.15 MB of data; here the five work
// vectors, the factors and (when it fits) the matrix live in shared memory, every reduction is a block reduction in a fixed
// order, and the only global traffic inside the loop is the part of the basis V (L2-resident) that does not fit beside them
// (reorthogonalisation re-reads the basis four times per step: its first vectors get the shared memory that is left).
// Same recurrence, statement by statement, as lanczos_run (readings 10-13):
//   v_1 = v0/||v0||;  for j = 1..m:  w = A^ v_j - beta_j v_{j-1};  alpha_j = v_j.w;  w -= alpha_j v_j;
//   [twice: c = V_j^T w; w -= V_j c];  beta_{j+1} = ||w||;  stop if beta_{j+1} <= tol max|alpha|;  v_{j+1} = w / beta_{j+1}.
// The operator is the arithmetic of solve_small_kernel (thread per block, interleaved packed factors) and of a row-per-thread
// CSR product summed left to right (the oracle's order).  Block sizes b <= 8 and b = 0; larger blocks take the multi-launch path.
#include <math.h>

#include <algorithm>
#include <atomic>

#include "bj_device.cuh"
#include "bj_internal.cuh"

namespace bj {

namespace {

constexpr int kSmallThreads = 1024;
constexpr int kSmallWarps = kSmallThreads / 32;
constexpr int kDotChunk = 8;
constexpr int kRowReg = 8;  // a thread keeps its row's entries in registers when no row is longer

struct SmallLzParams {
    int n, nnz, b, P, nblocks, m, reorth, mat_in_smem;
    int row_in_regs;     // n <= kSmallThreads and no row longer than kRowReg: thread i keeps row i of the CSR in registers
    int vcache;          // the first `vcache` basis vectors are also kept in shared memory
    double tol;
    const int32_t* rp;
    const int32_t* ci;
    const double* val;
    const double* fac;   // fac_small (interleaved packed, reciprocal diagonals) or null
    const double* v0;
    double* V;           // (reorth ? m : 0) x n, global: the stored basis
    double* alpha;       // [m] global
    double* beta;        // [m] global
    int* done;           // [0] stop flag, [1] m_eff, [2] invalid start vector
};

// sum over the CTA in a fixed order (shuffle tree per warp, warp sums added in index order), valid on every thread
__device__ __forceinline__ double cta_sum(double v, double* sh)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    // fixed pairwise tree over the warp sums: depth 5 instead of a chain of 32 dependent additions
    double s[kSmallWarps];
#pragma unroll
    for (int q = 0; q < kSmallWarps; ++q) s[q] = sh[q];
#pragma unroll
    for (int w = kSmallWarps / 2; w > 0; w >>= 1)
#pragma unroll
        for (int q = 0; q < w; ++q) s[q] += s[q + w];
    return s[0];
}

// x = L^-T y (DIR 1) or L^-1 y (DIR 0) on every diagonal block, thread per block, factors in shared memory;
// the arithmetic and its order are solve_small_kernel's
template <int B, int DIR>
__device__ __forceinline__ void small_solve(const SmallLzParams& p, const double* sf, const double* in, double* out)
{
    if constexpr (B == 0) {
        for (int i = threadIdx.x; i < p.n; i += kSmallThreads) out[i] = in[i];
    } else {
        constexpr int P = B * (B + 1) / 2;
        for (int k = threadIdx.x; k < p.nblocks; k += kSmallThreads) {
            const double* f = sf + (size_t)(k >> 5) * (P * kInterleave) + (k & 31);
            const int lo = k * B;
            double v[B];
#pragma unroll
            for (int i = 0; i < B; ++i) v[i] = (lo + i < p.n) ? in[lo + i] : 0.0;
            if (DIR == 0) {
#pragma unroll
                for (int i = 0; i < B; ++i) {
                    double s = v[i];
#pragma unroll
                    for (int j = 0; j < B; ++j)
                        if (j < i) s -= f[(i * (i + 1) / 2 + j) * kInterleave] * v[j];
                    v[i] = s * f[(i * (i + 1) / 2 + i) * kInterleave];
                }
            } else {
#pragma unroll
                for (int i = B - 1; i >= 0; --i) {
                    double s = v[i];
#pragma unroll
                    for (int j = 0; j < B; ++j)
                        if (j > i) s -= f[(j * (j + 1) / 2 + i) * kInterleave] * v[j];
                    v[i] = s * f[(i * (i + 1) / 2 + i) * kInterleave];
                }
            }
#pragma unroll
            for (int i = 0; i < B; ++i)
                if (lo + i < p.n) out[lo + i] = v[i];
        }
    }
}

template <int B>
__global__ void __launch_bounds__(kSmallThreads)
lanczos_small_kernel(const SmallLzParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = p.n, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // red | t | u | w | vc | vp | c[m + 1] | fac | (val | ci | rp) | Vs   (all dynamic: the opt-in limit counts static too)
    double* red = reinterpret_cast<double*>(smem_raw);
    double* t = red + kSmallWarps;
    double* u = t + n;
    double* w = u + n;
    double* vc = w + n;
    double* vp = vc + n;
    double* c = vp + n;
    double* sf = c + ((p.m + 2) & ~1);
    const size_t fac_doubles = B > 0 ? (size_t)((p.nblocks + kInterleave - 1) / kInterleave) * (B * (B + 1) / 2) * kInterleave : 0;
    double* sval = sf + fac_doubles;
    int* sci = reinterpret_cast<int*>(sval + (p.mat_in_smem ? p.nnz : 0));
    int* srp = sci + (p.mat_in_smem ? p.nnz : 0);
    double* Vs = reinterpret_cast<double*>(srp + (p.mat_in_smem ? ((n + 2) & ~1) : 0));  // vcache x n
    for (size_t e = tid; e < fac_doubles; e += kSmallThreads) sf[e] = p.fac[e];
    const double* val = p.val;
    const int* ci = p.ci;
    const int* rp = p.rp;
    if (p.mat_in_smem) {
        for (int e = tid; e < p.nnz; e += kSmallThreads) { sval[e] = p.val[e]; sci[e] = p.ci[e]; }
        for (int e = tid; e <= n; e += kSmallThreads) srp[e] = p.rp[e];
        val = sval; ci = sci; rp = srp;
    }
    // row `tid` of the matrix in registers
    double rv[kRowReg];
    int rc[kRowReg];
    int rlen = 0;
#pragma unroll
    for (int q = 0; q < kRowReg; ++q) { rv[q] = 0.0; rc[q] = 0; }
    if (p.row_in_regs && tid < n) {
        const int s0 = p.rp[tid];
        rlen = p.rp[tid + 1] - s0;
#pragma unroll
        for (int q = 0; q < kRowReg; ++q)
            if (q < rlen) { rv[q] = p.val[s0 + q]; rc[q] = p.ci[s0 + q]; }
    }
    // basis vector q: the shared-memory copy when it has one, else the global one
    auto vq = [&](int q) -> const double* { return q < p.vcache ? Vs + (size_t)q * n : p.V + (size_t)q * n; };
    auto store_v = [&](int q, int i, double x) {
        if (p.reorth) {
            if (q < p.vcache) Vs[(size_t)q * n + i] = x; else p.V[(size_t)q * n + i] = x;
        }
    };
    // v_1 = v0 / ||v0||
    double s = 0.0;
    for (int i = tid; i < n; i += kSmallThreads) { const double x = p.v0[i]; s = fma(x, x, s); }
    const double nrm = sqrt(cta_sum(s, red));
    if (!(nrm > 0.0) || isinf(nrm)) {  // zero or non-finite start vector: invalid argument
        if (tid == 0) { p.done[0] = 1; p.done[2] = 1; }
        return;
    }
    for (int i = tid; i < n; i += kSmallThreads) {
        const double x = p.v0[i] / nrm;
        vc[i] = x;
        vp[i] = 0.0;
        store_v(0, i, x);
    }
    double beta_j = 0.0, amax = 0.0;
    __syncthreads();
    for (int j = 0; j < p.m; ++j) {
        // ---- w = L^-1 A L^-T v_j ----
        small_solve<B, 1>(p, sf, vc, t);
        __syncthreads();
        if (p.row_in_regs) {
            if (tid < n) {
                double acc = 0.0;
#pragma unroll
                for (int q = 0; q < kRowReg; ++q)
                    if (q < rlen) acc = fma(rv[q], t[rc[q]], acc);  // left to right, the oracle's order
                u[tid] = acc;
            }
        } else {
            for (int i = tid; i < n; i += kSmallThreads) {
                double acc = 0.0;
                const int e = rp[i + 1];
                for (int q = rp[i]; q < e; ++q) acc = fma(val[q], t[ci[q]], acc);
                u[i] = acc;
            }
        }
        __syncthreads();
        small_solve<B, 0>(p, sf, u, w);
        __syncthreads();
        // ---- w -= beta_j v_{j-1};  alpha_j = v_j . w;  w -= alpha_j v_j ----
        double pa = 0.0;
        for (int i = tid; i < n; i += kSmallThreads) {
            double wi = w[i];
            if (j > 0) { wi -= beta_j * vp[i]; w[i] = wi; }
            pa = fma(vc[i], wi, pa);
        }
        const double a = cta_sum(pa, red);
        for (int i = tid; i < n; i += kSmallThreads) w[i] -= a * vc[i];
        // ---- full reorthogonalisation, classical Gram-Schmidt twice over v_1 .. v_j: c = V^T w, then w -= V c ----
        if (p.reorth) {
            const int nv = j + 1;
            __syncthreads();  // every row of w is final before another thread reads it
            for (int pass = 0; pass < 2; ++pass) {
                // one WARP per dot product: lanes stride over the rows, one shuffle tree per basis vector (a tree per
                // thread-row and vector, as in the multi-launch kernels, made this single SM shuffle-bound: 40 us per step)
                for (int q = warp; q < nv; q += kSmallWarps) {
                    const double* v = vq(q);
                    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;  // four independent chains, combined in a fixed order
                    int i = lane;
                    for (; i + 96 < n; i += 128) {
                        s0 = fma(v[i], w[i], s0);
                        s1 = fma(v[i + 32], w[i + 32], s1);
                        s2 = fma(v[i + 64], w[i + 64], s2);
                        s3 = fma(v[i + 96], w[i + 96], s3);
                    }
                    for (; i < n; i += 32) s0 = fma(v[i], w[i], s0);
                    double sq = (s0 + s1) + (s2 + s3);
#pragma unroll
                    for (int off = 16; off > 0; off >>= 1) sq += __shfl_down_sync(0xffffffffu, sq, off);
                    if (lane == 0) c[q] = sq;
                }
                __syncthreads();
                for (int i = tid; i < n; i += kSmallThreads) {
                    double wi = w[i];
                    int q = 0;
                    for (; q + kDotChunk <= nv; q += kDotChunk) {  // eight loads in flight, subtraction order q = 0, 1, .. unchanged
                        double x[kDotChunk];
#pragma unroll
                        for (int d = 0; d < kDotChunk; ++d) x[d] = vq(q + d)[i];
#pragma unroll
                        for (int d = 0; d < kDotChunk; ++d) wi -= c[q + d] * x[d];
                    }
                    for (; q < nv; ++q) wi -= c[q] * vq(q)[i];
                    w[i] = wi;
                }
                __syncthreads();
            }
        }
        // ---- beta_{j+1} = ||w||, bookkeeping, breakdown test ----
        double pb = 0.0;
        for (int i = tid; i < n; i += kSmallThreads) pb = fma(w[i], w[i], pb);
        const double bn = sqrt(cta_sum(pb, red));
        amax = fabs(a) > amax ? fabs(a) : amax;
        const bool brk = !(bn > p.tol * amax);
        if (tid == 0) {
            p.alpha[j] = a;
            p.beta[j] = bn;
            p.done[1] = j + 1;
            if (brk) p.done[0] = 1;
        }
        if (brk || j + 1 == p.m) break;  // uniform over the CTA
        for (int i = tid; i < n; i += kSmallThreads) {
            const double x = w[i] / bn;
            vp[i] = vc[i];
            vc[i] = x;
            store_v(j + 1, i, x);
        }
        beta_j = bn;
        __syncthreads();
    }
}

size_t small_smem_bytes(const bj_handle_s* h, int m, bool mat)
{
    const size_t fac = h->solve_kind == 1 ? (size_t)((h->nblocks + kInterleave - 1) / kInterleave) * h->packed * kInterleave * 8 : 0;
    size_t b = (size_t)kSmallWarps * 8 + (size_t)5 * h->n * 8 + (size_t)((m + 2) & ~1) * 8 + fac;
    if (mat) b += (size_t)h->nnz * 12 + (((size_t)h->n + 2) & ~(size_t)1) * 4;
    return b + 16;
}

}  // namespace

// The single-launch run is used when the vectors, the factors and the coefficient buffer fit one CTA's shared memory
// (the matrix joins them when it fits too, else it is read through L2): thread-per-block layouts only (b <= 8 dense packed,
// or b = 0), at most 1024 steps.
bool lanczos_small_usable(const bj_handle_s* h, int m)
{
    if (env_int("BJ_LANCZOS_SMALL", 1) == 0) return false;
    if (h->var_perm || !(h->solve_kind == 0 || (h->solve_kind == 1 && !h->tri)) || m > 1024 || h->n > 16384 || h->nnz == 0) return false;
    return small_smem_bytes(h, m, false) <= 200 * 1024;
}

int launch_lanczos_small(bj_handle_s* h, int m, bool reorth, double tol, const double* v0, double* V, double* alpha, double* beta,
                         int* done)
{
    SmallLzParams p;
    p.n = (int)h->n; p.nnz = (int)h->nnz; p.b = h->b; p.P = h->packed; p.nblocks = (int)h->nblocks; p.m = m;
    p.reorth = reorth ? 1 : 0;
    p.tol = tol;
    p.rp = h->row_ptr; p.ci = h->col_idx; p.val = h->val;
    p.fac = h->solve_kind == 1 ? h->fac_small : nullptr;
    p.v0 = v0; p.V = V; p.alpha = alpha; p.beta = beta; p.done = done;
    constexpr size_t kBudget = 222 * 1024;
    p.row_in_regs = (h->n <= kSmallThreads && h->max_row_nnz <= kRowReg) ? 1 : 0;
    // the basis is re-read four times per step by the reorthogonalisation: what shared memory is left after the work
    // vectors and the factors goes to its first vectors; the matrix (read once per step) joins only if everything fits
    const size_t vec_b = (size_t)h->n * 8;
    p.mat_in_smem = (!p.row_in_regs && small_smem_bytes(h, m, true) + (reorth ? (size_t)m * vec_b : 0) <= kBudget) ? 1 : 0;
    size_t smem = small_smem_bytes(h, m, p.mat_in_smem != 0);
    p.vcache = reorth ? (int)std::min<size_t>((size_t)m, (kBudget - smem) / vec_b) : 0;
    smem += (size_t)p.vcache * vec_b;
    cudaError_t e = cudaSuccess;
#define BJ_CASE(B)                                                                                              \
    case B: {                                                                                                   \
        static std::atomic<bool> configured[64];                                                                \
        e = ensure_big_smem(lanczos_small_kernel<B>, configured);                                               \
        if (e == cudaSuccess) lanczos_small_kernel<B><<<1, kSmallThreads, smem, h->stream>>>(p);                \
        break;                                                                                                  \
    }
    switch (h->solve_kind == 1 ? h->b : 0) {
        BJ_CASE(0) BJ_CASE(1) BJ_CASE(2) BJ_CASE(3) BJ_CASE(4) BJ_CASE(5) BJ_CASE(6) BJ_CASE(7) BJ_CASE(8)
        default: return BJ_ERR_INVALID_ARG;
    }
#undef BJ_CASE
    if (e != cudaSuccess) { set_cuda_error(e, "lanczos_small_kernel"); return BJ_ERR_CUDA; }
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

}  // namespace bj
