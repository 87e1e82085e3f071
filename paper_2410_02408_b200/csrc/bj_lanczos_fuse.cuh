// Fused Lanczos step (a8, fast mode): the vector work of one Lanczos iteration rides on the two ends of
// the operator apply, so an iteration is the operator's own kernels and nothing else, and both grid
// reductions of the step (alpha, beta) come out of kernels that run anyway.
//
// Notation: w' = A^ v_j - beta_j v_{j-1} (before the alpha correction), w = w' - alpha_j v_j (unnormalised
// next vector), beta_{j+1} = ||w||, v_{j+1} = w / beta_{j+1}.  The operator is linear, so the apply runs on
// the UNNORMALISED w and its result is divided by beta_{j+1} afterwards:
//
//   prologue (first kernel of the apply, t~ = L^-T w):  alpha_j = sum of the previous epilogue's partials;
//       w = w' - alpha_j v_j  built on the fly as the solve's input and stored in place of w';
//       per-CTA partials of w.w.
//   epilogue (last kernel of the apply, y~ = L^-1 A t~):  beta_{j+1} = sqrt(sum of the prologue's partials);
//       v_{j+1} = w / beta_{j+1} stored;  w'_new = y~ / beta_{j+1} - beta_{j+1} v_j  stored in place of w;
//       per-CTA partials of v_{j+1}.w'_new.
//
// In both kernels the last CTA to finish adds the partials in index order (deterministic, no float atomics)
// and leaves the sum in device memory for the next kernel.  Same arithmetic as the classical ordering up to
// the rounding of the 1/beta scaling.  The parity mode (full reorthogonalisation) does not use this file.
#pragma once

#include <math.h>
#include <stdint.h>

namespace bj {

struct LzReduce {
    double* part;      // [cap] per-CTA partials
    double* out;       // the finished sum
    unsigned* ticket;  // zero on entry, zero on exit
    int cap;
};

struct LzPrologue {
    const double* w0;     // raw start vector (first step only, else null)
    double* w;            // in: w' of the previous step; out: w   (first: out only)
    const double* vcur;   // v_j (unused when first)
    const double* sum_a;  // v_j . w'  (finished by the previous epilogue kernel)
    double* alpha;        // alpha[] (device): entry j written by CTA 0
    const int* done;      // [0] stop flag
    LzReduce red;         // -> w . w
    int j;                // step whose alpha is being closed (ignored when first)
    int first;
};

struct LzEpilogue {
    double* w;             // in: w; out: w'_new
    const double* vprev;   // v_j  (null on the first step: no beta term)
    double* vnew;          // v_{j+1} out
    const double* sum_b;   // w . w  (finished by the prologue kernel of this apply)
    const double* alpha;   // alpha[] (device)
    double* beta;          // beta[]  (device): entry j written by CTA 0
    double* amax;          // two slots, ping-pong: running max |alpha|
    int* done;             // [0] stop flag, [1] m_eff, [2] invalid start vector
    LzReduce red;          // -> v_{j+1} . w'_new
    double tol;
    int j;                 // step whose beta is being closed (ignored when first)
    int first;
};

// prologue scalars: alpha (0 on the first step) and the uniform stop flag
__device__ __forceinline__ bool lz_prologue_begin(const LzPrologue& q, double& alpha)
{
    alpha = 0.0;
    if (q.done[0]) return true;
    if (!q.first) {
        alpha = *q.sum_a;
        if (blockIdx.x == 0 && threadIdx.x == 0) q.alpha[q.j] = alpha;
    }
    return false;
}

// element i of the unnormalised next vector: stored in place, squared into pn
__device__ __forceinline__ double lz_prologue_elem(const LzPrologue& q, double alpha, int64_t i, double& pn)
{
    const double wi = q.first ? q.w0[i] : q.w[i] - alpha * q.vcur[i];
    q.w[i] = wi;
    pn = fma(wi, wi, pn);
    return wi;
}

// epilogue scalars: beta, 1/beta and the uniform stop flag (breakdown: beta <= tol max|alpha|)
__device__ __forceinline__ bool lz_epilogue_begin(const LzEpilogue& e, double& beta, double& inv_beta)
{
    beta = 0.0; inv_beta = 0.0;
    if (e.done[0]) return true;
    const double s = *e.sum_b;
    beta = sqrt(s > 0.0 ? s : 0.0);
    inv_beta = 1.0 / beta;
    if (e.first) {
        // beta_1 = ||v0||: a zero or non-finite start vector is an invalid argument (done[2]), not a breakdown
        const bool bad = !(beta > 0.0) || isinf(beta);
        if (bad && blockIdx.x == 0 && threadIdx.x == 0) { e.done[0] = 1; e.done[2] = 1; }
        return bad;
    }
    const double a = fabs(e.alpha[e.j]);
    const double prev = e.amax[e.j & 1];
    const double amax = a > prev ? a : prev;
    const bool brk = !(beta > e.tol * amax);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        e.beta[e.j] = beta;
        e.amax[(e.j + 1) & 1] = amax;
        e.done[1] = e.j + 1;
        if (brk) e.done[0] = 1;
    }
    return brk;
}

// row i of the apply's result: stores v_{j+1}[i] and w'_new[i], accumulates v_{j+1}.w'_new
__device__ __forceinline__ void lz_epilogue_elem(const LzEpilogue& e, double beta, double inv_beta, int64_t i, double y, double& pa)
{
    const double vn = e.w[i] * inv_beta;
    e.vnew[i] = vn;
    double wi = y * inv_beta;
    if (e.vprev) wi -= beta * e.vprev[i];
    pa = fma(vn, wi, pa);
    e.w[i] = wi;
}

// End of a kernel that carries a reduction.  EVERY thread of the CTA must call it (threads without data
// pass zero).  sh: shared scratch of at least blockDim.x / 32 doubles.
__device__ __forceinline__ void lz_reduce_finish(const LzReduce& r, double p, double* sh)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) p += __shfl_down_sync(0xffffffffu, p, off);
    __syncthreads();
    if (lane == 0) sh[warp] = p;
    __syncthreads();
    __shared__ int is_last;
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int q = 0; q < nw; ++q) a += sh[q];
        r.part[blockIdx.x] = a;
        __threadfence();
        const unsigned t = atomicAdd(r.ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    // the last CTA adds the partials in index order: thread-strided sums, then the fixed tree above
    double a = 0.0;
    for (unsigned q = threadIdx.x; q < gridDim.x; q += blockDim.x) a += __ldcg(r.part + q);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) a += __shfl_down_sync(0xffffffffu, a, off);
    __syncthreads();
    if (lane == 0) sh[warp] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double sa = 0.0;
        for (int q = 0; q < nw; ++q) sa += sh[q];
        *r.out = sa;
        *r.ticket = 0u;
    }
}

// Two reductions of one kernel closed by ONE ticket (one fence, one atomic, one round of barriers): ra's ticket and cap serve
// both; rb.part / rb.out receive the second sum.  Same fixed order of additions as two calls of lz_reduce_finish.
// sh: at least 2 * blockDim.x / 32 doubles.
__device__ __forceinline__ void lz_reduce_finish2(const LzReduce& ra, double pa, const LzReduce& rb, double pb, double* sh)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        pa += __shfl_down_sync(0xffffffffu, pa, off);
        pb += __shfl_down_sync(0xffffffffu, pb, off);
    }
    __syncthreads();
    if (lane == 0) { sh[warp] = pa; sh[nw + warp] = pb; }
    __syncthreads();
    __shared__ int is_last2;
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int q = 0; q < nw; ++q) { a += sh[q]; b += sh[nw + q]; }
        ra.part[blockIdx.x] = a;
        rb.part[blockIdx.x] = b;
        __threadfence();
        const unsigned t = atomicAdd(ra.ticket, 1u);
        is_last2 = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last2) return;
    __threadfence();
    double a = 0.0, b = 0.0;
    for (unsigned q = threadIdx.x; q < gridDim.x; q += blockDim.x) { a += __ldcg(ra.part + q); b += __ldcg(rb.part + q); }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, off);
        b += __shfl_down_sync(0xffffffffu, b, off);
    }
    __syncthreads();
    if (lane == 0) { sh[warp] = a; sh[nw + warp] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double sa = 0.0, sb = 0.0;
        for (int q = 0; q < nw; ++q) { sa += sh[q]; sb += sh[nw + q]; }
        *ra.out = sa;
        *rb.out = sb;
        *ra.ticket = 0u;
    }
}

}  // namespace bj
