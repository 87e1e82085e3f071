// Device-resident Lanczos on A^ = L^-1 A L^-T (a8) and the extreme eigenvalues of the Lanczos
// tridiagonal (a9).  kappa = lambda_max / lambda_min.  Lanczos itself is not in
// the paper; the variant is fixed in DESIGN.md section 3 (readings 10-13):
//   v_1 = v0/||v0||;  for j = 1..m:  w = A^ v_j - beta_j v_{j-1};  alpha_j = v_j.w;  w -= alpha_j v_j;
//   [full reorthogonalisation, twice: c = V_j^T w; w -= V_j c];  beta_{j+1} = ||w||;
//   stop if beta_{j+1} <= tol max|alpha|;  v_{j+1} = w / beta_{j+1}.
// The loop never synchronises with the host: alpha, beta, the breakdown flag and every
// intermediate scalar stay in device memory; grid reductions are two-stage with a fixed
// summation order (bitwise reproducible run to run).
#include <math.h>
#include <stdlib.h>

#include <algorithm>

#include "bj_internal.cuh"

namespace bj {

__device__ __forceinline__ uint64_t mix64(uint64_t seed, uint64_t i)
{
    uint64_t z = seed + (i + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__global__ void seeded_vector_kernel(uint64_t seed, int64_t n, double* __restrict__ v)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const double u = (double)(mix64(seed, (uint64_t)i) >> 11) * (1.0 / 9007199254740992.0);
        v[i] = 2.0 * u - 1.0;
    }
}

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

// partial[blockIdx.x * stride + slot] = sum over the CTA's chunk of a[i] * b[i]
__global__ void __launch_bounds__(kReduceThreads)
dot_partial_kernel(int64_t n, const double* __restrict__ a, const double* __restrict__ b,
                   double* __restrict__ partial, int stride, const int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32];
    if (done && done[0]) return;
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) s = fma(a[i], b[i], s);
    s = block_sum(s, sh);
    if (threadIdx.x == 0) partial[(int64_t)blockIdx.x * stride] = s;
}

// w -= beta_j * vprev (when vprev != null);  partial of v . w
__global__ void __launch_bounds__(kReduceThreads)
alpha_partial_kernel(int64_t n, double* __restrict__ w, const double* __restrict__ vprev,
                     const double* __restrict__ v, const double* __restrict__ scal,
                     double* __restrict__ partial, int stride, const int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32];
    if (done[0]) return;
    const Chunk c = my_chunk(n);
    const double beta = scal[0];
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        double wi = w[i];
        if (vprev) {
            wi -= beta * vprev[i];
            w[i] = wi;
        }
        s = fma(v[i], wi, s);
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) partial[(int64_t)blockIdx.x * stride] = s;
}

// w -= alpha * v;  optional partial of w . w
__global__ void __launch_bounds__(kReduceThreads)
axpy_norm_kernel(int64_t n, double* __restrict__ w, const double* __restrict__ v,
                 const double* __restrict__ scal, double* __restrict__ partial, int stride,
                 int want_norm, const int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32];
    if (done[0]) return;
    const Chunk c = my_chunk(n);
    const double alpha = scal[3];
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        const double wi = w[i] - alpha * v[i];
        w[i] = wi;
        s = fma(wi, wi, s);
    }
    if (want_norm) {
        s = block_sum(s, sh);
        if (threadIdx.x == 0) partial[(int64_t)blockIdx.x * stride] = s;
    }
}

// partial[cta * stride + q] = sum over chunk of V_q[i] * w[i],  q = 0..nv-1
__global__ void __launch_bounds__(kReduceThreads)
multidot_partial_kernel(int64_t n, int nv, const double* __restrict__ V, const double* __restrict__ w,
                        double* __restrict__ partial, int stride, const int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32];
    if (done[0]) return;
    const Chunk c = my_chunk(n);
    for (int q0 = 0; q0 < nv; q0 += 4) {
        double s[4] = {0.0, 0.0, 0.0, 0.0};
        for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
            const double wi = w[i];
#pragma unroll
            for (int d = 0; d < 4; ++d)
                if (q0 + d < nv) s[d] = fma(V[(int64_t)(q0 + d) * n + i], wi, s[d]);
        }
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            if (q0 + d < nv) {
                const double r = block_sum(s[d], sh);
                if (threadIdx.x == 0) partial[(int64_t)blockIdx.x * stride + q0 + d] = r;
            }
        }
    }
}

// w[i] -= c_0 V_0[i]; w[i] -= c_1 V_1[i]; ... in that order; optional partial of w . w
__global__ void __launch_bounds__(kReduceThreads)
multiaxpy_kernel(int64_t n, int nv, const double* __restrict__ V, double* __restrict__ w,
                 const double* __restrict__ coef, double* __restrict__ partial, int stride, int want_norm,
                 const int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32];
    if (done[0]) return;
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        double wi = w[i];
        for (int q = 0; q < nv; ++q) wi -= coef[q] * V[(int64_t)q * n + i];
        w[i] = wi;
        s = fma(wi, wi, s);
    }
    if (want_norm) {
        s = block_sum(s, sh);
        if (threadIdx.x == 0) partial[(int64_t)blockIdx.x * stride] = s;
    }
}

// one CTA: out[q] = sum_cta partial[cta * stride + q]  (sequential over cta: fixed order)
__global__ void __launch_bounds__(256)
finalize_multi_kernel(int nparts, int nv, const double* __restrict__ partial, int stride,
                      double* __restrict__ out, const int* __restrict__ done)
{
    if (done[0]) return;
    for (int q = threadIdx.x; q < nv; q += blockDim.x) {
        double s = 0.0;
        for (int p = 0; p < nparts; ++p) s += partial[(int64_t)p * stride + q];
        out[q] = s;
    }
}

// one CTA reduces `nparts` partials (slot 0) and applies the scalar step `what`:
//   0: scal[2] = sqrt(sum)                       (||v0||)
//   1: alpha[j] = scal[3] = sum
//   2: beta[j] = scal[0] = sqrt(sum); amax; m_eff = j+1; breakdown flag
__global__ void __launch_bounds__(256)
finalize_scalar_kernel(int nparts, const double* __restrict__ partial, int stride, int what, int j,
                       double tol, double* __restrict__ scal, double* __restrict__ alpha,
                       double* __restrict__ beta, int* __restrict__ done)
{
    __shared__ double sh[8];
    if (done[0]) return;
    double s = 0.0;
    for (int p = threadIdx.x; p < nparts; p += blockDim.x) s += partial[(int64_t)p * stride];
    s = block_sum(s, sh);
    if (threadIdx.x != 0) return;
    if (what == 0) {
        scal[2] = sqrt(s);
    } else if (what == 1) {
        alpha[j] = s;
        scal[3] = s;
    } else {
        const double bn = sqrt(s);
        beta[j] = bn;
        scal[0] = bn;
        const double a = fabs(scal[3]);
        const double amax = a > scal[1] ? a : scal[1];
        scal[1] = amax;
        done[1] = j + 1;
        if (!(bn > tol * amax)) done[0] = 1;
    }
}

// out[i] = in[i] / scal[slot]
__global__ void __launch_bounds__(256)
scale_div_kernel(int64_t n, const double* __restrict__ in, double* __restrict__ out,
                 const double* __restrict__ scal, int slot, const int* __restrict__ done)
{
    if (done[0]) return;
    const double d = scal[slot];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        out[i] = in[i] / d;
}

int launch_seeded_vector(bj_handle_s* h, uint64_t seed, double* v)
{
    const int64_t want = (h->n + 255) / 256;
    const unsigned blocks = (unsigned)std::min<int64_t>(want, 148 * 16);
    seeded_vector_kernel<<<blocks, 256, 0, h->stream>>>(seed, h->n, v);
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

void lanczos_free(bj_handle_s* h)
{
    LanczosWs& z = h->lz;
    cudaFree(z.V); cudaFree(z.w); cudaFree(z.partial); cudaFree(z.coef);
    cudaFree(z.alpha); cudaFree(z.beta); cudaFree(z.scal); cudaFree(z.done);
    h->workspace_bytes -= z.bytes;
    z = LanczosWs();
}

static int lanczos_alloc(bj_handle_s* h, int iters, int64_t nvec)
{
    LanczosWs& z = h->lz;
    if (z.cap_vectors >= nvec && z.cap_iters >= iters) return BJ_OK;
    lanczos_free(h);
    const size_t vb = (size_t)h->n * sizeof(double);
    int64_t bytes = 0;
    auto A = [&](void** p, size_t sz) { cudaError_t e = cudaMalloc(p, sz); if (e == cudaSuccess) bytes += sz; return e; };
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = A((void**)&z.V, vb * nvec);
    if (e == cudaSuccess) e = A((void**)&z.w, vb);
    if (e == cudaSuccess) e = A((void**)&z.partial, sizeof(double) * kMaxPartials * (size_t)(iters + 1));
    if (e == cudaSuccess) e = A((void**)&z.coef, sizeof(double) * (size_t)(iters + 1));
    if (e == cudaSuccess) e = A((void**)&z.alpha, sizeof(double) * (size_t)iters);
    if (e == cudaSuccess) e = A((void**)&z.beta, sizeof(double) * (size_t)iters);
    if (e == cudaSuccess) e = A((void**)&z.scal, sizeof(double) * 8);
    if (e == cudaSuccess) e = A((void**)&z.done, sizeof(int) * 4);
    z.bytes = bytes;
    h->workspace_bytes += bytes;
    if (e != cudaSuccess) {
        cudaGetLastError();
        lanczos_free(h);
        return BJ_ERR_ALLOC;
    }
    z.cap_vectors = nvec;
    z.cap_iters = iters;
    return BJ_OK;
}

// ------------------------------------------------------------------------------------------------
// host: extreme eigenvalues of the symmetric tridiagonal T (diag a[0..m-1], off-diagonal e[0..m-2])
// by bisection on the inertia of T - x I, and the last eigenvector component by twisted factorisation.
// ------------------------------------------------------------------------------------------------
static int negcount(int m, const double* a, const double* e, double x)
{
    int cnt = 0;
    double piv = a[0] - x;
    cnt += piv < 0.0;
    for (int i = 1; i < m; ++i) {
        if (piv == 0.0) piv = 1e-300;
        piv = (a[i] - x) - (e[i - 1] * e[i - 1]) / piv;
        cnt += piv < 0.0;
    }
    return cnt;
}

static double eig_k(int m, const double* a, const double* e, int k)
{
    double lo = a[0], hi = a[0];
    for (int i = 0; i < m; ++i) {
        const double r = (i ? fabs(e[i - 1]) : 0.0) + (i + 1 < m ? fabs(e[i]) : 0.0);
        lo = std::min(lo, a[i] - r);
        hi = std::max(hi, a[i] + r);
    }
    for (int it = 0; it < 4000; ++it) {
        const double mid = 0.5 * lo + 0.5 * hi;
        if (!(mid > lo) || !(mid < hi)) break;
        if (negcount(m, a, e, mid) >= k + 1) hi = mid; else lo = mid;
    }
    return 0.5 * lo + 0.5 * hi;
}

static double last_comp(int m, const double* a, const double* e, double th)
{
    if (m == 1) return 1.0;
    std::vector<double> up(m), dn(m), z(m);
    up[0] = a[0] - th;
    for (int i = 1; i < m; ++i) up[i] = (a[i] - th) - e[i - 1] * e[i - 1] / (up[i - 1] != 0.0 ? up[i - 1] : 1e-300);
    dn[m - 1] = a[m - 1] - th;
    for (int i = m - 2; i >= 0; --i) dn[i] = (a[i] - th) - e[i] * e[i] / (dn[i + 1] != 0.0 ? dn[i + 1] : 1e-300);
    int tw = 0;
    double best = INFINITY;
    for (int i = 0; i < m; ++i) {
        const double g = fabs(up[i] + dn[i] - (a[i] - th));
        if (g < best) { best = g; tw = i; }
    }
    z[tw] = 1.0;
    for (int i = tw - 1; i >= 0; --i) z[i] = -e[i] * z[i + 1] / (up[i] != 0.0 ? up[i] : 1e-300);
    for (int i = tw + 1; i < m; ++i) z[i] = -e[i - 1] * z[i - 1] / (dn[i] != 0.0 ? dn[i] : 1e-300);
    double nn = 0.0;
    for (int i = 0; i < m; ++i) nn += z[i] * z[i];
    return fabs(z[m - 1]) / sqrt(nn);
}

// ------------------------------------------------------------------------------------------------
int lanczos_run(bj_handle_s* h, const bj_lanczos_opts_t* o, bj_lanczos_result_t* res)
{
    const int m = o->iters;
    const bool reorth = o->reorth != 0;
    const double tol = o->breakdown_tol > 0.0 ? o->breakdown_tol : BJ_DEFAULT_BREAKDOWN_TOL;
    const int64_t n = h->n;
    const int64_t nvec = reorth ? m : 2;
    int rc = lanczos_alloc(h, m, nvec);
    if (rc != BJ_OK) return rc;
    LanczosWs& z = h->lz;
    cudaStream_t st = h->stream;
    const int stride = m + 1;
    const int G = (int)std::max<int64_t>(1, std::min<int64_t>(kMaxPartials, (n + 1023) / 1024));
    const unsigned EG = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);

    BJ_CUDA(cudaMemsetAsync(z.scal, 0, sizeof(double) * 8, st));
    BJ_CUDA(cudaMemsetAsync(z.done, 0, sizeof(int) * 4, st));
    BJ_CUDA(cudaMemsetAsync(z.alpha, 0, sizeof(double) * m, st));
    BJ_CUDA(cudaMemsetAsync(z.beta, 0, sizeof(double) * m, st));

    auto vcol = [&](int j) { return z.V + (size_t)(reorth ? j : (j & 1)) * (size_t)n; };

    // v_1 = v0 / ||v0||
    const double* v0 = o->v0;
    if (!v0) {
        rc = launch_seeded_vector(h, o->seed, z.w);
        if (rc != BJ_OK) return rc;
        v0 = z.w;
    }
    dot_partial_kernel<<<G, kReduceThreads, 0, st>>>(n, v0, v0, z.partial, stride, nullptr);
    finalize_scalar_kernel<<<1, 256, 0, st>>>(G, z.partial, stride, 0, 0, tol, z.scal, z.alpha, z.beta, z.done);
    scale_div_kernel<<<EG, 256, 0, st>>>(n, v0, vcol(0), z.scal, 2, z.done);
    h->launches += 3;
    BJ_CUDA(cudaGetLastError());

    for (int j = 0; j < m; ++j) {
        double* vj = vcol(j);
        rc = op_apply_device(h, vj, z.w);
        if (rc != BJ_OK) return rc;
        alpha_partial_kernel<<<G, kReduceThreads, 0, st>>>(n, z.w, j > 0 ? vcol(j - 1) : nullptr, vj, z.scal,
                                                           z.partial, stride, z.done);
        finalize_scalar_kernel<<<1, 256, 0, st>>>(G, z.partial, stride, 1, j, tol, z.scal, z.alpha, z.beta, z.done);
        axpy_norm_kernel<<<G, kReduceThreads, 0, st>>>(n, z.w, vj, z.scal, z.partial, stride, reorth ? 0 : 1, z.done);
        h->launches += 3;
        if (reorth) {
            for (int pass = 0; pass < 2; ++pass) {
                multidot_partial_kernel<<<G, kReduceThreads, 0, st>>>(n, j + 1, z.V, z.w, z.partial, stride, z.done);
                finalize_multi_kernel<<<1, 256, 0, st>>>(G, j + 1, z.partial, stride, z.coef, z.done);
                multiaxpy_kernel<<<G, kReduceThreads, 0, st>>>(n, j + 1, z.V, z.w, z.coef, z.partial, stride,
                                                               pass == 1 ? 1 : 0, z.done);
                h->launches += 3;
            }
        }
        finalize_scalar_kernel<<<1, 256, 0, st>>>(G, z.partial, stride, 2, j, tol, z.scal, z.alpha, z.beta, z.done);
        h->launches += 1;
        if (j + 1 < m) {
            scale_div_kernel<<<EG, 256, 0, st>>>(n, z.w, vcol(j + 1), z.scal, 0, z.done);
            h->launches += 1;
        }
        BJ_CUDA(cudaGetLastError());
    }

    std::vector<double> a(m), b(m);
    int done[4] = {0, 0, 0, 0};
    BJ_CUDA(cudaMemcpyAsync(a.data(), z.alpha, sizeof(double) * m, cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaMemcpyAsync(b.data(), z.beta, sizeof(double) * m, cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaMemcpyAsync(done, z.done, sizeof(int) * 4, cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaStreamSynchronize(st));
    const int me = done[1];
    if (me < 1) return BJ_ERR_CUDA;
    res->iters_done = me;
    res->lmin = eig_k(me, a.data(), b.data(), 0);
    res->lmax = eig_k(me, a.data(), b.data(), me - 1);
    res->res_min = fabs(b[me - 1]) * last_comp(me, a.data(), b.data(), res->lmin);
    res->res_max = fabs(b[me - 1]) * last_comp(me, a.data(), b.data(), res->lmax);
    if (res->alpha_host) std::copy(a.begin(), a.begin() + me, res->alpha_host);
    if (res->beta_host) std::copy(b.begin(), b.begin() + me, res->beta_host);
    return BJ_OK;
}

}  // namespace bj
