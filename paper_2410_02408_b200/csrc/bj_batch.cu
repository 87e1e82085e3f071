// Batched small systems: the paper's own sizes (N = 2^10 .. 2^14) as MANY
// independent systems in one launch -- its "solve each block separately" picture.
// The batch is one block-diagonal CSR (system s owns rows s*seg .. (s+1)*seg - 1), so setup, bj_apply and bj_op_apply
// work on it unchanged; what differs is that every system has its OWN Lanczos scalars.  One CTA per system does the
// whole vector part of a Lanczos step for its system -- alpha, the two axpys, beta, the breakdown test, the scaling --
// with block-level reductions only: no grid reduction, no partials, no host synchronisation inside the loop.
// An iteration is the operator apply on the whole batch plus ONE launch of lz_batch_step_kernel.
// Variant: DESIGN.md reading 10-12 without reorthogonalisation (the systems are small and the preconditioned
// spectra tame); per system it is exactly the recurrence of bj_lanczos.cu.
#include <math.h>

#include <algorithm>
#include <vector>

#include "bj_device.cuh"
#include "bj_internal.cuh"
#include "bj_reduce.cuh"

namespace bj {

namespace {

constexpr int kBatchThreads = 256;

// rows of system s: equal sizes (off == nullptr) or explicit offsets off[0..nsys]
__device__ __forceinline__ void batch_range(const int64_t* off, int64_t seg, int s, int64_t& base, int64_t& len)
{
    if (off) { base = off[s]; len = off[s + 1] - base; }
    else { base = (int64_t)s * seg; len = seg; }
}

// sum over the CTA, valid on every thread
__device__ __forceinline__ double block_sum_all(double v, double* sh)
{
    v = block_sum(v, sh);
    __syncthreads();
    if (threadIdx.x == 0) sh[0] = v;
    __syncthreads();
    const double r = sh[0];
    __syncthreads();
    return r;
}

// The batch entry points treat the matrix as block diagonal with respect to the systems: SpMV and the operator run on the
// whole matrix while every reduction is per system.  An entry that couples two systems would make every per-system result
// silently wrong, so each call checks it: CTA s flags any column outside [base_s, base_s + len_s) in the rows of system s
// (one coalesced pass over the column indices, 4 nnz bytes: microseconds beside the iterations that follow).
__global__ void __launch_bounds__(kBatchThreads)
batch_coupling_kernel(int64_t seg_, const int64_t* __restrict__ off, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci,
                      int* __restrict__ flag)
{
    int64_t base, seg;
    batch_range(off, seg_, blockIdx.x, base, seg);
    const int p0 = rp[base], p1 = rp[base + seg];
    bool bad = false;
    for (int p = p0 + threadIdx.x; p < p1; p += blockDim.x) {
        const int64_t c = ci[p];
        bad |= (c < base) | (c >= base + seg);
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flag, 1);
}

// v_1 = v0 / ||v0|| per system
__global__ void __launch_bounds__(kBatchThreads)
lz_batch_start_kernel(int64_t seg_, const int64_t* __restrict__ off, const double* __restrict__ v0, double* __restrict__ v)
{
    __shared__ double sh[kBatchThreads / 32];
    int64_t base, seg;
    batch_range(off, seg_, blockIdx.x, base, seg);
    double s = 0.0;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) {
        const double x = v0[base + i];
        s = fma(x, x, s);
    }
    const double nrm = sqrt(block_sum_all(s, sh));
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) v[base + i] = v0[base + i] / nrm;
}

// one Lanczos step of system blockIdx.x:  w -= beta_j v_{j-1};  alpha_j = v_j.w;  w -= alpha_j v_j;  beta_{j+1} = ||w||;
// stop this system if beta_{j+1} <= tol max|alpha|;  v_{j+1} = w / beta_{j+1}.  alpha/beta: [nsys][m] (device).
// A stopped system writes zeros into v_{j+1}, so the shared operator apply keeps producing zeros for it.
__global__ void __launch_bounds__(kBatchThreads)
lz_batch_step_kernel(int64_t seg_, const int64_t* __restrict__ off, int m, int j, double tol, double* __restrict__ w, const double* vprev,
                     const double* __restrict__ vcur, double* vnext,  // vprev and vnext share one buffer
                     double* __restrict__ alpha,
                     double* __restrict__ beta, double* __restrict__ amax, int* __restrict__ m_eff, int* __restrict__ stopped)
{
    __shared__ double sh[kBatchThreads / 32];
    pdl_trigger();
    pdl_wait();
    const int s = blockIdx.x;
    int64_t base, seg;
    batch_range(off, seg_, s, base, seg);
    if (stopped[s]) {
        if (vnext)
            for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) vnext[base + i] = 0.0;
        return;
    }
    const double bj = j > 0 ? beta[(int64_t)s * m + j - 1] : 0.0;
    double a = 0.0;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) {
        double wi = w[base + i];
        if (j > 0) {
            wi -= bj * vprev[base + i];
            w[base + i] = wi;
        }
        a = fma(vcur[base + i], wi, a);
    }
    a = block_sum_all(a, sh);
    double bb = 0.0;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) {
        const double wi = w[base + i] - a * vcur[base + i];
        w[base + i] = wi;
        bb = fma(wi, wi, bb);
    }
    const double bn = sqrt(block_sum_all(bb, sh));
    const double am = fmax(amax[s], fabs(a));
    const bool brk = !(bn > tol * am);
    if (threadIdx.x == 0) {
        alpha[(int64_t)s * m + j] = a;
        beta[(int64_t)s * m + j] = bn;
        amax[s] = am;
        m_eff[s] = j + 1;
        if (brk) stopped[s] = 1;
    }
    if (!vnext) return;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) vnext[base + i] = brk ? 0.0 : w[base + i] / bn;
}

// extreme eigenvalues of every system's Lanczos tridiagonal by bisection on the inertia of T - x I (the algorithm of
// tridiag_eig_k in bj_lanczos.cu), one THREAD per system: thousands of tiny tridiagonals are a device job, not a host loop
__device__ __forceinline__ int batch_negcount(int m, const double* a, const double* e, double x)
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
__device__ __forceinline__ double batch_eig_k(int m, const double* a, const double* e, int k)
{
    double lo = a[0], hi = a[0];
    for (int i = 0; i < m; ++i) {
        const double r = (i ? fabs(e[i - 1]) : 0.0) + (i + 1 < m ? fabs(e[i]) : 0.0);
        lo = fmin(lo, a[i] - r);
        hi = fmax(hi, a[i] + r);
    }
    for (int it = 0; it < 4000; ++it) {
        const double mid = 0.5 * lo + 0.5 * hi;
        if (!(mid > lo) || !(mid < hi)) break;
        if (batch_negcount(m, a, e, mid) >= k + 1) hi = mid; else lo = mid;
    }
    return 0.5 * lo + 0.5 * hi;
}
__global__ void __launch_bounds__(128)
batch_extremes_kernel(int64_t nsys, int m, const double* __restrict__ alpha, const double* __restrict__ beta,
                      const int* __restrict__ m_eff, double* __restrict__ lmin, double* __restrict__ lmax)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nsys) return;
    const int me = m_eff[s];
    if (me < 1) { lmin[s] = lmax[s] = 0.0; return; }
    lmin[s] = batch_eig_k(me, alpha + s * m, beta + s * m, 0);
    lmax[s] = batch_eig_k(me, alpha + s * m, beta + s * m, me - 1);
}

// ---- batched PCG: per-system scalars, one CTA per system for the vector parts ------------------------------------
// r = b, x = 0, bb[s] = ||b_s||^2 (a zero right-hand side stops its system at once)
__global__ void __launch_bounds__(kBatchThreads)
pcg_batch_init_kernel(int64_t seg_, const int64_t* __restrict__ off, const double* __restrict__ b, double* __restrict__ r, double* __restrict__ x,
                      double* __restrict__ bb, int* __restrict__ stopped, int* __restrict__ nstopped)
{
    __shared__ double sh[kBatchThreads / 32];
    const int s = blockIdx.x;
    int64_t base, seg;
    batch_range(off, seg_, s, base, seg);
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) {
        const double bi = b[base + i];
        r[base + i] = bi;
        x[base + i] = 0.0;
        acc = fma(bi, bi, acc);
    }
    acc = block_sum_all(acc, sh);
    if (threadIdx.x == 0) {
        bb[s] = acc;
        if (!(acc > 0.0)) { stopped[s] = 1; atomicAdd(nstopped, 1); }
    }
}

// first == 1: p = z, rho = r.z.   else: bt = (r.z) / rho, p = z + bt p, rho = r.z.   A stopped system keeps p = 0.
__global__ void __launch_bounds__(kBatchThreads)
pcg_batch_direction_kernel(int64_t seg_, const int64_t* __restrict__ off, int first, const double* __restrict__ r, const double* __restrict__ z,
                           double* __restrict__ p, double* __restrict__ rho, const int* __restrict__ stopped)
{
    __shared__ double sh[kBatchThreads / 32];
    pdl_trigger();
    pdl_wait();
    const int s = blockIdx.x;
    int64_t base, seg;
    batch_range(off, seg_, s, base, seg);
    if (stopped[s]) {
        for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) p[base + i] = 0.0;
        return;
    }
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) acc = fma(r[base + i], z[base + i], acc);
    const double rz = block_sum_all(acc, sh);
    const double bt = first ? 0.0 : rz / rho[s];
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) p[base + i] = first ? z[base + i] : fma(bt, p[base + i], z[base + i]);
    if (threadIdx.x == 0) rho[s] = rz;
}

// a = rho / (p.q); x += a p; r -= a q; relres = ||r|| / ||b||; the system stops when relres <= rtol
__global__ void __launch_bounds__(kBatchThreads)
pcg_batch_update_kernel(int64_t seg_, const int64_t* __restrict__ off, int k, double rtol, double* __restrict__ x, double* __restrict__ r,
                        const double* __restrict__ p, const double* __restrict__ q, const double* __restrict__ rho,
                        const double* __restrict__ bb, double* __restrict__ relres, int* __restrict__ iters,
                        int* __restrict__ stopped, int* __restrict__ converged, int* __restrict__ nstopped)
{
    __shared__ double sh[kBatchThreads / 32];
    pdl_trigger();
    pdl_wait();
    const int s = blockIdx.x;
    if (stopped[s]) return;
    int64_t base, seg;
    batch_range(off, seg_, s, base, seg);
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) acc = fma(p[base + i], q[base + i], acc);
    const double pq = block_sum_all(acc, sh);
    const double rh = rho[s];
    if (!(pq > 0.0) || rh == 0.0) {
        // p.Ap <= 0 (not SPD along p) or r.z = 0 (the residual is exactly zero although rtol = 0 kept the system going):
        // a = rho / (p.q) would be 0/0 or a step in a wrong direction; freeze the system where it stands
        if (threadIdx.x == 0) { stopped[s] = 1; converged[s] = rh == 0.0 ? 1 : 0; atomicAdd(nstopped, 1); }
        return;
    }
    const double a = rh / pq;
    acc = 0.0;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) {
        x[base + i] = fma(a, p[base + i], x[base + i]);
        const double ri = r[base + i] - a * q[base + i];
        r[base + i] = ri;
        acc = fma(ri, ri, acc);
    }
    const double rel = sqrt(block_sum_all(acc, sh) / bb[s]);
    if (threadIdx.x == 0) {
        relres[s] = rel;
        iters[s] = k + 1;
        if (rel <= rtol) { stopped[s] = 1; converged[s] = 1; atomicAdd(nstopped, 1); }
    }
}

// true_relres[s] = ||q_s - b_s|| / ||b_s||  with q = A x
__global__ void __launch_bounds__(kBatchThreads)
pcg_batch_residual_kernel(int64_t seg_, const int64_t* __restrict__ off, const double* __restrict__ q, const double* __restrict__ b,
                          const double* __restrict__ bb, double* __restrict__ out)
{
    __shared__ double sh[kBatchThreads / 32];
    pdl_trigger();
    pdl_wait();
    const int s = blockIdx.x;
    int64_t base, seg;
    batch_range(off, seg_, s, base, seg);
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < seg; i += blockDim.x) {
        const double d = q[base + i] - b[base + i];
        acc = fma(d, d, acc);
    }
    acc = block_sum_all(acc, sh);
    if (threadIdx.x == 0) out[s] = bb[s] > 0.0 ? sqrt(acc / bb[s]) : 0.0;
}

}  // namespace
}  // namespace bj

namespace bj {
void batch_free(bj_handle_s* h)
{
    if (h->batch_ws) { cudaFree(h->batch_ws); h->workspace_bytes -= (int64_t)h->batch_ws_bytes; }
    h->batch_ws = nullptr;
    h->batch_ws_bytes = 0;
}
// one allocation kept by the handle (a cudaMalloc of ~100 MB per call costs up to 0.2 s on a cold heap)
static void* batch_workspace(bj_handle_s* h, size_t bytes)
{
    if (h->batch_ws_bytes >= bytes) return h->batch_ws;
    batch_free(h);
    if (cudaMalloc(&h->batch_ws, bytes) != cudaSuccess) { cudaGetLastError(); h->batch_ws = nullptr; return nullptr; }
    h->batch_ws_bytes = bytes;
    h->workspace_bytes += (int64_t)bytes;
    return h->batch_ws;
}
// offsets_host == nullptr: nsys equal systems (n must divide).  Else offsets_host[0..nsys], 0 = off[0] < off[1] < .. = n,
// every system a whole number of Jacobi blocks.  Uploads the offsets to `dst` (device, nsys + 1 entries); *seg = n / nsys
// or 0.  Returns the device pointer to use (nullptr for equal sizes) through *off_dev.
static int batch_layout(bj_handle_s* h, int64_t nsys, const int64_t* offsets_host, int64_t* dst, int64_t* seg,
                        const int64_t** off_dev)
{
    *off_dev = nullptr;
    *seg = 0;
    if (h->solve_kind == 4 || h->var_perm) return BJ_ERR_INVALID_ARG;  // variable-size / permuted blocks: alignment with the systems is not checked here
    if (!offsets_host) {
        if (h->n % nsys) return BJ_ERR_INVALID_ARG;
        *seg = h->n / nsys;
        if (h->b > 0 && *seg % h->b) return BJ_ERR_INVALID_ARG;  // a Jacobi block must not straddle two systems
        return BJ_OK;
    }
    if (offsets_host[0] != 0 || offsets_host[nsys] != h->n) return BJ_ERR_INVALID_ARG;
    for (int64_t s = 0; s < nsys; ++s) {
        if (offsets_host[s + 1] <= offsets_host[s]) return BJ_ERR_INVALID_ARG;
        if (h->b > 0 && offsets_host[s] % h->b) return BJ_ERR_INVALID_ARG;
    }
    BJ_CUDA(cudaMemcpyAsync(dst, offsets_host, (size_t)(nsys + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, h->stream));
    *off_dev = dst;
    return BJ_OK;
}
// BJ_ERR_INVALID_ARG when an entry of the matrix couples two systems of the batch (see batch_coupling_kernel).  Synchronises.
static int batch_check_decoupled(bj_handle_s* h, int64_t nsys, int64_t seg, const int64_t* off, int* flag_dev)
{
    BJ_CUDA(cudaMemsetAsync(flag_dev, 0, sizeof(int), h->stream));
    batch_coupling_kernel<<<(unsigned)nsys, kBatchThreads, 0, h->stream>>>(seg, off, h->row_ptr, h->col_idx, flag_dev);
    h->launches++;
    int bad = 0;
    BJ_CUDA(cudaMemcpyAsync(&bad, flag_dev, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    BJ_CUDA(cudaStreamSynchronize(h->stream));
    return bad ? BJ_ERR_INVALID_ARG : BJ_OK;
}
}  // namespace bj

using namespace bj;

extern "C" int bj_pcg_solve_batch(bj_handle_t h, int64_t nsys, const int64_t* offsets_host, const double* b_dev, double* x_dev,
                                  int max_iters, double rtol, int32_t* iters_host, double* relres_host, double* true_relres_host)
{
    if (!h || h->failed || nsys < 1 || nsys > (1ll << 30) || max_iters < 1 || !b_dev || !x_dev || b_dev == x_dev) return BJ_ERR_INVALID_ARG;
    const int64_t n = h->n;
    cudaStream_t st = h->stream;
    // workspace: r, z, p, q; rho, bb, relres, true_relres [nsys each]; iters, stopped, converged [nsys each], nstopped
    const size_t vec_b = (size_t)4 * n * sizeof(double);
    const size_t scal_b = (size_t)4 * nsys * sizeof(double);
    const size_t int_b = (((size_t)3 * nsys + 4) * sizeof(int) + 7) & ~(size_t)7;
    const size_t off_b = (size_t)(nsys + 1) * sizeof(int64_t);
    char* ws = (char*)batch_workspace(h, vec_b + scal_b + int_b + off_b);
    if (!ws) return BJ_ERR_ALLOC;
    double* vec = (double*)ws;
    double* scal = (double*)(ws + vec_b);
    int* ints = (int*)(ws + vec_b + scal_b);
    auto cleanup = [&]() {};
    int64_t seg = 0;
    const int64_t* off = nullptr;
    {
        const int lrc = batch_layout(h, nsys, offsets_host, (int64_t*)(ws + vec_b + scal_b + int_b), &seg, &off);
        if (lrc != BJ_OK) return lrc;
    }
    double *r = vec, *z = vec + n, *p = vec + 2 * n, *q = vec + 3 * n;
    double *rho = scal, *bb = scal + nsys, *relres = scal + 2 * nsys, *truerel = scal + 3 * nsys;
    int *iters = ints, *stopped = ints + nsys, *converged = ints + 2 * nsys, *nstopped = ints + 3 * nsys;
    {
        const int crc = batch_check_decoupled(h, nsys, seg, off, nstopped + 1);
        if (crc != BJ_OK) return crc;
    }
    cudaError_t e = cudaMemsetAsync(scal, 0, (size_t)4 * nsys * sizeof(double), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(ints, 0, ((size_t)3 * nsys + 4) * sizeof(int), st);
    if (e != cudaSuccess) { set_cuda_error(e, "batch memset"); cleanup(); return BJ_ERR_CUDA; }
    const unsigned G = (unsigned)nsys;
    const bool pdl = h->pdl;
    int rc = BJ_OK;
    auto spmv = [&](const double* in, double* out) {
        return launch_spmv(h, in, out);
    };
#define BJ_BL(kernel, ...)                                                                                 \
    do {                                                                                                   \
        e = launch_kernel(kernel, dim3(G), dim3(kBatchThreads), 0, st, pdl, __VA_ARGS__);                  \
        if (e != cudaSuccess) { set_cuda_error(e, #kernel); rc = BJ_ERR_CUDA; }                            \
        h->launches++;                                                                                     \
    } while (0)
    pcg_batch_init_kernel<<<G, kBatchThreads, 0, st>>>(seg, off, b_dev, r, x_dev, bb, stopped, nstopped);
    h->launches++;
    rc = launch_solve(h, 2, r, z);
    if (rc == BJ_OK) BJ_BL(pcg_batch_direction_kernel, seg, off, 1, (const double*)r, (const double*)z, p, rho, (const int*)stopped);
    for (int k = 0; k < max_iters && rc == BJ_OK; ++k) {
        rc = spmv(p, q);
        if (rc != BJ_OK) break;
        BJ_BL(pcg_batch_update_kernel, seg, off, k, rtol, x_dev, r, (const double*)p, (const double*)q, (const double*)rho,
              (const double*)bb, relres, iters, stopped, converged, nstopped);
        if (rc != BJ_OK) break;
        rc = launch_solve(h, 2, r, z);
        if (rc != BJ_OK) break;
        BJ_BL(pcg_batch_direction_kernel, seg, off, 0, (const double*)r, (const double*)z, p, rho, (const int*)stopped);
        if ((k + 1) % 16 == 0 && k + 1 < max_iters && rc == BJ_OK) {  // every system done?
            int ns = 0;
            e = cudaMemcpyAsync(&ns, nstopped, sizeof(int), cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) { set_cuda_error(e, "batch poll"); rc = BJ_ERR_CUDA; break; }
            if (ns >= nsys) break;
        }
    }
    if (rc == BJ_OK) rc = spmv(x_dev, q);
    if (rc == BJ_OK) BJ_BL(pcg_batch_residual_kernel, seg, off, (const double*)q, b_dev, (const double*)bb, truerel);
#undef BJ_BL
    if (rc == BJ_OK) {
        e = cudaSuccess;
        if (iters_host) e = cudaMemcpyAsync(iters_host, iters, (size_t)nsys * sizeof(int), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && relres_host) e = cudaMemcpyAsync(relres_host, relres, (size_t)nsys * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && true_relres_host) e = cudaMemcpyAsync(true_relres_host, truerel, (size_t)nsys * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { set_cuda_error(e, "batch readback"); rc = BJ_ERR_CUDA; }
    }
    cleanup();
    return rc;
}

extern "C" int bj_cond_estimate_batch(bj_handle_t h, int64_t nsys, const int64_t* offsets_host, int iters, uint64_t seed,
                                      double* lmin_host, double* lmax_host, int32_t* iters_done_host)
{
    if (!h || h->failed || nsys < 1 || iters < 1 || !lmin_host || !lmax_host) return BJ_ERR_INVALID_ARG;
    const int64_t n = h->n;
    if (nsys > (1ll << 30)) return BJ_ERR_TOO_LARGE;
    const int m = iters;
    cudaStream_t st = h->stream;
    const double tol = BJ_DEFAULT_BREAKDOWN_TOL;

    // workspace: v_prev, v_cur (rotating), w; alpha/beta [nsys][m]; amax, lmin, lmax [nsys]; m_eff, stopped [nsys]
    const size_t vec_b = (size_t)3 * n * sizeof(double);
    const size_t scal_b = ((size_t)2 * nsys * m + 3 * nsys) * sizeof(double);
    const size_t int_b = ((size_t)2 * nsys * sizeof(int) + 7) & ~(size_t)7;
    const size_t off_b = (size_t)(nsys + 1) * sizeof(int64_t);
    char* ws = (char*)batch_workspace(h, vec_b + scal_b + int_b + off_b);
    if (!ws) return BJ_ERR_ALLOC;
    double* vec = (double*)ws;
    double* scal = (double*)(ws + vec_b);
    int* ints = (int*)(ws + vec_b + scal_b);
    auto cleanup = [&]() {};
    int64_t seg = 0;
    const int64_t* off = nullptr;
    {
        const int lrc = batch_layout(h, nsys, offsets_host, (int64_t*)(ws + vec_b + scal_b + int_b), &seg, &off);
        if (lrc != BJ_OK) return lrc;
    }
    {
        const int crc = batch_check_decoupled(h, nsys, seg, off, ints);
        if (crc != BJ_OK) return crc;
    }
    double* V[2] = {vec, vec + n};
    double* w = vec + 2 * n;
    double* alpha = scal;
    double* beta = scal + (size_t)nsys * m;
    double* amax = beta + (size_t)nsys * m;
    int* m_eff = ints;
    int* stopped = ints + nsys;
    int rc = BJ_OK;
    double* dlmin = amax + nsys;
    double* dlmax = dlmin + nsys;
    cudaError_t e = cudaMemsetAsync(scal, 0, ((size_t)2 * nsys * m + 3 * nsys) * sizeof(double), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(ints, 0, (size_t)2 * nsys * sizeof(int), st);
    if (e != cudaSuccess) { set_cuda_error(e, "batch memset"); cleanup(); return BJ_ERR_CUDA; }

    rc = launch_seeded_vector(h, seed, w);  // the start vector of system s is this vector's slice s
    if (rc == BJ_OK) {
        lz_batch_start_kernel<<<(unsigned)nsys, kBatchThreads, 0, st>>>(seg, off, w, V[0]);
        h->launches++;
    }
    for (int j = 0; j < m && rc == BJ_OK; ++j) {
        double* vj = V[j & 1];
        double* vn = V[(j + 1) & 1];
        rc = op_apply_device(h, vj, w);  // the whole batch at once: the matrix is block diagonal
        if (rc != BJ_OK) break;
        e = launch_kernel(lz_batch_step_kernel, dim3((unsigned)nsys), dim3(kBatchThreads), 0, st, h->pdl, seg, off, m, j, tol, w,
                          (const double*)vn, (const double*)vj, j + 1 < m ? vn : (double*)nullptr, alpha, beta, amax, m_eff,
                          stopped);
        if (e != cudaSuccess) { set_cuda_error(e, "lz_batch_step_kernel"); rc = BJ_ERR_CUDA; break; }
        h->launches++;
    }
    std::vector<int> hm((size_t)nsys);
    if (rc == BJ_OK) {
        batch_extremes_kernel<<<(unsigned)((nsys + 127) / 128), 128, 0, st>>>(nsys, m, alpha, beta, m_eff, dlmin, dlmax);
        h->launches++;
        e = cudaMemcpyAsync(lmin_host, dlmin, (size_t)nsys * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(lmax_host, dlmax, (size_t)nsys * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(hm.data(), m_eff, hm.size() * sizeof(int), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { set_cuda_error(e, "batch readback"); rc = BJ_ERR_CUDA; }
    }
    cleanup();
    if (rc != BJ_OK) return rc;
    for (int64_t s = 0; s < nsys; ++s) {
        if (hm[s] < 1) return BJ_ERR_CUDA;
        if (iters_done_host) iters_done_host[s] = hm[s];
    }
    return BJ_OK;
}
