// Preconditioned conjugate gradients: the classical stand-in for the solve stage
// that follows the preconditioning path, built from the path's own kernels --
// q = A p is the CSR SpMV (a6), z = M^-1 r is the batched block solve pair (a5) -- plus the vector
// kernels below.  Textbook Hestenes-Stiefel ordering from x_0 = 0:
//   r = b; z = M^-1 r; p = z; rho = r.z
//   repeat: q = A p; a = rho / (p.q); x += a p; r -= a q; stop if ||r|| / ||b|| <= rtol;
//           z = M^-1 r; rho' = r.z; bt = rho' / rho; p = z + bt p; rho = rho'
// Every scalar (rho, p.q, ||r||^2, a, bt, the stop flag) stays in device memory: a kernel that needs one
// re-sums the producer's per-CTA partials in a fixed order (bj_reduce.cuh), so the loop has no host
// synchronisation except a poll of the stop flag every `check_every` iterations.
// Reported: the paper's accuracy metric ||Ax - b|| / ||b|| recomputed from x, and the
// extreme Ritz values of M^-1 A from the CG coefficients (CG-Lanczos equivalence).
#include <math.h>

#include <string.h>

#include <algorithm>
#include <cmath>
#include <vector>

#include "bj_device.cuh"
#include "bj_internal.cuh"
#include "bj_pcg_fuse.cuh"
#include "bj_reduce.cuh"

namespace bj {

namespace {

// device scalar slots
enum { S_BB = 0, S_RHO_A = 1, S_RHO_B = 2, S_PQ = 3, S_RR = 4, S_COUNT = 8 };
// int flags: [0] stop, [1] iterations done, [2] converged

// r = b; x = 0; P0[cta] = partial of b.b
__global__ void __launch_bounds__(kReduceThreads)
pcg_init_kernel(int64_t n, const double* __restrict__ b, double* __restrict__ r, double* __restrict__ x,
                double* __restrict__ P0)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        const double bi = b[i];
        r[i] = bi;
        x[i] = 0.0;
        s = fma(bi, bi, s);
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) P0[blockIdx.x] = s;
}

// bb = sum P0 (kept in scal[S_BB]); zero right-hand side stops the run; p = z; PR[cta] = partial of r.z
__global__ void __launch_bounds__(kReduceThreads)
pcg_start_kernel(int64_t n, const double* __restrict__ r, const double* __restrict__ z, double* __restrict__ p,
                 const double* __restrict__ P0, int nparts, double* __restrict__ scal, double* __restrict__ PR,
                 int* __restrict__ flags)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    const double bb = reduce_partials(P0, nparts, sh);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        scal[S_BB] = bb;
        if (!(bb > 0.0)) flags[0] = 1;
    }
    if (!(bb > 0.0)) return;
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        const double zi = z[i];
        p[i] = zi;
        s = fma(r[i], zi, s);
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) PR[blockIdx.x] = s;
}

// PQ[cta] = partial of p.q
__global__ void __launch_bounds__(kReduceThreads)
pcg_pq_kernel(int64_t n, const double* __restrict__ p, const double* __restrict__ q, double* __restrict__ PQ,
              const int* __restrict__ flags)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (flags[0]) return;
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) s = fma(p[i], q[i], s);
    s = block_sum(s, sh);
    if (threadIdx.x == 0) PQ[blockIdx.x] = s;
}

// a = (sum PR) / (sum PQ); x += a p; r -= a q; PRR[cta] = partial of r.r; CTA 0 records alpha[k]
__global__ void __launch_bounds__(kReduceThreads)
pcg_update_kernel(int64_t n, double* __restrict__ x, double* __restrict__ r, const double* __restrict__ p,
                  const double* __restrict__ q, const double* __restrict__ PR, const double* __restrict__ PQ,
                  int nparts, int k, double* __restrict__ alpha, double* __restrict__ PRR, const int* __restrict__ flags)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (flags[0]) return;
    const double rho = reduce_partials(PR, nparts, sh);
    const double pq = reduce_partials(PQ, nparts, sh);
    const double a = rho / pq;
    if (blockIdx.x == 0 && threadIdx.x == 0) alpha[k] = a;
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        x[i] = fma(a, p[i], x[i]);
        const double ri = r[i] - a * q[i];
        r[i] = ri;
        s = fma(ri, ri, s);
    }
    __syncthreads();
    s = block_sum(s, sh);
    if (threadIdx.x == 0) PRR[blockIdx.x] = s;
}

// relres_k = sqrt(sum PRR / bb): CTA 0 records it and the iteration count; all CTAs stop together when it is
// <= rtol.  Otherwise PR2[cta] = partial of r.z (z = M^-1 r of the updated residual).
__global__ void __launch_bounds__(kReduceThreads)
pcg_rz_kernel(int64_t n, const double* __restrict__ r, const double* __restrict__ z, const double* __restrict__ PRR,
              int nparts, const double* __restrict__ scal, double rtol, int k, double* __restrict__ relres,
              double* __restrict__ PR2, int* __restrict__ flags)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (flags[0]) return;
    const double rr = reduce_partials(PRR, nparts, sh);
    const double rel = sqrt(rr / scal[S_BB]);
    const bool stop = rel <= rtol;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        relres[k] = rel;
        flags[1] = k + 1;
        if (stop) { flags[0] = 1; flags[2] = 1; }
    }
    if (stop) return;
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) s = fma(r[i], z[i], s);
    __syncthreads();
    s = block_sum(s, sh);
    if (threadIdx.x == 0) PR2[blockIdx.x] = s;
}

// bt = (sum PR2) / (sum PR); p = z + bt p; CTA 0 records beta[k]
__global__ void __launch_bounds__(kReduceThreads)
pcg_direction_kernel(int64_t n, double* __restrict__ p, const double* __restrict__ z, const double* __restrict__ PR,
                     const double* __restrict__ PR2, int nparts, int k, double* __restrict__ beta,
                     const int* __restrict__ flags)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (flags[0]) return;
    const double rho = reduce_partials(PR, nparts, sh);
    const double rho_new = reduce_partials(PR2, nparts, sh);
    const double bt = rho_new / rho;
    if (blockIdx.x == 0 && threadIdx.x == 0) beta[k] = bt;
    const Chunk c = my_chunk(n);
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) p[i] = fma(bt, p[i], z[i]);
}

// PD[cta] = partial of ||q - b||^2  (q = A x)
__global__ void __launch_bounds__(kReduceThreads)
pcg_residual_kernel(int64_t n, const double* __restrict__ q, const double* __restrict__ b, double* __restrict__ PD)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        const double d = q[i] - b[i];
        s = fma(d, d, s);
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) PD[blockIdx.x] = s;
}

// fused path: out[0] = sum PR (one CTA): the first rho as a finished scalar
__global__ void __launch_bounds__(kReduceThreads)
pcg_scalar_kernel(const double* __restrict__ PR, int nparts, double* __restrict__ out, const int* __restrict__ flags)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (flags[0]) return;
    const double s = reduce_partials(PR, nparts, sh);
    if (threadIdx.x == 0) out[0] = s;
}

// fused path, K3: stopping test on sqrt(rr / bb) (CTA 0 records relres[k] and the iteration count), then
// bt = rho_new / rho, p = z + bt p (CTA 0 records beta[k]).  All scalars are finished sums in scal[].
__global__ void __launch_bounds__(kReduceThreads)
pcg_direction_fused_kernel(int64_t n, double* __restrict__ p, const double* __restrict__ z, const double* __restrict__ scal,
                           int rho_cur, int rho_new, double rtol, int k, double* __restrict__ relres,
                           double* __restrict__ beta, int* __restrict__ flags)
{
    pdl_trigger();
    pdl_wait();
    if (flags[0]) return;
    const double rel = sqrt(scal[S_RR] / scal[S_BB]);
    const bool stop = rel <= rtol;
    const double bt = scal[rho_new] / scal[rho_cur];
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        relres[k] = rel;
        flags[1] = k + 1;
        if (stop) { flags[0] = 1; flags[2] = 1; }
        else beta[k] = bt;
    }
    if (stop) return;
    const Chunk c = my_chunk(n);
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) p[i] = fma(bt, p[i], z[i]);
}

// workspace of a run with up to m iterations: r, z, p, q (4 n doubles, kept by the handle); scalars, six partial arrays,
// alpha / beta / relres, flags, three partial arrays of the fused path
struct PcgWs {
    double *r, *z, *p, *q, *scal, *P0, *PRa, *PRb, *PQ, *PRR, *PD, *alpha, *beta, *relres, *FP;
    int* flags;  // 16 ints: [0..2] flags, [4..6] tickets of the fused path
    size_t fcap;
};

int pcg_workspace(bj_handle_s* h, int m, PcgWs& w)
{
    const int64_t n = h->n;
    w.fcap = (size_t)std::max<int64_t>(kMaxPartials, (h->nblocks + 127) / 128 + 1);
    if (!h->pcg_vec) {
        BJ_CUDA(cudaMalloc((void**)&h->pcg_vec, (size_t)4 * n * sizeof(double)));
        h->workspace_bytes += (int64_t)4 * n * (int64_t)sizeof(double);
    }
    if (h->pcg_cap_iters < m) {
        cudaFree(h->pcg_scal);
        h->pcg_scal = nullptr;
        h->pcg_cap_iters = 0;
        BJ_CUDA(cudaMalloc((void**)&h->pcg_scal, sizeof(double) * (S_COUNT + 6 * (size_t)kMaxPartials + 3 * (size_t)m + 8 + 3 * w.fcap)));
        h->pcg_cap_iters = m;
    }
    w.r = h->pcg_vec;
    w.z = w.r + n;
    w.p = w.z + n;
    w.q = w.p + n;
    w.scal = h->pcg_scal;
    w.P0 = w.scal + S_COUNT;
    w.PRa = w.P0 + kMaxPartials;
    w.PRb = w.PRa + kMaxPartials;
    w.PQ = w.PRb + kMaxPartials;
    w.PRR = w.PQ + kMaxPartials;
    w.PD = w.PRR + kMaxPartials;
    w.alpha = w.PD + kMaxPartials;
    w.beta = w.alpha + h->pcg_cap_iters;
    w.relres = w.beta + h->pcg_cap_iters;
    w.flags = reinterpret_cast<int*>(w.relres + h->pcg_cap_iters);
    w.FP = w.relres + h->pcg_cap_iters + 8;
    BJ_CUDA(cudaMemsetAsync(w.scal, 0, sizeof(double) * S_COUNT, h->stream));
    BJ_CUDA(cudaMemsetAsync(w.alpha, 0, sizeof(double) * (3 * (size_t)h->pcg_cap_iters + 8), h->stream));
    return BJ_OK;
}

// unfused step of Lanczos on M^-1 A (bj_pcg_fuse.cuh, mode 1): zp = sum PQ, the three coefficients, r_{k+1} written over r_{k-1}
__global__ void __launch_bounds__(kReduceThreads)
mlz_combine_kernel(int64_t n, const double* __restrict__ q, const double* __restrict__ r, double* __restrict__ x,
                   const double* __restrict__ PQ, int nparts, const double* __restrict__ bsq, int k, double* __restrict__ alpha)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    const double zp = reduce_partials(PQ, nparts, sh);
    const double b2 = bsq[k];
    const double bt = sqrt(b2);
    const double al = zp / b2;
    const double cq = 1.0 / bt, cr = -al / bt, cx = k > 0 ? -bt / sqrt(bsq[k - 1]) : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) alpha[k] = al;
    const Chunk c = my_chunk(n);
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) x[i] = mlz_combine(cq, cr, cx, q[i], r[i], x[i]);
}

}  // namespace

void pcg_free(bj_handle_s* h)
{
    if (h->pcg_vec) { h->workspace_bytes -= (int64_t)4 * h->n * (int64_t)sizeof(double); cudaFree(h->pcg_vec); }
    cudaFree(h->pcg_scal);
    h->pcg_vec = nullptr;
    h->pcg_scal = nullptr;
    h->pcg_cap_iters = 0;
}

int pcg_run(bj_handle_s* h, const double* b, double* x, const bj_pcg_opts_t* o, bj_pcg_result_t* res)
{
    const int64_t n = h->n;
    const int m = o->max_iters;
    const int check = o->check_every > 0 ? o->check_every : 16;
    const double rtol = o->rtol > 0.0 ? o->rtol : 0.0;
    cudaStream_t st = h->stream;

    PcgWs ws;
    int rc = pcg_workspace(h, m, ws);
    if (rc != BJ_OK) return rc;
    double *r = ws.r, *z = ws.z, *p = ws.p, *q = ws.q, *scal = ws.scal, *P0 = ws.P0, *PRa = ws.PRa, *PRb = ws.PRb, *PQ = ws.PQ,
           *PRR = ws.PRR, *PD = ws.PD, *alpha = ws.alpha, *beta = ws.beta, *relres = ws.relres, *FP = ws.FP;
    int* flags = ws.flags;
    const size_t fcap = ws.fcap;

    const int G = (int)std::max<int64_t>(1, std::min<int64_t>(kMaxPartials, (n + 1023) / 1024));
    const bool pdl = h->pdl;
    cudaError_t e = cudaSuccess;
#define BJ_LAUNCH(kernel, ...)                                                                  \
    do {                                                                                        \
        e = launch_kernel(kernel, dim3(G), dim3(kReduceThreads), 0, st, pdl, __VA_ARGS__);      \
        if (e != cudaSuccess) { set_cuda_error(e, #kernel); return BJ_ERR_CUDA; }               \
        h->launches++;                                                                          \
    } while (0)
    auto spmv = [&](const double* in, double* out) {
        return launch_spmv(h, in, out);
    };

    // launch-bound sizes: the whole run is ONE kernel of one cluster (bj_pcg_cluster.cu)
    const bool single = h->opt_pcg_small != 0 && pcg_cluster_usable(h);
    int G_read = G;  // partials of ||A x - b||^2 to add on the host
    if (single) {
        rc = launch_pcg_cluster(h, b, x, m, rtol, alpha, beta, relres, scal, PD, flags);
        if (rc != BJ_OK) return rc;
        G_read = 1;
    }
    int hflags[4] = {0, 0, 0, 0};
    if (!single) {
    BJ_LAUNCH(pcg_init_kernel, n, b, r, x, P0);
    rc = launch_solve(h, 2, r, z);  // z = M^-1 r  (b = 0: copy)
    if (rc != BJ_OK) return rc;
    BJ_LAUNCH(pcg_start_kernel, n, (const double*)r, (const double*)z, p, (const double*)P0, G, scal, PRa, flags);

    // Fused iteration (bj_pcg_fuse.cuh): needs the tile SpMV (dot hook) and a solve kernel that carries the PCG hook
    const bool fused = h->spmv_kernel == 1 && lanczos_fusable(h) && h->opt_pcg_fuse != 0;
    if (fused) {
        unsigned* tickets = reinterpret_cast<unsigned*>(flags + 4);
        LzReduce red_pq{FP, scal + S_PQ, tickets + 0, (int)fcap};
        PcgHook hook{};
        hook.x = x; hook.p = p; hook.r = r; hook.q = q; hook.pq = scal + S_PQ; hook.alpha = alpha; hook.flags = flags;
        hook.red_rr = LzReduce{FP + fcap, scal + S_RR, tickets + 1, (int)fcap};
        int rho_cur = S_RHO_A, rho_new = S_RHO_B;
        e = launch_kernel(pcg_scalar_kernel, dim3(1), dim3(kReduceThreads), 0, st, pdl, (const double*)PRa, G, scal + rho_cur,
                          (const int*)flags);
        if (e != cudaSuccess) { set_cuda_error(e, "pcg_scalar_kernel"); return BJ_ERR_CUDA; }
        h->launches++;
        for (int k = 0; k < m; ++k) {
            rc = launch_spmv_stream(h, p, q, false, nullptr, p, &red_pq);  // K1: q = A p, p.q
            if (rc != BJ_OK) return rc;
            hook.rho = scal + rho_cur;
            hook.red_rz = LzReduce{FP + 2 * fcap, scal + rho_new, tickets + 2, (int)fcap};
            hook.k = k;
            rc = launch_solve(h, 2, nullptr, z, nullptr, nullptr, &hook);  // K2: x, r updates, z = M^-1 r, r.r, r.z
            if (rc != BJ_OK) return rc;
            BJ_LAUNCH(pcg_direction_fused_kernel, n, p, (const double*)z, (const double*)scal, rho_cur, rho_new, rtol, k, relres,
                      beta, flags);  // K3
            std::swap(rho_cur, rho_new);
            if ((k + 1) % check == 0 && k + 1 < m) {
                BJ_CUDA(cudaMemcpyAsync(hflags, flags, sizeof(hflags), cudaMemcpyDeviceToHost, st));
                BJ_CUDA(cudaStreamSynchronize(st));
                if (hflags[0]) break;
            }
        }
    }
    double* PR = PRa;   // partials of the current rho = r.z
    double* PR2 = PRb;  // partials of the next one
    for (int k = 0; k < m && !fused; ++k) {
        rc = spmv(p, q);  // q = A p
        if (rc != BJ_OK) return rc;
        BJ_LAUNCH(pcg_pq_kernel, n, (const double*)p, (const double*)q, PQ, (const int*)flags);
        BJ_LAUNCH(pcg_update_kernel, n, x, r, (const double*)p, (const double*)q, (const double*)PR, (const double*)PQ, G, k,
                  alpha, PRR, (const int*)flags);
        rc = launch_solve(h, 2, r, z);  // z = M^-1 r
        if (rc != BJ_OK) return rc;
        BJ_LAUNCH(pcg_rz_kernel, n, (const double*)r, (const double*)z, (const double*)PRR, G, (const double*)scal, rtol, k,
                  relres, PR2, flags);
        BJ_LAUNCH(pcg_direction_kernel, n, p, (const double*)z, (const double*)PR, (const double*)PR2, G, k, beta,
                  (const int*)flags);
        std::swap(PR, PR2);
        if ((k + 1) % check == 0 && k + 1 < m) {
            BJ_CUDA(cudaMemcpyAsync(hflags, flags, sizeof(hflags), cudaMemcpyDeviceToHost, st));
            BJ_CUDA(cudaStreamSynchronize(st));
            if (hflags[0]) break;
        }
    }
    // the paper's metric from x itself: ||A x - b|| / ||b||
    rc = spmv(x, q);
    if (rc != BJ_OK) return rc;
    BJ_LAUNCH(pcg_residual_kernel, n, (const double*)q, b, PD);
    }  // !single
#undef BJ_LAUNCH

    // alpha | beta | relres | flags are one block of the workspace: one copy (a copy costs ~10 us of host time)
    const size_t cap = (size_t)h->pcg_cap_iters;
    std::vector<double> hblk(3 * cap + 8), hpd(G_read);
    double hscal[S_COUNT];
    BJ_CUDA(cudaMemcpyAsync(hblk.data(), alpha, sizeof(double) * hblk.size(), cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaMemcpyAsync(hpd.data(), PD, sizeof(double) * G_read, cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaMemcpyAsync(hscal, scal, sizeof(hscal), cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaStreamSynchronize(st));
    const double *ha = hblk.data(), *hb = hblk.data() + cap, *hr = hblk.data() + 2 * cap;
    memcpy(hflags, hblk.data() + 3 * cap, sizeof(hflags));

    const int it = hflags[1];
    res->iters = it;
    res->converged = hflags[2];
    res->relres = it > 0 ? hr[it - 1] : 0.0;
    double dd = 0.0;
    for (int g = 0; g < G_read; ++g) dd += hpd[g];
    res->true_relres = hscal[S_BB] > 0.0 ? sqrt(dd / hscal[S_BB]) : 0.0;
    res->lmin = res->lmax = 0.0;
    // CG-Lanczos: T = tridiag(e; d) with d_0 = 1/a_0, d_j = 1/a_j + bt_{j-1}/a_{j-1}, e_j = sqrt(bt_j)/a_j
    const int nb = (it > 0 && hflags[2]) ? it - 1 : it;  // a run stopped by rtol has one beta fewer
    const int kt = std::min(it, nb + 1);
    if (kt >= 1) {
        std::vector<double> d(kt), off(kt > 1 ? kt - 1 : 1);
        for (int j = 0; j < kt; ++j) d[j] = 1.0 / ha[j] + (j > 0 ? hb[j - 1] / ha[j - 1] : 0.0);
        for (int j = 0; j + 1 < kt; ++j) off[j] = sqrt(hb[j] > 0.0 ? hb[j] : 0.0) / ha[j];
        res->lmin = tridiag_eig_k(kt, d.data(), off.data(), 0);
        res->lmax = tridiag_eig_k(kt, d.data(), off.data(), kt - 1);
    }
    if (res->alpha_host) std::copy(ha, ha + it, res->alpha_host);
    if (res->beta_host) std::copy(hb, hb + std::max(nb, 0), res->beta_host);
    if (res->relres_host) std::copy(hr, hr + it, res->relres_host);
    return BJ_OK;
}

// Lanczos on M^-1 A in the M inner product: one pass over the factor per step.  With z_k = M^-1 r_k,
// bt_k^2 = r_k . z_k (bt_0 only normalises):
//   q = A z_k;  al_k = (z_k . q) / bt_k^2;  r_{k+1} = q / bt_k - (al_k / bt_k) r_k - (bt_k / bt_{k-1}) r_{k-1};  z_{k+1} = M^-1 r_{k+1}
// T = tridiag(bt_1..; al_0..) is the Lanczos matrix of L^-1 A L^-T started at L^-1 r_0.  Vectors stay unnormalised (the
// scalars carry the scaling), so a step is TWO kernels on the fused path: the tile SpMV with its dot hook, and the solve
// pair whose input is combined on the fly (PcgHook mode 1) and which finishes r_{k+1} . z_{k+1}.  No reorthogonalisation.
int mlanczos_run(bj_handle_s* h, const bj_lanczos_opts_t* o, bj_lanczos_result_t* res)
{
    const int64_t n = h->n;
    const int m = o->iters;
    const double tol = o->breakdown_tol > 0.0 ? o->breakdown_tol : BJ_DEFAULT_BREAKDOWN_TOL;
    cudaStream_t st = h->stream;
    PcgWs ws;
    int rc = pcg_workspace(h, m + 1, ws);
    if (rc != BJ_OK) return rc;
    double* rcur = ws.r;
    double* rprev = ws.p;
    double *z = ws.z, *q = ws.q, *alpha = ws.alpha, *bsq = ws.beta, *scal = ws.scal;  // bsq[0..m]
    int* flags = ws.flags;
    const size_t fcap = ws.fcap;
    const int G = (int)std::max<int64_t>(1, std::min<int64_t>(kMaxPartials, (n + 1023) / 1024));
    const bool pdl = h->pdl;
    cudaError_t e = cudaSuccess;
#define BJ_LAUNCH(grid, kernel, ...)                                                            \
    do {                                                                                        \
        e = launch_kernel(kernel, dim3(grid), dim3(kReduceThreads), 0, st, pdl, __VA_ARGS__);   \
        if (e != cudaSuccess) { set_cuda_error(e, #kernel); return BJ_ERR_CUDA; }               \
        h->launches++;                                                                          \
    } while (0)
    if (o->v0) {
        BJ_CUDA(cudaMemcpyAsync(rcur, o->v0, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
    } else {
        rc = launch_seeded_vector(h, o->seed, rcur);
        if (rc != BJ_OK) return rc;
    }
    BJ_CUDA(cudaMemsetAsync(rprev, 0, sizeof(double) * n, st));
    rc = launch_solve(h, 2, rcur, z);  // z_0 = M^-1 r_0  (b = 0: copy)
    if (rc != BJ_OK) return rc;
    BJ_LAUNCH(G, pcg_pq_kernel, n, (const double*)rcur, (const double*)z, ws.PRa, (const int*)flags);
    BJ_LAUNCH(1, pcg_scalar_kernel, (const double*)ws.PRa, G, bsq, (const int*)flags);  // bt_0^2

    const bool fused = h->spmv_kernel == 1 && lanczos_fusable(h) && h->opt_pcg_fuse != 0;
    unsigned* tickets = reinterpret_cast<unsigned*>(flags + 4);
    LzReduce red_zp{ws.FP, scal + S_PQ, tickets + 0, (int)fcap};
    PcgHook hook{};
    hook.mode = 1; hook.q = q; hook.pq = scal + S_PQ; hook.alpha = alpha; hook.flags = flags; hook.bsq = bsq;
    hook.red_rr = LzReduce{ws.FP + fcap, scal + S_RR, tickets + 1, (int)fcap};
    for (int k = 0; k < m; ++k) {
        if (fused) {
            rc = launch_spmv_stream(h, z, q, false, nullptr, z, &red_zp);  // K1: q = A z_k, z_k . q
            if (rc != BJ_OK) return rc;
            hook.r = rcur; hook.x = rprev; hook.k = k;
            hook.red_rz = LzReduce{ws.FP + 2 * fcap, bsq + k + 1, tickets + 2, (int)fcap};
            rc = launch_solve(h, 2, nullptr, z, nullptr, nullptr, &hook);  // K2: r_{k+1}, z_{k+1}, bt_{k+1}^2
            if (rc != BJ_OK) return rc;
        } else {
            rc = launch_spmv(h, z, q);
            if (rc != BJ_OK) return rc;
            BJ_LAUNCH(G, pcg_pq_kernel, n, (const double*)z, (const double*)q, ws.PQ, (const int*)flags);
            BJ_LAUNCH(G, mlz_combine_kernel, n, (const double*)q, (const double*)rcur, rprev, (const double*)ws.PQ, G,
                      (const double*)bsq, k, alpha);
            rc = launch_solve(h, 2, rprev, z);
            if (rc != BJ_OK) return rc;
            BJ_LAUNCH(G, pcg_pq_kernel, n, (const double*)rprev, (const double*)z, ws.PRa, (const int*)flags);
            BJ_LAUNCH(1, pcg_scalar_kernel, (const double*)ws.PRa, G, bsq + k + 1, (const int*)flags);
        }
        std::swap(rcur, rprev);  // r_{k+1} was written over r_{k-1}
    }
#undef BJ_LAUNCH
    std::vector<double> a(m), b2(m + 1), b(m);
    BJ_CUDA(cudaMemcpyAsync(a.data(), alpha, sizeof(double) * m, cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaMemcpyAsync(b2.data(), bsq, sizeof(double) * (m + 1), cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaStreamSynchronize(st));
    if (!(b2[0] > 0.0) || !std::isfinite(b2[0])) return BJ_ERR_INVALID_ARG;  // r_0 = 0 (or not finite)
    int me = 0;
    double amax = 0.0;
    for (int j = 0; j < m; ++j) {
        if (!std::isfinite(a[j])) break;
        b[j] = b2[j + 1] > 0.0 ? sqrt(b2[j + 1]) : 0.0;
        amax = std::max(amax, fabs(a[j]));
        me = j + 1;
        if (!(b[j] > tol * amax)) break;  // breakdown: the steps after it computed nothing meaningful and are dropped
    }
    if (me < 1) return BJ_ERR_CUDA;
    lanczos_fill_result(me, a.data(), b.data(), res);
    return BJ_OK;
}

}  // namespace bj
