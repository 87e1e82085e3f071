// Launch-bound sizes (the paper's N = 2^10, 2^12: PAPER.md:365): the WHOLE preconditioned CG run of bj_pcg.cu -- start,
// iterations, stopping test, the paper's residual ||A x - b|| / ||b|| -- as ONE kernel of one thread-block cluster
// (8 CTAs, or 16 when 8 cannot hold their share).  Same design as bj_lanczos_cluster.cu: CTA r owns a contiguous range of
// diagonal blocks and their rows; x, r, z, p, q are local slices in shared memory; per iteration the CTAs exchange the
// slice of p (the SpMV reads arbitrary columns: one bulk DSMEM copy per peer) and three scalars in two exchanges
// (p.q; r.r together with r.z), each pushed with st.async from registers and counted on the receiver's mbarrier.
// Same recurrence and the same scalar formulas as the multi-launch iteration of pcg_run (Hestenes-Stiefel; a_k = rho / p.q,
// relres_k = sqrt(r.r / b.b), bt_k = rho_new / rho); sums are grouped per CTA instead of per 1184 chunks (rounding only).
// An iteration of the multi-launch path is three to seven launches of ~4 us for 0.15 MB of data.
#include <cooperative_groups.h>
#include <math.h>

#include <algorithm>
#include <atomic>

#include "bj_cluster.cuh"

namespace cg = cooperative_groups;

namespace bj {

namespace {

struct ClusterPcgParams {
    int n, nblocks, m;
    int bpc, nl_max, groups_max, row_in_regs;
    double rtol;
    const int32_t* rp;
    const int32_t* ci;
    const double* val;
    const double* fac;
    const double* b;
    double* x;
    double* alpha;   // [m]
    double* beta;    // [m]
    double* relres;  // [m]
    double* scal;    // [0] = b.b
    double* pd;      // [0] = ||A x - b||^2
    int* flags;      // [0] stop, [1] iterations done, [2] converged
};

constexpr int kPcgPm = 2;  // doubles per exchange slot

template <int B, int CS>
__global__ void __launch_bounds__(kClThreads)
pcg_cluster_kernel(const ClusterPcgParams p)  // launched as one cluster of CS CTAs
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cg::cluster_group cl = cg::this_cluster();
    const int rank = (int)cl.block_rank();
    const int n = p.n, tid = threadIdx.x;
    constexpr int BB = B > 0 ? B : 1;
    constexpr int P = B * (B + 1) / 2;
    const int units = B > 0 ? p.nblocks : n;
    const int k_lo = min(units, rank * p.bpc), k_hi = min(units, k_lo + p.bpc);
    const int row_lo = k_lo * BB;
    const int nl = min(n, k_hi * BB) - row_lo;
    const int g_lo = k_lo >> 5;
    // red | xch[2][CS][2] | t_full[n] | x | r | z | p | q | u (nl_max each) | fac | 2 mbarriers
    double* red = reinterpret_cast<double*>(smem_raw);
    double* xch = red + kClWarps;
    double* t_full = xch + 2 * CS * kPcgPm;
    double* xs = t_full + ((n + 1) & ~1);
    double* r = xs + p.nl_max;
    double* z = r + p.nl_max;
    double* pv = z + p.nl_max;
    double* q = pv + p.nl_max;
    double* u = q + p.nl_max;
    double* sf = u + p.nl_max;
    Exchange x;
    x.bar = reinterpret_cast<uint64_t*>(sf + (size_t)p.groups_max * P * kInterleave);
    x.e = 0;
    x.rank = rank;
    if (tid == 0) {
        mbar_init(&x.bar[0], 1);
        mbar_init(&x.bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cl.sync();
    if constexpr (B > 0) {
        const int g_hi = k_hi > k_lo ? ((k_hi - 1) >> 5) + 1 : g_lo;
        const double* src = p.fac + (size_t)g_lo * (P * kInterleave);
        for (int e = tid; e < (g_hi - g_lo) * P * kInterleave; e += kClThreads) sf[e] = src[e];
    }
    double rv[kClRowReg];
    int rc[kClRowReg];
    int rlen = 0;
#pragma unroll
    for (int e = 0; e < kClRowReg; ++e) { rv[e] = 0.0; rc[e] = 0; }
    if (p.row_in_regs && tid < nl) {
        const int s0 = p.rp[row_lo + tid];
        rlen = p.rp[row_lo + tid + 1] - s0;
#pragma unroll
        for (int e = 0; e < kClRowReg; ++e)
            if (e < rlen) { rv[e] = p.val[s0 + e]; rc[e] = p.ci[s0 + e]; }
    }
    // out = A t_full on the own rows, left to right (the oracle's order)
    auto spmv_own = [&](double* out) {
        if (p.row_in_regs) {
            if (tid < nl) {
                double acc = 0.0;
#pragma unroll
                for (int e = 0; e < kClRowReg; ++e)
                    if (e < rlen) acc = fma(rv[e], t_full[rc[e]], acc);
                out[tid] = acc;
            }
        } else {
            for (int i = tid; i < nl; i += kClThreads) {
                double acc = 0.0;
                const int e1 = p.rp[row_lo + i + 1];
                for (int e = p.rp[row_lo + i]; e < e1; ++e) acc = fma(p.val[e], t_full[p.ci[e]], acc);
                out[i] = acc;
            }
        }
    };
    // z = M^-1 r on the own blocks (b = 0: copy)
    auto precond = [&]() {
        cluster_solve<B, 0>(n, k_lo, k_hi, g_lo, sf, r, u);
        __syncthreads();
        cluster_solve<B, 1>(n, k_lo, k_hi, g_lo, sf, u, z);
        __syncthreads();
    };
    // ---- start: x = 0, r = b, b.b, z = M^-1 r, p = z, rho = r.z ----
    double s = 0.0;
    for (int i = tid; i < nl; i += kClThreads) {
        const double bi = p.b[row_lo + i];
        r[i] = bi;
        xs[i] = 0.0;
        s = fma(bi, bi, s);
    }
    s = cl_cta_sum(s, red);
    const double bb = cluster_allreduce_scalar<CS>(x, s, xch, kPcgPm);
    if (rank == 0 && tid == 0) { p.scal[0] = bb; p.pd[0] = 0.0; }
    if (!(bb > 0.0)) {  // zero (or non-finite) right-hand side: x = 0, no iteration (uniform over the cluster)
        for (int i = tid; i < nl; i += kClThreads) p.x[row_lo + i] = 0.0;
        if (rank == 0 && tid == 0) p.flags[0] = 1;
        cl.sync();
        return;
    }
    __syncthreads();
    precond();
    s = 0.0;
    for (int i = tid; i < nl; i += kClThreads) {
        const double zi = z[i];
        pv[i] = zi;
        s = fma(r[i], zi, s);
    }
    s = cl_cta_sum(s, red);
    double rho = cluster_allreduce_scalar<CS>(x, s, xch, kPcgPm);
    for (int k = 0; k < p.m; ++k) {
        // ---- q = A p ----
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // pv is read by the async proxy (bulk copies)
        __syncthreads();
        exchange_all_bulk<CS>(x, pv, nl, t_full, row_lo, n);
        spmv_own(q);
        __syncthreads();
        s = 0.0;
        for (int i = tid; i < nl; i += kClThreads) s = fma(pv[i], q[i], s);
        s = cl_cta_sum(s, red);
        const double pq = cluster_allreduce_scalar<CS>(x, s, xch, kPcgPm);
        const double a = rho / pq;
        // ---- x += a p, r -= a q, z = M^-1 r ----
        double srr = 0.0;
        for (int i = tid; i < nl; i += kClThreads) {
            xs[i] = fma(a, pv[i], xs[i]);
            const double ri = r[i] - a * q[i];
            r[i] = ri;
            srr = fma(ri, ri, srr);
        }
        __syncthreads();
        precond();
        double srz = 0.0;
        for (int i = tid; i < nl; i += kClThreads) srz = fma(r[i], z[i], srz);
        srr = cl_cta_sum(srr, red);
        srz = cl_cta_sum(srz, red);
        cluster_allreduce_scalar2<CS>(x, srr, srz, xch, kPcgPm);
        const double rel = sqrt(srr / bb);
        const bool stop = rel <= p.rtol;
        const double bt = srz / rho;
        if (rank == 0 && tid == 0) {
            p.alpha[k] = a;
            p.relres[k] = rel;
            p.flags[1] = k + 1;
            if (stop) { p.flags[0] = 1; p.flags[2] = 1; }
            else p.beta[k] = bt;
        }
        if (stop) break;  // uniform: every CTA holds the same bits
        for (int i = tid; i < nl; i += kClThreads) pv[i] = fma(bt, pv[i], z[i]);
        rho = srz;
    }
    // ---- the paper's metric from x itself: ||A x - b||^2, and x to the caller ----
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    exchange_all_bulk<CS>(x, xs, nl, t_full, row_lo, n);
    spmv_own(q);
    __syncthreads();
    s = 0.0;
    for (int i = tid; i < nl; i += kClThreads) {
        const double d = q[i] - p.b[row_lo + i];
        s = fma(d, d, s);
        p.x[row_lo + i] = xs[i];
    }
    s = cl_cta_sum(s, red);
    const double dd = cluster_allreduce_scalar<CS>(x, s, xch, kPcgPm);
    if (rank == 0 && tid == 0) p.pd[0] = dd;
    cl.sync();  // no CTA leaves while another may still address its shared memory
}

struct PcgGeom {
    int bpc, nl_max, groups_max;
    size_t smem;
};

PcgGeom pcg_geometry(const bj_handle_s* h, int cs)
{
    PcgGeom g;
    const int bb = h->solve_kind == 1 ? h->b : 1;
    const int64_t units = h->solve_kind == 1 ? h->nblocks : h->n;
    g.bpc = (int)((units + cs - 1) / cs);
    g.nl_max = g.bpc * bb;
    g.groups_max = h->solve_kind == 1 ? (g.bpc + kInterleave - 1) / kInterleave + 1 : 0;
    const size_t d = kClWarps + 2 * (size_t)cs * kPcgPm + (((size_t)h->n + 1) & ~(size_t)1) + 6 * (size_t)g.nl_max +
                     (size_t)g.groups_max * h->packed * kInterleave;
    g.smem = d * 8 + 16 + 16;
    return g;
}

template <int B, int CS>
cudaError_t pcg_cluster_prepare(size_t smem, int* max_clusters)
{
    static std::atomic<bool> configured[64];
    cudaError_t e = ensure_big_smem(pcg_cluster_kernel<B, CS>, configured);
    if (e == cudaSuccess && CS > 8) e = cudaFuncSetAttribute(pcg_cluster_kernel<B, CS>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess || !max_clusters) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(CS);
    cfg.blockDim = dim3(kClThreads);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CS;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaOccupancyMaxActiveClusters(max_clusters, pcg_cluster_kernel<B, CS>, &cfg);
}

template <int B, int CS>
cudaError_t pcg_cluster_launch(const ClusterPcgParams& p, size_t smem, cudaStream_t st)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(CS);
    cfg.blockDim = dim3(kClThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CS;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, pcg_cluster_kernel<B, CS>, p);
}

// 8 CTAs when a CTA's share fits, else 16 (opt-in cluster size) with the CTA's rows of the matrix in registers, else 0;
// the answer is kept in the handle
int pcg_cluster_pick(bj_handle_s* h)
{
    if (h->pcg_cl_cs >= 0) return h->pcg_cl_cs;
    int cs = 0;
    constexpr size_t kBudget = 220 * 1024;
    const bool shape_ok = env_int("BJ_PCG_CLUSTER", 1) != 0 && !h->var_perm && (h->solve_kind == 0 || (h->solve_kind == 1 && !h->tri)) &&
                          h->n <= 16384 && h->n >= kClusterMax && h->nnz > 0;
    if (shape_ok) {
        if (pcg_geometry(h, 8).smem <= kBudget && (pcg_geometry(h, 8).nl_max <= kClThreads || h->n <= 2048)) {
            cs = 8;
        } else if (pcg_geometry(h, 16).smem <= kBudget && pcg_geometry(h, 16).nl_max <= kClThreads && h->max_row_nnz <= kClRowReg) {
            const size_t smem = pcg_geometry(h, 16).smem;
            int nc = 0;
            cudaError_t e = cudaSuccess;
#define BJ_CASE(B) case B: e = pcg_cluster_prepare<B, 16>(smem, &nc); break;
            switch (h->solve_kind == 1 ? h->b : 0) {
                BJ_CASE(0) BJ_CASE(1) BJ_CASE(2) BJ_CASE(3) BJ_CASE(4) BJ_CASE(5) BJ_CASE(6) BJ_CASE(7) BJ_CASE(8)
                default: break;
            }
#undef BJ_CASE
            if (e != cudaSuccess) cudaGetLastError();
            cs = (e == cudaSuccess && nc >= 1) ? 16 : 0;
        }
    }
    h->pcg_cl_cs = cs;
    return cs;
}

}  // namespace

bool pcg_cluster_usable(bj_handle_s* h) { return pcg_cluster_pick(h) != 0; }

// fills alpha / beta / relres / flags / scal[0] = b.b / pd[0] = ||A x - b||^2 and x; the caller reads them back
int launch_pcg_cluster(bj_handle_s* h, const double* b, double* x, int m, double rtol, double* alpha, double* beta, double* relres,
                       double* scal, double* pd, int* flags)
{
    const int cs = pcg_cluster_pick(h);
    if (cs == 0) return BJ_ERR_INVALID_ARG;
    const PcgGeom g = pcg_geometry(h, cs);
    ClusterPcgParams p;
    p.n = (int)h->n; p.nblocks = (int)h->nblocks; p.m = m;
    p.bpc = g.bpc; p.nl_max = g.nl_max; p.groups_max = g.groups_max;
    p.row_in_regs = (g.nl_max <= kClThreads && h->max_row_nnz <= kClRowReg) ? 1 : 0;
    p.rtol = rtol;
    p.rp = h->row_ptr; p.ci = h->col_idx; p.val = h->val;
    p.fac = h->solve_kind == 1 ? h->fac_small : nullptr;
    p.b = b; p.x = x; p.alpha = alpha; p.beta = beta; p.relres = relres; p.scal = scal; p.pd = pd; p.flags = flags;
    cudaError_t e = cudaSuccess;
#define BJ_CASE(B)                                                                                  \
    case B:                                                                                         \
        if (cs == 8) {                                                                              \
            e = pcg_cluster_prepare<B, 8>(g.smem, nullptr);                                         \
            if (e == cudaSuccess) e = pcg_cluster_launch<B, 8>(p, g.smem, h->stream);               \
        } else {                                                                                    \
            e = pcg_cluster_prepare<B, 16>(g.smem, nullptr);                                        \
            if (e == cudaSuccess) e = pcg_cluster_launch<B, 16>(p, g.smem, h->stream);              \
        }                                                                                           \
        break;
    switch (h->solve_kind == 1 ? h->b : 0) {
        BJ_CASE(0) BJ_CASE(1) BJ_CASE(2) BJ_CASE(3) BJ_CASE(4) BJ_CASE(5) BJ_CASE(6) BJ_CASE(7) BJ_CASE(8)
        default: return BJ_ERR_INVALID_ARG;
    }
#undef BJ_CASE
    if (e != cudaSuccess) { set_cuda_error(e, "pcg_cluster_kernel"); return BJ_ERR_CUDA; }
    h->launches++;
    return BJ_OK;
}

}  // namespace bj
