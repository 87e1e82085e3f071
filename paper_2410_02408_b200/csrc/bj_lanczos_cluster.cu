// Launch-bound sizes, second form: the whole m-step Lanczos run of bj_lanczos.cu as ONE kernel of ONE thread-block CLUSTER
// of eight CTAs -- sixteen when eight cannot hold the basis (N = 4096 at m = 50) -- (bj_lanczos_small.cu runs it on one CTA: its reorthogonalisation re-reads the basis four times per step and
// only ~20 basis vectors of N = 1024 fit beside the work vectors, the rest comes through one SM's L2 port: 17 us per step).
// Here CTA r owns a contiguous range of diagonal blocks and their rows; its slice of EVERY basis vector stays in its
// shared memory (8 x 200 KB for the basis), the operator's block solves and all vector updates are local, and the CTAs
// exchange through distributed shared memory only
//   * the slice of t = L^-T v_j (the SpMV reads arbitrary columns: every CTA keeps the full vector),
//   * the partial sums of alpha_j, of the reorthogonalisation coefficients (two passes) and of beta_{j+1}:
// each CTA pushes its partials into slot r of every CTA's exchange buffer, every CTA adds the eight slots in the same
// order, so all CTAs hold bit-identical scalars and take the same branches.  Per step: five exchanges of ~500 cycles and
// about twenty __syncthreads-separated phases of a few hundred cycles each -- the kernel is a latency chain (5.5 us per
// step with full reorthogonalisation over 25 vectors on average, 3.3 us without), not bandwidth-bound anywhere.
// Same recurrence, statement by statement, as lanczos_run (readings 10-13); the operator is the
// arithmetic of solve_small_kernel (thread per block, interleaved packed factors) and of a row-per-thread CSR product
// summed left to right.  Block sizes b <= 8 and b = 0.
#include <cooperative_groups.h>
#include <math.h>
#include <stdio.h>

#include <algorithm>
#include <atomic>

#include "bj_cluster.cuh"

namespace cg = cooperative_groups;

namespace bj {

namespace {

struct ClusterLzParams {
    int n, nnz, nblocks, m, reorth;
    int bpc;          // diagonal blocks per CTA (the last CTAs may own fewer, or none)
    int nl_max;       // rows per CTA at most (bpc * b, or bpc for b = 0)
    int ld;           // leading dimension of the basis slice Vt[row][vector] (odd: conflict-free in both passes)
    int row_in_regs;  // nl_max <= kClThreads and no row longer than kClRowReg
    int groups_max;   // interleave groups of factors a CTA copies at most
    double tol;
    const int32_t* rp;
    const int32_t* ci;
    const double* val;
    const double* fac;  // fac_small (interleaved packed, reciprocal diagonals) or null
    const double* v0;
    double* alpha;      // [m] global
    double* beta;       // [m] global
    int* done;          // [0] stop flag, [1] m_eff, [2] invalid start vector
};

template <int B, int CS>
__global__ void __launch_bounds__(kClThreads)
lanczos_cluster_kernel(const ClusterLzParams p)  // launched as clusters of CS CTAs (launch attribute)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cg::cluster_group cl = cg::this_cluster();
    const int rank = (int)cl.block_rank();
    const int n = p.n, tid = threadIdx.x;
    constexpr int BB = B > 0 ? B : 1;                  // rows per unit (a "block" of the b = 0 handle is one row)
    constexpr int P = B * (B + 1) / 2;
    const int units = B > 0 ? p.nblocks : n;
    const int k_lo = min(units, rank * p.bpc), k_hi = min(units, k_lo + p.bpc);
    const int row_lo = k_lo * BB;
    const int nl = min(n, k_hi * BB) - row_lo;          // rows of this CTA (0 for a CTA beyond the last block)
    const int g_lo = k_lo >> 5;
    const int pm = (p.m + 2) & ~1;
    // red | dpart | c | xch[2][8][pm] | t_full[n] | tl | u | w | vc | vp (nl_max each) | fac | Vt[nl_max][ld] | 2 mbarriers
    double* red = reinterpret_cast<double*>(smem_raw);
    double* dpart = red + kClWarps;                     // (slice, vector) partials of a dot sweep
    double* c = dpart + kClThreads;
    double* xch = c + pm;
    double* t_full = xch + 2 * CS * pm;
    double* tl = t_full + ((n + 1) & ~1);
    double* u = tl + p.nl_max;
    double* w = u + p.nl_max;
    double* vc = w + p.nl_max;
    double* vp = vc + p.nl_max;
    double* sf = vp + p.nl_max;
    double* Vt = sf + (size_t)p.groups_max * P * kInterleave;
    Exchange x;
    x.bar = reinterpret_cast<uint64_t*>(Vt + (p.reorth ? (size_t)p.nl_max * p.ld : 0));
    x.e = 0;
    x.rank = rank;
    if (tid == 0) {
        mbar_init(&x.bar[0], 1);
        mbar_init(&x.bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cl.sync();  // every CTA's barriers exist before a peer signals them
    if constexpr (B > 0) {
        const int g_hi = k_hi > k_lo ? ((k_hi - 1) >> 5) + 1 : g_lo;
        const double* src = p.fac + (size_t)g_lo * (P * kInterleave);
        for (int e = tid; e < (g_hi - g_lo) * P * kInterleave; e += kClThreads) sf[e] = src[e];
    }
    // row `row_lo + tid` of the matrix in registers
    double rv[kClRowReg];
    int rc[kClRowReg];
    int rlen = 0;
#pragma unroll
    for (int q = 0; q < kClRowReg; ++q) { rv[q] = 0.0; rc[q] = 0; }
    if (p.row_in_regs && tid < nl) {
        const int s0 = p.rp[row_lo + tid];
        rlen = p.rp[row_lo + tid + 1] - s0;
#pragma unroll
        for (int q = 0; q < kClRowReg; ++q)
            if (q < rlen) { rv[q] = p.val[s0 + q]; rc[q] = p.ci[s0 + q]; }
    }
    // v_1 = v0 / ||v0||
    double s = 0.0;
    for (int i = tid; i < nl; i += kClThreads) { const double x0 = p.v0[row_lo + i]; s = fma(x0, x0, s); }
    s = cl_cta_sum(s, red);
    const double nrm = sqrt(cluster_allreduce_scalar<CS>(x, s, xch, pm));
    if (!(nrm > 0.0) || isinf(nrm)) {  // zero or non-finite start vector: invalid argument (uniform over the cluster)
        if (rank == 0 && tid == 0) { p.done[0] = 1; p.done[2] = 1; }
        cl.sync();
        return;
    }
    for (int i = tid; i < nl; i += kClThreads) {
        const double x0 = p.v0[row_lo + i] / nrm;
        vc[i] = x0;
        vp[i] = 0.0;
        if (p.reorth) Vt[(size_t)i * p.ld] = x0;
    }
    double beta_j = 0.0, amax = 0.0;
    __syncthreads();
#ifdef BJ_CL_PROF
    long long tk[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, t0 = clock64(), t1;
#define BJ_TICK(k) do { t1 = clock64(); tk[k] += t1 - t0; t0 = t1; } while (0)
#else
#define BJ_TICK(k) do { } while (0)
#endif
    for (int j = 0; j < p.m; ++j) {
        // ---- t = L^-T v_j on the own blocks, then to every CTA (the SpMV reads arbitrary columns) ----
        cluster_solve<B, 1>(n, k_lo, k_hi, g_lo, sf, vc, tl);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // tl is read by the async proxy (bulk copies)
        __syncthreads();
        BJ_TICK(0);
        exchange_all_bulk<CS>(x, tl, nl, t_full, row_lo, n);
        BJ_TICK(1);
        // ---- u = A t (own rows, left to right: the oracle's order), w = L^-1 u ----
        if (p.row_in_regs) {
            if (tid < nl) {
                double acc = 0.0;
#pragma unroll
                for (int q = 0; q < kClRowReg; ++q)
                    if (q < rlen) acc = fma(rv[q], t_full[rc[q]], acc);
                u[tid] = acc;
            }
        } else {
            for (int i = tid; i < nl; i += kClThreads) {
                double acc = 0.0;
                const int e = p.rp[row_lo + i + 1];
                for (int q = p.rp[row_lo + i]; q < e; ++q) acc = fma(p.val[q], t_full[p.ci[q]], acc);
                u[i] = acc;
            }
        }
        __syncthreads();
        cluster_solve<B, 0>(n, k_lo, k_hi, g_lo, sf, u, w);
        __syncthreads();
        BJ_TICK(2);
        // ---- w -= beta_j v_{j-1};  alpha_j = v_j . w;  w -= alpha_j v_j ----
        double pa = 0.0;
        for (int i = tid; i < nl; i += kClThreads) {
            double wi = w[i];
            if (j > 0) { wi -= beta_j * vp[i]; w[i] = wi; }
            pa = fma(vc[i], wi, pa);
        }
        pa = cl_cta_sum(pa, red);
        BJ_TICK(3);
        const double a = cluster_allreduce_scalar<CS>(x, pa, xch, pm);
        BJ_TICK(4);
        for (int i = tid; i < nl; i += kClThreads) w[i] -= a * vc[i];
        __syncthreads();
        // ---- full reorthogonalisation, classical Gram-Schmidt twice over v_1 .. v_j: c = V^T w, then w -= V c ----
        if (p.reorth) {
            const int nv = j + 1;
            // dots: thread = (vector q, row slice): consecutive lanes read consecutive vectors of one row of Vt
            // (conflict-free), w[row] is a broadcast; no shuffles.  64 vectors per sweep, four row slices whose partials
            // are added in slice order.  (Measured and dropped: narrower sweeps with more slices for few vectors, four
            // accumulators with eight loads in flight, 512 threads -- all slower; the pass is a latency chain.)
            constexpr int cols = kClDotCols, slices = kClThreads / kClDotCols;
            const int per = (nl + slices - 1) / slices;
            const int qc = tid & (cols - 1), sl = tid / cols;
            const int i0 = min(nl, sl * per), i1 = min(nl, i0 + per);
            BJ_TICK(5);
            for (int pass = 0; pass < 2; ++pass) {
                // the coefficient exchange is armed first; the thread that finishes a vector's CTA sum pushes it straight
                // from its register into slot `rank` of the eight CTAs
                double* xb = xch + (size_t)(x.e & 1) * CS * pm;
                uint64_t* bar = x.bar + (x.e & 1);
                const uint32_t parity = (uint32_t)((x.e >> 1) & 1);
                if (tid == 0) mbar_expect_tx(bar, (uint32_t)nv * 8u * CS);
                for (int q0 = 0; q0 < nv; q0 += cols) {
                    const int q = q0 + qc;
                    double s0 = 0.0, s1 = 0.0;
                    if (q < nv) {
                        const double* col = Vt + q;
                        int i = i0;
                        for (; i + 1 < i1; i += 2) {
                            s0 = fma(col[(size_t)i * p.ld], w[i], s0);
                            s1 = fma(col[(size_t)(i + 1) * p.ld], w[i + 1], s1);
                        }
                        if (i < i1) s0 = fma(col[(size_t)i * p.ld], w[i], s0);
                    }
                    if (q0 > 0) __syncthreads();  // dpart is reused by the next sweep (more than 64 vectors)
                    dpart[sl * cols + qc] = s0 + s1;
                    __syncthreads();
                    if (tid < cols && q < nv) {
                        double sq = dpart[tid];
#pragma unroll
                        for (int r = 1; r < slices; ++r) sq += dpart[r * cols + tid];
                        const uint32_t dst = smem_u32(xb + rank * pm + q), bar_s = smem_u32(bar);
#pragma unroll
                        for (int r = 0; r < CS; ++r) st_async_f64(mapa_u32(dst, r), sq, mapa_u32(bar_s, r));
                    }
                }
                BJ_TICK(6);
                mbar_wait(bar, parity);
                ++x.e;
                for (int q = tid; q < nv; q += kClThreads) {
                    double sc = 0.0;
#pragma unroll
                    for (int r = 0; r < CS; ++r) sc += xb[r * pm + q];
                    c[q] = sc;
                }
                __syncthreads();
                BJ_TICK(7);
                // w -= V c: thread per row, the row of Vt is contiguous; lanes are ld (odd) doubles apart: conflict-free
                for (int i = tid; i < nl; i += kClThreads) {
                    const double* row = Vt + (size_t)i * p.ld;
                    double wi = w[i];
                    int q = 0;
                    for (; q < nv; ++q) wi -= c[q] * row[q];
                    w[i] = wi;
                }
                __syncthreads();
                BJ_TICK(8);
            }
        }
        // ---- beta_{j+1} = ||w||, bookkeeping, breakdown test ----
        double pb = 0.0;
        for (int i = tid; i < nl; i += kClThreads) pb = fma(w[i], w[i], pb);
        pb = cl_cta_sum(pb, red);
        BJ_TICK(9);
        const double bn = sqrt(cluster_allreduce_scalar<CS>(x, pb, xch, pm));
        BJ_TICK(10);
        amax = fabs(a) > amax ? fabs(a) : amax;
        const bool brk = !(bn > p.tol * amax);
        if (rank == 0 && tid == 0) {
            p.alpha[j] = a;
            p.beta[j] = bn;
            p.done[1] = j + 1;
            if (brk) p.done[0] = 1;
        }
        if (brk || j + 1 == p.m) break;  // uniform over the cluster: every CTA holds the same bits
        __syncthreads();
        for (int i = tid; i < nl; i += kClThreads) {
            const double x1 = w[i] / bn;
            vp[i] = vc[i];
            vc[i] = x1;
            if (p.reorth) Vt[(size_t)i * p.ld + (j + 1)] = x1;
        }
        beta_j = bn;
        __syncthreads();
        BJ_TICK(11);
    }
#ifdef BJ_CL_PROF
    if (tid == 0 && rank == 0)
        printf("solveT %lld xchT %lld spmv+solve %lld asum %lld axch %lld axpy %lld | dot %lld cxch %lld upd %lld | bsum %lld bxch %lld norm %lld (cycles/step)\n",
               tk[0] / p.m, tk[1] / p.m, tk[2] / p.m, tk[3] / p.m, tk[4] / p.m, tk[5] / p.m, tk[6] / p.m, tk[7] / p.m, tk[8] / p.m, tk[9] / p.m,
               tk[10] / p.m, tk[11] / p.m);
#endif
    cl.sync();  // no CTA leaves while another may still address its shared memory
}

struct ClusterGeom {
    int bpc, nl_max, ld, groups_max;
    size_t smem;
};

ClusterGeom cluster_geometry(const bj_handle_s* h, int m, bool reorth, int cs)
{
    ClusterGeom g;
    const int bb = h->solve_kind == 1 ? h->b : 1;
    const int64_t units = h->solve_kind == 1 ? h->nblocks : h->n;
    g.bpc = (int)((units + cs - 1) / cs);
    g.nl_max = g.bpc * bb;
    g.ld = m | 1;
    g.groups_max = h->solve_kind == 1 ? (g.bpc + kInterleave - 1) / kInterleave + 1 : 0;
    const size_t pm = (size_t)((m + 2) & ~1);
    size_t d = kClWarps + kClThreads + pm + 2 * (size_t)cs * pm + (((size_t)h->n + 1) & ~(size_t)1) + 5 * (size_t)g.nl_max +
               (size_t)g.groups_max * h->packed * kInterleave;
    if (reorth) d += (size_t)g.nl_max * g.ld;
    g.smem = d * 8 + 16 + 16;
    return g;
}

template <int B, int CS>
cudaError_t cluster_prepare(size_t smem, int* max_clusters)
{
    static std::atomic<bool> configured[64];
    cudaError_t e = ensure_big_smem(lanczos_cluster_kernel<B, CS>, configured);
    if (e == cudaSuccess && CS > 8) e = cudaFuncSetAttribute(lanczos_cluster_kernel<B, CS>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
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
    return cudaOccupancyMaxActiveClusters(max_clusters, lanczos_cluster_kernel<B, CS>, &cfg);
}

template <int B, int CS>
cudaError_t cluster_launch(const ClusterLzParams& p, size_t smem, cudaStream_t st)
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
    return cudaLaunchKernelEx(&cfg, lanczos_cluster_kernel<B, CS>, p);
}

// which cluster size serves (h, m, reorth): 8 when a CTA's share fits its shared memory, else 16 (opt-in size: half the
// share per CTA) when that fits and the device can place such a cluster, else 0.  The answer is kept in the handle.
int cluster_pick(bj_handle_s* h, int m, bool reorth)
{
    if (env_int("BJ_LANCZOS_CLUSTER", 1) == 0) return 0;
    if (h->var_perm || !(h->solve_kind == 0 || (h->solve_kind == 1 && !h->tri)) || m > 1024 || h->n > 16384 || h->n < kClusterMax ||
        h->nnz == 0)
        return 0;
    if (h->cl_m == m && h->cl_reorth == (reorth ? 1 : 0)) return h->cl_cs;
    int cs = 0;
    constexpr size_t kBudget = 220 * 1024;
    if (cluster_geometry(h, m, reorth, 8).smem <= kBudget) {
        cs = 8;
    } else if (cluster_geometry(h, m, reorth, 16).smem <= kBudget && cluster_geometry(h, m, reorth, 16).nl_max <= kClThreads &&
               h->max_row_nnz <= kClRowReg && env_int("BJ_LANCZOS_CLUSTER16", 1) != 0) {
        // (only with the CTA's rows of the matrix in registers: N = 16384 without them measured 0.82 ms for 50 steps
        // against 0.67 ms on the multi-launch path)
        const size_t smem = cluster_geometry(h, m, reorth, 16).smem;
        int nc = 0;
        cudaError_t e = cudaSuccess;
#define BJ_CASE(B) case B: e = cluster_prepare<B, 16>(smem, &nc); break;
        switch (h->solve_kind == 1 ? h->b : 0) {
            BJ_CASE(0) BJ_CASE(1) BJ_CASE(2) BJ_CASE(3) BJ_CASE(4) BJ_CASE(5) BJ_CASE(6) BJ_CASE(7) BJ_CASE(8)
            default: break;
        }
#undef BJ_CASE
        if (e != cudaSuccess) cudaGetLastError();  // the device cannot place it: not an error of the call
        cs = (e == cudaSuccess && nc >= 1) ? 16 : 0;
    }
    h->cl_m = m;
    h->cl_reorth = reorth ? 1 : 0;
    h->cl_cs = cs;
    return cs;
}

}  // namespace

// The cluster form is used when a CTA's share of the basis fits its shared memory beside the work vectors (N = 1024, m = 50:
// 52 KB of basis per CTA of an eight-CTA cluster; N = 4096: 104 KB per CTA of a sixteen-CTA cluster); otherwise the
// single-CTA kernel (basis through L2) or the multi-launch path run.
bool lanczos_cluster_usable(bj_handle_s* h, int m, bool reorth) { return cluster_pick(h, m, reorth) != 0; }

int launch_lanczos_cluster(bj_handle_s* h, int m, bool reorth, double tol, const double* v0, double* alpha, double* beta, int* done)
{
    const int cs = cluster_pick(h, m, reorth);
    if (cs == 0) return BJ_ERR_INVALID_ARG;
    const ClusterGeom g = cluster_geometry(h, m, reorth, cs);
    ClusterLzParams p;
    p.n = (int)h->n; p.nnz = (int)h->nnz; p.nblocks = (int)h->nblocks; p.m = m;
    p.reorth = reorth ? 1 : 0;
    p.bpc = g.bpc; p.nl_max = g.nl_max; p.ld = g.ld; p.groups_max = g.groups_max;
    p.row_in_regs = (g.nl_max <= kClThreads && h->max_row_nnz <= kClRowReg) ? 1 : 0;
    p.tol = tol;
    p.rp = h->row_ptr; p.ci = h->col_idx; p.val = h->val;
    p.fac = h->solve_kind == 1 ? h->fac_small : nullptr;
    p.v0 = v0; p.alpha = alpha; p.beta = beta; p.done = done;
    cudaError_t e = cudaSuccess;
#define BJ_CASE(B)                                                                                  \
    case B:                                                                                         \
        if (cs == 8) {                                                                              \
            e = cluster_prepare<B, 8>(g.smem, nullptr);                                             \
            if (e == cudaSuccess) e = cluster_launch<B, 8>(p, g.smem, h->stream);                   \
        } else {                                                                                    \
            e = cluster_prepare<B, 16>(g.smem, nullptr);                                            \
            if (e == cudaSuccess) e = cluster_launch<B, 16>(p, g.smem, h->stream);                  \
        }                                                                                           \
        break;
    switch (h->solve_kind == 1 ? h->b : 0) {
        BJ_CASE(0) BJ_CASE(1) BJ_CASE(2) BJ_CASE(3) BJ_CASE(4) BJ_CASE(5) BJ_CASE(6) BJ_CASE(7) BJ_CASE(8)
        default: return BJ_ERR_INVALID_ARG;
    }
#undef BJ_CASE
    if (e != cudaSuccess) { set_cuda_error(e, "lanczos_cluster_kernel"); return BJ_ERR_CUDA; }
    h->launches++;
    return BJ_OK;
}

}  // namespace bj
