// CSR SpMV  u = A t  (a6), the dominant byte stream of the preconditioned operator (a7).
//
// Kernel 0  (spmv_vector_kernel): one sub-warp of LPR lanes per row; column/value loads of
//   consecutive rows are contiguous, so a warp's loads coalesce; partial sums are combined with
//   warp shuffles.  It needs no plan and no alignment, handles any row length, and is the
//   fall-back for matrices the streamed kernel cannot take.
// Kernel 1  (spmv_stream_kernel, below): persistent CTAs; a producer thread streams each tile's
//   contiguous col/val (and factor) ranges into a shared-memory ring with 1-D bulk async copies
//   (cp.async.bulk + mbarrier, i.e. the TMA engine: no registers staged, deep memory-level
//   parallelism), consumer warps reduce rows out of shared memory, gather t through L1/L2, and can
//   run the forward block solve y = L^-1 u on the tile before y is written (fuses a7's last factor).
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>
#include <atomic>

#include "bj_device.cuh"
#include "bj_internal.cuh"
#include "bj_lanczos_fuse.cuh"

namespace bj {

int env_int(const char* name, int dflt)
{
    const char* v = getenv(name);
    return v && *v ? atoi(v) : dflt;
}

// ------------------------------------------------------------------------------------------------
// Kernel 0: LPR lanes per row
// ------------------------------------------------------------------------------------------------
template <int LPR>
__global__ void __launch_bounds__(256)
spmv_vector_kernel(int64_t n, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci,
                   const double* __restrict__ val, const double* __restrict__ x, double* __restrict__ y)
{
    pdl_trigger();
    pdl_wait();
    const int64_t gtid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t row = gtid / LPR;
    const int lane = threadIdx.x & (LPR - 1);
    double acc = 0.0;
    if (row < n) {
        const int s = rp[row], e = rp[row + 1];
        for (int p = s + lane; p < e; p += LPR) {
            const int c = ld_stream(ci + p);
            const double v = ld_stream(val + p);
            acc = fma(v, __ldg(x + c), acc);
        }
    }
#pragma unroll
    for (int off = LPR / 2; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off, LPR);
    if (row < n && lane == 0) y[row] = acc;
}

int launch_spmv_vector(bj_handle_s* h, const double* x, double* y)
{
    const int threads = 256;
    const int lpr = h->spmv_lanes;
    const unsigned blocks = (unsigned)((h->n * lpr + threads - 1) / threads);
    KernelScope scope(h, BJ_K_SPMV);
    const bool pdl = h->pdl && !h->prof_on;
    cudaError_t e = cudaSuccess;
#define BJ_CASE(L)                                                                                            \
    case L:                                                                                                   \
        e = launch_kernel(spmv_vector_kernel<L>, blocks, threads, 0, h->stream, pdl, h->n, h->row_ptr, h->col_idx, \
                          h->val, x, y);                                                                      \
        break;
    switch (lpr) {
        BJ_CASE(1) BJ_CASE(2) BJ_CASE(4) BJ_CASE(8) BJ_CASE(16) BJ_CASE(32)
        default: return BJ_ERR_INVALID_ARG;
    }
#undef BJ_CASE
    if (e != cudaSuccess) { set_cuda_error(e, "spmv_vector_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}

// ------------------------------------------------------------------------------------------------
// Kernel 1: persistent, TMA-streamed tiles
//
// A tile is `R` consecutive rows.  Its column indices, values, row pointers and (when fused) the
// packed factors of its diagonal blocks are each ONE contiguous byte range, so one elected
// producer thread moves them with four 1-D bulk async copies (cp.async.bulk -> UBLKCP) into one
// stage of a shared-memory ring; completion is tracked by an mbarrier transaction count.  Bulk
// copies need 16-byte aligned addresses and sizes: ranges are widened to multiples of four
// elements, and the (at most three) elements that would fall past the end of a caller array are
// copied by the producer with plain loads instead.
// Eight consumer warps then (A) reduce the rows out of shared memory, LPR lanes per row, gathering
// t[col] through L1/L2, and (B, fused) run the forward substitution of the tile's diagonal blocks
// from the staged factors, one thread per block, before y is written.  The stage is handed back
// through a second mbarrier.  Tiles are dealt round-robin to the CTAs, so the CTAs resident at any
// time stream neighbouring tiles (DRAM page and gather locality).
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int kMaxConsumerThreads = 512;
constexpr int kMaxStreamThreads = kMaxConsumerThreads + 32;

struct StreamParams {
    int64_t n, nnz;
    const int32_t* rp;
    const int32_t* ci;
    const int16_t* ci16;  // LZ == 3: 16-bit column deltas col - row (handle-owned copy)
    const double* val;
    const double* x;
    double* y;
    const double* fac;   // fac_small (fused) or null
    int b, P, bs;        // block size, packed size, padded block stride in su
    int R, cap, stages;
    int64_t ntiles;
    int rp_ints;         // ints reserved per stage for row pointers (R + 4)
    int fac_bytes;       // bytes reserved per stage for factors
    int stage_bytes;
    int su_doubles;      // doubles per su buffer
    int su_bufs;         // number of su buffers (2; FUSE 3: one per stage)
    unsigned b_magic;    // ceil(2^32 / b): i / b == (i * b_magic) >> 32 for 0 <= i < 65536
    int early_trigger;   // programmatic dependent launch: release the next kernel at entry (else at exit)
    int lz;              // 1: fused Lanczos epilogue on the rows this kernel writes (FUSE 0 and 1); 2: dot hook (FUSE 0)
    LzEpilogue epi;
    const double* dot_with;  // lz == 2: per-CTA partials of dot_with . y go to dot_red (PCG: p . A p)
    LzReduce dot_red;
    int64_t fac_keep_from;   // FUSE 1: tiles >= this load their factors as ordinary L2 lines (serpentine walk, launch_group_t)
};

__device__ __forceinline__ void consumer_bar_sync(int nthreads)
{
    asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}

// LPR lanes per row; kBatch entries per lane in flight per round;
// FUSE: 0 = SpMV only, 1 = + forward solve, thread per block (b <= 8);  TRI (FUSE 1 only): the blocks are tridiagonal and
//       the factors compact, element (i, j) at slot i + j
// LZ (compile time, so that the plain operator kernel carries none of it): 0 plain, 1 fused Lanczos epilogue, 2 dot hook,
// 3 plain with 16-bit column deltas (opts.col16: the column stream is col - row in int16, 10 bytes per entry instead of 12)
constexpr int kBatch = 8;
template <int LPR, int FUSE, bool TRI, int LZ>
__global__ void __launch_bounds__(kMaxStreamThreads)
spmv_stream_kernel(const StreamParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);
    uint64_t* empty = full + p.stages;
    double* su = reinterpret_cast<double*>(smem_raw + 128);               // su_bufs x su_doubles (fused only)
    unsigned char* stage0 = smem_raw + 128 + (size_t)p.su_bufs * p.su_doubles * sizeof(double);
    // per stage: val[cap] | fac[fac_bytes] | col[cap] | rp[rp_ints]
    auto s_val = [&](int s) { return reinterpret_cast<double*>(stage0 + (size_t)s * p.stage_bytes); };
    auto s_fac = [&](int s) { return reinterpret_cast<double*>(stage0 + (size_t)s * p.stage_bytes + (size_t)p.cap * 8); };
    constexpr bool C16 = LZ == 3;
    constexpr int Q = C16 ? 8 : 4;            // ranges are widened to whole groups of Q entries (16-byte bulk copies)
    constexpr int kColBytes = C16 ? 2 : 4;
    auto s_col = [&](int s) { return reinterpret_cast<int*>(stage0 + (size_t)s * p.stage_bytes + (size_t)p.cap * 8 + p.fac_bytes); };
    auto s_col16 = [&](int s) { return reinterpret_cast<int16_t*>(stage0 + (size_t)s * p.stage_bytes + (size_t)p.cap * 8 + p.fac_bytes); };
    auto s_rp = [&](int s) { return reinterpret_cast<int*>(stage0 + (size_t)s * p.stage_bytes + (size_t)p.cap * (8 + kColBytes) + p.fac_bytes); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (p.early_trigger) pdl_trigger();
    if (threadIdx.x == 0) {
        for (int s = 0; s < p.stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], (blockDim.x - 32) / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int R = p.R;
    __shared__ double lz_sh[kMaxStreamThreads / 32];
    double pa = 0.0, beta = 0.0, inv_beta = 0.0;
    if (LZ == 1) {  // beta and the stop flag come from the previous kernel: every thread waits for it
        pdl_wait();
        if (lz_epilogue_begin(p.epi, beta, inv_beta)) return;  // uniform over the grid, nothing in flight yet
    }
    if (warp == 0) {
        // ------------------------------ producer ------------------------------------------------
        const uint64_t pol = policy_evict_first();
        const uint64_t pol_keep = policy_evict_normal();
        const int nnz4 = (int)(p.nnz & ~(long long)(Q - 1));
        int pb0 = 0, pb1 = 0;
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x, ++it) {
            if ((it & 31) == 0) {  // each lane fetches the nnz bounds of one of the next 32 tiles
                const int64_t tl = tile + (int64_t)lane * gridDim.x;
                if (tl < p.ntiles) {
                    const int64_t q0 = tl * R;
                    const int64_t q1 = q0 + R < p.n ? q0 + R : p.n;
                    pb0 = __ldg(p.rp + q0);
                    pb1 = __ldg(p.rp + q1);
                }
            }
            const int p0 = __shfl_sync(0xffffffffu, pb0, it & 31);
            const int p1 = __shfl_sync(0xffffffffu, pb1, it & 31);
            if (lane == 0) {
                const int s = it % p.stages;
                const uint32_t ph = (uint32_t)((it / p.stages) & 1);
                mbar_wait(&empty[s], ph ^ 1u);
                const int64_t r0 = tile * R;
                const int rows = (int)(r0 + R <= p.n ? R : p.n - r0);
                // nnz range widened to multiples of 4, clamped to the last whole quad of the arrays
                const int a0 = p0 & ~(Q - 1);
                int a1 = (p1 + Q - 1) & ~(Q - 1);
                if (a1 > nnz4) a1 = nnz4;
                if (a1 < a0) a1 = a0;
                double* dv = s_val(s);
                int* dc = s_col(s);
                int16_t* dc16 = s_col16(s);
                int* dr = s_rp(s);
                for (int q = (a1 > p0 ? a1 : p0); q < p1; ++q) {  // tail past the last whole group of the arrays
                    dv[q - a0] = p.val[q];
                    if (C16) dc16[q - a0] = p.ci16[q]; else dc[q - a0] = p.ci[q];
                }
                // row pointers r0 .. r0+rows (rows+1 ints), whole quads by bulk copy, rest by hand
                const int64_t np1 = p.n + 1;
                int want = rows + 1;
                int rq = (want + 3) & ~3;
                if (r0 + rq > np1) rq = (int)((np1 - r0) & ~3ll);
                for (int q = rq; q < want; ++q) dr[q] = p.rp[r0 + q];
                uint32_t bytes = (uint32_t)(a1 - a0) * (uint32_t)(8 + kColBytes) + (uint32_t)rq * 4u;
                uint32_t fbytes = 0;
                const double* fsrc = nullptr;
                if (FUSE == 1) {
                    const int nblk = (rows + p.b - 1) / p.b;
                    const int groups = (nblk + kInterleave - 1) / kInterleave;
                    fbytes = (uint32_t)groups * (uint32_t)p.P * kInterleave * 8u;
                    fsrc = p.fac + (r0 / p.b / kInterleave) * (int64_t)p.P * kInterleave;
                    bytes += fbytes;
                }
                mbar_expect_tx(&full[s], bytes);
                if (a1 > a0) {
                    bulk_g2s(dv, p.val + a0, (uint32_t)(a1 - a0) * 8u, &full[s], pol);
                    if (C16) bulk_g2s(dc16, p.ci16 + a0, (uint32_t)(a1 - a0) * 2u, &full[s], pol);
                    else bulk_g2s(dc, p.ci + a0, (uint32_t)(a1 - a0) * 4u, &full[s], pol);
                }
                if (rq > 0) bulk_g2s(dr, p.rp + r0, (uint32_t)rq * 4u, &full[s], pol);
                if (FUSE && fbytes) bulk_g2s(s_fac(s), fsrc, fbytes, &full[s], tile >= p.fac_keep_from ? pol_keep : pol);
            }
        }
    } else {
        // ------------------------------ consumers -----------------------------------------------
        const int ctid = threadIdx.x - 32;
        const int nct = blockDim.x - 32;
        const int sub = ctid & (LPR - 1);
        const int kRowsPerPass = nct / LPR;
        pdl_wait();  // x (= t) comes from the previous kernel; the producer streams only setup-time constants
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x, ++it) {
            const int s = it % p.stages;
            const uint32_t ph = (uint32_t)((it / p.stages) & 1);
            const int64_t r0 = tile * R;
            const int rows = (int)(r0 + R <= p.n ? R : p.n - r0);
            double* sub_u = su + (size_t)(it & 1) * p.su_doubles;
            mbar_wait(&full[s], ph);
            const double* sv = s_val(s);
            const int* sc = s_col(s);
            const int16_t* sc16 = s_col16(s);
            const int* sr = s_rp(s);
            const int a0 = sr[0] & ~(Q - 1);
            // (A) rows out of shared memory
            for (int base = 0; base < rows; base += kRowsPerPass) {
                const int i = base + ctid / LPR;
                const bool valid = i < rows;
                double acc = 0.0;
                if (valid) {
                    // BATCH entries per lane per round: all their gathers are in flight together
                    const int e = sr[i + 1] - a0;
                    for (int q = sr[i] - a0 + sub; q < e; q += kBatch * LPR) {
                        int c[kBatch];
                        double xv[kBatch], av[kBatch];
#pragma unroll
                        for (int k = 0; k < kBatch; ++k) {
                            const int qq = q + k * LPR;
                            c[k] = C16 ? (int)(r0 + i) + (int)sc16[qq < e ? qq : q] : sc[qq < e ? qq : q];
                        }
#pragma unroll
                        for (int k = 0; k < kBatch; ++k)  // predicated: a masked lane costs no L1 wavefront
                            xv[k] = (q + k * LPR < e) ? __ldg(p.x + c[k]) : 0.0;
#pragma unroll
                        for (int k = 0; k < kBatch; ++k) {
                            const int qq = q + k * LPR;
                            av[k] = qq < e ? sv[qq] : 0.0;
                        }
#pragma unroll
                        for (int k = 0; k < kBatch; ++k) acc = fma(av[k], xv[k], acc);
                    }
                }
#pragma unroll
                for (int off = LPR / 2; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off, LPR);
                if (valid && sub == 0) {
                    if (FUSE == 1) {
                        const int k = (int)__umulhi((unsigned)i, p.b_magic);
                        sub_u[k * p.bs + (i - k * p.b)] = acc;
                    } else {
                        if (LZ == 1) {
                            lz_epilogue_elem(p.epi, beta, inv_beta, r0 + i, acc, pa);
                        } else {
                            if (LZ == 2) pa = fma(p.dot_with[r0 + i], acc, pa);
                            p.y[r0 + i] = acc;
                        }
                    }
                }
            }
            if (FUSE == 1) {
                // (B) forward substitution y = L^-1 u on the tile's diagonal blocks, one thread per block
                consumer_bar_sync(nct);
                const int nblk = (rows + p.b - 1) / p.b;
                const int b = p.b;
                const double* sf = s_fac(s);
                int rot = ctid - 32 * (it & 7);  // rotate the solving warps from tile to tile
                if (rot < 0) rot += nct;
                for (int k = rot; k < nblk; k += nct) {
                    const double* f = sf + (size_t)(k >> 5) * p.P * kInterleave + (k & 31);
                    double* uk = sub_u + k * p.bs;
                    const int64_t lo = r0 + (int64_t)k * b;
                    double v[kSmallMax];
#pragma unroll
                    for (int i = 0; i < kSmallMax; ++i) v[i] = (i < b && lo + i < p.n) ? uk[i] : 0.0;
                    if (TRI) {  // compact bidiagonal factors (tridiagonal blocks): compile-time variant
#pragma unroll
                        for (int i = 0; i < kSmallMax; ++i) {
                            if (i < b) {
                                double acc = v[i];
                                if (i > 0) acc -= f[(2 * i - 1) * kInterleave] * v[i - 1];
                                v[i] = acc * f[(2 * i) * kInterleave];
                            }
                        }
                    } else {
#pragma unroll
                    for (int i = 0; i < kSmallMax; ++i) {
                        if (i < b) {
                            double acc = v[i];
#pragma unroll
                            for (int j = 0; j < i; ++j) acc -= f[(i * (i + 1) / 2 + j) * kInterleave] * v[j];
                            v[i] = acc * f[(i * (i + 1) / 2 + i) * kInterleave];
                        }
                    }
                    }
#pragma unroll
                    for (int i = 0; i < kSmallMax; ++i)
                        if (i < b) uk[i] = v[i];
                }
                // (C) rows leave COALESCED: thread q takes rows q, q + nct, .. of the tile (and, inside a Lanczos
                // step, their w / v_j / v_{j+1} elements)
                consumer_bar_sync(nct);
                for (int i = ctid; i < rows; i += nct) {
                    const int k = (int)__umulhi((unsigned)i, p.b_magic);
                    const double yv = sub_u[k * p.bs + (i - k * b)];
                    if (LZ == 1) lz_epilogue_elem(p.epi, beta, inv_beta, r0 + i, yv, pa);
                    else p.y[r0 + i] = yv;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }
    }
    if (LZ == 1) lz_reduce_finish(p.epi.red, pa, lz_sh);
    if (LZ == 2) lz_reduce_finish(p.dot_red, pa, lz_sh);
}

template <int LPR, int FUSE, bool TRI, int LZ>
int launch_stream_t(bj_handle_s* h, const StreamParams& sp, int want_per_sm, int threads, size_t smem)
{
    static std::atomic<bool> configured[64];
    {
        cudaError_t e = ensure_big_smem(spmv_stream_kernel<LPR, FUSE, TRI, LZ>, configured);
        if (e != cudaSuccess) { set_cuda_error(e, "cudaFuncSetAttribute(spmv_stream_kernel)"); return BJ_ERR_CUDA; }
    }
    int occ = 1;  // persistent grid: exactly the CTAs that are resident at once
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, spmv_stream_kernel<LPR, FUSE, TRI, LZ>, threads, smem);
    const int per_sm = std::max(1, std::min(occ, want_per_sm));
    const int grid = (int)std::min<int64_t>(sp.ntiles, (int64_t)h->num_sms * per_sm);
    cudaError_t e = launch_kernel(spmv_stream_kernel<LPR, FUSE, TRI, LZ>, grid, threads, smem, h->stream,
                                  h->pdl && !h->prof_on, sp);
    if (e != cudaSuccess) { set_cuda_error(e, "spmv_stream_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}


}  // namespace

namespace {
// shared-memory layout of one launch; the single source of truth for configure and launch
void fill_layout(const bj_handle_s* h, bool fuse, StreamParams& sp, size_t& smem, bool c16 = false)
{
    sp.b = h->b > 0 ? h->b : 1;
    sp.P = h->packed;
    sp.bs = (sp.b % 2) ? sp.b : sp.b + 1;
    sp.R = h->tile_rows;
    sp.cap = h->tile_cap;
    sp.stages = h->tile_stages;
    sp.ntiles = h->ntiles;
    sp.rp_ints = sp.R + 4;
    sp.su_bufs = 2;
    sp.fac_bytes = fuse ? (((sp.R / sp.b) * sp.P * 8 + 15) & ~15) : 0;
    sp.su_doubles = !fuse ? 0 : (((sp.R / sp.b) * sp.bs + 1) & ~1);
    sp.stage_bytes = (sp.cap * (c16 ? 10 : 12) + sp.fac_bytes + sp.rp_ints * 4 + 15) & ~15;
    sp.b_magic = (unsigned)(((1ull << 32) + sp.b - 1) / sp.b);
    smem = 128 + (size_t)sp.su_bufs * sp.su_doubles * 8 + (size_t)sp.stages * sp.stage_bytes;
}
constexpr size_t kSmemTwoPerSm = 110 * 1024;
constexpr size_t kSmemOnePerSm = 224 * 1024;
}  // namespace

// Tile geometry (rows per tile, fusion, lanes per row) for a matrix whose columns are / are not coherent between
// neighbouring rows.  rows == 0: the streamed kernel cannot be used.
StreamGeometry spmv_stream_geometry(const bj_handle_s* h, bool random_cols)
{
    StreamGeometry g;
    if (h->nnz == 0) return g;
    if (((uintptr_t)h->val & 15) || ((uintptr_t)h->col_idx & 15) || ((uintptr_t)h->row_ptr & 15)) return g;
    const double mean = (double)h->nnz / (double)h->n;
    {
        // lanes per row in the tile kernel: rows come out of shared memory, so one thread per row
        // (coalesced gathers for banded matrices, oracle summation order) up to ~12 entries per row
        int l = 1;
        while (l < 32 && (double)l * 12.0 < mean) l *= 2;
        // Random column structure (no coherence between neighbouring rows): the kernel is bound by the
        // L1/LSU gather rate, not by HBM; what helps is many warps with gathers in flight, one row per thread.
        if (random_cols && mean <= 48.0) l = 1;
        g.lanes = env_int("BJ_STREAM_LANES", l);
        g.warps = std::max(1, std::min(env_int("BJ_CONSUMER_WARPS", random_cols ? 16 : 8), kMaxConsumerThreads / 32));
    }
    const int target_nnz = env_int("BJ_TILE_NNZ", 2048);
    int R = (int)((double)target_nnz / (mean > 1.0 ? mean : 1.0));
    R = std::max(32, std::min(R, 1024));
    bool fuse = false;
    if (h->solve_kind == 1 && !random_cols && !h->var_perm) {  // (a permuted handle's blocks are not row ranges of A)
        const int unit = kInterleave * h->b;  // fused tiles must hold whole interleave groups
        int Rf = ((R + unit / 2) / unit) * unit;
        if (Rf < unit) Rf = unit;
        if ((double)Rf * mean <= 1.6 * target_nnz && Rf <= 1024) { R = Rf; fuse = true; }
    }
    if (!fuse) R = ((R + 31) / 32) * 32;
    R = env_int("BJ_TILE_ROWS", R);
    if (fuse && (R % (kInterleave * h->b)) != 0) fuse = false;
    if (R % 4) return g;
    g.rows = R;
    g.fuse = fuse;
    return g;
}

void spmv_stream_adopt(bj_handle_s* h, const StreamGeometry& g)
{
    h->stream_ok = false;
    h->fuse_ok = g.rows > 0 && g.fuse;
    h->ntiles = g.rows > 0 ? (h->n + g.rows - 1) / g.rows : 0;
    h->tile_rows = g.rows;
    h->stream_lanes = g.lanes;
    h->stream_warps = g.warps;
}

// Decide the tile geometry from the handle's coherence statistic and launch the kernel that measures the fullest tile.
int spmv_stream_configure(bj_handle_s* h)
{
    const StreamGeometry g = spmv_stream_geometry(h, h->coherence < 0.25);
    spmv_stream_adopt(h, g);
    // measure the fullest tile (result is read back with the rest of the setup status)
    return launch_spmv_plan(h, g.rows);
}

// second half of the plan, once the fullest tile is known
int spmv_stream_finish(bj_handle_s* h, int max_tile)
{
    if (h->ntiles <= 0) return BJ_OK;
    const bool fuse = h->fuse_ok;
    h->tile_cap = ((max_tile + 16) + 7) & ~7;  // ranges are widened to groups of up to 8 entries on both sides
    int stages = env_int("BJ_STAGES", 2);
    StreamParams sp;
    size_t smem = 0;
    h->tile_stages = stages;
    fill_layout(h, fuse, sp, smem);
    if (smem > kSmemTwoPerSm) {
        // one CTA per SM: as many stages as fit, at least two
        while (stages > 2 && smem > kSmemOnePerSm) { h->tile_stages = --stages; fill_layout(h, fuse, sp, smem); }
        if (smem > kSmemOnePerSm) { h->ntiles = 0; h->fuse_ok = false; return BJ_OK; }
    }
    h->tile_stages = stages;
    h->stream_ok = true;
    if (env_int("BJ_VERBOSE", 0))
        fprintf(stderr, "[bj] spmv plan: rows/tile %d cap %d stages %d smem %zu B lanes/row %d consumer warps %d fuse %d coherence %.3f\n",
                h->tile_rows, h->tile_cap, h->tile_stages, smem, h->stream_lanes, h->stream_warps, (int)h->fuse_ok, h->coherence);
    return BJ_OK;
}

int launch_spmv_stream(bj_handle_s* h, const double* x, double* y, bool fuse_forward, const LzEpilogue* epi,
                       const double* dot_with, const LzReduce* dot_red)
{
    if (!h->stream_ok) return BJ_ERR_INVALID_ARG;
    const bool fuse = fuse_forward && h->fuse_ok;
    if (fuse_forward && !fuse) return BJ_ERR_INVALID_ARG;
    StreamParams sp;
    size_t smem = 0;
    // 16-bit column deltas: plain operator kernels only (no hooks), thread-per-block fusion or none
    const bool c16 = h->col16 != nullptr && !epi && !dot_with;
    fill_layout(h, fuse, sp, smem, c16);
    sp.n = h->n; sp.nnz = h->nnz; sp.rp = h->row_ptr; sp.ci = h->col_idx; sp.val = h->val;
    sp.ci16 = h->col16;
    sp.x = x; sp.y = y;
    sp.early_trigger = (h->tune.pdl_early >> 1) & 1;
    if ((h->tune.pdl_early & 4) && !fuse && !epi && !dot_with) sp.early_trigger = 1;
    sp.lz = epi ? 1 : (dot_with && dot_red) ? 2 : 0;
    sp.dot_with = dot_with;
    sp.dot_red = dot_red ? *dot_red : LzReduce{};
    if (sp.lz == 2 && (fuse || h->num_sms * 4 > dot_red->cap)) return BJ_ERR_INVALID_ARG;
    sp.epi = epi ? *epi : LzEpilogue{};
    if (epi && h->num_sms * 4 > epi->red.cap) return BJ_ERR_INVALID_ARG;
    sp.fac = fuse ? h->fac_small : nullptr;
    sp.fac_keep_from = sp.ntiles;
    if (fuse && h->tune.serp_keep_mb > 0 && sp.lz == 0) {
        const int64_t tile_bytes = (int64_t)(sp.R / sp.b) * sp.P * 8;
        sp.fac_keep_from = sp.ntiles - std::min<int64_t>(sp.ntiles, (int64_t)h->tune.serp_keep_mb * 1000000 / tile_bytes);
    }
    const int threads = 32 + 32 * h->stream_warps;
    const int grid = h->tune.ctas_per_sm;  // wanted CTAs per SM; clipped to the real occupancy at launch
    int rc = BJ_OK;
    {
        KernelScope scope(h, fuse ? BJ_K_SPMV_SOLVE_L : BJ_K_SPMV);
#define BJ_CASE(L)                                                                                 \
    case L:                                                                                        \
        rc = !fuse    ? (sp.lz == 1   ? launch_stream_t<L, 0, false, 1>(h, sp, grid, threads, smem)  \
                         : sp.lz == 2 ? launch_stream_t<L, 0, false, 2>(h, sp, grid, threads, smem)  \
                         : c16        ? launch_stream_t<L, 0, false, 3>(h, sp, grid, threads, smem)  \
                                      : launch_stream_t<L, 0, false, 0>(h, sp, grid, threads, smem)) \
             : h->tri ? (sp.lz == 1   ? launch_stream_t<L, 1, true, 1>(h, sp, grid, threads, smem)   \
                         : c16        ? launch_stream_t<L, 1, true, 3>(h, sp, grid, threads, smem)   \
                                      : launch_stream_t<L, 1, true, 0>(h, sp, grid, threads, smem))  \
                      : (sp.lz == 1   ? launch_stream_t<L, 1, false, 1>(h, sp, grid, threads, smem)  \
                         : c16        ? launch_stream_t<L, 1, false, 3>(h, sp, grid, threads, smem)  \
                                      : launch_stream_t<L, 1, false, 0>(h, sp, grid, threads, smem)); \
        break;
        switch (h->stream_lanes) {
            BJ_CASE(1) BJ_CASE(2) BJ_CASE(4) BJ_CASE(8) BJ_CASE(16) BJ_CASE(32)
            default: rc = BJ_ERR_INVALID_ARG;
        }
#undef BJ_CASE
    }
    if (rc != BJ_OK) return rc;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

}  // namespace bj
