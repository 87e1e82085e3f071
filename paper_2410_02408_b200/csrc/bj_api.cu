// C ABI of the bj library (include/bj.h): handle life cycle, setup orchestration (a1-a4),
// operator composition (a7) and the host-buffer / profiling helpers.  All arithmetic lives in
// the kernels of the sibling .cu files; there is no CPU fallback.
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>

#include "bj_internal.cuh"
#include "bj_lanczos_fuse.cuh"

namespace bj {

static thread_local char g_cuda_msg[512] = "no CUDA error recorded";

void set_cuda_error(cudaError_t e, const char* where)
{
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), where);
    cudaGetLastError();  // clear the non-sticky error state
}

KernelScope::KernelScope(bj_handle_s* h_, int kind_) : h(h_), kind(kind_)
{
    h->launches++;
    if (!h->prof_on) return;
    auto get = [&]() {
        cudaEvent_t e = nullptr;
        if (!h->event_pool.empty()) { e = h->event_pool.back(); h->event_pool.pop_back(); }
        else cudaEventCreate(&e);
        return e;
    };
    a = get();
    b = get();
    cudaEventRecord(a, h->stream);
}

KernelScope::~KernelScope()
{
    if (!a) return;
    cudaEventRecord(b, h->stream);
    h->spans.push_back(ProfSpan{kind, a, b});
}

static int resolve_spans(bj_handle_s* h)
{
    if (h->spans.empty()) return BJ_OK;
    BJ_CUDA(cudaStreamSynchronize(h->stream));
    for (auto& s : h->spans) {
        float ms = 0.f;
        BJ_CUDA(cudaEventElapsedTime(&ms, s.a, s.b));
        h->prof_ms[s.kind] += ms;
        h->prof_cnt[s.kind] += 1;
        h->event_pool.push_back(s.a);
        h->event_pool.push_back(s.b);
    }
    h->spans.clear();
    return BJ_OK;
}

int launch_spmv(bj_handle_s* h, const double* x, double* y)
{
    if (h->spmv_kernel == 2) return launch_spmv_bsr(h, x, y);
    return h->spmv_kernel == 1 ? launch_spmv_stream(h, x, y, false) : launch_spmv_vector(h, x, y);
}

// y = L^-1 A L^-T x.  x == y allowed.
int op_apply_device(bj_handle_s* h, const double* x, double* y)
{
    int rc;
    if (h->solve_kind == 0) {  // identity preconditioner: A^ = A
        if (x == y) {
            BJ_CUDA(cudaMemcpyAsync(h->t, x, (size_t)h->n * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
            x = h->t;
        }
        return launch_spmv(h, x, y);
    }
    rc = launch_solve(h, 1, x, h->t);  // t = L^-T x
    if (rc != BJ_OK) return rc;
    const bool fuse = h->spmv_kernel == 1 && h->fuse_ok && h->opt_fuse != 0;
    if (fuse) return launch_spmv_stream(h, h->t, y, true);  // y = L^-1 (A t) in one kernel
    rc = launch_spmv(h, h->t, h->u);
    if (rc != BJ_OK) return rc;
    return launch_solve(h, 0, h->u, y);  // y = L^-1 u
}

int op_apply_lanczos(bj_handle_s* h, const LzPrologue* pro, const LzEpilogue* epi, double* w)
{
    if (!lanczos_fusable(h)) return BJ_ERR_INVALID_ARG;
    int rc = launch_solve(h, 1, nullptr, h->t, pro, nullptr);  // v_next on the fly, t = L^-T v_next
    if (rc != BJ_OK) return rc;
    const bool fuse = h->solve_kind == 1 && h->spmv_kernel == 1 && h->fuse_ok && h->opt_fuse != 0;
    if (fuse) return launch_spmv_stream(h, h->t, w, true, epi);  // w' and the dot partials in the SpMV's epilogue
    rc = launch_spmv(h, h->t, h->u);
    if (rc != BJ_OK) return rc;
    return launch_solve(h, 0, h->u, w, nullptr, epi);
}

// Device memory for a handle comes from a private stream-ordered pool (cudaMallocFromPoolAsync) whose
// release threshold keeps freed slabs cached: repeated setups (block-size sweeps) then cost microseconds
// instead of a cudaMalloc each.  bj_release_cached_memory() returns the cache to the driver.
// BJ_POOL=0 selects plain cudaMalloc.
static cudaMemPool_t g_pool[64] = {};
static std::once_flag g_pool_once[64];

static cudaMemPool_t get_pool(int dev)
{
    if (dev < 0 || dev >= 64 || env_int("BJ_POOL", 1) == 0) return nullptr;
    std::call_once(g_pool_once[dev], [dev]() {  // two threads setting up at once create ONE pool
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) == cudaSuccess) {
            uint64_t keep = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
            g_pool[dev] = pool;
        } else {
            cudaGetLastError();
        }
    });
    return g_pool[dev];
}

static void* slab_alloc(size_t bytes, int dev, cudaStream_t stream, bool* pooled)
{
    void* p = nullptr;
    *pooled = false;
    if (cudaMemPool_t pool = get_pool(dev)) {
        if (cudaMallocFromPoolAsync(&p, bytes, pool, stream) == cudaSuccess) { *pooled = true; return p; }
        cudaGetLastError();
    }
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}

static void free_handle(bj_handle_s* h)
{
    if (!h) return;
    lanczos_free(h);
    pcg_free(h);
    batch_free(h);
    bsr_free(h);
    col16_free(h);
    if (h->slab) {
        // stream-ordered free on the handle's stream; if that stream is gone (a destroyed torch side stream after
        // bj_set_stream) fall back to a synchronous free so that the slab is not leaked
        if (!h->slab_pooled || cudaFreeAsync(h->slab, h->stream) != cudaSuccess) {
            cudaGetLastError();
            cudaDeviceSynchronize();
            cudaFree(h->slab);
        }
    }
    var_free(h);
    cudaFree(h->stage_in); cudaFree(h->stage_out);
    for (auto& s : h->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
    for (auto e : h->event_pool) cudaEventDestroy(e);
    delete h;
}

static void choose_spmv(bj_handle_s* h)
{
    int k = 0;
    if (h->stream_ok) k = 1;
    if (h->bsr_ok) k = 2;  // opt-in (opts.bsr) and the matrix is 3x3-blocked: fewer bytes than either CSR kernel
    if (h->opt_spmv_kernel == 0) k = 0;
    if (h->opt_spmv_kernel == 1 && h->stream_ok) k = 1;
    h->spmv_kernel = k;
}

}  // namespace bj

using namespace bj;

extern "C" {

const char* bj_strerror(int code)
{
    switch (code) {
        case BJ_OK: return "ok";
        case BJ_ERR_INVALID_ARG: return "invalid argument";
        case BJ_ERR_NOT_CANONICAL: return "CSR is not canonical (row_ptr not monotone from 0 to nnz, column out of range, or columns not strictly increasing in a row)";
        case BJ_ERR_TOO_LARGE: return "n or nnz does not fit 32-bit indices";
        case BJ_ERR_NOT_SPD: return "a diagonal block is not positive definite (see bj_get_info bad_block)";
        case BJ_ERR_ALLOC: return "allocation failed";
        case BJ_ERR_CUDA: return g_cuda_msg;
        case BJ_ERR_LIMIT: return "bj_cond_estimate_noalloc: beyond the limits of the fixed device scratch (n <= 16384, iters <= 1024, "
                                  "uniform blocks b <= 8 or b = 0 without permutation or band storage, basis share fits shared memory)";
        default: return "unknown bj status";
    }
}

}  // extern "C"

static int setup_impl(const bj_csr_t* csr, int b, const bj_setup_opts_t& o, bj_handle_t* out, const int32_t* perm_dev = nullptr)
{
    if (!out) return BJ_ERR_INVALID_ARG;
    *out = nullptr;
    for (int r : o.reserved) if (r != 0) return BJ_ERR_INVALID_ARG;
    void* cuda_stream = o.cuda_stream;
    if (!csr || !csr->row_ptr || csr->n <= 0 || csr->nnz < 0 || b < 0 || b > BJ_B_MAX) return BJ_ERR_INVALID_ARG;
    if (csr->nnz > 0 && (!csr->col_idx || !csr->val)) return BJ_ERR_INVALID_ARG;
    if (csr->n >= (1ll << 31) - 64 || csr->nnz >= (1ll << 31) - 64) return BJ_ERR_TOO_LARGE;

    int dev = 0;
    BJ_CUDA(cudaGetDevice(&dev));
    bj_handle_s* h = new (std::nothrow) bj_handle_s();
    if (!h) return BJ_ERR_ALLOC;
    h->n = csr->n; h->nnz = csr->nnz; h->b = b;
    h->row_ptr = csr->row_ptr; h->col_idx = csr->col_idx; h->val = csr->val;
    h->stream = (cudaStream_t)cuda_stream;
    h->nblocks = b > 0 ? (csr->n + b - 1) / b : 0;
    h->packed = b * (b + 1) / 2;
    cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev);
    h->opts = o;
    h->pdl = env_int("BJ_PDL", 1) != 0;
    {
        Tuning& t = h->tune;  // launch shapes only (see bj_internal.cuh)
        t.solve_warps = env_int("BJ_SOLVE_WARPS", t.solve_warps);
        t.solve_stage_kb = env_int("BJ_SOLVE_STAGE_KB", t.solve_stage_kb);
        t.solve_stages = env_int("BJ_SOLVE_STAGES", t.solve_stages);
        t.solve_ctas = env_int("BJ_SOLVE_CTAS", t.solve_ctas);
        t.group_stages = env_int("BJ_GROUP_STAGES", t.group_stages);
        t.group_smem_kb = env_int("BJ_GROUP_SMEM_KB", t.group_smem_kb);
        t.group_warps = env_int("BJ_GROUP_WARPS", t.group_warps);
        t.group_lanes = env_int("BJ_GROUP_LANES", t.group_lanes);
        t.pdl_early = env_int("BJ_PDL_EARLY", t.pdl_early);
        t.ctas_per_sm = env_int("BJ_CTAS_PER_SM", t.ctas_per_sm);
        if (o.serp_keep_mb != 0) t.serp_keep_mb = o.serp_keep_mb < 0 ? 0 : o.serp_keep_mb;
    }

    auto fail = [&](int code) { free_handle(h); return code; };

    // one slab holds t, u, the status words and the factors (one allocation instead of five)
    auto up256 = [](size_t v) { return (v + 255) & ~(size_t)255; };
    const size_t vb = up256((size_t)h->n * sizeof(double));
    size_t fac_a = 0, fac_b = 0;
    if (b > 0 && b <= kSmallMax) {
        h->solve_kind = 1;
        const int64_t groups = (h->nblocks + kInterleave - 1) / kInterleave;
        fac_a = (size_t)groups * h->packed * kInterleave * sizeof(double);
    } else if (b > 0) {
        h->solve_kind = 2;
        h->lanes = b <= 16 ? 16 : 32;
        fac_a = fac_b = (size_t)h->nblocks * h->packed * sizeof(double) + 16;  // 16 B slack: bulk copies round up
        // the group kernel (b = 16, 24, 32) runs the backward substitution from the forward copy too: one copy is kept
        h->single_copy = b == 16 || b == 24 || b == 32;
        if (h->single_copy) fac_b = 0;
    }
    const size_t total = 2 * vb + 256 + up256(fac_a) + up256(fac_b);
    h->slab = slab_alloc(total, dev, h->stream, &h->slab_pooled);
    if (!h->slab) return fail(BJ_ERR_ALLOC);
    {
        char* base = (char*)h->slab;
        h->t = (double*)base;
        h->u = (double*)(base + vb);
        h->status = (Status*)(base + 2 * vb);
        char* f = base + 2 * vb + 256;
        if (h->solve_kind == 1) h->fac_small = (double*)f;
        if (h->solve_kind == 2) { h->fac_fwd = (double*)f; h->fac_bwd = h->single_copy ? nullptr : (double*)(f + up256(fac_a)); }
        h->workspace_bytes = (int64_t)(2 * vb + 256);
        h->factor_bytes = (int64_t)(fac_a + fac_b);
    }
    Status init;
    memset(&init, 0, sizeof(init));
    init.bad_block = 0x7fffffffffffffffll;
    cudaError_t ce = cudaMemcpyAsync(h->status, &init, sizeof(init), cudaMemcpyHostToDevice, h->stream);
    if (ce != cudaSuccess) { set_cuda_error(ce, "status init"); return fail(BJ_ERR_CUDA); }

    // lanes per row for the CSR-vector kernel: power of two near the mean row length
    {
        const double mean = (double)h->nnz / (double)h->n;
        int l = 1;
        while (l < 32 && (double)l * 1.15 < mean) l *= 2;
        h->spmv_lanes = l;
    }
    // only the padding the extraction kernels do not write needs zeroing
    auto zero_padding = [&]() -> cudaError_t {
        cudaError_t e = cudaSuccess;
        if (h->solve_kind == 1) {
            const size_t group_bytes = (size_t)h->packed * kInterleave * sizeof(double);
            const int64_t groups = (h->nblocks + kInterleave - 1) / kInterleave;  // (packed may be the compact tridiagonal size)
            if (h->nblocks % kInterleave) e = cudaMemsetAsync((char*)h->fac_small + (size_t)(groups - 1) * group_bytes, 0, group_bytes, h->stream);
        } else if (h->solve_kind == 3) {
            // the last interleave group may be partly unused: zero it so that no lane ever reads an uninitialised factor
            const size_t group_bytes = (size_t)(h->band + 1) * b * kInterleave * sizeof(double);
            if (h->nblocks % kInterleave)
                e = cudaMemsetAsync((char*)h->fac_band + (size_t)(h->nblocks / kInterleave) * group_bytes, 0, group_bytes, h->stream);
        } else if (h->solve_kind == 2) {
            e = cudaMemsetAsync((char*)h->fac_fwd + fac_a - 16, 0, 16, h->stream);
            if (e == cudaSuccess && h->fac_bwd) e = cudaMemsetAsync((char*)h->fac_bwd + fac_b - 16, 0, 16, h->stream);
        }
        return e;
    };
    auto read_status = [&](Status& dst, const char* where) -> int {
        cudaError_t e = cudaMemcpyAsync(&dst, h->status, sizeof(dst), cudaMemcpyDeviceToHost, h->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
        if (e != cudaSuccess) { set_cuda_error(e, where); return BJ_ERR_CUDA; }
        return BJ_OK;
    };

    SetupTimer timer(h->stream);
    h->setup_timer = &timer;  // the launch helpers of the setup kernels bracket each kernel with events
    struct TimerGuard { bj_handle_s* h; ~TimerGuard() { h->setup_timer = nullptr; } } timer_guard{h};
    Status stt;
    int rc = BJ_OK;
    // opts.band: the factor layout depends on the band statistic, so the extraction follows the validation pass
    const bool want_band = o.band != 0 && !perm_dev && ((h->solve_kind == 1 && b >= 4) || (h->solve_kind == 2 && h->nblocks >= 64));

    // b <= 8, short rows, no permutation, no band detection: validation rides on the entry-parallel extraction
    // (bj_setup_rows.cu) and the factorisation follows without a host round trip.  Its cost follows nnz (6.5 ns per entry and
    // SM-microsecond): measured against the three passes it wins for up to 8 entries per row (config 2 b = 8 0.140 -> 0.120 ms,
    // b = 7 0.148 -> 0.122, config 1 0.031 -> 0.016) and loses beyond (config 4 b = 8, 9 per row: 0.30 vs 0.26 ms; config 5
    // b = 3, 81 per row: 0.59 vs 0.44), except for incoherent columns (config 3 b = 8: 0.12 vs 0.22 ms), which setup cannot
    // know before it has read them.  BJ_SETUP_ROWWISE = 0 / 2 forces the three passes / the one kernel.
    const int rowwise_env = env_int("BJ_SETUP_ROWWISE", 1);
    const bool rowwise = h->solve_kind == 1 && !perm_dev && !want_band && rowwise_env != 0 && (rowwise_env == 2 || h->nnz <= 8 * h->n);
    // a1 validate (also longest row and the column-coherence statistic)
    if (rowwise) {  // (the unused slots of a partly filled last interleave group are zeroed first)
        ce = zero_padding();
        if (ce != cudaSuccess) { set_cuda_error(ce, "factor memset"); return fail(BJ_ERR_CUDA); }
    }
    rc = rowwise ? launch_setup_rows(h) : launch_validate(h);
    if (rc != BJ_OK) return fail(rc);
    rc = read_status(stt, "validate");
    if (rc != BJ_OK) return fail(rc);
    if (stt.flags & (ST_BAD_ROWPTR | ST_BAD_COL | ST_UNSORTED)) return fail(BJ_ERR_NOT_CANONICAL);
    if (stt.descents != stt.legal_descents) return fail(BJ_ERR_NOT_CANONICAL);  // a descent inside a row

    h->coherence = stt.compared ? (double)stt.coherent / (double)stt.compared : 1.0;
    h->max_row_nnz = stt.max_row_nnz;
    if (perm_dev) {  // bj_setup_perm: blocks of P A P^T, vectors in the original ordering (reading 23)
        rc = perm_install(h, perm_dev);
        if (rc != BJ_OK) return fail(rc);
    }

    // NEXT-2, opt-in: banded diagonal blocks keep banded factors -- (w+1) b doubles per block instead of b(b+1)/2.
    if (want_band) {
        rc = launch_band_width(h);
        if (rc != BJ_OK) return fail(rc);
        rc = read_status(stt, "band width");
        if (rc != BJ_OK) return fail(rc);
        if (h->solve_kind == 1 && stt.max_band >= 0 && stt.max_band <= 1) {
            // b <= 8: tridiagonal blocks keep bidiagonal factors, 2b - 1 doubles per block instead of b(b+1)/2; same kernels
            // (thread per block, fused into the SpMV tile kernel, Lanczos / PCG hooks), compile-time / uniform index switch
            h->tri = true;
            h->band = stt.max_band;
            h->packed = 2 * b - 1;
            h->factor_bytes = (int64_t)((h->nblocks + kInterleave - 1) / kInterleave) * h->packed * kInterleave * (int64_t)sizeof(double);
        } else if (h->solve_kind == 2 && stt.max_band >= 0 && stt.max_band <= 2) {
            h->solve_kind = 3;
            h->band = stt.max_band;
            h->fac_band = h->fac_fwd;  // (w+1) b <= 3 b < b(b+1)/2 for b > 8: fits the forward copy's storage
            h->factor_bytes = (int64_t)((h->nblocks + kInterleave - 1) / kInterleave) * kInterleave * (h->band + 1) * b * (int64_t)sizeof(double);
        }
    }

    if (b > 0 && !rowwise) {
        // a2-a4 extract + factor
        ce = zero_padding();
        if (ce != cudaSuccess) { set_cuda_error(ce, "factor memset"); return fail(BJ_ERR_CUDA); }
        rc = h->solve_kind == 3 ? launch_extract_factor_band(h) : launch_extract_factor(h);
        if (rc != BJ_OK) return fail(rc);
    }
    // SpMV plan for the streamed kernel: tile rows now, stage capacity once the fullest tile is known
    rc = spmv_stream_configure(h);
    if (rc != BJ_OK) return fail(rc);
    rc = read_status(stt, "setup");
    if (rc != BJ_OK) return fail(rc);
    const int max_tile = stt.max_tile_nnz;
    h->setup_kernel_ms = timer.total_ms();
    rc = spmv_stream_finish(h, max_tile);
    if (rc != BJ_OK) return fail(rc);
    if (o.col16 != 0 && h->stream_ok) {  // NEXT-2, opt-in: 16-bit column deltas for the tile kernel
        rc = col16_build(h);
        if (rc != BJ_OK) return fail(rc);
    }
    if (o.bsr != 0) {  // NEXT-2, opt-in: 3x3-blocked copy of the matrix when its structure allows
        h->bsr_max_row_nnz = stt.max_row_nnz;
        rc = bsr_build(h);
        if (rc != BJ_OK) return fail(rc);
    }
    choose_spmv(h);
    *out = h;
    if (stt.flags & ST_NOT_SPD) {
        h->failed = true;
        h->bad_block = (int64_t)stt.bad_block;
        return BJ_ERR_NOT_SPD;
    }
    return BJ_OK;
}

extern "C" {

int bj_setup_ex(const bj_csr_t* csr, int b, const bj_setup_opts_t* opts, bj_handle_t* out)
{
    bj_setup_opts_t o;
    memset(&o, 0, sizeof(o));
    if (opts) o = *opts;
    return setup_impl(csr, b, o, out);
}

int bj_setup_on_stream(const bj_csr_t* csr, int b, void* cuda_stream, bj_handle_t* out)
{
    bj_setup_opts_t o;
    memset(&o, 0, sizeof(o));
    o.cuda_stream = cuda_stream;
    return setup_impl(csr, b, o, out);
}

int bj_setup(const bj_csr_t* csr, int b, bj_handle_t* out) { return bj_setup_on_stream(csr, b, nullptr, out); }

int bj_get_setup_time(bj_handle_t h, double* kernel_ms, int64_t* alg_bytes)
{
    if (!h) return BJ_ERR_INVALID_ARG;
    if (kernel_ms) *kernel_ms = h->setup_kernel_ms;
    if (alg_bytes) *alg_bytes = 12 * h->nnz + 4 * (h->n + 1) + h->factor_bytes;
    return BJ_OK;
}

int bj_setup_blocks_perm(const bj_csr_t* csr, const int64_t* block_ptr_host, int64_t nblocks, const int32_t* perm_dev,
                         void* cuda_stream, bj_handle_t* out)
{
    if (!out) return BJ_ERR_INVALID_ARG;
    *out = nullptr;
    if (!csr || !block_ptr_host || nblocks < 1 || nblocks > csr->n) return BJ_ERR_INVALID_ARG;
    if (block_ptr_host[0] != 0 || block_ptr_host[nblocks] != csr->n) return BJ_ERR_INVALID_ARG;
    for (int64_t k = 0; k < nblocks; ++k) {
        const int64_t s = block_ptr_host[k + 1] - block_ptr_host[k];
        if (s < 1 || s > BJ_B_MAX) return BJ_ERR_INVALID_ARG;
    }
    bj_handle_t h = nullptr;
    int rc = bj_setup_on_stream(csr, 0, cuda_stream, &h);  // validation and the SpMV plan of a b = 0 handle
    if (rc != BJ_OK) return rc;
    rc = var_setup(h, block_ptr_host, nblocks, perm_dev);
    if (rc != BJ_OK && rc != BJ_ERR_NOT_SPD) { free_handle(h); return rc; }
    *out = h;  // after BJ_ERR_NOT_SPD the handle only answers bj_get_info / bj_destroy, like bj_setup
    return rc;
}

int bj_setup_blocks(const bj_csr_t* csr, const int64_t* block_ptr_host, int64_t nblocks, void* cuda_stream, bj_handle_t* out)
{
    return bj_setup_blocks_perm(csr, block_ptr_host, nblocks, nullptr, cuda_stream, out);
}

int bj_setup_perm(const bj_csr_t* csr, int b, const int32_t* perm_dev, void* cuda_stream, bj_handle_t* out)
{
    if (!out) return BJ_ERR_INVALID_ARG;
    *out = nullptr;
    if (!csr || csr->n <= 0 || b < 1 || b > BJ_B_MAX || !perm_dev) return BJ_ERR_INVALID_ARG;
    bj_setup_opts_t o;
    memset(&o, 0, sizeof(o));
    o.cuda_stream = cuda_stream;
    return setup_impl(csr, b, o, out, perm_dev);  // the uniform-block kernels, vectors gathered / scattered through perm
}

int bj_release_cached_memory(void)
{
    int dev = 0;
    BJ_CUDA(cudaGetDevice(&dev));
    if (dev >= 0 && dev < 64 && g_pool[dev]) {
        BJ_CUDA(cudaDeviceSynchronize());
        BJ_CUDA(cudaMemPoolTrimTo(g_pool[dev], 0));
    }
    return BJ_OK;
}

int bj_set_stream(bj_handle_t h, void* cuda_stream)
{
    if (!h) return BJ_ERR_INVALID_ARG;
    h->stream = (cudaStream_t)cuda_stream;
    return BJ_OK;
}

int bj_set_option(bj_handle_t h, int option, int value)
{
    if (!h || h->failed) return BJ_ERR_INVALID_ARG;
    switch (option) {
        case BJ_OPT_SPMV_KERNEL:
            if (value < -1 || value > 1) return BJ_ERR_INVALID_ARG;
            h->opt_spmv_kernel = value;
            choose_spmv(h);
            return BJ_OK;
        case BJ_OPT_FUSE_FORWARD:
            if (value < -1 || value > 1) return BJ_ERR_INVALID_ARG;
            h->opt_fuse = value;
            return BJ_OK;
        case BJ_OPT_LANCZOS_FUSE:
            if (value < -1 || value > 1) return BJ_ERR_INVALID_ARG;
            h->opt_lanczos_fuse = value;
            return BJ_OK;
        case BJ_OPT_PCG_FUSE:
            if (value < -1 || value > 1) return BJ_ERR_INVALID_ARG;
            h->opt_pcg_fuse = value;
            return BJ_OK;
        case BJ_OPT_PCG_SINGLE_LAUNCH:
            if (value < -1 || value > 1) return BJ_ERR_INVALID_ARG;
            h->opt_pcg_small = value;
            return BJ_OK;
        case BJ_OPT_LANCZOS_SINGLE_LAUNCH:
            if (value < -1 || value > 2) return BJ_ERR_INVALID_ARG;
            h->opt_lanczos_small = value;
            return BJ_OK;
        default: return BJ_ERR_INVALID_ARG;
    }
}

int bj_destroy(bj_handle_t h)
{
    if (!h) return BJ_ERR_INVALID_ARG;
    cudaStreamSynchronize(h->stream);
    free_handle(h);
    return BJ_OK;
}

int bj_get_info(bj_handle_t h, bj_info_t* info)
{
    if (!h || !info) return BJ_ERR_INVALID_ARG;
    memset(info, 0, sizeof(*info));
    info->n = h->n; info->nnz = h->nnz; info->b = h->solve_kind == 4 ? -1 : h->b; info->nblocks = h->nblocks;
    info->bad_block = h->bad_block;
    info->factor_bytes = h->factor_bytes;
    info->workspace_bytes = h->workspace_bytes;
    info->kernel_launches = h->launches;
    info->spmv_kernel = h->spmv_kernel;
    info->spmv_lanes = h->spmv_lanes;
    info->solve_kernel = h->solve_kind == 4 ? 4 : h->solve_kind;
    info->band_width = (h->solve_kind == 3 || h->tri) ? h->band : -1;
    info->col16 = h->col16 ? 1 : 0;
    info->permuted = h->var_perm ? 1 : 0;
    info->fused_forward = (h->spmv_kernel == 1 && h->fuse_ok && h->opt_fuse != 0 && h->solve_kind != 0) ? 1 : 0;
    return BJ_OK;
}

#define BJ_CHECK_H(h) do { if (!(h) || (h)->failed) return BJ_ERR_INVALID_ARG; } while (0)

int bj_apply(bj_handle_t h, const double* r, double* z)
{
    BJ_CHECK_H(h);
    if (!r || !z) return BJ_ERR_INVALID_ARG;
    return launch_solve(h, 2, r, z);
}

int bj_solve_L(bj_handle_t h, const double* r, double* y)
{
    BJ_CHECK_H(h);
    if (!r || !y) return BJ_ERR_INVALID_ARG;
    return launch_solve(h, 0, r, y);
}

int bj_solve_Lt(bj_handle_t h, const double* y, double* x)
{
    BJ_CHECK_H(h);
    if (!y || !x) return BJ_ERR_INVALID_ARG;
    return launch_solve(h, 1, y, x);
}

int bj_spmv(bj_handle_t h, const double* x, double* y)
{
    BJ_CHECK_H(h);
    if (!x || !y || x == y) return BJ_ERR_INVALID_ARG;
    return launch_spmv(h, x, y);
}

int bj_op_apply(bj_handle_t h, const double* x, double* y)
{
    BJ_CHECK_H(h);
    if (!x || !y) return BJ_ERR_INVALID_ARG;
    return op_apply_device(h, x, y);
}

int bj_pcg_solve(bj_handle_t h, const double* b_dev, double* x_dev, const bj_pcg_opts_t* o, bj_pcg_result_t* res)
{
    if (!h || h->failed || !b_dev || !x_dev || !o || !res || o->max_iters < 1 || b_dev == x_dev) return BJ_ERR_INVALID_ARG;
    const int rc = pcg_run(h, b_dev, x_dev, o, res);
    if (rc != BJ_OK) return rc;
    return resolve_spans(h);
}

int bj_seeded_vector(bj_handle_t h, uint64_t seed, double* v)
{
    BJ_CHECK_H(h);
    if (!v) return BJ_ERR_INVALID_ARG;
    return launch_seeded_vector(h, seed, v);
}

int bj_cond_estimate_ex(bj_handle_t h, const bj_lanczos_opts_t* o, bj_lanczos_result_t* res)
{
    BJ_CHECK_H(h);
    if (!o || !res || o->iters < 1 || o->iters > (1 << 20)) return BJ_ERR_INVALID_ARG;
    return lanczos_run(h, o, res);
}

int bj_cond_estimate_minv(bj_handle_t h, const bj_lanczos_opts_t* o, bj_lanczos_result_t* res)
{
    BJ_CHECK_H(h);
    if (!o || !res || o->iters < 1 || o->iters > (1 << 20)) return BJ_ERR_INVALID_ARG;
    return mlanczos_run(h, o, res);
}

int bj_cond_estimate(bj_handle_t h, int iters, double* lmin, double* lmax)
{
    BJ_CHECK_H(h);
    if (iters < 1 || !lmin || !lmax) return BJ_ERR_INVALID_ARG;
    bj_lanczos_opts_t o;
    memset(&o, 0, sizeof(o));
    o.iters = iters;
    o.seed = BJ_DEFAULT_SEED;
    o.reorth = 1;
    if (h->lz.cap_vectors < iters) {  // the basis is not there yet: full reorthogonalisation only if it fits (the query costs ~50 us)
        size_t free_b = 0, total_b = 0;
        BJ_CUDA(cudaMemGetInfo(&free_b, &total_b));
        const double need = ((double)iters + 2.0) * (double)h->n * 8.0;
        o.reorth = need < 0.8 * (double)free_b ? 1 : 0;
    }
    bj_lanczos_result_t r;
    memset(&r, 0, sizeof(r));
    int rc = lanczos_run(h, &o, &r);
    if (rc != BJ_OK) return rc;
    *lmin = r.lmin;
    *lmax = r.lmax;
    return BJ_OK;
}

static int ensure_staging(bj_handle_s* h)
{
    if (h->stage_in) return BJ_OK;
    const size_t vb = (size_t)h->n * sizeof(double);
    if (cudaMalloc((void**)&h->stage_in, vb) != cudaSuccess || cudaMalloc((void**)&h->stage_out, vb) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(h->stage_in);
        h->stage_in = nullptr;
        return BJ_ERR_ALLOC;
    }
    h->workspace_bytes += 2 * (int64_t)vb;
    return BJ_OK;
}

int bj_op_apply_host(bj_handle_t h, const double* x_host, double* y_host)
{
    BJ_CHECK_H(h);
    if (!x_host || !y_host) return BJ_ERR_INVALID_ARG;
    int rc = ensure_staging(h);
    if (rc != BJ_OK) return rc;
    const size_t vb = (size_t)h->n * sizeof(double);
    BJ_CUDA(cudaMemcpyAsync(h->stage_in, x_host, vb, cudaMemcpyHostToDevice, h->stream));
    rc = op_apply_device(h, h->stage_in, h->stage_out);
    if (rc != BJ_OK) return rc;
    BJ_CUDA(cudaMemcpyAsync(y_host, h->stage_out, vb, cudaMemcpyDeviceToHost, h->stream));
    BJ_CUDA(cudaStreamSynchronize(h->stream));
    return BJ_OK;
}

int bj_apply_host(bj_handle_t h, const double* r_host, double* z_host)
{
    BJ_CHECK_H(h);
    if (!r_host || !z_host) return BJ_ERR_INVALID_ARG;
    int rc = ensure_staging(h);
    if (rc != BJ_OK) return rc;
    const size_t vb = (size_t)h->n * sizeof(double);
    BJ_CUDA(cudaMemcpyAsync(h->stage_in, r_host, vb, cudaMemcpyHostToDevice, h->stream));
    rc = launch_solve(h, 2, h->stage_in, h->stage_out);
    if (rc != BJ_OK) return rc;
    BJ_CUDA(cudaMemcpyAsync(z_host, h->stage_out, vb, cudaMemcpyDeviceToHost, h->stream));
    BJ_CUDA(cudaStreamSynchronize(h->stream));
    return BJ_OK;
}

int bj_profile_enable(bj_handle_t h, int on)
{
    BJ_CHECK_H(h);
    int rc = resolve_spans(h);
    if (rc != BJ_OK) return rc;
    h->prof_on = on != 0;
    if (on) {
        for (int k = 0; k < BJ_K_COUNT; ++k) { h->prof_ms[k] = 0.0; h->prof_cnt[k] = 0; }
    }
    return BJ_OK;
}

int bj_profile_get(bj_handle_t h, int kind, double* ms_total, int64_t* launches)
{
    BJ_CHECK_H(h);
    if (kind < 0 || kind >= BJ_K_COUNT) return BJ_ERR_INVALID_ARG;
    int rc = resolve_spans(h);
    if (rc != BJ_OK) return rc;
    if (ms_total) *ms_total = h->prof_ms[kind];
    if (launches) *launches = h->prof_cnt[kind];
    return BJ_OK;
}

}  // extern "C"
