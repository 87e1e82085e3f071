// Internal declarations of the bj CUDA library (sm_100a only).  Not installed; the public
// boundary is include/bj.h.  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <utility>
#include <vector>

#include "bj.h"

namespace bj {

constexpr int kSmallMax = 8;        // b <= kSmallMax: one thread per block, factor in registers
constexpr int kInterleave = 32;     // blocks per interleave group in the small layout
constexpr int kReduceThreads = 256;
constexpr int kMaxPartials = 1184;  // 148 SMs x 8: upper bound on reduction grids

// status word bits written by the setup kernels
enum : int { ST_BAD_ROWPTR = 1, ST_BAD_COL = 2, ST_UNSORTED = 4, ST_NOT_SPD = 8 };

struct Status {
    int flags;
    int pad;
    long long bad_block;  // atomicMin target
    int max_tile_nnz;     // SpMV plan
    int max_row_nnz;
    unsigned long long coherent;  // entries whose column is within 16 of the same-position column of the next row
    unsigned long long compared;  // entries compared
    unsigned long long descents;        // entries with col[p] <= col[p-1]
    unsigned long long legal_descents;  // ... of which at the start of a non-empty row
    int max_band;                       // largest lower bandwidth of a diagonal block (band_width_kernel, opts.band)
    int pad2;
};

// Launch-shape knobs: defaults are the measured best on B200; each can be overridden by the environment variable
// BJ_<NAME>, read ONCE by bj_setup (sweeps re-run the setup).  They change launch geometry only -- never a storage
// format or an algorithm (those are bj_setup_opts_t / bj_set_option).
struct Tuning {
    int solve_warps = 8, solve_stage_kb = 32, solve_stages = 2, solve_ctas = 4;  // solve_stream_kernel
    int group_stages = 2, group_smem_kb = 220, group_warps = 12, group_lanes = 0;  // solve_group_kernel
    int serp_keep_mb = 48;  // bj_setup_opts_t.serp_keep_mb: serpentine walk of the block solves, megabytes of factor kept in L2 per walk
    int pdl_early = 4;      // bit 0: stream solves, bit 1: stream SpMV release their dependents at entry; bit 2 (default): the
                            // plain UNFUSED tile SpMV does (its dependent, the forward solve, then starts on the SMs the SpMV's
                            // tail frees and prefetches its factors: cfg 3 131.8 -> 128.9 us, cfg 4 184.7 -> 182.7; the fused
                            // SpMV + solve kernel measured 0.6 us slower with it and keeps the exit trigger)
    int ctas_per_sm = 4;    // wanted CTAs per SM of the SpMV tile kernel
};

// CUDA events right around each kernel of bj_setup (bj_get_setup_time): host work between launches and the read-backs
// between the phases are not device time
struct SetupTimer {
    cudaStream_t st;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> spans;
    explicit SetupTimer(cudaStream_t s) : st(s) {}
    void begin() { cudaEvent_t a = nullptr, b = nullptr; cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, st); spans.push_back({a, b}); }
    void end() { if (!spans.empty()) cudaEventRecord(spans.back().second, st); }
    double total_ms() {  // call after a stream synchronisation
        double t = 0.0;
        for (auto& sp : spans) { float ms = 0.f; if (cudaEventElapsedTime(&ms, sp.first, sp.second) == cudaSuccess) t += ms; else cudaGetLastError(); }
        return t;
    }
    ~SetupTimer() { for (auto& sp : spans) { cudaEventDestroy(sp.first); cudaEventDestroy(sp.second); } }
};

struct ProfSpan {
    int kind;
    cudaEvent_t a, b;
};

struct LanczosWs {
    int64_t cap_vectors = 0;  // vectors of length n held in V
    double* V = nullptr;      // basis (reorth) or 2 rotating vectors
    double* w = nullptr;
    double* partial = nullptr;  // kMaxPartials x (cap+1)
    double* coef = nullptr;     // reorth coefficients c[0..cap)
    double* alpha = nullptr;    // device alpha[iters]
    double* beta = nullptr;
    double* scal = nullptr;     // [0]=beta_j (current), [1]=amax, [2]=1/||v0||, [3]=alpha_j
    int* done = nullptr;        // [0]=stop flag, [1]=m_eff
    double* lz_part = nullptr;  // fused fast mode: [2][lz_cap] per-CTA partials of the epilogue kernel
    double* lz_sums = nullptr;  // [0] = v.w', [1] = w'.w'
    unsigned* lz_ticket = nullptr;
    int lz_cap = 0;
    int cap_iters = 0;
    size_t cap_partial = 0;  // doubles held in `partial`
    int64_t bytes = 0;
};

}  // namespace bj

struct bj_handle_s {
    // problem
    int64_t n = 0, nnz = 0;
    int b = 0;
    int64_t nblocks = 0;
    const int32_t* row_ptr = nullptr;
    const int32_t* col_idx = nullptr;
    const double* val = nullptr;
    cudaStream_t stream = nullptr;
    bool failed = false;  // NOT_SPD: only get_info / destroy allowed
    int64_t bad_block = -1;

    // factors
    int solve_kind = 0;  // 0 none, 1 small (interleaved), 2 warp (fwd + bwd packed copies), 3 banded (interleaved band), 4 variable-size blocks
    int32_t* var_bptr = nullptr;  // kind 4: block pointers (nblocks + 1), factor offsets (nblocks + 1), packed factors
    int64_t* var_foff = nullptr;
    double* var_fac = nullptr;
    int var_smax = 0;
    int32_t* var_perm = nullptr;  // permuted handle (bj_setup_perm, bj_setup_blocks_perm): perm and its inverse (handle-owned, n ints each)
    int32_t* var_pinv = nullptr;
    int band = -1;       // kind 3: lower bandwidth w of every diagonal block (0..2)
    double* fac_band = nullptr;  // kind 3: aliases the dense factor storage of the slab
    bool tri = false;    // kind 1 with opts.band: every block is (at most) tridiagonal, compact bidiagonal factors, packed = 2b - 1
    int lanes = 0;       // lanes per block for kind 2 (8, 16 or 32)
    int packed = 0;      // b(b+1)/2
    double* fac_small = nullptr;
    double* fac_fwd = nullptr;
    double* fac_bwd = nullptr;   // null when single_copy
    bool single_copy = false;    // b = 16, 24, 32 (group kernel): both substitutions run from the forward copy, the only one kept
    int64_t factor_bytes = 0;

    // temporaries
    void* slab = nullptr;     // one allocation holds t, u, status and the factors
    bool slab_pooled = false;
    double* t = nullptr;
    double* u = nullptr;
    bj::Status* status = nullptr;  // device
    int64_t workspace_bytes = 0;

    // SpMV plan
    int spmv_lanes = 8;       // lanes per row, CSR-vector kernel
    int stream_lanes = 1;     // lanes per row, reduce phase of the tile kernel
    int stream_warps = 8;     // consumer warps of the tile kernel
    int max_row_nnz = 0;      // longest row (validation pass)
    double coherence = 1.0;   // fraction of entries with |col(i+1, j) - col(i, j)| <= 16: ~1 banded/stencil, ~0 random
    int spmv_kernel = 0;      // chosen kernel: 0 CSR-vector, 1 TMA tile kernel, 2 BSR(3) copy
    int opt_spmv_kernel = -1; // user override
    int opt_fuse = -1;
    int opt_lanczos_fuse = -1;  // BJ_OPT_LANCZOS_FUSE / BJ_OPT_PCG_FUSE: 0 selects the unfused iterations
    int pcg_cl_cs = -1;  // cluster size of the single-launch PCG (bj_pcg_cluster.cu): -1 not asked yet, 0 not usable
    int opt_pcg_small = -1;  // BJ_OPT_PCG_SINGLE_LAUNCH: 0 keeps launch-bound sizes on the multi-launch iteration
    int cl_m = -1, cl_reorth = -1, cl_cs = 0;  // last answer of the cluster-size choice of bj_lanczos_cluster.cu
    int opt_lanczos_small = -1; // BJ_OPT_LANCZOS_SINGLE_LAUNCH: 0 keeps launch-bound sizes on the multi-launch path
    int opt_pcg_fuse = -1;
    bj_setup_opts_t opts = {};  // the options this handle was set up with
    double setup_kernel_ms = 0.0;  // device time of the setup kernels (bj_get_setup_time)
    bj::SetupTimer* setup_timer = nullptr;  // non-null while bj_setup runs
    int tile_rows = 0;        // rows per tile of the streamed kernel (multiple of b)
    int tile_cap = 0;         // nnz capacity per stage
    int tile_stages = 0;
    int64_t ntiles = 0;
    bool stream_ok = false;   // streamed kernel usable (alignment, capacity)
    bool fuse_ok = false;
    int num_sms = 148;
    bool pdl = true;          // chain the library's kernels with programmatic dependent launch
    bj::Tuning tune;

    // Lanczos
    bj::LanczosWs lz;

    // PCG workspace (bj_pcg.cu): r, z, p, q and the device scalars, allocated by the first bj_pcg_solve
    double* pcg_vec = nullptr;
    double* pcg_scal = nullptr;
    int pcg_cap_iters = 0;

    int16_t* col16 = nullptr;  // opt-in (opts.col16): column stream as 16-bit deltas col - row (owned by the handle)

    // BSR(3) copy of the matrix (bj_bsr.cu), opt-in (opts.bsr): owned by the handle
    double* bsr_val = nullptr;
    int32_t* bsr_col = nullptr;
    int32_t* bsr_rp = nullptr;
    bool bsr_ok = false;
    int64_t bsr_bytes = 0;
    int bsr_tile_rows = 0, bsr_tile_cap = 0, bsr_max_row_nnz = 0;

    // batched-systems workspace (bj_batch.cu): one allocation kept by the handle, grown on demand
    void* batch_ws = nullptr;
    size_t batch_ws_bytes = 0;

    // e2e staging
    double* stage_in = nullptr;
    double* stage_out = nullptr;

    // accounting
    int64_t launches = 0;
    bool prof_on = false;
    std::vector<bj::ProfSpan> spans;
    std::vector<cudaEvent_t> event_pool;
    double prof_ms[BJ_K_COUNT] = {0};
    int64_t prof_cnt[BJ_K_COUNT] = {0};
};

namespace bj {

// RAII bracket around ONE setup kernel launch (events only while bj_setup is timing)
struct SetupSpan {
    SetupTimer* t;
    explicit SetupSpan(bj_handle_s* h) : t(h->setup_timer) { if (t) t->begin(); }
    ~SetupSpan() { if (t) t->end(); }
};

// error plumbing -------------------------------------------------------------------------------
void set_cuda_error(cudaError_t e, const char* where);
#define BJ_CUDA(call)                                   \
    do {                                                \
        cudaError_t e__ = (call);                       \
        if (e__ != cudaSuccess) {                       \
            bj::set_cuda_error(e__, #call);             \
            return BJ_ERR_CUDA;                         \
        }                                               \
    } while (0)

// profiling brackets: RAII around one kernel launch
struct KernelScope {
    bj_handle_s* h;
    int kind;
    cudaEvent_t a = nullptr, b = nullptr;
    KernelScope(bj_handle_s* h_, int kind_);
    ~KernelScope();
};


// setup (bj_setup_kernels.cu)
int launch_validate(bj_handle_s* h);
int launch_extract_factor(bj_handle_s* h);
int launch_setup_rows(bj_handle_s* h);  // a1-a3 in one kernel for b <= 8, short rows, no permutation / band detection (bj_setup_rows.cu)
int launch_spmv_plan(bj_handle_s* h, int tile_rows);  // Status.max_tile_nnz for tiles of tile_rows rows
int col16_build(bj_handle_s* h);       // 16-bit column deltas when every |col - row| < 32768
void col16_free(bj_handle_s* h);

struct LzPrologue;
struct LzEpilogue;
struct PcgHook;

// banded block factors (bj_band_kernels.cu), opt-in
int launch_band_width(bj_handle_s* h);            // Status.max_band
int launch_extract_factor_band(bj_handle_s* h);   // a2 + a3 into fac_band
int launch_solve_band(bj_handle_s* h, int dir, const double* in, double* out, const LzPrologue* pro, const LzEpilogue* epi,
                      const PcgHook* pcg);

// solves (bj_solve_kernels.cu): dir 0 = forward (L^-1), 1 = backward (L^-T), 2 = both (apply)
// pro (dir 1 only) / epi (dir 0 only): fused Lanczos hooks of bj_lanczos_fuse.cuh, null for a plain solve
int launch_solve(bj_handle_s* h, int dir, const double* in, double* out, const LzPrologue* pro = nullptr,
                 const LzEpilogue* epi = nullptr, const PcgHook* pcg = nullptr);  // pcg: dir 2 only (bj_pcg_fuse.cuh)
bool lanczos_fusable(const bj_handle_s* h);

// SpMV (bj_spmv_kernels.cu)
int launch_spmv_vector(bj_handle_s* h, const double* x, double* y);
int launch_spmv_bsr(bj_handle_s* h, const double* x, double* y);  // bj_bsr.cu
int bsr_build(bj_handle_s* h);
void bsr_free(bj_handle_s* h);
// plain y = A x with the handle's chosen kernel (0 CSR-vector, 1 TMA tile kernel, 2 BSR(3))
int launch_spmv(bj_handle_s* h, const double* x, double* y);
struct LzReduce;
// epi: fused Lanczos epilogue; dot_with / dot_red: per-CTA partials of dot_with . y finished into *dot_red->out (unfused only)
int launch_spmv_stream(bj_handle_s* h, const double* x, double* y, bool fuse_forward, const LzEpilogue* epi = nullptr,
                       const double* dot_with = nullptr, const LzReduce* dot_red = nullptr);
struct StreamGeometry { int rows = 0; bool fuse = false; int lanes = 1, warps = 8; };
StreamGeometry spmv_stream_geometry(const bj_handle_s* h, bool random_cols);  // tile rows / fusion / lanes for a column structure
int spmv_stream_configure(bj_handle_s* h);  // geometry from h->coherence, launch tile_nnz_kernel (async)
void spmv_stream_adopt(bj_handle_s* h, const StreamGeometry& g);  // take a geometry whose fullest tile was measured already
int spmv_stream_finish(bj_handle_s* h, int max_tile);  // stage capacity and count, sets stream_ok

// Lanczos (bj_lanczos.cu)
int lanczos_run(bj_handle_s* h, const bj_lanczos_opts_t* o, bj_lanczos_result_t* r);
void lanczos_free(bj_handle_s* h);
int launch_seeded_vector(bj_handle_s* h, uint64_t seed, double* v);
// k-th smallest eigenvalue (k = 0 .. m-1) of the symmetric tridiagonal (diag a[0..m-1], off-diagonal e[0..m-2]), bisection
double tridiag_eig_k(int m, const double* a, const double* e, int k);
void lanczos_fill_result(int me, const double* a, const double* b, bj_lanczos_result_t* res);
// the whole run as one kernel of one eight-CTA cluster, the basis distributed over their shared memory (bj_lanczos_cluster.cu)
bool lanczos_cluster_usable(bj_handle_s* h, int m, bool reorth);
int launch_lanczos_cluster(bj_handle_s* h, int m, bool reorth, double tol, const double* v0, double* alpha, double* beta, int* done);
// the whole run as one single-CTA kernel for launch-bound sizes (bj_lanczos_small.cu)
bool lanczos_small_usable(const bj_handle_s* h, int m);
int launch_lanczos_small(bj_handle_s* h, int m, bool reorth, double tol, const double* v0, double* V, double* alpha, double* beta,
                         int* done);
// Lanczos on M^-1 A in the M inner product (bj_pcg.cu; shares the PCG workspace and the PCG hook of the solve kernels)
int mlanczos_run(bj_handle_s* h, const bj_lanczos_opts_t* o, bj_lanczos_result_t* res);

// preconditioned CG (bj_pcg.cu)
// variable-size blocks (bj_var_kernels.cu)
int var_setup(bj_handle_s* h, const int64_t* ptr_host, int64_t nblocks, const int32_t* perm_dev);  // perm_dev: device, or null
void var_free(bj_handle_s* h);
int perm_install(bj_handle_s* h, const int32_t* perm_dev);  // handle-owned copies of perm and its inverse; validates
void perm_free(bj_handle_s* h);
int launch_solve_var(bj_handle_s* h, int dir, const double* in, double* out);
int pcg_run(bj_handle_s* h, const double* b, double* x, const bj_pcg_opts_t* o, bj_pcg_result_t* r);
// the whole run as one kernel of one cluster for launch-bound sizes (bj_pcg_cluster.cu)
bool pcg_cluster_usable(bj_handle_s* h);
int launch_pcg_cluster(bj_handle_s* h, const double* b, double* x, int m, double rtol, double* alpha, double* beta, double* relres,
                       double* scal, double* pd, int* flags);
void pcg_free(bj_handle_s* h);
void batch_free(bj_handle_s* h);

int env_int(const char* name, int dflt);  // tuning knobs BJ_* (read at setup / launch)

// operator (bj_api.cu)
int op_apply_device(bj_handle_s* h, const double* x, double* y);
// one fused Lanczos step: t = L^-T v_next (v_next built by the prologue), w = L^-1 A t - beta v_cur with the dot partials
int op_apply_lanczos(bj_handle_s* h, const LzPrologue* pro, const LzEpilogue* epi, double* w);

}  // namespace bj
