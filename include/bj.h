/*
 * bj.h -- C ABI of the B200-native block-Jacobi preconditioning path of arxiv 2410.02408.
 *
 * What the library computes (citations: PAPER.md line numbers of /root/reference/PAPER.md,
 * and the readings fixed in DESIGN.md section 3):
 *   - A is a sparse symmetric positive-definite matrix (sec 3.1), here fp64 CSR.
 *   - It is partitioned into contiguous index blocks of size b (sec 3.2; the
 *     listing at 160-208 slices A[i:i+bs, j:j+bs], ragged at the edge).  Only the DIAGONAL tiles
 *     D_k enter the preconditioner M = blockdiag(D_k).
 *   - The paper's Jacobi preconditioner M_i = diag(A_i)^-1, A~ = M A, b~ = M b (PAPER.md:84-90,
 *     sec 3.3; kernel M[idx] = 1/A[idx*N+idx] at 214-235) is the case b = 1.  For general b each
 *     D_k = L_k L_k^T is factored by Cholesky and the preconditioned operator is taken in the
 *     symmetric split form  A^ = L^-1 A L^-T  (same spectrum as M^-1 A; HHL needs Hermitian input,
 *     PAPER.md:68).
 *   - kappa(A) = ||A|| ||A^-1|| = lambda_max / lambda_min is estimated by Lanczos
 *     on A (b = 0) and on A^; the paper's cost argument is O(log N kappa^2).
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer unless the parameter name ends in `_host` or the comment
 *     says "host".  The library never frees or reallocates caller memory.
 *   - CSR arrays passed to bj_setup are BORROWED and must outlive the handle.  They must be
 *     canonical: row_ptr[0] = 0, row_ptr[n] = nnz, row_ptr non-decreasing, 0 <= col < n, columns
 *     strictly increasing within each row, both triangles stored.  Symmetry is a precondition
 *     and is not checked.  Only the lower triangle of each diagonal block is read
 *     by the factorisation.
 *   - Vector arguments are length-n fp64 arrays.  In-place calls (output == input) are allowed
 *     for bj_apply, bj_solve_L, bj_solve_Lt and bj_op_apply; bj_spmv requires y != x.
 *   - bj_apply / bj_op_apply / bj_spmv / bj_solve_* only ENQUEUE work on the handle's stream and
 *     return without synchronising.  bj_setup, bj_cond_estimate*, bj_*_host synchronise.
 *   - All functions return BJ_OK (0) or a negative bj_status code; bj_strerror gives text.  A
 *     CUDA runtime failure returns BJ_ERR_CUDA and leaves the CUDA error string in bj_strerror.
 *   - No CPU fallback exists: without a CUDA device every compute entry point fails with BJ_ERR_CUDA.
 *   - A handle is not thread-safe; different handles may be used concurrently on different streams.
 *
 * Opt-in storage variants are ARGUMENTS (bj_setup_opts_t, bj_setup_ex), per handle: banded / compact factors, 16-bit
 * column deltas, a BSR(3) copy of the matrix.  Each moves fewer bytes than the CSR / dense-block counts of SURVEY.md 8(d)
 * and has its own byte accounting; each falls back silently to the default layout when the matrix
 * does not have the structure; results stay within the same tolerances.  bj_get_info reports which are in use.
 * Environment variables (BJ_*) only tune LAUNCH SHAPES (tile sizes, stages, warps per CTA); they
 * never select a storage format or an algorithm, and every result is independent of them up to summation order.
 */
#ifndef BJ_H_
#define BJ_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BJ_B_MAX 32                        /* largest supported block size on the GPU path      */
#define BJ_DEFAULT_SEED 0x241002408ull      /* default Lanczos start-vector seed                  */
#define BJ_DEFAULT_BREAKDOWN_TOL 1e-12      /* beta_{j+1} <= tol * max|alpha_i| ends the run      */

typedef enum {
    BJ_OK = 0,
    BJ_ERR_INVALID_ARG = -1,   /* null pointer, n <= 0, b < 0, b > BJ_B_MAX, iters < 1, y == x in bj_spmv */
    BJ_ERR_NOT_CANONICAL = -2, /* CSR validation failed (see Conventions)                                  */
    BJ_ERR_TOO_LARGE = -3,     /* n or nnz >= 2^31                                                         */
    BJ_ERR_NOT_SPD = -4,       /* a diagonal block has a pivot <= 0 or non-finite; see bj_info_t.bad_block  */
    BJ_ERR_ALLOC = -5,         /* device or host allocation failed                                         */
    BJ_ERR_CUDA = -6,          /* CUDA runtime error (sticky text in bj_strerror)                           */
    BJ_ERR_LIMIT = -7          /* bj_cond_estimate_noalloc: outside the limits of its fixed device scratch  */
} bj_status;

typedef struct bj_handle_s* bj_handle_t;

typedef struct {
    int64_t n, nnz;
    const int32_t* row_ptr; /* device, n+1 */
    const int32_t* col_idx; /* device, nnz */
    const double* val;      /* device, nnz */
} bj_csr_t;

/* Per-handle setup options (bj_setup_ex).  Zero-initialise, then set fields: 0 / NULL is the default everywhere, so
 * `bj_setup_opts_t o = {0};` reproduces bj_setup.  The three storage variants are SURVEY.md 8(f) NEXT-2: each is used
 * only when the matrix has the structure (otherwise the default layout, silently) and has its own byte model. */
typedef struct {
    void* cuda_stream;      /* cudaStream_t the setup runs on and the handle keeps (NULL: the default stream)               */
    int32_t band;           /* 1: banded diagonal blocks (lower bandwidth <= 2; b <= 8: tridiagonal) keep banded factors    */
    int32_t col16;          /* 1: the tile SpMV streams 16-bit column deltas col - row when every |col - row| < 32768       */
    int32_t bsr;            /* 1: a handle-owned BSR(3) copy of a 3x3-blocked matrix (three unknowns per node)              */
    int32_t serp_keep_mb;   /* serpentine walk of the factor array in chains of applies: megabytes of each walk left as
                               ordinary L2 lines for the next kernel (results bit-identical).  0: default (48); < 0: off   */
    int32_t reserved[8];    /* must be zero                                                                               */
} bj_setup_opts_t;

typedef struct {
    int32_t iters;        /* number of Lanczos steps = operator applies = dim of T (>= 1)           */
    int32_t reorth;       /* 0: none (fused fast mode), 1: full reorthogonalisation, twice (parity)  */
    uint64_t seed;        /* start vector v0[i] = 2 u_i - 1, u_i = (mix64(seed,i) >> 11) 2^-53       */
    const double* v0;     /* device, optional: caller-supplied start vector (overrides seed)         */
    double breakdown_tol; /* <= 0 selects BJ_DEFAULT_BREAKDOWN_TOL                                   */
} bj_lanczos_opts_t;

typedef struct {
    int32_t iters_done;   /* m_eff <= iters (smaller after a breakdown; not an error)                */
    double lmin, lmax;    /* extreme Ritz values of T_{m_eff}                                        */
    double res_min, res_max; /* Ritz residual bounds beta_{m+1} |s_{m,i}| for both ends               */
    double* alpha_host;   /* host, optional, caller-allocated, >= iters doubles: alpha_1..           */
    double* beta_host;    /* host, optional, caller-allocated, >= iters doubles: beta_2..beta_{m+1}   */
} bj_lanczos_result_t;

typedef struct {
    int64_t n, nnz;
    int32_t b;
    int64_t nblocks;
    int64_t bad_block;        /* first non-SPD block after BJ_ERR_NOT_SPD, else -1                   */
    int64_t factor_bytes;     /* device bytes held for the factors                                   */
    int64_t workspace_bytes;  /* device bytes held for temporaries and Lanczos workspace             */
    int64_t kernel_launches;  /* number of kernels this handle has launched so far                   */
    int32_t spmv_kernel;      /* 0: row-per-subwarp CSR-vector kernel, 1: TMA-streamed tile kernel,
                                 2: TMA-streamed BSR(3) kernel (opts.bsr)                              */
    int32_t spmv_lanes;       /* lanes per row chosen at setup                                       */
    int32_t solve_kernel;     /* 0: none (b=0), 1: thread-per-block (b<=8), 2: group/subwarp-per-block, 3: banded */
    int32_t fused_forward;    /* 1 if bj_op_apply fuses y = L^-1 u into the SpMV kernel               */
    int32_t band_width;       /* >= 0: banded factors in use (opts.band at setup), the lower bandwidth of every
                                 diagonal block; -1: dense packed factors                                   */
    int32_t col16;            /* 1: the tile SpMV streams 16-bit column deltas (opts.col16 at setup)            */
    int32_t permuted;         /* 1: the blocks are those of P A P^T (bj_setup_perm, bj_setup_blocks_perm)        */
} bj_info_t;

typedef struct {
    int32_t max_iters;    /* >= 1                                                                     */
    int32_t check_every;  /* the host reads the device stop flag every this many iterations; <= 0: 16 */
    double rtol;          /* stop when ||r_k|| / ||b|| <= rtol (recurrence residual); 0: run max_iters */
} bj_pcg_opts_t;

typedef struct {
    int32_t iters;        /* iterations done                                                          */
    int32_t converged;    /* 1 if the rtol test stopped the run                                       */
    double relres;        /* ||r_k|| / ||b|| from the recurrence at exit                              */
    double true_relres;   /* ||A x - b|| / ||b|| recomputed from x: the paper's accuracy metric */
    double lmin, lmax;    /* extreme Ritz values of M^-1 A from the CG coefficients (CG-Lanczos); 0 if iters < 1 */
    double* alpha_host;   /* host, optional, caller-allocated, >= max_iters doubles: step lengths a_k  */
    double* beta_host;    /* host, optional, >= max_iters doubles: bt_k                                */
    double* relres_host;  /* host, optional, >= max_iters doubles: ||r_{k+1}|| / ||b||                 */
} bj_pcg_result_t;

/* kernel-kind indices for bj_profile_get */
enum { BJ_K_SOLVE_LT = 0, BJ_K_SPMV = 1, BJ_K_SOLVE_L = 2, BJ_K_APPLY = 3, BJ_K_SPMV_SOLVE_L = 4, BJ_K_COUNT = 5 };

/* options for bj_set_option */
enum {
    BJ_OPT_SPMV_KERNEL = 1,   /* 0 / 1 as in bj_info_t.spmv_kernel; -1 = automatic (default) */
    BJ_OPT_FUSE_FORWARD = 2,  /* 0: three kernels, 1: fuse forward solve into SpMV, -1 = automatic    */
    BJ_OPT_LANCZOS_FUSE = 3,  /* 0: fast-mode Lanczos runs the unfused vector kernels; 1 / -1: the fused step (default) */
    BJ_OPT_PCG_FUSE = 4,      /* 0: PCG / M^-1 A Lanczos run the unfused iteration; 1 / -1: the fused one (default)     */
    BJ_OPT_PCG_SINGLE_LAUNCH = 6, /* 0: launch-bound sizes keep the multi-launch PCG iteration; 1 / -1 (default): bj_pcg_solve runs as ONE
                                 kernel of one cluster of 8 (or 16) CTAs when the vectors fit their shared memory (b <= 8 or 0) */
    BJ_OPT_LANCZOS_SINGLE_LAUNCH = 5 /* 0: launch-bound sizes (vectors + factors fit one CTA's shared memory, b <= 8) keep the
                                 multi-launch Lanczos; 1 / -1 (default): the whole run is ONE kernel -- of one cluster of 8
                                 (or 16) CTAs with the basis distributed over their shared memory when a CTA's share fits,
                                 else of one CTA; 2: always the single-CTA form                                         */
};

/* a1-a4. Validate the CSR, extract the diagonal b x b blocks, factor each
 * by Cholesky (b = 1: PAPER.md:234) and build the launch plan.  b >= 1; b == 0 builds an identity
 * preconditioner (A^ = A) used to estimate kappa(A).  The last block is ragged when b does not divide n.
 * On BJ_ERR_NOT_SPD a handle is still returned in *out so that bj_get_info can report bad_block; it
 * accepts only bj_get_info and bj_destroy.  Uses the default stream until bj_set_stream.  Synchronises. */
int bj_setup(const bj_csr_t* csr, int b, bj_handle_t* out);

/* Same as bj_setup but enqueues on `cuda_stream` (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream) and keeps it as the handle's stream. */
int bj_setup_on_stream(const bj_csr_t* csr, int b, void* cuda_stream, bj_handle_t* out);

/* Same as bj_setup with per-handle options (host struct, read during the call only; NULL = all defaults).  Two
 * handles of one process may differ in every option.  A non-zero reserved field is BJ_ERR_INVALID_ARG. */
int bj_setup_ex(const bj_csr_t* csr, int b, const bj_setup_opts_t* opts_host, bj_handle_t* out);

/* Device time of the setup kernels of THIS handle (a1-a3: validation, plan, extraction + Cholesky; CUDA events on the
 * handle's stream around the kernel sequence, host round trips between them excluded) and the bytes they must move
 * (12 nnz + 4 (n + 1) read once + factor bytes written).  Host out-pointers, either may be NULL. */
int bj_get_setup_time(bj_handle_t h, double* kernel_ms_host, int64_t* algorithmic_bytes_host);

/* Handle memory comes from a private stream-ordered pool that keeps freed slabs cached for the next
 * bj_setup (block-size sweeps); this returns the cache to the driver.  Synchronises the device. */
int bj_release_cached_memory(void);

/* diagonal blocks of DIFFERENT sizes (supervariable blocks).  block_ptr_host[0..nblocks] (host, int64):
 * 0 = p_0 < p_1 < .. < p_nblocks = n, every size p_{k+1} - p_k in 1..BJ_B_MAX; block k is the dense diagonal slice
 * A[p_k:p_{k+1}, p_k:p_{k+1}] (the listing of PAPER.md:191-197 with a per-block size).  The array is read during the call
 * only.  Every other entry point works on the handle unchanged (bj_apply, bj_solve_L/Lt, bj_op_apply, bj_cond_estimate*,
 * bj_pcg_solve; the Lanczos / PCG iterations run unfused); the batch entry points return BJ_ERR_INVALID_ARG.  One warp per
 * block (lane = row), packed lower triangles back to back.  bj_get_info reports b = -1, solve_kernel = 4.  Errors as
 * bj_setup; a layout that breaks the rules above is BJ_ERR_INVALID_ARG.  Synchronises. */
int bj_setup_blocks(const bj_csr_t* csr, const int64_t* block_ptr_host, int64_t nblocks, void* cuda_stream, bj_handle_t* out);

/* SURVEY 8(f) NEXT-3, the permutation argument ("RCM or strong-coupling lines"): the paper's partition into diagonal blocks
 * presupposes an ordering in which contiguous index ranges are the intended blocks.  perm_dev (device,
 * n int32, read during the call only: the handle keeps its own copy) is a permutation of 0..n-1, perm[i] = ORIGINAL index of
 * the unknown at permuted position i.  The diagonal blocks are those of P A P^T, (P A P^T)[i, j] = A[perm[i], perm[j]]:
 *     M = P^T blockdiag(D_k) P,   D_k = (P A P^T)[kb:(k+1)b, kb:(k+1)b] = L_k L_k^T      (ragged last block as in bj_setup)
 * and every vector of every entry point stays in the ORIGINAL ordering:
 *     bj_solve_L: y = P^T L^-1 P r,  bj_solve_Lt: x = P^T L^-T P y,  bj_apply: z = M^-1 r,  bj_op_apply: y = (P^T L^-1 P) A (P^T L^-T P) x
 * (orthogonally similar to the split operator of the permuted matrix: same spectrum, so bj_cond_estimate* report its
 * kappa).  No permuted copy of A is made: the extraction looks columns up through the inverse permutation, the block solves
 * gather and scatter through perm, the SpMV runs on A as it is.  bj_setup_perm runs on the uniform-block kernels of bj_setup
 * (bj_get_info: permuted = 1; plain solves and SpMV, unfused Lanczos / PCG iterations; the opt-in storage variants and the
 * batch entry points do not apply).  bj_setup_blocks_perm combines a permutation with block sizes 1..BJ_B_MAX given by
 * block_ptr_host (positions in the PERMUTED ordering) on the warp-per-block kernels of bj_setup_blocks (b = -1, solve_kernel = 4).  A sequence that is not a permutation is BJ_ERR_INVALID_ARG; other errors as bj_setup.  Synchronises. */
int bj_setup_perm(const bj_csr_t* csr, int b, const int32_t* perm_dev, void* cuda_stream, bj_handle_t* out);
int bj_setup_blocks_perm(const bj_csr_t* csr, const int64_t* block_ptr_host, int64_t nblocks, const int32_t* perm_dev,
                         void* cuda_stream, bj_handle_t* out);
int bj_set_stream(bj_handle_t h, void* cuda_stream);
int bj_set_option(bj_handle_t h, int option, int value);
int bj_destroy(bj_handle_t h);
int bj_get_info(bj_handle_t h, bj_info_t* info_host);
const char* bj_strerror(int code);

/* a5. z = M^-1 r = L^-T (L^-1 r), M = blockdiag(D_k)  (b~ = M b of PAPER.md:88-90).  b = 0: z = r. */
int bj_apply(bj_handle_t h, const double* r, double* z);
/* a6. y = A x (CSR SpMV). */
int bj_spmv(bj_handle_t h, const double* x, double* y);
/* y = L^-1 r (forward substitution per block) and x = L^-T y (backward). b = 0: copy. */
int bj_solve_L(bj_handle_t h, const double* r, double* y);
int bj_solve_Lt(bj_handle_t h, const double* y, double* x);
/* a7. y = L^-1 A L^-T x, the split-preconditioned operator (symmetric form of A~ = M A). */
int bj_op_apply(bj_handle_t h, const double* x, double* y);

/* a8-a9. Lanczos on A^ with the default options (full reorthogonalisation when the basis fits in
 * free device memory, else none; default seed); extreme Ritz values to host out-pointers.  Synchronises. */
int bj_cond_estimate(bj_handle_t h, int iters, double* lmin_host, double* lmax_host);
int bj_cond_estimate_ex(bj_handle_t h, const bj_lanczos_opts_t* opts_host, bj_lanczos_result_t* res_host);

/* the same spectrum from Lanczos on M^-1 A in the M inner product -- ONE pass over the factor per step
 * (z = M^-1 r, bj_apply) instead of the two of L^-1 A L^-T (A^ is similar to M^-1 A).  Three-term recurrence
 *   r_{j+1} = A u_j - al_j rh_j - bt_j rh_{j-1},  al_j = u_j . A u_j,  z_{j+1} = M^-1 r_{j+1},  bt_{j+1} = sqrt(r_{j+1} . z_{j+1}),
 *   u_j = z_j / bt_j,  rh_j = r_j / bt_j,
 * started from r_0 = the seeded vector (or opts.v0, device, length n) -- T = tridiag(bt_1..; al_0..) equals the tridiagonal of
 * bj_cond_estimate_ex started at v0 = L^-1 r_0.  opts.reorth is ignored (no reorthogonalisation: the fast-mode estimate);
 * iters, seed, v0, breakdown_tol and every field of the result mean what they mean for bj_cond_estimate_ex.  Two kernels per
 * step on the fused path (tile SpMV with a dot hook; block-solve pair with the combination built on the fly), vectors
 * unnormalised, scalars on the device, one synchronisation at the end.  Workspace: the PCG workspace (4 n doubles, kept).
 * A zero start vector returns BJ_ERR_INVALID_ARG.  Synchronises. */
int bj_cond_estimate_minv(bj_handle_t h, const bj_lanczos_opts_t* opts_host, bj_lanczos_result_t* res_host);

/* bj_cond_estimate_ex for callers that cannot allocate device memory at call time (CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same options, same result fields, the same single-launch cluster kernel
 * (DESIGN.md section 5), but its device scratch (start vector, alpha, beta, status words) is ONE file-scope device array
 * of fixed size, 147 488 bytes, which every GPU that loads the library holds until the process exits.  The call makes no
 * cudaMalloc / cudaFree / pool call and no allocating library call.
 * Limits: n <= BJ_NOALLOC_MAX_N, iters <= BJ_NOALLOC_MAX_ITERS, uniform blocks b <= 8 or b = 0 without permutation
 * or band storage, and a CTA's share of the basis must fit its shared memory (a cluster of 8 CTAs, or of 16 when the rows fit registers:
 * N = 1024 and N = 4096 at iters = 50 do, N = 16384 does not);
 * anything beyond returns BJ_ERR_LIMIT and does nothing.  The handle comes from bj_setup as usual (setup does allocate).
 * Every call on a device shares the array, which keeps the previous call's contents (the call clears what must start at
 * zero): calls that OVERLAP on the GPU -- two handles on two streams of one device -- race on it; serialise them.
 * The device must be current.  Synchronises. */
#define BJ_NOALLOC_MAX_N 16384
#define BJ_NOALLOC_MAX_ITERS 1024
int bj_cond_estimate_noalloc(bj_handle_t h, const bj_lanczos_opts_t* opts_host, bj_lanczos_result_t* res_host);

/* preconditioned conjugate gradients for A x = b from x_0 = 0 with M = blockdiag(D_k)
 * (z = M^-1 r is bj_apply; b = 0 handle: plain CG), the classical stand-in for the solve stage that follows
 * the preconditioning path.  b_dev and x_dev are device vectors of length n (x_dev out).
 * Textbook Hestenes-Stiefel ordering; every scalar stays on the device, the host only polls the stop flag every
 * check_every iterations.  Reports the paper's residual ||Ax-b||/||b|| (its bar is 1e-3,
 * PAPER.md:388) and a second estimate of the spectrum of M^-1 A from the CG coefficients.  Synchronises.
 * Workspace (4 n doubles) is allocated by the first call and kept by the handle.  b_dev = 0 returns x = 0, iters = 0. */
int bj_pcg_solve(bj_handle_t h, const double* b_dev, double* x_dev, const bj_pcg_opts_t* opts_host, bj_pcg_result_t* res_host);

/* Fill a device vector with the seeded start-vector sequence (see bj_lanczos_opts_t.seed). */
int bj_seeded_vector(bj_handle_t h, uint64_t seed, double* v);

/* End-to-end variants with HOST buffers (pinned or pageable): copy x to the device, run the device
 * path, copy the result back, synchronise.  Staging buffers belong to the handle. */
int bj_op_apply_host(bj_handle_t h, const double* x_host, double* y_host);
int bj_apply_host(bj_handle_t h, const double* r_host, double* z_host);

/* Per-kernel timing: when enabled, every kernel launched by the calls above is bracketed by CUDA
 * events on the handle's stream; bj_profile_get synchronises and returns the accumulated device
 * milliseconds and launch count of one kernel kind (BJ_K_*), then leaves the totals unchanged;
 * enabling again resets them. */
int bj_profile_enable(bj_handle_t h, int on);
int bj_profile_get(bj_handle_t h, int kind, double* ms_total_host, int64_t* launches_host);

/* many small independent systems in one launch (the paper's own sizes N = 2^10 .. 2^14,
 * PAPER.md:365, and its "solve each block separately" picture).  The handle's matrix is a batch of
 * `nsys` systems stored as ONE block-diagonal CSR.  offsets_host == NULL: equal sizes seg = n / nsys (system s owns rows
 * s*seg .. (s+1)*seg - 1; the block size b must divide seg).  Else offsets_host[0..nsys] (host, 0 = off[0] < .. < off[nsys] = n,
 * every offset a multiple of b): systems of different sizes, e.g. the paper's 2^10, 2^12 and 2^14 mixed in one batch.
 * bj_apply / bj_op_apply work on the batch unchanged.  This runs `iters`
 * Lanczos steps (no reorthogonalisation) on every system at once -- one CTA per system does the vector part of a step
 * with block-level reductions only -- and returns the extreme Ritz values per system: host arrays of nsys doubles
 * (kappa_s = lmax[s] / lmin[s]); iters_done_host (optional, nsys ints) is smaller than iters after a breakdown.
 * Start vector of system s: slice s of the seeded vector (bj_seeded_vector).  Synchronises. */
int bj_cond_estimate_batch(bj_handle_t h, int64_t nsys, const int64_t* offsets_host, int iters, uint64_t seed,
                           double* lmin_host, double* lmax_host, int32_t* iters_done_host);

/* NEXT-4, the solve side: PCG on every system of the batch at once (same layout rules as bj_cond_estimate_batch), each
 * system with its own step lengths and its own stopping test ||r_s|| / ||b_s|| <= rtol; a finished system is frozen
 * (its direction is zeroed) while the others go on.  b_dev / x_dev: device vectors of length n (x out).  Host outputs
 * (each optional, nsys entries): iterations taken, recurrence residual, and the paper's ||A x - b|| / ||b|| per system.
 * Synchronises. */
int bj_pcg_solve_batch(bj_handle_t h, int64_t nsys, const int64_t* offsets_host, const double* b_dev, double* x_dev,
                       int max_iters, double rtol, int32_t* iters_host, double* relres_host, double* true_relres_host);

#ifdef __cplusplus
}
#endif
#endif /* BJ_H_ */
