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
#include <string.h>

#include <algorithm>
#include <atomic>

#include "bj_device.cuh"
#include "bj_internal.cuh"
#include "bj_lanczos_fuse.cuh"
#include "bj_reduce.cuh"

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

// P[cta] = sum over the CTA's chunk of a[i] * b[i]
__global__ void __launch_bounds__(kReduceThreads)
dot_partial_kernel(int64_t n, const double* __restrict__ a, const double* __restrict__ b, double* __restrict__ P)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) s = fma(a[i], b[i], s);
    s = block_sum(s, sh);
    if (threadIdx.x == 0) P[blockIdx.x] = s;
}

// Closes step j_prev and opens the next one:  beta = sqrt(sum PB);  out = in / beta.
//   mode 0: start vector, v_1 = v0 / ||v0||, no bookkeeping.
//   mode 1: beta_{j_prev+2} = ||w||: CTA 0 records beta[j_prev], max|alpha|, m_eff and the breakdown flag
//           (beta <= tol max|alpha|); on breakdown nothing is written.  out == nullptr: bookkeeping only.
__global__ void __launch_bounds__(kReduceThreads)
scale_kernel(int64_t n, const double* __restrict__ in, double* __restrict__ out, const double* __restrict__ PB,
             int nparts, int mode, int j_prev, double tol, const double* __restrict__ alpha,
             double* __restrict__ beta, double* __restrict__ amax_buf, int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (done[0]) return;
    const double bn = sqrt(reduce_partials(PB, nparts, sh));
    if (mode == 0 && (!(bn > 0.0) || isinf(bn))) {  // zero or non-finite start vector: invalid argument, nothing is written
        if (blockIdx.x == 0 && threadIdx.x == 0) { done[0] = 1; done[2] = 1; }
        return;
    }
    if (mode == 1) {
        const double a = fabs(alpha[j_prev]);
        const double prev = amax_buf[j_prev & 1];
        const double amax = a > prev ? a : prev;
        const bool brk = !(bn > tol * amax);
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            beta[j_prev] = bn;
            amax_buf[(j_prev + 1) & 1] = amax;
            done[1] = j_prev + 1;
            if (brk) done[0] = 1;
        }
        if (brk) return;
    }
    if (!out) return;
    const Chunk c = my_chunk(n);
    const double rb = __drcp_rn(bn);  // in / bn as one multiplication and a residual correction (div_by): the correctly rounded quotient
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) out[i] = div_by(in[i], bn, rb);
}

// w -= beta_j v_{j-1} (j > 0);  PA[cta] = partial of v_j . w
__global__ void __launch_bounds__(kReduceThreads)
alpha_partial_kernel(int64_t n, double* __restrict__ w, const double* __restrict__ vprev,
                     const double* __restrict__ v, const double* __restrict__ beta, int j,
                     double* __restrict__ PA, const int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (done[0]) return;
    const Chunk c = my_chunk(n);
    const double bj = j > 0 ? beta[j - 1] : 0.0;
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        double wi = w[i];
        if (j > 0) {
            wi -= bj * vprev[i];
            w[i] = wi;
        }
        s = fma(v[i], wi, s);
    }
    s = block_sum(s, sh);
    if (threadIdx.x == 0) PA[blockIdx.x] = s;
}

// alpha_j = sum PA (CTA 0 records it);  w -= alpha_j v_j;  optional PB[cta] = partial of w . w
__global__ void __launch_bounds__(kReduceThreads)
axpy_norm_kernel(int64_t n, double* __restrict__ w, const double* __restrict__ v, const double* __restrict__ PA,
                 int nparts, int j, double* __restrict__ alpha, double* __restrict__ PB, int want_norm,
                 const int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (done[0]) return;
    const double a = reduce_partials(PA, nparts, sh);
    if (blockIdx.x == 0 && threadIdx.x == 0) alpha[j] = a;
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
        const double wi = w[i] - a * v[i];
        w[i] = wi;
        s = fma(wi, wi, s);
    }
    if (want_norm) {
        __syncthreads();
        s = block_sum(s, sh);
        if (threadIdx.x == 0) PB[blockIdx.x] = s;
    }
}

// partial[cta * stride + q] = sum over chunk of V_q[i] * w[i],  q = 0..nv-1.
// Eight columns per sweep of the chunk (w is read once per eight columns, eight independent load streams per thread),
// one combined block reduction per sweep: shuffle tree per value, then thread d adds the warp sums of value d in order.
constexpr int kDotCols = 8;
__global__ void __launch_bounds__(kReduceThreads)
multidot_partial_kernel(int64_t n, int nv, const double* __restrict__ V, const double* __restrict__ w,
                        double* __restrict__ partial, int stride, const int* __restrict__ done)
{
    __shared__ double sh[kReduceThreads / 32][kDotCols];
    pdl_trigger();
    pdl_wait();
    if (done[0]) return;
    const Chunk c = my_chunk(n);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // The sweeps run from the LAST eight columns to the first (each dot product is independent: same bits in any order):
    // the kernel ends on the columns multiaxpy_kernel starts with, and starts on the ones it ended with in the previous
    // pass: a few columns per kernel come out of L2 (parity mode, m = 50, config 2: 21.5 -> 21.25 ms).  Explicit L2 policies
    // on top (keep the 2..6 boundary columns as ordinary lines, everything else evict_first) were measured and dropped:
    // the hinted loads run the two kernels 25 % slower (26.2 ms).  Also measured and dropped: alpha_j and w -= alpha_j v_j folded
    // into the first sweep of the first pass (saves the axpy_norm_kernel launch, but w then needs coherent loads and a
    // write-back inside the sweep: 20.9 -> 21.1 ms).
    for (int q0 = ((nv - 1) / kDotCols) * kDotCols; q0 >= 0; q0 -= kDotCols) {
        double s[kDotCols];
#pragma unroll
        for (int d = 0; d < kDotCols; ++d) s[d] = 0.0;
        const int live = nv - q0 < kDotCols ? nv - q0 : kDotCols;
        if (live == kDotCols) {
            for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
                const double wi = w[i];
                double vq[kDotCols];
#pragma unroll
                for (int d = 0; d < kDotCols; ++d) vq[d] = V[(int64_t)(q0 + d) * n + i];
#pragma unroll
                for (int d = 0; d < kDotCols; ++d) s[d] = fma(vq[d], wi, s[d]);
            }
        } else {
            for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += blockDim.x) {
                const double wi = w[i];
#pragma unroll
                for (int d = 0; d < kDotCols; ++d)
                    if (d < live) s[d] = fma(V[(int64_t)(q0 + d) * n + i], wi, s[d]);
            }
        }
#pragma unroll
        for (int d = 0; d < kDotCols; ++d) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) s[d] += __shfl_down_sync(0xffffffffu, s[d], off);
        }
        __syncthreads();  // the previous sweep's readers are done with sh
        if (lane == 0) {
#pragma unroll
            for (int d = 0; d < kDotCols; ++d) sh[warp][d] = s[d];
        }
        __syncthreads();
        if (threadIdx.x < live) {
            double r = 0.0;
            for (int q = 0; q < (int)(blockDim.x >> 5); ++q) r += sh[q][threadIdx.x];
            partial[(int64_t)blockIdx.x * stride + q0 + threadIdx.x] = r;
        }
    }
}

// w[i] -= c_0 V_0[i]; w[i] -= c_1 V_1[i]; ... in that order; optional partial of w . w.
// Same sweep structure as multidot_partial_kernel: eight columns at a time over the CTA's whole chunk of rows, so that every
// column is read in one contiguous run per CTA (a first version walked all columns row by row: 50 interleaved 2 KB pieces per
// CTA, 4.25 TB/s against the 6.3 TB/s of the dot kernel); the chunk of w waits in shared memory between the sweeps.
constexpr int kAxpyRowsPerThread = 8;                               // rows of w a thread holds in registers at a time
constexpr int kAxpyRowsMax = kAxpyRowsPerThread * kReduceThreads;   // rows of a piece (longer chunks go piece by piece)
__global__ void __launch_bounds__(kReduceThreads)
multiaxpy_kernel(int64_t n, int nv, const double* __restrict__ V, double* __restrict__ w,
                 const double* __restrict__ coef, double* __restrict__ PB, int want_norm,
                 const int* __restrict__ done, int piece)
{
    __shared__ double sh[kReduceThreads / 32];
    pdl_trigger();
    pdl_wait();
    if (done[0]) return;
    const Chunk c = my_chunk(n);
    double s = 0.0;
    for (int64_t lo = c.lo; lo < c.hi; lo += kAxpyRowsMax) {
        // the thread's rows lo + tid + k * 256 of the piece wait in registers between the sweeps (a first version kept the
        // piece in shared memory: one LDS + STS per row and sweep, 5.5 TB/s against the 6.3 TB/s of the dot kernel)
        double wr[kAxpyRowsPerThread];
        const int64_t base = lo + threadIdx.x;
#pragma unroll
        for (int k = 0; k < kAxpyRowsPerThread; ++k) wr[k] = base + k * kReduceThreads < c.hi ? w[base + k * kReduceThreads] : 0.0;
        for (int q0 = 0; q0 < nv; q0 += kDotCols) {
            const int live = nv - q0 < kDotCols ? nv - q0 : kDotCols;
            double cq[kDotCols];
#pragma unroll
            for (int d = 0; d < kDotCols; ++d) cq[d] = d < live ? coef[q0 + d] : 0.0;
            const double* Vq = V + (int64_t)q0 * n + base;
            if (live == kDotCols) {
#pragma unroll
                for (int k = 0; k < kAxpyRowsPerThread; ++k) {
                    if (base + k * kReduceThreads < c.hi) {
                        double vq[kDotCols];
#pragma unroll
                        for (int d = 0; d < kDotCols; ++d) vq[d] = Vq[(int64_t)d * n + k * kReduceThreads];
#pragma unroll
                        for (int d = 0; d < kDotCols; ++d) wr[k] -= cq[d] * vq[d];
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < kAxpyRowsPerThread; ++k) {
                    if (base + k * kReduceThreads < c.hi) {
#pragma unroll
                        for (int d = 0; d < kDotCols; ++d)
                            if (d < live) wr[k] -= cq[d] * Vq[(int64_t)d * n + k * kReduceThreads];
                    }
                }
            }
        }
#pragma unroll
        for (int k = 0; k < kAxpyRowsPerThread; ++k) {
            if (base + k * kReduceThreads < c.hi) {
                w[base + k * kReduceThreads] = wr[k];
                s = fma(wr[k], wr[k], s);
            }
        }
    }
    if (want_norm) {
        s = block_sum(s, sh);
        if (threadIdx.x == 0) PB[blockIdx.x] = s;
    }
}

// Reorthogonalisation, middle of a step: w -= V c (the first pass' update) AND the second pass' dot products c2 = V^T w in
// ONE pass over the basis.  Four kernels per step read V four times (dot, axpy, dot, axpy: 4 x 16.8 MB x j on config 2);
// the update of one pass and the dots of the next need the same tile of V and nothing global in between, so a persistent
// CTA brings a tile of R rows of every column into shared memory ONCE (one bulk async copy per column and stage, two
// stages of 100 KB), updates its rows of w (thread per row, subtraction order q = 0, 1, ..: the oracle's),
// writes them back, and adds the tile's contribution to its running c2 (warp per column, fixed order).  Three reads of V
// per step instead of four.  Partials: partial[cta * stride + q], closed by finalize_multi_kernel as before.
constexpr int kFuseThreads = 512;
constexpr int kFuseCtasPerSm = 1;
constexpr int kFuseWarps = kFuseThreads / 32;
constexpr int kFuseSlots = 208 / kFuseWarps;   // columns per warp at most: nv <= 208
constexpr int kFuseStages = 2;                 // measured on config 2, m = 50 (BJ_REORTH_STAGES / BJ_REORTH_STAGE_KB): 2 x 100 KB 19.4 ms,
                                               // 3 x 66 KB 21.4, 4 x 50 KB 23.4, two 256-thread CTAs per SM 22.3: a tile costs ~1 us
                                               // whatever its height (barriers, the nv-step update chain, the shuffle trees), so
                                               // tall tiles win although two stages keep only one tile in flight
constexpr int kFuseStageBytes = 100 * 1024;
__global__ void __launch_bounds__(kFuseThreads, kFuseCtasPerSm)
reorth_axpy_dot_kernel(int64_t n, int nv, const double* __restrict__ V, double* __restrict__ w, const double* __restrict__ coef,
                       double* __restrict__ partial, int stride, const int* __restrict__ done, int R, int64_t ntiles, int S)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);            // [kFuseStages]
    double* cs = reinterpret_cast<double*>(smem_raw + 64);              // coefficients of the update, nv (<= 208)
    double* w1 = cs + 208;                                              // the tile's updated rows, R (<= 512)
    double* stage0 = w1 + 512;                                          // [kFuseStages][(nv + 1) * R]: columns 0..nv-1, then w
    const size_t stage_doubles = (size_t)(nv + 1) * R;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    pdl_trigger();
    if (tid == 0) {
        for (int q = 0; q < S; ++q) mbar_init(&full[q], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_wait();  // w and the coefficients come from the previous kernels
    if (done[0]) return;
    for (int q = tid; q < nv; q += kFuseThreads) cs[q] = coef[q];
    // a full tile (R rows) arrives by bulk copies; the ragged last tile is read with ordinary loads
    auto issue = [&](int64_t tile, int s) {  // warp 0
        const int64_t r0 = tile * R;
        if (r0 + R > n) return;
        double* dst = stage0 + (size_t)s * stage_doubles;
        const uint32_t bytes = (uint32_t)R * 8u;
        if (lane == 0) mbar_expect_tx(&full[s], bytes * (uint32_t)(nv + 1));
        __syncwarp();
        const uint64_t pol = policy_evict_first();
        for (int q = lane; q <= nv; q += 32)
            bulk_g2s(dst + (size_t)q * R, q < nv ? V + (int64_t)q * n + r0 : w + r0, bytes, &full[s], pol);
    };
    double acc[kFuseSlots];
#pragma unroll
    for (int k = 0; k < kFuseSlots; ++k) acc[k] = 0.0;
    if (warp == 0) {
        for (int q = 0; q < S; ++q)
            if ((int64_t)blockIdx.x + (int64_t)q * gridDim.x < ntiles) issue((int64_t)blockIdx.x + (int64_t)q * gridDim.x, q);
    }
    __syncthreads();  // cs is complete
    int it = 0;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        const int s = it % S;
        const int64_t r0 = tile * R;
        const int rows = (int)(r0 + R <= n ? R : n - r0);
        double* Vs = stage0 + (size_t)s * stage_doubles;
        if (rows == R) {
            mbar_wait(&full[s], (uint32_t)((it / S) & 1));
        } else {
            for (int e = tid; e < (nv + 1) * rows; e += kFuseThreads) {
                const int q = e / rows, r = e - q * rows;
                Vs[(size_t)q * R + r] = q < nv ? V[(int64_t)q * n + r0 + r] : w[r0 + r];
            }
            __syncthreads();
        }
        // ---- w -= V c on the tile's rows (thread per row) ----
        if (tid < rows) {
            double wi = Vs[(size_t)nv * R + tid];
            for (int q = 0; q < nv; ++q) wi -= cs[q] * Vs[(size_t)q * R + tid];
            w1[tid] = wi;
            w[r0 + tid] = wi;
        }
        __syncthreads();
        // ---- c2 += V^T w1 over the tile (warp per column, lanes stride the rows, fixed shuffle tree) ----
#pragma unroll
        for (int k = 0; k < kFuseSlots; ++k) {
            const int q = warp + k * kFuseWarps;
            if (q < nv) {
                const double* col = Vs + (size_t)q * R;
                double s0 = 0.0, s1 = 0.0;
                int r = lane;
                for (; r + 32 < rows; r += 64) {
                    s0 = fma(col[r], w1[r], s0);
                    s1 = fma(col[r + 32], w1[r + 32], s1);
                }
                if (r < rows) s0 = fma(col[r], w1[r], s0);
                double sq = s0 + s1;
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) sq += __shfl_down_sync(0xffffffffu, sq, off);
                acc[k] += sq;  // (meaningful on lane 0)
            }
        }
        __syncthreads();  // the stage and w1 are free
        if (warp == 0 && tile + S * (int64_t)gridDim.x < ntiles) issue(tile + S * (int64_t)gridDim.x, s);
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < kFuseSlots; ++k) {
            const int q = warp + k * kFuseWarps;
            if (q < nv) partial[(int64_t)blockIdx.x * stride + q] = acc[k];
        }
    }
}

// The same fused pass with the tile in REGISTERS (nv <= NVMAX <= 52): a thread takes one row at a time, requests its nv basis
// entries together (coalesced across the warp: consecutive threads, consecutive rows; ~100 KB in flight per SM), updates
// w_r in the oracle's order, writes it back, and adds V_qr w_r to its nv private accumulators; one reduction at the very
// end (shuffle tree per column inside each warp, then the warp sums in order).  No shared-memory tile, no bulk copies (a
// 1.8 KB copy per column and tile is what holds the kernel above at 3.4 TB/s), no barrier inside the stream.
constexpr int kRegFuseThreads = 256;
template <int NVMAX, int MINB>
__global__ void __launch_bounds__(kRegFuseThreads, MINB)
reorth_axpy_dot_reg_kernel(int64_t n, int nv, const double* __restrict__ V, double* __restrict__ w, const double* __restrict__ coef,
                           double* __restrict__ partial, int stride, const int* __restrict__ done)
{
    __shared__ double cs[NVMAX];
    __shared__ double sh[kRegFuseThreads / 32][NVMAX];
    pdl_trigger();
    pdl_wait();
    if (done[0]) return;
    for (int q = threadIdx.x; q < NVMAX; q += kRegFuseThreads) cs[q] = q < nv ? coef[q] : 0.0;
    __syncthreads();
    double acc[NVMAX];
#pragma unroll
    for (int q = 0; q < NVMAX; ++q) acc[q] = 0.0;
    const Chunk c = my_chunk(n);
    for (int64_t i = c.lo + threadIdx.x; i < c.hi; i += kRegFuseThreads) {
        double v[NVMAX];
#pragma unroll
        for (int q = 0; q < NVMAX; ++q) v[q] = q < nv ? V[(int64_t)q * n + i] : 0.0;
        double wi = w[i];
#pragma unroll
        for (int q = 0; q < NVMAX; ++q) wi -= cs[q] * v[q];  // (columns past nv: c = v = 0, exact)
        w[i] = wi;
#pragma unroll
        for (int q = 0; q < NVMAX; ++q) acc[q] = fma(v[q], wi, acc[q]);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int q = 0; q < NVMAX; ++q) {
        double sq = acc[q];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) sq += __shfl_down_sync(0xffffffffu, sq, off);
        if (lane == 0) sh[warp][q] = sq;
    }
    __syncthreads();
    if (threadIdx.x < nv) {
        double r = 0.0;
#pragma unroll
        for (int k = 0; k < kRegFuseThreads / 32; ++k) r += sh[k][threadIdx.x];
        partial[(int64_t)blockIdx.x * stride + threadIdx.x] = r;
    }
}

// out[q] = sum_cta partial[cta * stride + q]: one CTA per coefficient (a single CTA for all of them took 39 us at 50 vectors,
// one tenth of a parity-mode step).  Thread t adds the partials of CTAs t, t + 256, .. in that order, then the fixed block
// tree: bitwise reproducible.
__global__ void __launch_bounds__(256)
finalize_multi_kernel(int nparts, int nv, const double* __restrict__ partial, int stride,
                      double* __restrict__ out, const int* __restrict__ done)
{
    __shared__ double sh[8];
    pdl_trigger();
    pdl_wait();
    if (done[0]) return;
    const int q = blockIdx.x;
    double s = 0.0;
    for (int p = threadIdx.x; p < nparts; p += blockDim.x) s += partial[(int64_t)p * stride + q];
    s = block_sum(s, sh);
    if (threadIdx.x == 0) out[q] = s;
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
    cudaFree(z.alpha);  // one block: done | scal | alpha | beta
    cudaFree(z.lz_part); cudaFree(z.lz_sums); cudaFree(z.lz_ticket);
    h->workspace_bytes -= z.bytes;
    z = LanczosWs();
}

static int lanczos_alloc(bj_handle_s* h, int iters, int64_t nvec, bool reorth)
{
    LanczosWs& z = h->lz;
    // partials: two rows for alpha / beta; the reorthogonalisation coefficients need kMaxPartials x (iters + 1) more,
    // which only the parity mode touches (9.5 KB per iteration: not reserved for fast-mode runs of 10^5 steps)
    const size_t want_partial = (size_t)kMaxPartials * (reorth ? (size_t)iters + 3 : 2);
    if (z.cap_vectors >= nvec && z.cap_iters >= iters && z.cap_partial >= want_partial) return BJ_OK;
    lanczos_free(h);
    const size_t vb = (size_t)h->n * sizeof(double);
    int64_t bytes = 0;
    auto A = [&](void** p, size_t sz) { cudaError_t e = cudaMalloc(p, sz); if (e == cudaSuccess) bytes += sz; return e; };
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = A((void**)&z.V, vb * nvec);
    if (e == cudaSuccess) e = A((void**)&z.w, vb);
    if (e == cudaSuccess) e = A((void**)&z.partial, sizeof(double) * want_partial);
    if (e == cudaSuccess) e = A((void**)&z.coef, sizeof(double) * (size_t)(iters + 1));
    // one block (one memset before a run, one copy back after it): alpha[iters] | beta[iters] | scal[8] | done[4 ints]
    if (e == cudaSuccess) e = A((void**)&z.alpha, sizeof(double) * (2 * (size_t)iters + 8 + 2));
    if (e == cudaSuccess) {
        z.beta = z.alpha + iters;
        z.scal = z.beta + iters;
        z.done = reinterpret_cast<int*>(z.scal + 8);
    }
    // fused fast mode: the epilogue kernel with the largest grid is the thread-per-block solve (nblocks / 128 CTAs)
    z.lz_cap = (int)std::max<int64_t>(kMaxPartials, (h->nblocks + 127) / 128 + 1);
    if (e == cudaSuccess) e = A((void**)&z.lz_part, sizeof(double) * 2 * (size_t)z.lz_cap);
    if (e == cudaSuccess) e = A((void**)&z.lz_sums, sizeof(double) * 4);
    if (e == cudaSuccess) e = A((void**)&z.lz_ticket, sizeof(unsigned) * 4);
    z.bytes = bytes;
    h->workspace_bytes += bytes;
    if (e != cudaSuccess) {
        cudaGetLastError();
        lanczos_free(h);
        return BJ_ERR_ALLOC;
    }
    z.cap_vectors = nvec;
    z.cap_iters = iters;
    z.cap_partial = want_partial;
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

double tridiag_eig_k(int m, const double* a, const double* e, int k)
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

// one D2H copy of alpha[], beta[] and the flags at the end of a run; extremes of T on the host
static int lanczos_readback(bj_handle_s* h, int m, bj_lanczos_result_t* res)
{
    LanczosWs& z = h->lz;
    cudaStream_t st = h->stream;
    const size_t cap = (size_t)z.cap_iters, words = 2 * cap + 8 + 2;
    std::vector<double> blk(words);
    BJ_CUDA(cudaMemcpyAsync(blk.data(), z.alpha, sizeof(double) * words, cudaMemcpyDeviceToHost, st));  // one copy: alpha | beta | scal | done
    BJ_CUDA(cudaStreamSynchronize(st));
    const double* ap = blk.data();
    const double* bp = blk.data() + cap;
    int done[4];
    memcpy(done, blk.data() + 2 * cap + 8, sizeof(done));
    std::vector<double> a(ap, ap + m), b(bp, bp + m);
    if (done[2]) return BJ_ERR_INVALID_ARG;  // ||v0|| is zero or not finite
    const int me = done[1];
    if (me < 1) return BJ_ERR_CUDA;
    lanczos_fill_result(me, a.data(), b.data(), res);
    return BJ_OK;
}

// ------------------------------------------------------------------------------------------------
int lanczos_run(bj_handle_s* h, const bj_lanczos_opts_t* o, bj_lanczos_result_t* res)
{
    const int m = o->iters;
    const bool reorth = o->reorth != 0;
    const double tol = o->breakdown_tol > 0.0 ? o->breakdown_tol : BJ_DEFAULT_BREAKDOWN_TOL;
    const int64_t n = h->n;
    const int64_t nvec = reorth ? m : 2;
    int rc = lanczos_alloc(h, m, nvec, reorth);
    if (rc != BJ_OK) return rc;
    LanczosWs& z = h->lz;
    cudaStream_t st = h->stream;
    const int stride = m + 1;
    const int G = (int)std::max<int64_t>(1, std::min<int64_t>(kMaxPartials, (n + 1023) / 1024));
    const int64_t chunk_rows = (n + G - 1) / G;  // rows per CTA of the vector kernels (my_chunk)
    const int axpy_piece = (int)std::min<int64_t>(chunk_rows, kAxpyRowsMax);
    const size_t axpy_smem = 0;
    bool fuse_reorth = reorth && env_int("BJ_REORTH_FUSE", 1) != 0;
    const int fuse_stages = std::max(2, std::min(8, env_int("BJ_REORTH_STAGES", kFuseStages)));
    const int fuse_stage_bytes = std::min(env_int("BJ_REORTH_STAGE_KB", kFuseStageBytes / 1024) * 1024, 200 * 1024 / fuse_stages) / kFuseCtasPerSm;
    if (fuse_reorth) {
        static std::atomic<bool> configured[64];
        if (ensure_big_smem(reorth_axpy_dot_kernel, configured) != cudaSuccess) { cudaGetLastError(); fuse_reorth = false; }
    }

    BJ_CUDA(cudaMemsetAsync(z.alpha, 0, sizeof(double) * (2 * (size_t)z.cap_iters + 8 + 2), st));  // alpha, beta, scal, done

    auto vcol = [&](int j) { return z.V + (size_t)(reorth ? j : (j & 1)) * (size_t)n; };
    double* PA = z.partial;                 // per-CTA partials of v_j . w
    double* PB = z.partial + kMaxPartials;  // per-CTA partials of w . w
    double* PM = z.partial + 2 * kMaxPartials;  // reorthogonalisation partials, G x stride
    double* amax_buf = z.scal;              // two slots, ping-pong
    const bool pdl = h->pdl;
    cudaError_t e = cudaSuccess;
#define BJ_LAUNCH(kernel, grid, block, ...)                                          \
    do {                                                                             \
        e = launch_kernel(kernel, dim3(grid), dim3(block), 0, st, pdl, __VA_ARGS__); \
        if (e != cudaSuccess) { set_cuda_error(e, #kernel); return BJ_ERR_CUDA; }    \
        h->launches++;                                                               \
    } while (0)

    // v_1 = v0 / ||v0||
    const double* v0 = o->v0;
    if (!v0) {
        rc = launch_seeded_vector(h, o->seed, z.w);
        if (rc != BJ_OK) return rc;
        v0 = z.w;
    }
    const bool cluster_ok = h->opt_lanczos_small != 0 && h->opt_lanczos_small != 2 && lanczos_cluster_usable(h, m, reorth);
    if (h->opt_lanczos_small != 0 && (cluster_ok || lanczos_small_usable(h, m))) {
        // launch-bound sizes: the whole run is ONE single-CTA kernel (bj_lanczos_small.cu)
        // (option value 2 keeps the single-CTA form; by default the eight-CTA cluster form runs when a CTA's share of the basis fits)
        if (cluster_ok)
            rc = launch_lanczos_cluster(h, m, reorth, tol, v0, z.alpha, z.beta, z.done);
        else
            rc = launch_lanczos_small(h, m, reorth, tol, v0, z.V, z.alpha, z.beta, z.done);
        if (rc != BJ_OK) return rc;
        return lanczos_readback(h, m, res);
    }
    const bool fused_mode = !reorth && lanczos_fusable(h) && h->opt_lanczos_fuse != 0;
    if (!fused_mode) BJ_LAUNCH(dot_partial_kernel, G, kReduceThreads, n, v0, v0, PB);
    if (!fused_mode)
        BJ_LAUNCH(scale_kernel, G, kReduceThreads, n, v0, vcol(0), (const double*)PB, G, 0, 0, tol,
                  (const double*)z.alpha, z.beta, amax_buf, z.done);

    const bool fused = fused_mode;
    if (fused) {
        // Fast mode, fused: an iteration is exactly the kernels of one operator apply (bj_lanczos_fuse.cuh).
        BJ_CUDA(cudaMemsetAsync(z.lz_ticket, 0, sizeof(unsigned) * 4, st));
        LzPrologue pro;
        LzEpilogue epi;
        pro.w = z.w; pro.sum_a = z.lz_sums; pro.alpha = z.alpha; pro.done = z.done;
        pro.red.part = z.lz_part; pro.red.out = z.lz_sums + 1; pro.red.ticket = z.lz_ticket; pro.red.cap = z.lz_cap;
        epi.w = z.w; epi.sum_b = z.lz_sums + 1; epi.alpha = z.alpha; epi.beta = z.beta; epi.amax = amax_buf;
        epi.done = z.done; epi.tol = tol;
        epi.red.part = z.lz_part; epi.red.out = z.lz_sums; epi.red.ticket = z.lz_ticket; epi.red.cap = z.lz_cap;
        for (int j = 0; j < m; ++j) {
            pro.w0 = j == 0 ? v0 : nullptr;
            pro.vcur = j > 0 ? vcol(j - 1) : nullptr;
            pro.j = j - 1;
            pro.first = j == 0;
            epi.vprev = j > 0 ? vcol(j - 1) : nullptr;
            epi.vnew = vcol(j);
            epi.j = j - 1;
            epi.first = j == 0;
            rc = op_apply_lanczos(h, &pro, &epi, z.w);
            if (rc != BJ_OK) return rc;
        }
        // close the last step with the unfused kernels: alpha_m, w = w' - alpha_m v_m, beta_{m+1} = ||w||
        BJ_LAUNCH(axpy_norm_kernel, G, kReduceThreads, n, z.w, (const double*)vcol(m - 1), (const double*)z.lz_sums, 1, m - 1,
                  z.alpha, PB, 1, (const int*)z.done);
        BJ_LAUNCH(scale_kernel, G, kReduceThreads, n, (const double*)z.w, (double*)nullptr, (const double*)PB, G, 1, m - 1, tol,
                  (const double*)z.alpha, z.beta, amax_buf, z.done);
    }
    for (int j = 0; j < m && !fused; ++j) {
        double* vj = vcol(j);
        rc = op_apply_device(h, vj, z.w);  // w = A^ v_j
        if (rc != BJ_OK) return rc;
        BJ_LAUNCH(alpha_partial_kernel, G, kReduceThreads, n, z.w, (const double*)(j > 0 ? vcol(j - 1) : vj),
                  (const double*)vj, (const double*)z.beta, j, PA, (const int*)z.done);
        BJ_LAUNCH(axpy_norm_kernel, G, kReduceThreads, n, z.w, (const double*)vj, (const double*)PA, G, j, z.alpha,
                  PB, reorth ? 0 : 1, (const int*)z.done);
        if (reorth) {
            const int nv = j + 1;
            // the first pass' update and the second pass' dots in one pass over V (reorth_axpy_dot_kernel) when a tile of
            // at least 32 rows of all nv columns fits a stage and the arrays are 16-byte aligned for the bulk copies
            int R = (int)(((size_t)fuse_stage_bytes / ((size_t)(nv + 1) * 8)) & ~(size_t)31);
            if (R > kFuseThreads) R = kFuseThreads;  // a thread per row of the tile
            const bool fuse_mid = fuse_reorth && R >= 32 && nv <= kFuseWarps * kFuseSlots && n % 2 == 0 &&
                                  ((uintptr_t)z.V % 16) == 0 && ((uintptr_t)z.w % 16) == 0;
            for (int pass = 0; pass < 2; ++pass) {
                const bool fused_before = pass == 1 && (fuse_mid || (fuse_reorth && nv <= 52 && env_int("BJ_REORTH_REG", 1) != 0));
                if (!fused_before) {
                    BJ_LAUNCH(multidot_partial_kernel, G, kReduceThreads, n, nv, (const double*)z.V,
                              (const double*)z.w, PM, stride, (const int*)z.done);
                    BJ_LAUNCH(finalize_multi_kernel, nv, 256, G, nv, (const double*)PM, stride, z.coef,
                              (const int*)z.done);
                }
                if (pass == 0 && fuse_reorth && nv <= 52 && env_int("BJ_REORTH_REG", 1) != 0) {
                    // the tile in registers (no alignment condition: ordinary loads)
                    // the kernel's cost follows NVMAX (padding columns are multiplied by zeros) and, for few columns, the
                    // memory latency of a row: narrower variants run more CTAs per SM
                    int grid = 0;
#define BJ_REG_FUSE(NVM, MB)                                                                                                   \
    do {                                                                                                                       \
        grid = (int)std::min<int64_t>((n + kRegFuseThreads - 1) / kRegFuseThreads, (int64_t)h->num_sms * MB);                  \
        e = launch_kernel(reorth_axpy_dot_reg_kernel<NVM, MB>, dim3(grid), dim3(kRegFuseThreads), 0, st, pdl, n, nv,           \
                          (const double*)z.V, z.w, (const double*)z.coef, PM, stride, (const int*)z.done);                     \
    } while (0)
                    if (nv <= 8) BJ_REG_FUSE(8, 4);
                    else if (nv <= 16) BJ_REG_FUSE(16, 3);
                    else if (nv <= 24) BJ_REG_FUSE(24, 2);
                    else if (nv <= 32) BJ_REG_FUSE(32, 1);
                    else if (nv <= 40) BJ_REG_FUSE(40, 1);
                    else BJ_REG_FUSE(52, 1);
#undef BJ_REG_FUSE
                    if (e != cudaSuccess) { set_cuda_error(e, "reorth_axpy_dot_reg_kernel"); return BJ_ERR_CUDA; }
                    h->launches++;
                    BJ_LAUNCH(finalize_multi_kernel, nv, 256, grid, nv, (const double*)PM, stride, z.coef,
                              (const int*)z.done);
                    continue;
                }
                if (pass == 0 && fuse_mid) {
                    const int64_t ntiles = (n + R - 1) / R;
                    const int grid = (int)std::min<int64_t>(ntiles, (int64_t)h->num_sms * kFuseCtasPerSm);
                    const size_t smem = 64 + (208 + 512) * sizeof(double) + fuse_stages * (size_t)(nv + 1) * R * sizeof(double);
                    e = launch_kernel(reorth_axpy_dot_kernel, dim3(grid), dim3(kFuseThreads), smem, st, pdl, n, nv,
                                      (const double*)z.V, z.w, (const double*)z.coef, PM, stride, (const int*)z.done, R, ntiles, fuse_stages);
                    if (e != cudaSuccess) { set_cuda_error(e, "reorth_axpy_dot_kernel"); return BJ_ERR_CUDA; }
                    h->launches++;
                    BJ_LAUNCH(finalize_multi_kernel, nv, 256, grid, nv, (const double*)PM, stride, z.coef,
                              (const int*)z.done);
                    continue;
                }
                e = launch_kernel(multiaxpy_kernel, dim3(G), dim3(kReduceThreads), axpy_smem, st, pdl, n, nv,
                                  (const double*)z.V, z.w, (const double*)z.coef, PB, pass == 1 ? 1 : 0, (const int*)z.done,
                                  axpy_piece);
                if (e != cudaSuccess) { set_cuda_error(e, "multiaxpy_kernel"); return BJ_ERR_CUDA; }
                h->launches++;
            }
        }
        // beta_{j+2} = ||w||, bookkeeping, and v_{j+2} = w / beta (not needed after the last step)
        BJ_LAUNCH(scale_kernel, G, kReduceThreads, n, (const double*)z.w, j + 1 < m ? vcol(j + 1) : (double*)nullptr,
                  (const double*)PB, G, 1, j, tol, (const double*)z.alpha, z.beta, amax_buf, z.done);
    }
#undef BJ_LAUNCH

    return lanczos_readback(h, m, res);
}

// extreme Ritz values, their residual bounds and the optional coefficient copies from alpha[0..me-1], beta[0..me-1]
void lanczos_fill_result(int me, const double* a, const double* b, bj_lanczos_result_t* res)
{
    res->iters_done = me;
    res->lmin = tridiag_eig_k(me, a, b, 0);
    res->lmax = tridiag_eig_k(me, a, b, me - 1);
    res->res_min = fabs(b[me - 1]) * last_comp(me, a, b, res->lmin);
    res->res_max = fabs(b[me - 1]) * last_comp(me, a, b, res->lmax);
    if (res->alpha_host) std::copy(a, a + me, res->alpha_host);
    if (res->beta_host) std::copy(b, b + me, res->beta_host);
}

}  // namespace bj
