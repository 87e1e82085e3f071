// Setup for b <= 8 and short rows, without a permutation or band detection: ONE kernel instead of three passes over the CSR.
// tile_validate_extract_kernel<B> (a1 + a2 + a3): a CTA takes a tile of consecutive rows (a multiple of b, at most 256) --
// whose entries are one contiguous range of col_idx / val -- and keeps the tile's row pointers and its diagonal blocks
// (packed lower triangles, zero-filled) in shared memory.
//   * ENTRY-parallel walk: a thread takes eight consecutive entries (two 16-byte loads of columns; a warp covers 1 KB), finds
//     the row of the first by binary search in the shared row pointers and walks them from there; per entry the checks of a1
//     (column range, strictly ascending inside the row) and, if it lies in the lower triangle of the row's diagonal block, one
//     store into the shared tile.  The row-pointer checks, the longest row and the column-coherence statistic of the SpMV plan
//     ride on the threads that load the row pointers.
//   * then thread t factors block t of the tile in place in shared memory (the arithmetic of extract_factor_small_kernel)
//     and writes it in the interleaved layout of solve_small_kernel.
// The CSR is read once, nothing intermediate goes through global memory, and one host synchronisation goes away.  The
// thread-per-BLOCK extraction it replaces walked b rows per thread with ~100 registers (16 warps per SM, 31 sectors per warp
// load): 90 us on config 2 at 14 % issue utilisation.  An invalid CSR is flagged in the status word and reported as
// BJ_ERR_NOT_CANONICAL by bj_setup; reads stay in bounds (a tile with a bad row pointer is skipped).
#include <algorithm>

#include "bj_device.cuh"
#include "bj_internal.cuh"

namespace bj {

namespace {

constexpr int kTileThreads = 256;
constexpr int kTileUnroll = 8;   // entries per thread requested together

// (four CTAs per SM: the entry walk needs the warps, the factorisation -- one warp per tile -- pays a few spilled bytes;
// measured on config 2 b = 8: 2 / 3 / 4 / 5 / 6 CTAs per SM 0.189 / 0.163 / 0.120 / 0.129 / 0.134 ms)
template <int B>
__global__ void __launch_bounds__(kTileThreads, 4)
tile_validate_extract_kernel(int64_t n, int64_t nnz, int64_t ntiles, int64_t nblocks, const int32_t* __restrict__ rp,
                             const int32_t* __restrict__ ci, const double* __restrict__ val, double* __restrict__ fac, Status* st)
{
    constexpr int P = B * (B + 1) / 2;
    constexpr int PS = P | 1;                   // odd stride of a block in the shared tile: thread-per-block accesses hit different banks
    constexpr int TR = (kTileThreads / B) * B;  // rows per tile: whole blocks only, so that a block belongs to ONE CTA
    constexpr int NB = TR / B;                  // blocks per tile
    __shared__ int rps[TR + 1];
    __shared__ double raws[NB * PS];            // the tile's diagonal blocks, packed lower triangles by rows
    __shared__ unsigned sh[2][kTileThreads / 32];
    __shared__ int tile_bad;
    int flags = 0, len = 0;
    unsigned coh = 0, cmp = 0;
    const int tid = threadIdx.x, lane = tid & 31;
    const bool vec_ok = (reinterpret_cast<uintptr_t>(ci) & 15) == 0;  // 16-byte loads of the columns
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t r0 = tile * TR;
        const int rows = (int)(r0 + TR <= n ? TR : n - r0);
        __syncthreads();  // the previous tile's readers of rps / tile_bad are done
        if (tid == 0) tile_bad = 0;
        __syncthreads();
        // ---- row pointers of the tile; a1 for them ----
        if (tid < rows) {
            const int64_t i = r0 + tid;
            const int64_t s = rp[i];
            rps[tid] = (int)s;
            {
                const int64_t e = rp[i + 1];
                if (tid == rows - 1) rps[rows] = (int)e;
                if (s > e || s < 0 || e > nnz || (i == 0 && s != 0) || (i == n - 1 && e != nnz)) {
                    flags |= ST_BAD_ROWPTR;
                    tile_bad = 1;
                } else {
                    const int l = (int)(e - s);
                    len = l > len ? l : len;
                    if ((tile & 7) == 0 && i + 1 < n) {  // every eighth tile also gathers the column-coherence statistic
                        const int64_t e2 = rp[i + 2];
                        if (e2 >= e && e2 <= nnz) {
                            int64_t m = (e2 - e) < (e - s) ? (e2 - e) : (e - s);
                            if (m > 8) m = 8;  // a sample: the first entries of the two rows
                            for (int64_t q = 0; q < m; ++q) {
                                const int d = ci[e + q] - ci[s + q];
                                ++cmp;
                                coh += (d >= -16 && d <= 16);
                            }
                        }
                    }
                }
            }
        }
        // ---- zero the tile's blocks (TR is a multiple of B: they are this CTA's alone) ----
        const int64_t kb0 = r0 / B, kb1 = (r0 + rows + B - 1) / B;
        for (int e = tid; e < NB * PS; e += kTileThreads) raws[e] = 0.0;
        __syncthreads();
        if (tile_bad) continue;  // uniform: nothing of this tile is read through its row pointers
        // ---- the entries of the tile: one contiguous range; a thread takes EIGHT CONSECUTIVE entries (two 16-byte loads of
        // columns; a warp covers 1 KB), finds the row of the first by binary search and walks the row pointers from there ----
        const int e0 = rps[0], e1 = rps[rows];
        for (int base = e0 & ~7; base < e1; base += kTileThreads * kTileUnroll) {
            const int p0 = base + tid * kTileUnroll;
            int c[kTileUnroll];
            if (vec_ok && p0 >= e0 && p0 + kTileUnroll <= e1) {
                const int4 a4 = *reinterpret_cast<const int4*>(ci + p0);
                const int4 b4 = *reinterpret_cast<const int4*>(ci + p0 + 4);
                c[0] = a4.x; c[1] = a4.y; c[2] = a4.z; c[3] = a4.w;
                c[4] = b4.x; c[5] = b4.y; c[6] = b4.z; c[7] = b4.w;
            } else {
#pragma unroll
                for (int u = 0; u < kTileUnroll; ++u) c[u] = (p0 + u >= e0 && p0 + u < e1) ? ci[p0 + u] : -1;
            }
            int cprev = __shfl_up_sync(0xffffffffu, c[kTileUnroll - 1], 1);  // entry p0 - 1 is the last one of the lane below
            if (lane == 0 && p0 > e0 && p0 < e1) cprev = ci[p0 - 1];
            // the row of the first entry: the last r with rps[r] <= p (rows <= 256: eight steps)
            int r = 0;
            {
                const int pf = p0 < e0 ? e0 : p0;
                int lo = 0, hi = rows;
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (rps[mid] <= pf) lo = mid; else hi = mid;
                }
                r = lo;
            }
            int next = rps[r + 1], start = rps[r];
            // everything below is 32-bit and tile-local: block kl = r / B of the tile, row rr of it, first column of the block lob
            int kl = r / B, rr = r - kl * B;
            const int r0i = (int)r0;
            int lob = r0i + kl * B;
            int dst[kTileUnroll];  // offset of the entry in the tile's raw blocks, or -1
#pragma unroll
            for (int u = 0; u < kTileUnroll; ++u) {
                const int p = p0 + u;
                dst[u] = -1;
                if (p >= e0 && p < e1) {
                    while (p >= next) {  // next row (empty rows are stepped over)
                        ++r;
                        start = next;
                        next = rps[r + 1];
                        if (++rr == B) { rr = 0; ++kl; lob += B; }
                    }
                    const int cc = c[u];
                    if ((unsigned)cc >= (unsigned)n) flags |= ST_BAD_COL;
                    if (p != start && cc <= cprev) flags |= ST_UNSORTED;  // columns ascend strictly inside a row
                    const unsigned d = (unsigned)(cc - lob);                 // in the block's lower triangle: 0 <= d <= rr
                    if (cc >= lob && d <= (unsigned)rr) dst[u] = kl * PS + rr * (rr + 1) / 2 + (int)d;
                }
                cprev = c[u];
            }
            double v[kTileUnroll];  // the values of the entries inside the blocks, requested together
#pragma unroll
            for (int u = 0; u < kTileUnroll; ++u) v[u] = dst[u] >= 0 ? val[p0 + u] : 0.0;
#pragma unroll
            for (int u = 0; u < kTileUnroll; ++u)
                if (dst[u] >= 0) raws[dst[u]] = v[u];
        }
        __syncthreads();
        // ---- a3: thread t factors block kb0 + t in place in the shared tile (the arithmetic of extract_factor_small_kernel)
        // and writes it in the interleaved layout of solve_small_kernel ----
        if (tid < (int)(kb1 - kb0)) {
            const int64_t k = kb0 + tid;
            double* D = raws + tid * PS;  // packed lower triangle, e = i (i + 1) / 2 + j
            const int64_t lo = k * B;
#pragma unroll
            for (int i = 0; i < B; ++i) {
                if (lo + i >= n) {  // identity rows pad a ragged last block
#pragma unroll
                    for (int j = 0; j <= i; ++j) D[i * (i + 1) / 2 + j] = (j == i) ? 1.0 : 0.0;
                }
            }
            bool bad = false;
            double rinv[B];
#pragma unroll
            for (int j = 0; j < B; ++j) {
                double sjj = D[j * (j + 1) / 2 + j];
#pragma unroll
                for (int q = 0; q < j; ++q) sjj -= D[j * (j + 1) / 2 + q] * D[j * (j + 1) / 2 + q];
                if (!(sjj > 0.0) || isinf(sjj)) { bad = true; sjj = 1.0; }
                const double ljj = sqrt(sjj);
                const double rjj = __drcp_rn(ljj);  // also the stored diagonal slot 1 / l_jj
                rinv[j] = rjj;
                D[j * (j + 1) / 2 + j] = ljj;
#pragma unroll
                for (int i = j + 1; i < B; ++i) {
                    double t = D[i * (i + 1) / 2 + j];
#pragma unroll
                    for (int q = 0; q < j; ++q) t -= D[i * (i + 1) / 2 + q] * D[j * (j + 1) / 2 + q];
                    D[i * (i + 1) / 2 + j] = div_by(t, ljj, rjj);
                }
            }
            if (bad) {
                atomicOr(&st->flags, ST_NOT_SPD);
                atomicMin(&st->bad_block, (long long)k);
            }
            double* f = fac + (k >> 5) * (int64_t)(P * kInterleave) + (k & 31);
#pragma unroll
            for (int i = 0; i < B; ++i)
#pragma unroll
                for (int j = 0; j <= i; ++j) f[(i * (i + 1) / 2 + j) * kInterleave] = (i == j) ? rinv[i] : D[i * (i + 1) / 2 + j];
        }
    }
    flags = __reduce_or_sync(0xffffffffu, flags);
    len = __reduce_max_sync(0xffffffffu, len);
    coh = __reduce_add_sync(0xffffffffu, coh);
    cmp = __reduce_add_sync(0xffffffffu, cmp);
    const int warp = tid >> 5;
    if (lane == 0) {
        if (flags) atomicOr(&st->flags, flags);
        if (len > *(volatile int*)&st->max_row_nnz) atomicMax(&st->max_row_nnz, len);
        sh[0][warp] = coh; sh[1][warp] = cmp;
    }
    __syncthreads();
    if (tid == 0) {
        unsigned a = 0, c2 = 0;
        for (int w = 0; w < kTileThreads / 32; ++w) { a += sh[0][w]; c2 += sh[1][w]; }
        if (c2) { atomicAdd(&st->coherent, (unsigned long long)a); atomicAdd(&st->compared, (unsigned long long)c2); }
    }
}

// The same kernel with the factorisation taken off the critical path: warps 0..6 (224 threads) are the EXTRACT group and
// walk tile after tile, warp 7 is the FACTOR group and factors the blocks of the previous tile meanwhile (in the one-group
// form a third of the warp time was seven warps waiting at the barrier while one factored).  Two shared tiles alternate;
// the groups hand them over through two pairs of mbarriers (full: 7 arrivals, one per extract warp; empty: 1 arrival).
constexpr int kExtractThreads = kTileThreads - 32;
constexpr int kStageCap = 4096;  // entries of a tile staged in shared memory
__device__ __forceinline__ void bar_extract() { asm volatile("bar.sync 1, %0;" ::"n"(kExtractThreads) : "memory"); }

template <int B>
__global__ void __launch_bounds__(kTileThreads, 4)
tile_setup_ws_kernel(int64_t n, int64_t nnz, int64_t ntiles, int64_t nblocks, const int32_t* __restrict__ rp,
                     const int32_t* __restrict__ ci, const double* __restrict__ val, double* __restrict__ fac, Status* st)
{
    constexpr int P = B * (B + 1) / 2;
    constexpr int PS = P | 1;
    constexpr int TR = (kTileThreads / B) * B;
    constexpr int NB = TR / B;
    __shared__ __align__(8) uint64_t full[2], empty[2];
    __shared__ int rps[TR + 1];
    __shared__ double raws[2][NB * PS];
    __shared__ unsigned sh[2][kTileThreads / 32];
    __shared__ int tile_bad, bad_buf[2];
    __shared__ int cis[kStageCap];              // the columns of the tile
    int flags = 0, len = 0;
    unsigned coh = 0, cmp = 0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool vec_ok = (reinterpret_cast<uintptr_t>(ci) & 15) == 0;
    if (tid == 0) {
        mbar_init(&full[0], kExtractThreads / 32);
        mbar_init(&full[1], kExtractThreads / 32);
        mbar_init(&empty[0], 1);
        mbar_init(&empty[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (warp == kExtractThreads / 32) {
        // ================= FACTOR group: one warp, thread per block, in place in the shared tile =================
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
            const int buf = it & 1;
            mbar_wait(&full[buf], (uint32_t)((it >> 1) & 1));
            const int64_t r0 = tile * TR;
            const int rows = (int)(r0 + TR <= n ? TR : n - r0);
            const int64_t kb0 = r0 / B, kb1 = (r0 + rows + B - 1) / B;
            if (!bad_buf[buf]) {
                for (int t = lane; t < (int)(kb1 - kb0); t += 32) {
                    const int64_t k = kb0 + t;
                    double* D = raws[buf] + t * PS;  // packed lower triangle, e = i (i + 1) / 2 + j
                    const int64_t lo = k * B;
#pragma unroll
                    for (int i = 0; i < B; ++i) {
                        if (lo + i >= n) {  // identity rows pad a ragged last block
#pragma unroll
                            for (int j = 0; j <= i; ++j) D[i * (i + 1) / 2 + j] = (j == i) ? 1.0 : 0.0;
                        }
                    }
                    bool bad = false;
                    double rinv[B];
#pragma unroll
                    for (int j = 0; j < B; ++j) {
                        double sjj = D[j * (j + 1) / 2 + j];
#pragma unroll
                        for (int q = 0; q < j; ++q) sjj -= D[j * (j + 1) / 2 + q] * D[j * (j + 1) / 2 + q];
                        if (!(sjj > 0.0) || isinf(sjj)) { bad = true; sjj = 1.0; }
                        const double ljj = sqrt(sjj);
                        const double rjj = __drcp_rn(ljj);
                        rinv[j] = rjj;
                        D[j * (j + 1) / 2 + j] = ljj;
#pragma unroll
                        for (int i = j + 1; i < B; ++i) {
                            double tt = D[i * (i + 1) / 2 + j];
#pragma unroll
                            for (int q = 0; q < j; ++q) tt -= D[i * (i + 1) / 2 + q] * D[j * (j + 1) / 2 + q];
                            D[i * (i + 1) / 2 + j] = div_by(tt, ljj, rjj);
                        }
                    }
                    if (bad) {
                        atomicOr(&st->flags, ST_NOT_SPD);
                        atomicMin(&st->bad_block, (long long)k);
                    }
                    double* f = fac + (k >> 5) * (int64_t)(P * kInterleave) + (k & 31);
#pragma unroll
                    for (int i = 0; i < B; ++i)
#pragma unroll
                        for (int j = 0; j <= i; ++j) f[(i * (i + 1) / 2 + j) * kInterleave] = (i == j) ? rinv[i] : D[i * (i + 1) / 2 + j];
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[buf]);
        }
    } else {
        // ================= EXTRACT group: 224 threads =================
        // The row pointers and the columns of the NEXT tile are requested while this tile is worked on and wait in
        // registers: a tile is then one global latency (the values) instead of a chain of three.
        constexpr int kPfRp = (TR + kExtractThreads) / kExtractThreads;  // row pointers per thread (TR + 1 in all)
        constexpr int kPfCi = 9;                                          // columns per thread: tiles of up to 2016 entries
        int pf_rp[kPfRp], pf_ci[kPfCi], pf_e0 = 0, pf_ne = -1;            // pf_ne < 0: the columns were not prefetched
        auto prefetch = [&](int64_t tnext) {
            pf_ne = -1;
            if (tnext >= ntiles) return;
            const int64_t r0n = tnext * TR;
            const int rowsn = (int)(r0n + TR <= n ? TR : n - r0n);
#pragma unroll
            for (int u = 0; u < kPfRp; ++u) {
                const int rl = tid + u * kExtractThreads;
                pf_rp[u] = rl <= rowsn ? rp[r0n + rl] : 0;
            }
            const int64_t e0n = rp[r0n], e1n = rp[r0n + rowsn];
            if (e0n >= 0 && e0n <= e1n && e1n <= nnz && e1n - e0n <= (int64_t)kExtractThreads * kPfCi) {
                pf_e0 = (int)e0n;
                pf_ne = (int)(e1n - e0n);
#pragma unroll
                for (int u = 0; u < kPfCi; ++u) {
                    const int q = tid + u * kExtractThreads;
                    pf_ci[u] = q < pf_ne ? ci[e0n + q] : 0;
                }
            }
        };
        prefetch(blockIdx.x);
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
            const int buf = it & 1;
            const int64_t r0 = tile * TR;
            const int rows = (int)(r0 + TR <= n ? TR : n - r0);
            bar_extract();  // the previous tile's readers of rps / cis / tile_bad are done
            if (tid == 0) tile_bad = 0;
#pragma unroll
            for (int u = 0; u < kPfRp; ++u) {
                const int rl = tid + u * kExtractThreads;
                if (rl <= rows) rps[rl] = pf_rp[u];
            }
            const int st_e0 = pf_e0, st_ne = pf_ne;  // what the staged columns cover (uniform over the group)
            if (st_ne >= 0) {
#pragma unroll
                for (int u = 0; u < kPfCi; ++u) {
                    const int q = tid + u * kExtractThreads;
                    if (q < st_ne) cis[q] = pf_ci[u];
                }
            }
            bar_extract();
            prefetch(tile + gridDim.x);  // in flight during this tile's work
            // ---- a1 for the row pointers; longest row; coherence sample ----
            for (int rl = tid; rl < rows; rl += kExtractThreads) {
                const int64_t i = r0 + rl;
                const int64_t sR = rps[rl], eR = rps[rl + 1];
                if (sR > eR || sR < 0 || eR > nnz || (i == 0 && sR != 0) || (i == n - 1 && eR != nnz)) {
                    flags |= ST_BAD_ROWPTR;
                    tile_bad = 1;
                } else {
                    const int l = (int)(eR - sR);
                    len = l > len ? l : len;
                    if ((tile & 7) == 0 && i + 1 < n) {  // every eighth tile also gathers the column-coherence statistic
                        const int64_t e2 = rp[i + 2];
                        if (e2 >= eR && e2 <= nnz) {
                            int64_t m = (e2 - eR) < (eR - sR) ? (e2 - eR) : (eR - sR);
                            if (m > 8) m = 8;
                            for (int64_t q = 0; q < m; ++q) {
                                const int d = ci[eR + q] - ci[sR + q];
                                ++cmp;
                                coh += (d >= -16 && d <= 16);
                            }
                        }
                    }
                }
            }
            // the tile two iterations ago has left this buffer
            if (it >= 2) mbar_wait(&empty[buf], (uint32_t)(((it >> 1) + 1) & 1));
            double* R = raws[buf];
            for (int e = tid; e < NB * PS; e += kExtractThreads) R[e] = 0.0;
            bar_extract();
            const bool skip = tile_bad != 0;
            if (tid == 0) bad_buf[buf] = skip ? 1 : 0;
            if (!skip) {
                // A thread takes a ROW: it scans the row's columns out of shared memory (checks of a1: range, strictly
                // ascending) and fetches the value of an entry only if it lies in the lower triangle of the row's diagonal
                // block.  (An entry-parallel walk with a binary search per eight entries cost ~80 instructions per entry.)
                const int e0 = rps[0], e1 = rps[rows];
                bool staged = st_ne >= 0 && st_e0 == e0 && st_ne == e1 - e0;  // (always, for a valid tile that was prefetched)
                if (!staged && e1 - e0 <= kStageCap) {  // a longer tile: staged now
                    for (int q = tid; q < e1 - e0; q += kExtractThreads) cis[q] = ci[e0 + q];
                    bar_extract();
                    staged = true;
                }
                for (int rl = tid; rl < rows; rl += kExtractThreads) {
                    const int sr = rps[rl], er = rps[rl + 1];
                    const int kl = rl / B, rr = rl - kl * B;
                    const int lob = (int)r0 + kl * B;
                    double* Rr = R + kl * PS + rr * (rr + 1) / 2;
                    int prev = -1;
                    for (int p = sr; p < er; ++p) {
                        const int cc = staged ? cis[p - e0] : ci[p];
                        if ((unsigned)cc >= (unsigned)n) flags |= ST_BAD_COL;
                        if (cc <= prev) flags |= ST_UNSORTED;
                        prev = cc;
                        const unsigned d = (unsigned)(cc - lob);
                        if (cc >= lob && d <= (unsigned)rr) Rr[d] = val[p];
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&full[buf]);  // this warp's part of the tile is in the buffer
        }
    }
    flags = __reduce_or_sync(0xffffffffu, flags);
    len = __reduce_max_sync(0xffffffffu, len);
    coh = __reduce_add_sync(0xffffffffu, coh);
    cmp = __reduce_add_sync(0xffffffffu, cmp);
    if (lane == 0) {
        if (flags) atomicOr(&st->flags, flags);
        if (len > *(volatile int*)&st->max_row_nnz) atomicMax(&st->max_row_nnz, len);
        sh[0][warp] = coh; sh[1][warp] = cmp;
    }
    __syncthreads();
    if (tid == 0) {
        unsigned a = 0, c2 = 0;
        for (int w = 0; w < kTileThreads / 32; ++w) { a += sh[0][w]; c2 += sh[1][w]; }
        if (c2) { atomicAdd(&st->coherent, (unsigned long long)a); atomicAdd(&st->compared, (unsigned long long)c2); }
    }
}

}  // namespace

// a1-a3 for solve_kind 1 without permutation and without band detection (see the header); the caller reads the status back.
// b >= 7: the warp-specialised form (measured on config 2: b = 8 0.122 -> 0.113 ms, b = 7 0.121 -> 0.118); smaller blocks
// factor too quickly to be worth a warp of their own (b = 4: 0.097 one group, 0.104 specialised).
template <int B>
static void launch_tile(bj_handle_s* h)
{
    constexpr int64_t tr = (kTileThreads / B) * B;
    const int64_t ntiles = (h->n + tr - 1) / tr;
    const unsigned grid = (unsigned)std::min<int64_t>(ntiles, (int64_t)h->num_sms * 8);
    SetupSpan span(h);
    if constexpr (B >= 7)
        tile_setup_ws_kernel<B><<<grid, kTileThreads, 0, h->stream>>>(h->n, h->nnz, ntiles, h->nblocks, h->row_ptr, h->col_idx, h->val,
                                                                     h->fac_small, h->status);
    else
        tile_validate_extract_kernel<B><<<grid, kTileThreads, 0, h->stream>>>(h->n, h->nnz, ntiles, h->nblocks, h->row_ptr, h->col_idx,
                                                                             h->val, h->fac_small, h->status);
}

int launch_setup_rows(bj_handle_s* h)
{
    switch (h->b) {
        case 1: launch_tile<1>(h); break;
        case 2: launch_tile<2>(h); break;
        case 3: launch_tile<3>(h); break;
        case 4: launch_tile<4>(h); break;
        case 5: launch_tile<5>(h); break;
        case 6: launch_tile<6>(h); break;
        case 7: launch_tile<7>(h); break;
        case 8: launch_tile<8>(h); break;
        default: return BJ_ERR_INVALID_ARG;
    }
    h->launches += 1;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

}  // namespace bj
