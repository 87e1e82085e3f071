// Batched block triangular solves (a5 and the two outer factors of a7):
//   forward  y = L^-1 r,   backward  x = L^-T y,   both  z = L^-T L^-1 r  (= M^-1 r).
// Diagonals are stored as reciprocals by the setup kernel.
//
// Two layouts, both HBM-bound by design (0.25 flop per byte):
//   b <= 8 : one THREAD per block.  The packed factor of 32 consecutive blocks is interleaved so that
//            element e of blocks 32g..32g+31 is one 256-byte line: every load of the warp is fully
//            coalesced and all P = b(b+1)/2 loads of a thread are independent (deep MLP).
//   b  > 8 : one SUB-WARP (16 or 32 lanes) per block, lane i owns row i.  Forward substitution is
//            column oriented: at step j lane j's y_j is final, is broadcast by shuffle, lanes i > j
//            subtract L_ij y_j.  The packed factors are streamed into shared memory by bulk async
//            copies (TMA) in a persistent producer/consumer ring, so HBM streaming never waits for
//            a block's dependent chain.
#include <algorithm>
#include <atomic>

#include "bj_device.cuh"
#include "bj_internal.cuh"
#include "bj_lanczos_fuse.cuh"
#include "bj_pcg_fuse.cuh"

namespace bj {

// ------------------------------------------------------------------------------------------------
// thread per block, compile-time B.  DIR: 0 forward, 1 backward, 2 both.
// ------------------------------------------------------------------------------------------------
template <int B, bool VEC>
__device__ __forceinline__ void load_rows(const double* src, int64_t lo, int64_t n, bool whole, double (&v)[B])
{
    if (whole) {
        if constexpr (VEC && B % 4 == 0) {
#pragma unroll
            for (int i = 0; i < B; i += 4) ld_v4(src + lo + i, v + i);
        } else if constexpr (VEC && B % 2 == 0) {
#pragma unroll
            for (int i = 0; i < B; i += 2) ld_v2(src + lo + i, v + i);
        } else {
#pragma unroll
            for (int i = 0; i < B; ++i) v[i] = src[lo + i];
        }
    } else {
#pragma unroll
        for (int i = 0; i < B; ++i) v[i] = (lo + i < n) ? src[lo + i] : 0.0;
    }
}

template <int B, bool VEC>
__device__ __forceinline__ void store_rows(double* dst, int64_t lo, int64_t n, bool whole, const double (&v)[B])
{
    if (whole) {
        if constexpr (VEC && B % 4 == 0) {
#pragma unroll
            for (int i = 0; i < B; i += 4) st_v4(dst + lo + i, v + i);
        } else if constexpr (VEC && B % 2 == 0) {
#pragma unroll
            for (int i = 0; i < B; i += 2) st_v2(dst + lo + i, v + i);
        } else {
#pragma unroll
            for (int i = 0; i < B; ++i) dst[lo + i] = v[i];
        }
    } else {
#pragma unroll
        for (int i = 0; i < B; ++i)
            if (lo + i < n) dst[lo + i] = v[i];
    }
}

// Permuted handles (bj_setup_perm, reading 23): the block's rows lo .. lo + B - 1 of the PERMUTED ordering live at
// perm[lo + i] in the caller's vectors; the index loads are coalesced, the vector accesses are gathers / scatters.
template <int B>
__device__ __forceinline__ void load_rows_perm(const double* src, const int32_t* __restrict__ perm, int64_t lo, int64_t n, double (&v)[B])
{
    int idx[B];
#pragma unroll
    for (int i = 0; i < B; ++i) idx[i] = (lo + i < n) ? perm[lo + i] : -1;
#pragma unroll
    for (int i = 0; i < B; ++i) v[i] = idx[i] >= 0 ? src[idx[i]] : 0.0;
}

template <int B>
__device__ __forceinline__ void store_rows_perm(double* dst, const int32_t* __restrict__ perm, int64_t lo, int64_t n, const double (&v)[B])
{
#pragma unroll
    for (int i = 0; i < B; ++i)
        if (lo + i < n) dst[perm[lo + i]] = v[i];
}

// LZ: 0 plain, 1 Lanczos prologue (DIR 1: the input is w built on the fly), 2 Lanczos epilogue (DIR 0),
//     3 PCG update + apply (DIR 2: x += a p, r -= a q on the fly, z = M^-1 r, partials of r.r and r.z)
//     TRI: tridiagonal blocks, compact bidiagonal factor of 2B - 1 elements, element (i, j) at slot i + j
#ifndef BJ_SMALL_HOOK_MINB
#define BJ_SMALL_HOOK_MINB 4
#endif
#define SMALL_MINB ((LZ == 3 && B >= 7 && !TRI) ? BJ_SMALL_HOOK_MINB : 1)
template <int B, int DIR, bool VEC, int LZ, bool TRI>
__global__ void __launch_bounds__(128, SMALL_MINB)
solve_small_kernel(int64_t n, int64_t nblocks, const double* __restrict__ fac,
                   const double* in, double* out,  // in == out allowed: a thread touches only its own block
                   const LzPrologue pro, const LzEpilogue epi, const PcgHook pcg,
                   const int serp,                 // 1: serpentine walk (launch_small): CTA q takes the q-th LAST slice of blocks
                   const unsigned serp_keep_from,  //    and CTAs q >= serp_keep_from load their factors as ordinary L2 lines instead of evict_first
                   const int32_t* __restrict__ perm)  // plain solves only (LZ == 0): vectors are accessed through perm, or null
{
    constexpr int P = TRI ? 2 * B - 1 : B * (B + 1) / 2;
    __shared__ double lz_sh[8];
    pdl_trigger();
    const unsigned bid = serp ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
    const int64_t k = (int64_t)bid * blockDim.x + threadIdx.x;
    const bool act = k < nblocks;
    if (LZ == 0 && !act) return;
    const int64_t kc = act ? k : 0;
    const double* f = fac + (kc >> 5) * (int64_t)(P * kInterleave) + (kc & 31);
    double l[P];
    if (serp) {
        const uint64_t pol = blockIdx.x >= serp_keep_from ? policy_evict_normal() : policy_evict_first();
#pragma unroll
        for (int e = 0; e < P; ++e) l[e] = ld_stream_hint(f + e * kInterleave, pol);
    } else {
#pragma unroll
        for (int e = 0; e < P; ++e) l[e] = ld_stream(f + e * kInterleave);   // factors never change after setup
    }
    pdl_wait();                                                          // `in` may come from the previous kernel
    const int64_t lo = kc * B;
    double v[B];
    const bool whole = lo + B <= n;
    double acc = 0.0, beta = 0.0, inv_beta = 0.0;  // Lanczos / PCG: running dot product of this thread
    double rin[LZ == 3 ? B : 1];                   // PCG: the residual rows, kept for r.z
    double acc2 = 0.0;
    if (LZ == 1) {
        double alpha, c[B];
        if (act) {  // operands first, the scalar (a dependent load) after them
            if (pro.first) {
                load_rows<B, VEC>(pro.w0, lo, n, whole, v);
            } else {
                load_rows<B, VEC>(pro.w, lo, n, whole, v);
                load_rows<B, VEC>(pro.vcur, lo, n, whole, c);
            }
        }
        if (lz_prologue_begin(pro, alpha)) return;  // uniform over the grid
        if (act) {
            if (!pro.first) {
#pragma unroll
                for (int i = 0; i < B; ++i) v[i] -= alpha * c[i];
            }
#pragma unroll
            for (int i = 0; i < B; ++i) acc = fma(v[i], v[i], acc);  // rows past n were loaded as zeros
            store_rows<B, VEC>(pro.w, lo, n, whole, v);
        }
    } else if (LZ == 3) {
        // every vector operand is requested BEFORE the scalars are read: the step length / the three coefficients hang on
        // a dependent load plus a division and a square root, and the loads do not depend on them
        double c[B], xs[B], pv[B];
        if (act) {
            load_rows<B, VEC>(pcg.r, lo, n, whole, v);
            load_rows<B, VEC>(pcg.q, lo, n, whole, c);
            load_rows<B, VEC>(pcg.x, lo, n, whole, xs);
            if (!pcg.mode) load_rows<B, VEC>(pcg.p, lo, n, whole, pv);
        }
        double a;
        if (pcg_hook_begin(pcg, a)) return;  // uniform over the grid
        if (pcg.mode) {  // three-term step of Lanczos on M^-1 A: r_{k+1} replaces r_{k-1} (uniform branch)
            double cq, cr, cx;
            mlz_hook_coeffs(pcg, cq, cr, cx);
            if (act) {
#pragma unroll
                for (int i = 0; i < B; ++i) {
                    v[i] = mlz_combine(cq, cr, cx, c[i], v[i], xs[i]);
                    rin[i] = v[i];
                }
                store_rows<B, VEC>(pcg.x, lo, n, whole, v);
            }
        } else if (act) {
#pragma unroll
            for (int i = 0; i < B; ++i) {
                v[i] = v[i] - a * c[i];             // r_new
                acc = fma(v[i], v[i], acc);
                rin[i] = v[i];
                xs[i] = fma(a, pv[i], xs[i]);
            }
            store_rows<B, VEC>(pcg.r, lo, n, whole, v);
            store_rows<B, VEC>(pcg.x, lo, n, whole, xs);
        }
    } else {
        if (LZ == 0 && perm) load_rows_perm<B>(in, perm, lo, n, v);
        else load_rows<B, VEC>(in, lo, n, whole, v);                    // before the scalars: independent of them
        if (LZ == 2 && lz_epilogue_begin(epi, beta, inv_beta)) return;  // uniform over the grid
    }
    if (DIR == 0 || DIR == 2) {
#pragma unroll
        for (int i = 0; i < B; ++i) {
            double s = v[i];
            if (TRI) {
                if (i > 0) s -= l[2 * i - 1] * v[i - 1];
                v[i] = s * l[2 * i];
            } else {
#pragma unroll
                for (int j = 0; j < i; ++j) s -= l[i * (i + 1) / 2 + j] * v[j];
                v[i] = s * l[i * (i + 1) / 2 + i];
            }
        }
    }
    if (DIR == 1 || DIR == 2) {
#pragma unroll
        for (int i = B - 1; i >= 0; --i) {
            double s = v[i];
            if (TRI) {
                if (i + 1 < B) s -= l[2 * i + 1] * v[i + 1];
                v[i] = s * l[2 * i];
            } else {
#pragma unroll
                for (int j = i + 1; j < B; ++j) s -= l[j * (j + 1) / 2 + i] * v[j];
                v[i] = s * l[i * (i + 1) / 2 + i];
            }
        }
    }
    if (LZ == 2) {
        if (act) {
            double c[B], d[B];  // w and v_j
            load_rows<B, VEC>(epi.w, lo, n, whole, c);
            if (epi.vprev) load_rows<B, VEC>(epi.vprev, lo, n, whole, d);
#pragma unroll
            for (int i = 0; i < B; ++i) {
                c[i] *= inv_beta;                       // v_{j+1}
                v[i] *= inv_beta;
                if (epi.vprev) v[i] -= beta * d[i];     // w'_new
                acc = fma(c[i], v[i], acc);             // rows past n: c = 0
            }
            store_rows<B, VEC>(epi.vnew, lo, n, whole, c);
            store_rows<B, VEC>(epi.w, lo, n, whole, v);
        }
        lz_reduce_finish(epi.red, acc, lz_sh);
    } else {
        if (act) {
            if (LZ == 0 && perm) store_rows_perm<B>(out, perm, lo, n, v);
            else store_rows<B, VEC>(out, lo, n, whole, v);
        }
        if (LZ == 1) lz_reduce_finish(pro.red, acc, lz_sh);
        if (LZ == 3) {
            if (act) {
#pragma unroll
                for (int i = 0; i < B; ++i) acc2 = fma(rin[i], v[i], acc2);
            }
            lz_reduce_finish2(pcg.red_rr, acc, pcg.red_rz, acc2, lz_sh);  // one ticket for both sums
        }
    }
}

// ------------------------------------------------------------------------------------------------
// 8 < b <= 32, b not in {16, 24, 32}: persistent CTAs, factors streamed through a shared-memory ring by the TMA engine.
// A tile is G consecutive blocks; their packed factors are one contiguous byte range, moved by ONE
// bulk async copy per stage (two when DIR == 2 needs both copies).  Each consumer sub-warp (W = 16
// or 32 lanes, lane i owns row i) takes blocks of the tile round-robin: its right-hand sides are
// fetched from global memory before it waits for the stage, the substitution runs out of shared
// memory (subwarp_block_solve), results go straight back to global memory.  HBM streaming is thereby
// decoupled from the b-step dependent chain of each block.
// ------------------------------------------------------------------------------------------------
constexpr int kMaxBlocksPerSub = 4;
#ifndef BJ_SOLVE_MINB
#define BJ_SOLVE_MINB 3  // registers capped so that three CTAs fit one SM
#endif

struct SolveStreamParams {
    int64_t n, nblocks, ntiles;
    const double* fac0;  // forward copy (DIR 0, 2) or backward copy (DIR 1)
    const double* fac1;  // backward copy (DIR 2 only)
    const double* in;
    double* out;
    int b, P, G, stages;
    int copy_doubles;    // doubles reserved per copy per stage (G * P rounded to even)
    int early_trigger;   // programmatic dependent launch: release the next kernel at entry (else at exit)
    const int32_t* perm; // permuted handle: vectors are accessed through perm, or null
};

template <int W, int DIR>
__global__ void __launch_bounds__(32 + 256, BJ_SOLVE_MINB)
solve_stream_kernel(const SolveStreamParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw);
    uint64_t* empty = full + p.stages;
    double* stage0 = reinterpret_cast<double*>(smem_raw + 128);
    constexpr int kCopies = DIR == 2 ? 2 : 1;
    const int stage_doubles = kCopies * p.copy_doubles;

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

    if (warp == 0) {
        if (lane == 0) {
            const uint64_t pol = policy_evict_first();
            int it = 0;
            for (int64_t tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x, ++it) {
                const int s = it % p.stages;
                const uint32_t ph = (uint32_t)((it / p.stages) & 1);
                mbar_wait(&empty[s], ph ^ 1u);
                const int64_t k0 = tile * p.G;
                const int nb = (int)(k0 + p.G <= p.nblocks ? p.G : p.nblocks - k0);
                const uint32_t bytes = (uint32_t)(((size_t)nb * p.P * 8 + 15) & ~(size_t)15);  // arrays carry 16 B of slack
                double* dst = stage0 + (size_t)s * stage_doubles;
                mbar_expect_tx(&full[s], bytes * kCopies);
                bulk_g2s(dst, p.fac0 + k0 * p.P, bytes, &full[s], pol);
                if (DIR == 2) bulk_g2s(dst + p.copy_doubles, p.fac1 + k0 * p.P, bytes, &full[s], pol);
            }
        }
    } else {
        const int ctid = threadIdx.x - 32;
        const int nsub = (blockDim.x - 32) / W;
        const int sub = ctid / W;
        const int i = ctid & (W - 1);
        const int b = p.b;
        pdl_wait();  // `in` may come from the previous kernel
        // right-hand sides are fetched one tile ahead: their HBM latency hides behind the current tile's solves
        auto fetch_rhs = [&](int64_t tile, double* dst) {
            const int64_t k0 = tile * p.G;
#pragma unroll
            for (int q = 0; q < kMaxBlocksPerSub; ++q) {
                const int64_t kb = k0 + sub + q * nsub;
                const int64_t row = kb * b + i;
                dst[q] = (tile < p.ntiles && q * nsub < p.G && kb < p.nblocks && i < b && row < p.n) ? p.in[p.perm ? p.perm[row] : row] : 0.0;
            }
        };
        double rn[kMaxBlocksPerSub];
        fetch_rhs(blockIdx.x, rn);
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x, ++it) {
            const int s = it % p.stages;
            const uint32_t ph = (uint32_t)((it / p.stages) & 1);
            const int64_t k0 = tile * p.G;
            const int nb = (int)(k0 + p.G <= p.nblocks ? p.G : p.nblocks - k0);
            double r[kMaxBlocksPerSub];
#pragma unroll
            for (int q = 0; q < kMaxBlocksPerSub; ++q) r[q] = rn[q];
            fetch_rhs(tile + gridDim.x, rn);
            mbar_wait(&full[s], ph);
            const double* f = stage0 + (size_t)s * stage_doubles;
#pragma unroll
            for (int q = 0; q < kMaxBlocksPerSub; ++q) {
                if (q * nsub < p.G) {  // uniform over the CTA
                    const int kb = sub + q * nsub;
                    const int kc = kb < nb ? kb : 0;  // idle sub-warps read block 0 (valid memory), result dropped
                    const double* fq = f + (size_t)kc * p.P;
                    double v = r[q];
                    if (DIR == 0 || DIR == 2) v = subwarp_block_solve<W, 0>(fq, b, i, v);
                    if (DIR == 1) v = subwarp_block_solve<W, 1>(fq, b, i, v);
                    if (DIR == 2) v = subwarp_block_solve<W, 1>(fq + p.copy_doubles, b, i, v);
                    const int64_t row = (k0 + kb) * b + i;
                    if (kb < nb && i < b && row < p.n) p.out[p.perm ? p.perm[row] : row] = v;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// b in {16, 24, 32}: a GROUP of LPB = 4 lanes per block, each lane owning the b / 4 rows i = 4k + l in
// registers, eight blocks per warp.  At step j the owner of row j broadcasts its finished value inside
// the group (one 64-bit shuffle serves b / 4 rows of eight blocks), every lane updates its rows below
// (above) j with one LDS + one DFMA each; which rows take part is known at compile time except in the
// one register row that holds row j.  About 2 instructions per block and step instead of 9 with one lane
// per row, no idle lanes for b = 24: the solve is HBM-bound again instead of issue-bound.
// Each warp owns a private ring of shared-memory stages; lane 0 refills a stage right after the warp
// has consumed it (one bulk async copy per block, blocks padded to a stride of 32 mod 128 bytes so the
// eight groups of a warp read different banks).  No producer warp, no CTA-wide barrier.
// ------------------------------------------------------------------------------------------------
struct GroupParams {
    int64_t n, nblocks, ntiles;  // a tile = the eight consecutive blocks one warp solves together
    const double* fac0;          // the forward copy: every direction runs from it (group_backward_fwdcopy)
    const double* in;
    double* out;
    int stages;
    int lz;              // 0 plain, 1 Lanczos prologue (DIR 1), 2 Lanczos epilogue (DIR 0), 3 PCG update + apply (DIR 2)
    int reverse;         // serpentine: this launch walks the tiles from the last to the first (see launch_group_t)
    int64_t keep_from;   // tiles at position >= keep_from of the walk are loaded as ordinary L2 lines instead of evict_first
    LzPrologue pro;
    LzEpilogue epi;
    PcgHook pcg;
    const int32_t* perm;  // plain solves of a permuted handle: vectors are accessed through perm, or null
};

__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// LZ (compile time: the plain solves carry none of the hooks): 0 plain, 1 Lanczos prologue (DIR 1), 2 Lanczos epilogue
// (DIR 0), 3 PCG update + apply (DIR 2)
template <int B, int LPB, int DIR, int LZ>
__global__ void __launch_bounds__(384)
solve_group_kernel(const GroupParams p)
{
    using Geo = GroupGeom<B, LPB>;
    constexpr int RPL = Geo::RPL;
    constexpr int NBW = Geo::NBW;
    constexpr int kCopies = 1;  // bj_apply (DIR 2) runs both substitutions from the forward copy
    constexpr int kStageDoubles = kCopies * NBW * Geo::STRIDE;
    constexpr uint32_t kBlockBytes = Geo::P * 8;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nwarps = blockDim.x >> 5;
    // per warp: `stages` mbarriers (64 bytes reserved), an exchange buffer for the tile's vector rows, then its ring
    constexpr int XB = B + 2;          // padded row of the exchange buffer (one block), in doubles
    constexpr int kXchg = NBW * XB;    // NBW * B = 32 * RPL rows per tile
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw) + warp * 8;
    double* xchg = reinterpret_cast<double*>(smem_raw + (size_t)nwarps * 64) + (size_t)warp * kXchg;
    double* ring = reinterpret_cast<double*>(smem_raw + (size_t)nwarps * 64) + (size_t)nwarps * kXchg +
                   (size_t)warp * p.stages * kStageDoubles;

    if (lane == 0) {
        for (int s = 0; s < p.stages; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    const int64_t stride = (int64_t)gridDim.x * nwarps;
    const int64_t first = (int64_t)blockIdx.x * nwarps + warp;
    const uint64_t pol_stream = policy_evict_first();
    const uint64_t pol_keep = policy_evict_normal();
    // `tile` counts positions of the walk; phys() is the tile of the factor array that sits there
    auto phys = [&](int64_t tile) { return p.reverse ? p.ntiles - 1 - tile : tile; };
    auto issue = [&](int64_t tile, int s) {  // lane 0 only: one bulk copy per block and copy
        if (tile >= p.ntiles) return;
        const uint64_t pol = tile >= p.keep_from ? pol_keep : pol_stream;
        const int64_t k0 = phys(tile) * NBW;
        const int nb = (int)(k0 + NBW <= p.nblocks ? NBW : p.nblocks - k0);
        double* dst = ring + (size_t)s * kStageDoubles;
        mbar_expect_tx(&full[s], (uint32_t)nb * kBlockBytes * kCopies);
        for (int q = 0; q < nb; ++q) {
            bulk_g2s(dst + q * Geo::STRIDE, p.fac0 + (k0 + q) * Geo::P, kBlockBytes, &full[s], pol);
        }
    };
    if (lane == 0)
        for (int s = 0; s < p.stages; ++s) issue(first + s * stride, s);  // factors are setup-time constants: no wait

    const int g = lane / LPB, l = lane % LPB;
    pdl_wait();  // `in` may come from the previous kernel
    __shared__ double lz_sh[24];
    double alpha = 0.0, beta = 0.0, inv_beta = 0.0, acc = 0.0;  // Lanczos scalars and this thread's dot product
    bool stop = false;
    if (DIR == 1 && LZ == 1) stop = lz_prologue_begin(p.pro, alpha);
    if (DIR == 0 && LZ == 2) stop = lz_epilogue_begin(p.epi, beta, inv_beta);
    double acc2 = 0.0;  // PCG: r.z
    if (DIR == 2 && LZ == 3) stop = pcg_hook_begin(p.pcg, alpha);  // alpha = the CG step length here
    double mcq = 0.0, mcr = 0.0, mcx = 0.0;  // mode 1 (Lanczos on M^-1 A): coefficients of q, r, r_prev
    const bool mlz = DIR == 2 && LZ == 3 && p.pcg.mode != 0;
    if (mlz && !stop) mlz_hook_coeffs(p.pcg, mcq, mcr, mcx);
    if (stop) {  // uniform over the grid; the bulk copies already issued must land before the CTA may exit
        for (int s = 0; s < p.stages; ++s)
            if (first + s * stride < p.ntiles) mbar_wait(&full[s], 0u);
        return;
    }
    // Vector rows move COALESCED: the tile's NBW * B = 32 * RPL rows are contiguous in memory, lane q takes rows
    // k * 32 + q; the exchange buffer turns that into the solve's (block g, row k * LPB + l) ownership and back.
    // Loads of one tile are issued together (all rows, all vectors) before anything is stored: the Lanczos
    // vectors may alias as far as the compiler knows, so interleaved stores would serialise the loads.
    auto fetch = [&](int64_t tile, double (&dst)[RPL], double (&ew)[RPL], double (&ev)[RPL]) {
        const int64_t row0 = phys(tile) * (NBW * B) + lane;
        double a[RPL], c[RPL];
#pragma unroll
        for (int k = 0; k < RPL; ++k) {
            const int64_t row = row0 + k * 32;
            const bool live = tile < p.ntiles && row < p.n;
            a[k] = c[k] = 0.0;
            if (DIR == 1 && LZ == 1) {
                if (live) a[k] = p.pro.first ? p.pro.w0[row] : p.pro.w[row];
                if (live && !p.pro.first) c[k] = p.pro.vcur[row];
            } else if (DIR == 2 && LZ == 3) {
                if (live) { a[k] = p.pcg.r[row]; c[k] = p.pcg.q[row]; ew[k] = p.pcg.x[row]; ev[k] = mlz ? 0.0 : p.pcg.p[row]; }
            } else {
                if (live) a[k] = p.in[(LZ == 0 && p.perm) ? p.perm[row] : row];
                if (DIR == 0 && LZ == 2) {  // the epilogue's own operands ride along one tile ahead
                    ew[k] = live ? p.epi.w[row] : 0.0;
                    ev[k] = (live && p.epi.vprev) ? p.epi.vprev[row] : 0.0;
                }
            }
        }
#pragma unroll
        for (int k = 0; k < RPL; ++k) {
            if (DIR == 1 && LZ == 1) {  // the solve's input is w = w' - alpha v_j, built here and stored once
                const int64_t row = row0 + k * 32;
                const double wi = a[k] - alpha * c[k];
                if (tile < p.ntiles && row < p.n) p.pro.w[row] = wi;
                acc = fma(wi, wi, acc);
                dst[k] = wi;
            } else if (DIR == 2 && LZ == 3) {  // r_new = r - a q (the solve's input, stored once), x += a p
                const int64_t row = row0 + k * 32;
                const double ri = mlz ? mlz_combine(mcq, mcr, mcx, c[k], a[k], ew[k]) : a[k] - alpha * c[k];
                if (tile < p.ntiles && row < p.n) {
                    if (mlz) {
                        p.pcg.x[row] = ri;  // r_{k+1} takes the place of r_{k-1}
                    } else {
                        p.pcg.r[row] = ri;
                        p.pcg.x[row] = fma(alpha, ev[k], ew[k]);
                    }
                    acc = fma(ri, ri, acc);
                }
                dst[k] = (tile < p.ntiles && row < p.n) ? ri : 0.0;
            } else {
                dst[k] = a[k];
            }
        }
    };
    double rn[RPL], ewn[RPL], evn[RPL];
    fetch(first, rn, ewn, evn);
    int it = 0;
    for (int64_t tile = first; tile < p.ntiles; tile += stride, ++it) {
        const int s = it % p.stages;
        const uint32_t ph = (uint32_t)((it / p.stages) & 1);
        double r[RPL];
#pragma unroll
        for (int k = 0; k < RPL; ++k) {
            const int e = k * 32 + lane;
            xchg[(e / B) * XB + e % B] = rn[k];
        }
        __syncwarp();
#pragma unroll
        for (int k = 0; k < RPL; ++k) r[k] = xchg[g * XB + k * LPB + l];
        double ew[RPL], ev[RPL];
#pragma unroll
        for (int k = 0; k < RPL; ++k) { ew[k] = (DIR == 2 && LZ == 3) ? rn[k] : ewn[k]; ev[k] = evn[k]; }  // PCG: ew = r_new rows
        fetch(tile + stride, rn, ewn, evn);  // one tile ahead: its latency hides behind this tile's solve
        mbar_wait(&full[s], ph);
        const double* f = ring + (size_t)s * kStageDoubles + g * Geo::STRIDE;
        if (DIR == 0 || DIR == 2) group_forward<B, LPB>(f, l, r);
        if (DIR == 1 || DIR == 2) group_backward_fwdcopy<B, LPB>(f, l, r);
        __syncwarp();
#pragma unroll
        for (int k = 0; k < RPL; ++k) xchg[g * XB + k * LPB + l] = r[k];
        __syncwarp();
        const int64_t row0 = phys(tile) * (NBW * B) + lane;
#pragma unroll
        for (int k = 0; k < RPL; ++k) {
            const int e = k * 32 + lane;
            const int64_t row = row0 + k * 32;
            const double y = xchg[(e / B) * XB + e % B];
            if (row < p.n) {
                if (DIR == 0 && LZ == 2) {
                    const double vn = ew[k] * inv_beta;              // v_{j+1}
                    const double wi = y * inv_beta - beta * ev[k];   // w'_new (ev = 0 on the first step)
                    p.epi.vnew[row] = vn;
                    p.epi.w[row] = wi;
                    acc = fma(vn, wi, acc);
                } else {
                    if (DIR == 2 && LZ == 3) acc2 = fma(ew[k], y, acc2);  // r_new . z
                    p.out[(LZ == 0 && p.perm) ? p.perm[row] : row] = y;
                }
            }
        }
        __syncwarp();
        if (lane == 0) {
            fence_proxy_async();  // the warp's generic reads of this stage precede the async refill
            issue(tile + (int64_t)p.stages * stride, s);
        }
    }
    if (DIR == 1 && LZ == 1) lz_reduce_finish(p.pro.red, acc, lz_sh);
    if (DIR == 0 && LZ == 2) lz_reduce_finish(p.epi.red, acc, lz_sh);
    if (DIR == 2 && LZ == 3) {
        lz_reduce_finish2(p.pcg.red_rr, acc, p.pcg.red_rz, acc2, lz_sh);  // one ticket for both sums
    }
}

// b == 1 fast path is just the B = 1 instance of solve_small_kernel.

template <int DIR, int LZ>
static int launch_small(bj_handle_s* h, const double* in, double* out, const LzPrologue* pro, const LzEpilogue* epi,
                        const PcgHook* pcg = nullptr)
{
    const int threads = 128;
    const unsigned blocks = (unsigned)((h->nblocks + threads - 1) / threads);
    uintptr_t al = (uintptr_t)in | (uintptr_t)out;
    if (pro) al |= (uintptr_t)pro->w0 | (uintptr_t)pro->w | (uintptr_t)pro->vcur;
    if (epi) al |= (uintptr_t)epi->w | (uintptr_t)epi->vprev | (uintptr_t)epi->vnew;
    if (pcg) al |= (uintptr_t)pcg->x | (uintptr_t)pcg->p | (uintptr_t)pcg->r | (uintptr_t)pcg->q;
    const bool vec = (al & 31) == 0;
    const bool pdl = h->pdl && !h->prof_on;
    const LzPrologue pr = pro ? *pro : LzPrologue{};
    const LzEpilogue ep = epi ? *epi : LzEpilogue{};
    const PcgHook pc = pcg ? *pcg : PcgHook{};
    if (pcg && ((int)blocks > pcg->red_rr.cap || (int)blocks > pcg->red_rz.cap)) return BJ_ERR_INVALID_ARG;
    if ((epi && (int)blocks > epi->red.cap) || (pro && (int)blocks > pro->red.cap)) return BJ_ERR_INVALID_ARG;
    cudaError_t e = cudaSuccess;
    // serpentine walk (see launch_group_t): the backward solve starts at the END of the factor array, where the fused
    // SpMV + forward-solve kernel of the previous operator apply stopped, and keeps the head of the array for the next one
    const int P = h->tri ? 2 * h->b - 1 : h->packed;
    const int64_t cta_bytes = (int64_t)threads * P * 8;
    const int64_t keep_ctas = std::min<int64_t>(blocks, (int64_t)h->tune.serp_keep_mb * 1000000 / cta_bytes);
    const int serp = (DIR == 1 && LZ == 0 && keep_ctas > 0) ? 1 : 0;  // plain kernels only (see launch_group_t)
    const unsigned serp_keep_from = (unsigned)(blocks - keep_ctas);
#define BJ_LAUNCH_SMALL(B, V, T)                                                                                  \
    launch_kernel(solve_small_kernel<B, DIR, V, LZ, T>, blocks, threads, 0, h->stream, pdl, h->n, h->nblocks,     \
                  (const double*)h->fac_small, in, out, pr, ep, pc, serp, serp_keep_from, (const int32_t*)(LZ == 0 ? h->var_perm : nullptr))
#define BJ_CASE(B)                                                                         \
    case B:                                                                                \
        e = vec ? BJ_LAUNCH_SMALL(B, true, false) : BJ_LAUNCH_SMALL(B, false, false);      \
        break;
#define BJ_CASE_T(B)                                                                       \
    case B:                                                                                \
        e = h->tri ? (vec ? BJ_LAUNCH_SMALL(B, true, true) : BJ_LAUNCH_SMALL(B, false, true)) \
                   : (vec ? BJ_LAUNCH_SMALL(B, true, false) : BJ_LAUNCH_SMALL(B, false, false)); \
        break;
    switch (h->b) {
        BJ_CASE(1) BJ_CASE(2) BJ_CASE(3) BJ_CASE_T(4) BJ_CASE_T(5) BJ_CASE_T(6) BJ_CASE_T(7) BJ_CASE_T(8)
        default: return BJ_ERR_INVALID_ARG;
    }
#undef BJ_CASE_T
#undef BJ_CASE
#undef BJ_LAUNCH_SMALL
    if (e != cudaSuccess) { set_cuda_error(e, "solve_small_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}

template <int W, int DIR>
static int launch_stream_solve(bj_handle_s* h, const SolveStreamParams& sp, int want_per_sm, int threads, size_t smem)
{
    static std::atomic<bool> configured[64];
    {
        cudaError_t e = ensure_big_smem(solve_stream_kernel<W, DIR>, configured);
        if (e != cudaSuccess) { set_cuda_error(e, "cudaFuncSetAttribute(solve_stream_kernel)"); return BJ_ERR_CUDA; }
    }
    int occ = 1;  // persistent grid: exactly the CTAs that are resident at once
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, solve_stream_kernel<W, DIR>, threads, smem);
    const int per_sm = std::max(1, std::min(occ, want_per_sm));
    const int grid = (int)std::min<int64_t>(sp.ntiles, (int64_t)h->num_sms * per_sm);
    cudaError_t e = launch_kernel(solve_stream_kernel<W, DIR>, grid, threads, smem, h->stream, h->pdl && !h->prof_on, sp);
    if (e != cudaSuccess) { set_cuda_error(e, "solve_stream_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}

template <int DIR>
static int launch_warp(bj_handle_s* h, const double* in, double* out)
{
    const int W = h->lanes;
    const int cwarps = std::max(1, std::min(h->tune.solve_warps, 8));
    const int threads = 32 + 32 * cwarps;
    const int nsub = cwarps * 32 / W;
    const int copies = DIR == 2 ? 2 : 1;
    const size_t block_bytes = (size_t)h->packed * 8;
    const int target = h->tune.solve_stage_kb * 1024;
    int bps = (int)((target / copies + nsub * block_bytes / 2) / (nsub * block_bytes));
    bps = std::max(1, std::min(bps, kMaxBlocksPerSub));
    SolveStreamParams sp;
    sp.n = h->n; sp.nblocks = h->nblocks; sp.b = h->b; sp.P = h->packed;
    sp.G = nsub * bps;
    if (sp.G % 2) sp.G += 1;  // keeps every tile's byte offset 16-byte aligned when P is odd
    sp.ntiles = (h->nblocks + sp.G - 1) / sp.G;
    sp.copy_doubles = (sp.G * sp.P + 1) & ~1;
    sp.fac0 = DIR == 1 ? h->fac_bwd : h->fac_fwd;
    sp.fac1 = h->fac_bwd;
    sp.in = in; sp.out = out;
    sp.perm = h->var_perm;
    sp.early_trigger = h->tune.pdl_early & 1;
    const size_t stage_bytes = (size_t)copies * sp.copy_doubles * 8;
    int stages = std::max(2, h->tune.solve_stages);
    while (stages > 2 && 128 + stages * stage_bytes > 110 * 1024) --stages;
    sp.stages = stages;
    const size_t smem = 128 + stages * stage_bytes;
    const int per_sm = h->tune.solve_ctas;
    return W == 16 ? launch_stream_solve<16, DIR>(h, sp, per_sm, threads, smem) : launch_stream_solve<32, DIR>(h, sp, per_sm, threads, smem);
}

template <int B, int LPB, int DIR>
static int launch_group_t(bj_handle_s* h, const double* in, double* out, const LzPrologue* pro, const LzEpilogue* epi,
                          const PcgHook* pcg)
{
    using Geo = GroupGeom<B, LPB>;
    constexpr int kGroupBlocksPerWarp = Geo::NBW;
    constexpr int kCopies = 1;  // DIR 2 uses the forward copy for both substitutions
    const size_t stage_bytes = (size_t)kCopies * kGroupBlocksPerWarp * Geo::STRIDE * 8;
    const int stages = std::max(2, std::min(8, h->tune.group_stages));
    // as many warps as fit one SM's shared memory (one CTA per SM), at most 12: the bytes in flight per SM are
    // what hides the ~2 us loaded DRAM latency (throughput ~ ring bytes / (latency + one tile's solve))
    const size_t budget = (size_t)h->tune.group_smem_kb * 1024;
    const size_t xchg_bytes = (size_t)kGroupBlocksPerWarp * (B + 2) * 8;
    int warps = (int)(budget / (stages * stage_bytes + 64 + xchg_bytes));
    warps = std::max(1, std::min(warps, h->tune.group_warps));
    const size_t smem = (size_t)warps * (64 + xchg_bytes + stages * stage_bytes);
    static std::atomic<bool> configured[64];
    static std::atomic<bool> configured_hook[64];
    {
        cudaError_t e = ensure_big_smem(solve_group_kernel<B, LPB, DIR, 0>, configured);
        if (e == cudaSuccess) e = ensure_big_smem(solve_group_kernel<B, LPB, DIR, (DIR == 1 ? 1 : DIR == 0 ? 2 : 3)>, configured_hook);
        if (e != cudaSuccess) { set_cuda_error(e, "cudaFuncSetAttribute(solve_group_kernel)"); return BJ_ERR_CUDA; }
    }
    GroupParams gp;
    gp.n = h->n; gp.nblocks = h->nblocks;
    gp.ntiles = (h->nblocks + kGroupBlocksPerWarp - 1) / kGroupBlocksPerWarp;
    gp.fac0 = h->fac_fwd;
    gp.in = in; gp.out = out; gp.stages = stages;
    // Serpentine walk (BJ_SERP_KEEP_MB > 0): the backward solve walks the factor array from its end to its start and the
    // forward solve from start to end, and the last `keep` megabytes of each walk are loaded as ordinary L2 lines instead
    // of evict_first.  In a chain of operator applies (back-to-back bj_op_apply, parity-mode Lanczos) the next backward
    // solve then finds the tail of the array, and the forward solve its head, still in the 126 MB L2: those bytes are not
    // read from HBM twice.  bj_apply (DIR 2) always walks forward and keeps nothing; the hooked kernels of the fused
    // Lanczos / PCG steps keep nothing either (their vectors are worth more L2 than the factors: measured).
    {
        const int64_t tile_bytes = (int64_t)kGroupBlocksPerWarp * Geo::P * 8;
        const int64_t keep_tiles = (DIR == 2 || pro || epi || pcg) ? 0 : std::min<int64_t>(gp.ntiles, (int64_t)h->tune.serp_keep_mb * 1000000 / tile_bytes);
        gp.reverse = (DIR == 1 && keep_tiles > 0) ? 1 : 0;
        gp.keep_from = gp.ntiles - keep_tiles;
    }
    gp.lz = (DIR == 1 && pro) ? 1 : (DIR == 0 && epi) ? 2 : (DIR == 2 && pcg) ? 3 : 0;
    gp.perm = h->var_perm;
    gp.pcg = pcg ? *pcg : PcgHook{};
    gp.pro = pro ? *pro : LzPrologue{};
    gp.epi = epi ? *epi : LzEpilogue{};
    constexpr int kLz = DIR == 1 ? 1 : DIR == 0 ? 2 : 3;  // the one hook this direction can carry
    int occ = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, solve_group_kernel<B, LPB, DIR, 0>, warps * 32, smem);
    const int64_t want = (gp.ntiles + warps - 1) / warps;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(want, (int64_t)h->num_sms * std::max(1, occ)));
    if ((gp.lz == 2 && grid > gp.epi.red.cap) || (gp.lz == 1 && grid > gp.pro.red.cap)) return BJ_ERR_INVALID_ARG;
    if (gp.lz == 3 && (grid > gp.pcg.red_rr.cap || grid > gp.pcg.red_rz.cap)) return BJ_ERR_INVALID_ARG;
    cudaError_t e = gp.lz ? launch_kernel(solve_group_kernel<B, LPB, DIR, kLz>, grid, warps * 32, smem, h->stream, h->pdl && !h->prof_on, gp)
                          : launch_kernel(solve_group_kernel<B, LPB, DIR, 0>, grid, warps * 32, smem, h->stream, h->pdl && !h->prof_on, gp);
    if (e != cudaSuccess) { set_cuda_error(e, "solve_group_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}

template <int DIR>
static int launch_group(bj_handle_s* h, const double* in, double* out, const LzPrologue* pro, const LzEpilogue* epi,
                        const PcgHook* pcg = nullptr)
{
    // lanes per block: small enough tiles that many warps fit one SM's shared memory (latency hiding)
    const int lpb = (h->tune.group_lanes > 0 ? h->tune.group_lanes : (h->b == 32 ? 8 : 4));
    switch (h->b) {
        case 16: return lpb == 8 ? launch_group_t<16, 8, DIR>(h, in, out, pro, epi, pcg) : launch_group_t<16, 4, DIR>(h, in, out, pro, epi, pcg);
        case 24: return lpb == 8 ? launch_group_t<24, 8, DIR>(h, in, out, pro, epi, pcg) : launch_group_t<24, 4, DIR>(h, in, out, pro, epi, pcg);
        case 32: return lpb == 16 ? launch_group_t<32, 16, DIR>(h, in, out, pro, epi, pcg)
                      : lpb == 8 ? launch_group_t<32, 8, DIR>(h, in, out, pro, epi, pcg) : launch_group_t<32, 4, DIR>(h, in, out, pro, epi, pcg);
        default: return BJ_ERR_INVALID_ARG;
    }
}

static bool use_group_kernel(const bj_handle_s* h)
{
    return h->single_copy;  // b = 16, 24, 32: one (forward) copy of the factors, group of lanes per block
}

// kind 1 always carries the hooks; kind 2 only in the group kernel (b = 16, 24, 32); b = 0 has no solve to ride on
bool lanczos_fusable(const bj_handle_s* h)
{
    if (h->var_perm) return false;  // the hooks address the vectors by block row: permuted handles run the unfused iterations
    return h->solve_kind == 1 || h->solve_kind == 3 || (h->solve_kind == 2 && use_group_kernel(h));
}

int launch_solve(bj_handle_s* h, int dir, const double* in, double* out, const LzPrologue* pro, const LzEpilogue* epi,
                 const PcgHook* pcg)
{
    if ((pro || epi || pcg) && !lanczos_fusable(h)) return BJ_ERR_INVALID_ARG;
    if (pcg && dir != 2) return BJ_ERR_INVALID_ARG;
    int rc = BJ_OK;
    if (h->solve_kind == 0) {
        if (in != out) BJ_CUDA(cudaMemcpyAsync(out, in, (size_t)h->n * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
        return BJ_OK;
    }
    const int kind = dir == 0 ? BJ_K_SOLVE_L : (dir == 1 ? BJ_K_SOLVE_LT : BJ_K_APPLY);
    {
        KernelScope scope(h, kind);
        if (h->solve_kind == 4) {
            rc = launch_solve_var(h, dir, in, out);
        } else if (h->solve_kind == 3) {
            rc = launch_solve_band(h, dir, in, out, pro, epi, pcg);
        } else if (h->solve_kind == 1) {
            rc = dir == 0   ? (epi ? launch_small<0, 2>(h, in, out, nullptr, epi) : launch_small<0, 0>(h, in, out, nullptr, nullptr))
                 : dir == 1 ? (pro ? launch_small<1, 1>(h, in, out, pro, nullptr) : launch_small<1, 0>(h, in, out, nullptr, nullptr))
                            : (pcg ? launch_small<2, 3>(h, in, out, nullptr, nullptr, pcg) : launch_small<2, 0>(h, in, out, nullptr, nullptr));
        } else if (use_group_kernel(h)) {
            rc = dir == 0 ? launch_group<0>(h, in, out, pro, epi) : dir == 1 ? launch_group<1>(h, in, out, pro, epi)
                          : launch_group<2>(h, in, out, nullptr, nullptr, pcg);
        } else {
            rc = dir == 0 ? launch_warp<0>(h, in, out) : dir == 1 ? launch_warp<1>(h, in, out) : launch_warp<2>(h, in, out);
        }
    }
    if (rc != BJ_OK) return rc;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

}  // namespace bj
