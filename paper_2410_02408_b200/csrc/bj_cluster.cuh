// Device helpers shared by the single-launch cluster kernels (bj_lanczos_cluster.cu, bj_pcg_cluster.cu): CTA-wide fixed-order
// sums, one-way exchanges between the CTAs of a thread-block cluster through distributed shared memory (st.async / bulk
// copies counted on the receiver's mbarrier), and the block solves on a CTA's own diagonal blocks.
#pragma once

#include <stdint.h>

#include "bj_device.cuh"
#include "bj_internal.cuh"

namespace bj {

namespace {

constexpr int kClusterMax = 16;  // eight CTAs (portable) or sixteen (opt-in: one GPC of a B200 holds them)
constexpr int kClThreads = 256;
constexpr int kClWarps = kClThreads / 32;
constexpr int kClRowReg = 8;   // a thread keeps its row's entries in registers when no row is longer
constexpr int kClDotCols = 64; // basis vectors per sweep of the dot pass


// sum over the CTA in a fixed order (shuffle tree per warp, pairwise tree over the warp sums), valid on every thread
__device__ __forceinline__ double cl_cta_sum(double v, double* sh)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    double s[kClWarps];
#pragma unroll
    for (int q = 0; q < kClWarps; ++q) s[q] = sh[q];
#pragma unroll
    for (int w = kClWarps / 2; w > 0; w >>= 1)
#pragma unroll
        for (int q = 0; q < w; ++q) s[q] += s[q + w];
    return s[0];
}

// Exchanges between the CTAs are one-way pushes: st.async writes 8 bytes into a peer's shared memory and counts them on
// the PEER's mbarrier (complete_tx), the receiver arms that barrier with the bytes it expects and waits for the phase --
// no cluster-wide barrier, no wait for store acknowledgements (a cluster barrier after remote stores measured ~1000
// cycles per exchange, three to five times per step).  Exchange e uses barrier e & 1 and buffer e & 1: a CTA can be at
// most one exchange ahead of a peer (it needs every peer's data of exchange e to finish e, and a peer sends e only after
// it has read the buffer of e - 1), so two alternate.
struct Exchange {
    uint64_t* bar;  // [2]
    int e;          // exchanges started so far (identical on every CTA)
    int rank;
};

__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, int rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_async_f64(uint32_t raddr, double v, uint32_t rbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];" ::"r"(raddr),
                 "l"(__double_as_longlong(v)), "r"(rbar)
                 : "memory");
}

// every CTA sends src[0..count) to dst_base[dst_off + 0..count) of EVERY CTA (itself included) and waits until the eight
// contributions (total_doubles in all) have arrived in its own copy
template <int CS>
__device__ __forceinline__ void exchange_all(Exchange& x, const double* src, int count, double* dst_base, int dst_off, int total_doubles)
{
    uint64_t* bar = x.bar + (x.e & 1);
    const uint32_t parity = (uint32_t)((x.e >> 1) & 1);
    if (threadIdx.x == 0) mbar_expect_tx(bar, (uint32_t)total_doubles * 8u);
    const uint32_t bar_s = smem_u32(bar), dst_s = smem_u32(dst_base + dst_off);
    for (int e = threadIdx.x; e < count * CS; e += kClThreads) {
        const int dst = e % CS, q = e / CS;
        st_async_f64(mapa_u32(dst_s + 8u * (uint32_t)q, dst), src[q], mapa_u32(bar_s, dst));
    }
    mbar_wait(bar, parity);
    ++x.e;
}

// The same exchange for a long slice (the CTA's rows of t): ONE bulk copy per peer through the async proxy instead of
// count st.async per peer (1240 -> ~500 cycles for 128 rows), when the slice is 16-byte aligned and sized; the caller
// has made src visible to the async proxy (fence.proxy.async before its __syncthreads).  src is not rewritten before
// every peer has passed the next exchange, i.e. long after the copies have read it.
template <int CS>
__device__ __forceinline__ void exchange_all_bulk(Exchange& x, const double* src, int count, double* dst_base, int dst_off, int total_doubles)
{
    if (((count | dst_off) & 1) != 0) return exchange_all<CS>(x, src, count, dst_base, dst_off, total_doubles);
    uint64_t* bar = x.bar + (x.e & 1);
    const uint32_t parity = (uint32_t)((x.e >> 1) & 1);
    if (threadIdx.x == 0) mbar_expect_tx(bar, (uint32_t)total_doubles * 8u);
    if (threadIdx.x < CS && count > 0) {
        const uint32_t dst = mapa_u32(smem_u32(dst_base + dst_off), threadIdx.x), rbar = mapa_u32(smem_u32(bar), threadIdx.x);
        asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                     "r"(smem_u32(src)), "r"((uint32_t)count * 8u), "r"(rbar)
                     : "memory");
    }
    mbar_wait(bar, parity);
    ++x.e;
}

// All-reduce of ONE double that every thread of the CTA already holds (cl_cta_sum): threads 0..7 push it straight from
// the register to the eight CTAs, every thread adds the eight slots itself -- no staging store, no __syncthreads.
// (The callers' next exchange is always behind a __syncthreads, so no thread still reads this buffer when a peer
// refills it two exchanges later.)
template <int CS>
__device__ __forceinline__ double cluster_allreduce_scalar(Exchange& x, double v, double* xch2, int pm)
{
    double* xch = xch2 + (size_t)(x.e & 1) * CS * pm;
    uint64_t* bar = x.bar + (x.e & 1);
    const uint32_t parity = (uint32_t)((x.e >> 1) & 1);
    if (threadIdx.x == 0) mbar_expect_tx(bar, 8u * CS);
    if (threadIdx.x < CS)
        st_async_f64(mapa_u32(smem_u32(xch + x.rank * pm), threadIdx.x), v, mapa_u32(smem_u32(bar), threadIdx.x));
    mbar_wait(bar, parity);
    ++x.e;
    double s = 0.0;
#pragma unroll
    for (int r = 0; r < CS; ++r) s += xch[r * pm];
    return s;
}

// x = L^-T y (DIR 1) or L^-1 y (DIR 0) on the CTA's own diagonal blocks k_lo .. k_hi, thread per block, factors in shared
// memory (the interleave groups that cover the range, g_lo first); in / out are the CTA's local slices.
// The arithmetic and its order are solve_small_kernel's.
template <int B, int DIR>
__device__ __forceinline__ void cluster_solve(int n, int k_lo, int k_hi, int g_lo, const double* sf, const double* in, double* out)
{
    if constexpr (B == 0) {
        for (int i = threadIdx.x; i < k_hi - k_lo; i += kClThreads) out[i] = in[i];
    } else {
        constexpr int P = B * (B + 1) / 2;
        for (int k = k_lo + threadIdx.x; k < k_hi; k += kClThreads) {
            const double* f = sf + (size_t)((k >> 5) - g_lo) * (P * kInterleave) + (k & 31);
            const int li = (k - k_lo) * B, lo = k * B;
            double v[B];
#pragma unroll
            for (int i = 0; i < B; ++i) v[i] = (lo + i < n) ? in[li + i] : 0.0;
            if (DIR == 0) {
#pragma unroll
                for (int i = 0; i < B; ++i) {
                    double s = v[i];
#pragma unroll
                    for (int j = 0; j < B; ++j)
                        if (j < i) s -= f[(i * (i + 1) / 2 + j) * kInterleave] * v[j];
                    v[i] = s * f[(i * (i + 1) / 2 + i) * kInterleave];
                }
            } else {
#pragma unroll
                for (int i = B - 1; i >= 0; --i) {
                    double s = v[i];
#pragma unroll
                    for (int j = 0; j < B; ++j)
                        if (j > i) s -= f[(j * (j + 1) / 2 + i) * kInterleave] * v[j];
                    v[i] = s * f[(i * (i + 1) / 2 + i) * kInterleave];
                }
            }
#pragma unroll
            for (int i = 0; i < B; ++i)
                if (lo + i < n) out[li + i] = v[i];
        }
    }
}

// All-reduce of TWO doubles that every thread already holds: one exchange, slots two doubles wide.
template <int CS>
__device__ __forceinline__ void cluster_allreduce_scalar2(Exchange& x, double& a, double& b, double* xch2, int pm)
{
    double* xch = xch2 + (size_t)(x.e & 1) * CS * pm;
    uint64_t* bar = x.bar + (x.e & 1);
    const uint32_t parity = (uint32_t)((x.e >> 1) & 1);
    if (threadIdx.x == 0) mbar_expect_tx(bar, 16u * CS);
    if (threadIdx.x < 2 * CS) {
        const int dst = threadIdx.x >> 1, which = threadIdx.x & 1;
        st_async_f64(mapa_u32(smem_u32(xch + x.rank * pm + which), dst), which ? b : a, mapa_u32(smem_u32(bar), dst));
    }
    mbar_wait(bar, parity);
    ++x.e;
    double sa = 0.0, sb = 0.0;
#pragma unroll
    for (int r = 0; r < CS; ++r) { sa += xch[r * pm]; sb += xch[r * pm + 1]; }
    a = sa;
    b = sb;
}

}  // namespace

}  // namespace bj
