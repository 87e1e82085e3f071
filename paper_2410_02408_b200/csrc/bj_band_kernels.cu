// Banded block factors (opt-in with bj_setup_opts_t.band), the b > 8 kernels.  (For b <= 8 the
// same switch compacts tridiagonal blocks inside the existing thread-per-block kernels: see `tri` in bj_api.cu.)
//
// When every diagonal block D_k is banded with lower bandwidth w <= 2 (stencil matrices whose blocks follow a grid
// line are tridiagonal: configs 2 and 4), its Cholesky factor has the same band (no fill outside it), so the
// packed-dense factor stream of b(b+1)/2 doubles per block shrinks to (w+1) b.  This moves FEWER bytes than the
// dense-block count of SURVEY.md 8(d) and therefore carries its own byte accounting:
//   one solve pass = 8 N (w+1) + 16 N bytes  instead of  4 N (b+1) + 16 N.
// Arithmetic: exactly the oracle's left-looking Cholesky and substitutions with the structurally zero terms
// skipped (adding a zero product changes nothing), so the parity bar is unchanged.
//
// Layout: element (i, d) = l_{i, i-d}, d = 0..w (d = 0 holds 1 / l_ii), of blocks 32 g .. 32 g + 31 is one 256-byte
// line: fac_band[g * 32 E + (i (w+1) + d) * 32 + k % 32], E = (w+1) b.  One THREAD per block: every load of a warp
// is one coalesced line and no load depends on the substitution chain.
#include <algorithm>

#include "bj_device.cuh"
#include "bj_internal.cuh"
#include "bj_pcg_fuse.cuh"

namespace bj {

namespace {

// lower bandwidth of the diagonal blocks: max over rows of (row - first in-block column of the row)
__global__ void __launch_bounds__(256)
band_width_kernel(int64_t n, int b, const int32_t* __restrict__ rp, const int32_t* __restrict__ ci, Status* st)
{
    const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int d = 0;
    if (row < n) {
        const int64_t lo = (row / b) * b;
        int s = rp[row], hi = rp[row + 1];
        const int e = hi;
        while (s < hi) {  // first entry with column >= lo
            const int mid = (s + hi) >> 1;
            if (ci[mid] < lo) s = mid + 1; else hi = mid;
        }
        if (s < e && ci[s] < row) d = (int)(row - ci[s]);
    }
    d = __reduce_max_sync(0xffffffffu, d);
    if ((threadIdx.x & 31) == 0 && d > *(volatile int*)&st->max_band) atomicMax(&st->max_band, d);
}

// a2 + a3 for banded blocks: one thread per block, rows in order, a window of the last W factor rows in registers
template <int W>
__global__ void __launch_bounds__(128)
extract_factor_band_kernel(int64_t n, int b, int64_t nblocks, const int32_t* __restrict__ rp,
                           const int32_t* __restrict__ ci, const double* __restrict__ val, double* __restrict__ fac,
                           Status* st)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nblocks) return;
    const int E = (W + 1) * b;
    double* f = fac + (k >> 5) * (int64_t)E * kInterleave + (k & 31);
    const int64_t lo = k * b;
    double prev[W > 0 ? W : 1][W + 1];  // prev[r][d] = l_{i-1-r, i-1-r-d}
#pragma unroll
    for (int r = 0; r < (W > 0 ? W : 1); ++r)
#pragma unroll
        for (int d = 0; d <= W; ++d) prev[r][d] = 0.0;
    bool bad = false;
    for (int i = 0; i < b; ++i) {
        const int64_t row = lo + i;
        double a[W + 1];
#pragma unroll
        for (int d = 0; d <= W; ++d) a[d] = 0.0;
        if (row < n) {
            const int64_t first = row - W > lo ? row - W : lo;
            int s = rp[row], hi = rp[row + 1];
            const int e = hi;
            while (s < hi) {
                const int mid = (s + hi) >> 1;
                if (ci[mid] < first) s = mid + 1; else hi = mid;
            }
#pragma unroll
            for (int q = 0; q <= W; ++q) {
                if (s + q < e) {
                    const int64_t c = ci[s + q];
                    if (c <= row) {
                        const int d = (int)(row - c);
#pragma unroll
                        for (int dd = 0; dd <= W; ++dd)
                            if (dd == d) a[dd] = val[s + q];
                    }
                }
            }
        } else {
            a[0] = 1.0;  // identity rows pad the ragged last block
        }
        // row i of the factor: l_{i,j} = (a_ij - sum_{p<j} l_ip l_jp) / l_jj for j = i-W .. i-1, then the diagonal
        double cur[W + 1];
#pragma unroll
        for (int d = W; d >= 1; --d) {
            double sres = a[d];
            // p runs over i-W .. i-d-1 (ascending): offsets i-p = W .. d+1 in this row, (i-d)-p = W-d .. 1 in row i-d
#pragma unroll
            for (int o = W; o > d; --o) sres -= cur[o] * prev[d - 1][o - d];
            cur[d] = (i - d >= 0) ? sres / prev[d - 1][0] : 0.0;
        }
        double dg = a[0];
#pragma unroll
        for (int d = W; d >= 1; --d) dg -= cur[d] * cur[d];
        if (!(dg > 0.0) || isinf(dg)) { bad = true; dg = 1.0; }
        cur[0] = sqrt(dg);
        f[(i * (W + 1)) * kInterleave] = 1.0 / cur[0];
#pragma unroll
        for (int d = 1; d <= W; ++d) f[(i * (W + 1) + d) * kInterleave] = cur[d];
        // slide the window
#pragma unroll
        for (int r = W - 1; r >= 1; --r)
#pragma unroll
            for (int d = 0; d <= W; ++d) prev[r][d] = prev[r - 1][d];
        if (W > 0) {
#pragma unroll
            for (int d = 0; d <= W; ++d) prev[0][d] = cur[d];
        }
    }
    if (bad) {
        atomicOr(&st->flags, ST_NOT_SPD);
        atomicMin(&st->bad_block, (long long)k);
    }
}

// rows lo .. lo + b - 1 of a vector <-> registers (b <= BMAX at run time); 256-bit accesses when `vec`
template <int BMAX>
__device__ __forceinline__ void load_rows_rt(const double* src, int64_t lo, int64_t n, int b, bool vec, double (&v)[BMAX])
{
    if (vec) {
#pragma unroll
        for (int i = 0; i < BMAX; i += 4)
            if (i < b) ld_v4(src + lo + i, v + i);
    } else {
#pragma unroll
        for (int i = 0; i < BMAX; ++i) v[i] = (i < b && lo + i < n) ? src[lo + i] : 0.0;
    }
}
template <int BMAX>
__device__ __forceinline__ void store_rows_rt(double* dst, int64_t lo, int64_t n, int b, bool vec, const double (&v)[BMAX])
{
    if (vec) {
#pragma unroll
        for (int i = 0; i < BMAX; i += 4)
            if (i < b) st_v4(dst + lo + i, v + i);
    } else {
#pragma unroll
        for (int i = 0; i < BMAX; ++i)
            if (i < b && lo + i < n) dst[lo + i] = v[i];
    }
}

// thread per block; BMAX bounds the register arrays (b <= BMAX); DIR 0 forward, 1 backward, 2 both.
// LZ (compile time): 0 plain, 1 Lanczos prologue (DIR 1), 2 Lanczos epilogue (DIR 0), 3 PCG update + apply (DIR 2) --
// the same hooks, in the same order of operations, as solve_small_kernel (bj_solve_kernels.cu).
template <int BMAX, int W, int DIR, int LZ>
__global__ void __launch_bounds__(128)
solve_band_kernel(int64_t n, int b, int64_t nblocks, const double* __restrict__ fac, const double* in, double* out,
                  const LzPrologue pro, const LzEpilogue epi, const PcgHook pcg)
{
    __shared__ double lz_sh[8];
    pdl_trigger();
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool act = k < nblocks;
    if (LZ == 0 && !act) return;
    const int64_t kc = act ? k : 0;
    const int E = (W + 1) * b;
    const double* f = fac + (kc >> 5) * (int64_t)E * kInterleave + (kc & 31);
    const int64_t lo = kc * b;
    uintptr_t al = (uintptr_t)in | (uintptr_t)out;
    if (LZ == 1) al = (uintptr_t)pro.w0 | (uintptr_t)pro.w | (uintptr_t)pro.vcur;
    if (LZ == 2) al |= (uintptr_t)epi.w | (uintptr_t)epi.vprev | (uintptr_t)epi.vnew;
    if (LZ == 3) al = (uintptr_t)out | (uintptr_t)pcg.x | (uintptr_t)pcg.p | (uintptr_t)pcg.r | (uintptr_t)pcg.q;
    const bool vec = (b % 4 == 0) && lo + b <= n && (al & 31) == 0;
    // the whole band goes to registers first: (W+1) b independent, coalesced loads in flight per thread
    double l[(W + 1) * BMAX];
#pragma unroll
    for (int e = 0; e < (W + 1) * BMAX; ++e) l[e] = (e < E) ? ld_const_stream(f + e * kInterleave) : 0.0;
    pdl_wait();  // `in` may come from the previous kernel
    double v[BMAX];
    double acc = 0.0, acc2 = 0.0, beta = 0.0, inv_beta = 0.0;
    double rin[LZ == 3 ? BMAX : 1];
    if (LZ == 1) {
        double alpha, c[BMAX];
        if (act) {  // operands first, the scalar (a dependent load) after them
            if (pro.first) {
                load_rows_rt<BMAX>(pro.w0, lo, n, b, vec, v);
            } else {
                load_rows_rt<BMAX>(pro.w, lo, n, b, vec, v);
                load_rows_rt<BMAX>(pro.vcur, lo, n, b, vec, c);
            }
        }
        if (lz_prologue_begin(pro, alpha)) return;  // uniform over the grid
        if (act) {
            if (!pro.first) {
#pragma unroll
                for (int i = 0; i < BMAX; ++i)
                    if (i < b) v[i] -= alpha * c[i];
            }
#pragma unroll
            for (int i = 0; i < BMAX; ++i)
                if (i < b && lo + i < n) acc = fma(v[i], v[i], acc);
            store_rows_rt<BMAX>(pro.w, lo, n, b, vec, v);
        }
    } else if (LZ == 3) {
        // vector operands are requested before the scalars are read (see solve_small_kernel)
        double c[BMAX], xs[BMAX], pv[BMAX];
        if (act) {
            load_rows_rt<BMAX>(pcg.r, lo, n, b, vec, v);
            load_rows_rt<BMAX>(pcg.q, lo, n, b, vec, c);
            load_rows_rt<BMAX>(pcg.x, lo, n, b, vec, xs);
            if (!pcg.mode) load_rows_rt<BMAX>(pcg.p, lo, n, b, vec, pv);
        }
        double a;
        if (pcg_hook_begin(pcg, a)) return;  // uniform over the grid
        if (pcg.mode) {  // three-term step of Lanczos on M^-1 A: r_{k+1} replaces r_{k-1} (uniform branch)
            double cq, cr, cx;
            mlz_hook_coeffs(pcg, cq, cr, cx);
            if (act) {
#pragma unroll
                for (int i = 0; i < BMAX; ++i) {
                    if (i < b) {
                        v[i] = mlz_combine(cq, cr, cx, c[i], v[i], xs[i]);
                        rin[i] = v[i];
                    }
                }
                store_rows_rt<BMAX>(pcg.x, lo, n, b, vec, v);
            }
        } else if (act) {
#pragma unroll
            for (int i = 0; i < BMAX; ++i) {
                if (i < b) {
                    v[i] = v[i] - a * c[i];
                    if (lo + i < n) acc = fma(v[i], v[i], acc);
                    rin[i] = v[i];
                    xs[i] = fma(a, pv[i], xs[i]);
                }
            }
            store_rows_rt<BMAX>(pcg.r, lo, n, b, vec, v);
            store_rows_rt<BMAX>(pcg.x, lo, n, b, vec, xs);
        }
    } else {
        load_rows_rt<BMAX>(in, lo, n, b, vec, v);                       // before the scalars: independent of them
        if (LZ == 2 && lz_epilogue_begin(epi, beta, inv_beta)) return;  // uniform over the grid
    }
    if (DIR == 0 || DIR == 2) {
#pragma unroll
        for (int i = 0; i < BMAX; ++i) {
            if (i < b) {
                double s = v[i];
#pragma unroll
                for (int d = W; d >= 1; --d)
                    if (i - d >= 0) s -= l[i * (W + 1) + d] * v[i - d];
                v[i] = s * l[i * (W + 1)];
            }
        }
    }
    if (DIR == 1 || DIR == 2) {
#pragma unroll
        for (int i = BMAX - 1; i >= 0; --i) {
            if (i < b) {
                double s = v[i];
#pragma unroll
                for (int d = 1; d <= W; ++d)
                    if (i + d < BMAX && i + d < b) s -= l[(i + d) * (W + 1) + d] * v[i + d];
                v[i] = s * l[i * (W + 1)];
            }
        }
    }
    if (LZ == 2) {
        if (act) {
            double c[BMAX], d[BMAX];  // w and v_j
            load_rows_rt<BMAX>(epi.w, lo, n, b, vec, c);
            if (epi.vprev) load_rows_rt<BMAX>(epi.vprev, lo, n, b, vec, d);
#pragma unroll
            for (int i = 0; i < BMAX; ++i) {
                if (i < b) {
                    c[i] *= inv_beta;                       // v_{j+1}
                    v[i] *= inv_beta;
                    if (epi.vprev) v[i] -= beta * d[i];     // w'_new
                    if (lo + i < n) acc = fma(c[i], v[i], acc);
                }
            }
            store_rows_rt<BMAX>(epi.vnew, lo, n, b, vec, c);
            store_rows_rt<BMAX>(epi.w, lo, n, b, vec, v);
        }
        lz_reduce_finish(epi.red, acc, lz_sh);
    } else {
        if (act) store_rows_rt<BMAX>(out, lo, n, b, vec, v);
        if (LZ == 1) lz_reduce_finish(pro.red, acc, lz_sh);
        if (LZ == 3) {
            if (act) {
#pragma unroll
                for (int i = 0; i < BMAX; ++i)
                    if (i < b && lo + i < n) acc2 = fma(rin[i], v[i], acc2);
            }
            lz_reduce_finish2(pcg.red_rr, acc, pcg.red_rz, acc2, lz_sh);  // one ticket for both sums
        }
    }
}

template <int BMAX, int W>
int launch_band_t(bj_handle_s* h, int dir, const double* in, double* out, const LzPrologue* pro, const LzEpilogue* epi,
                  const PcgHook* pcg)
{
    const unsigned blocks = (unsigned)((h->nblocks + 127) / 128);
    const bool pdl = h->pdl && !h->prof_on;
    const LzPrologue pr = pro ? *pro : LzPrologue{};
    const LzEpilogue ep = epi ? *epi : LzEpilogue{};
    const PcgHook pc = pcg ? *pcg : PcgHook{};
    if ((pro && (int)blocks > pro->red.cap) || (epi && (int)blocks > epi->red.cap) ||
        (pcg && ((int)blocks > pcg->red_rr.cap || (int)blocks > pcg->red_rz.cap)))
        return BJ_ERR_INVALID_ARG;
#define BJ_BAND_LAUNCH(D, L)                                                                                          \
    launch_kernel(solve_band_kernel<BMAX, W, D, L>, blocks, 128, 0, h->stream, pdl, h->n, h->b, h->nblocks,             \
                  (const double*)h->fac_band, in, out, pr, ep, pc)
    cudaError_t e = dir == 0   ? (epi ? BJ_BAND_LAUNCH(0, 2) : BJ_BAND_LAUNCH(0, 0))
                    : dir == 1 ? (pro ? BJ_BAND_LAUNCH(1, 1) : BJ_BAND_LAUNCH(1, 0))
                               : (pcg ? BJ_BAND_LAUNCH(2, 3) : BJ_BAND_LAUNCH(2, 0));
#undef BJ_BAND_LAUNCH
    if (e != cudaSuccess) { set_cuda_error(e, "solve_band_kernel launch"); return BJ_ERR_CUDA; }
    return BJ_OK;
}

}  // namespace

int launch_band_width(bj_handle_s* h)
{
    const unsigned blocks = (unsigned)((h->n + 255) / 256);
    { SetupSpan span(h); band_width_kernel<<<blocks, 256, 0, h->stream>>>(h->n, h->b, h->row_ptr, h->col_idx, h->status); }
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

int launch_extract_factor_band(bj_handle_s* h)
{
    const unsigned blocks = (unsigned)((h->nblocks + 127) / 128);
    SetupSpan span(h);
#define BJ_CASE(W)                                                                                                      \
    case W:                                                                                                             \
        extract_factor_band_kernel<W><<<blocks, 128, 0, h->stream>>>(h->n, h->b, h->nblocks, h->row_ptr, h->col_idx, h->val, \
                                                                     h->fac_band, h->status);                          \
        break;
    switch (h->band) {
        BJ_CASE(0) BJ_CASE(1) BJ_CASE(2)
        default: return BJ_ERR_INVALID_ARG;
    }
#undef BJ_CASE
    h->launches++;
    BJ_CUDA(cudaGetLastError());
    return BJ_OK;
}

int launch_solve_band(bj_handle_s* h, int dir, const double* in, double* out, const LzPrologue* pro, const LzEpilogue* epi,
                      const PcgHook* pcg)
{
    const bool small = h->b <= 16;
    switch (h->band) {
        case 0: return small ? launch_band_t<16, 0>(h, dir, in, out, pro, epi, pcg) : launch_band_t<32, 0>(h, dir, in, out, pro, epi, pcg);
        case 1: return small ? launch_band_t<16, 1>(h, dir, in, out, pro, epi, pcg) : launch_band_t<32, 1>(h, dir, in, out, pro, epi, pcg);
        case 2: return small ? launch_band_t<16, 2>(h, dir, in, out, pro, epi, pcg) : launch_band_t<32, 2>(h, dir, in, out, pro, epi, pcg);
        default: return BJ_ERR_INVALID_ARG;
    }
}

}  // namespace bj
