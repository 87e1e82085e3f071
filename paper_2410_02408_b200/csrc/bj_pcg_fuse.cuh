// Fused PCG iteration: the vector updates and all three dot products of one iteration
// ride on the two path kernels that run anyway, plus one direction kernel:
//   K1  q = A p            (CSR SpMV tile kernel)      + per-CTA partials of p.q
//   K2  z = M^-1 r_new     (block solve pair, a5)      a = rho / (p.q);  x += a p;  r_new = r - a q  built on the fly as
//                                                      the solve's input and stored;  partials of r_new.r_new and r_new.z
//   K3  p = z + bt p       (bj_pcg.cu)                 stopping test on ||r_new|| / ||b||,  bt = rho_new / rho
// Same arithmetic, in the same order, as the unfused kernels of bj_pcg.cu; reductions finish in the kernel that
// produces them (last CTA, fixed order: lz_reduce_finish of bj_lanczos_fuse.cuh).
#pragma once

#include <stdint.h>

#include "bj_lanczos_fuse.cuh"

namespace bj {

struct PcgHook {
    double* x;            // solution, updated in place
    const double* p;      // direction
    double* r;            // residual, updated in place
    const double* q;      // A p
    const double* rho;    // r.z of the current residual (finished sum)
    const double* pq;     // p.q (finished sum)
    double* alpha;        // alpha[] (device): entry k written by CTA 0
    const int* flags;     // [0] stop flag
    LzReduce red_rr;      // -> r_new . r_new
    LzReduce red_rz;      // -> r_new . z
    int k;
    // mode 1: one step of Lanczos on M^-1 A in the M inner product (bj_cond_estimate_minv) on the same
    // kernel: q = A z_k, r = r_k, x = r_{k-1} (overwritten by r_{k+1}), p unused;  bsq[j] = r_j . z_j = bt_j^2, pq = z_k . q
    //   al_k = pq / bt_k^2,   r_{k+1} = q / bt_k - (al_k / bt_k) r_k - (bt_k / bt_{k-1}) r_{k-1},   z_{k+1} = M^-1 r_{k+1} -> out
    int mode;
    const double* bsq;
};

// mode 1 coefficients of (q, r, x); uniform over the grid.  CTA 0 records al_k.
__device__ __forceinline__ void mlz_hook_coeffs(const PcgHook& c, double& cq, double& cr, double& cx)
{
    const double b2 = c.bsq[c.k];
    const double bt = sqrt(b2);
    const double al = *c.pq / b2;
    cq = 1.0 / bt;
    cr = -al / bt;
    cx = c.k > 0 ? -bt / sqrt(c.bsq[c.k - 1]) : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) c.alpha[c.k] = al;
}

// the three-term combination, one fixed order of operations for every kernel that carries the hook
__device__ __forceinline__ double mlz_combine(double cq, double cr, double cx, double q, double r, double x)
{
    return fma(cx, x, fma(cr, r, cq * q));
}

// step length (uniform) and the stop flag; CTA 0 records alpha[k]
__device__ __forceinline__ bool pcg_hook_begin(const PcgHook& c, double& a)
{
    a = 0.0;
    if (c.flags[0]) return true;
    if (c.mode) return false;
    a = *c.rho / *c.pq;
    if (blockIdx.x == 0 && threadIdx.x == 0) c.alpha[c.k] = a;
    return false;
}

}  // namespace bj
