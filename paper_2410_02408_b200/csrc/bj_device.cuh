// Device-side helpers shared by the bj kernels (sm_100a inline PTX) and the launch helper that
// chains the library's own kernels with programmatic dependent launch (PDL).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

namespace bj {

// streaming (read-once) loads: bypass L1 allocation
__device__ __forceinline__ double ld_stream(const double* p)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
// streaming load with an explicit L2 eviction policy (createpolicy): evict_first for read-once data, evict_last for the
// slice the next kernel starts with
__device__ __forceinline__ double ld_stream_hint(const double* p, uint64_t pol)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
    return v;
}
// same load, but schedulable: the compiler may hoist it above unrelated arithmetic (the data never changes after setup)
__device__ __forceinline__ double ld_const_stream(const double* p)
{
    double v;
    asm("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
// read-once stream with an L2 evict-first policy (createpolicy, see policy_evict_first): small reused arrays (row
// pointers, the gathered vector) stay L2-resident
__device__ __forceinline__ double ld_once(const double* p, uint64_t pol)
{
    double v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ int ld_once(const int* p, uint64_t pol)
{
    int v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.s32 %0, [%1], %2;" : "=r"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ int ld_stream(const int* p)
{
    int v;
    asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}

// a / l with r = RN(1 / l): one multiplication and one residual correction (Markstein) give the correctly rounded
// quotient.  The library division takes its ~55-instruction slow path for the whole warp as soon as ONE lane divides a
// zero or tiny numerator -- which a sparse block does in every column.
__device__ __forceinline__ double div_by(double a, double l, double r)
{
    const double q = a * r;
    return fma(fma(-l, q, a), r, q);
}

// 256-bit / 128-bit vector accesses (LDG.E.256 / STG.E.256 on sm_100); pointers must be 32 / 16 byte aligned
__device__ __forceinline__ void ld_v4(const double* p, double* v)
{
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3]) : "l"(p));
}
__device__ __forceinline__ void st_v4(double* p, const double* v)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(v[3]) : "memory");
}
__device__ __forceinline__ void ld_v2(const double* p, double* v)
{
    asm volatile("ld.global.v2.f64 {%0,%1}, [%2];" : "=d"(v[0]), "=d"(v[1]) : "l"(p));
}
__device__ __forceinline__ void st_v2(double* p, const double* v)
{
    asm volatile("st.global.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(v[0]), "d"(v[1]) : "memory");
}

// mbarrier + 1-D bulk async copy (TMA engine) primitives ------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// the slice of a read-once stream that the NEXT kernel starts with: ordinary LRU lines.  (evict_last was measured and
// dropped: the lines outlive the chain of applies and take L2 away from the Lanczos vectors and from bj_apply's input.)
__device__ __forceinline__ uint64_t policy_evict_normal()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t pol)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
        : "memory");
}

// the shared solve of one diagonal block by a sub-warp of W lanes (lane i owns row i), factor read from
// `f` (shared or global memory).  DIR 0: forward, f = column-major packed lower, rows scaled by 1/l_ii;
// DIR 1: backward, f = row-major packed lower, columns scaled by 1/l_ii; diagonal slots hold 1/l_ii.
//   forward : y_i = r_i/l_ii - sum_{j<i} (l_ij/l_ii) y_j      backward: x_i = y_i/l_ii - sum_{j>i} (l_ji/l_ii) x_j
// Column oriented: at step j lane j's value is final and is broadcast by shuffle; one SHFL + one DFMA
// per step on the dependent chain.  All W lanes must call (full-mask shuffles); lanes >= b return 0.
template <int W, int DIR>
__device__ __forceinline__ double subwarp_block_solve(const double* f, int b, int i, double r)
{
    // 1/l_ii sits in the diagonal slot of row/column i
    const int dslot = DIR == 0 ? i * b - i * (i - 1) / 2 : i * (i + 1) / 2 + i;
    r *= (i < b) ? f[dslot] : 0.0;
#pragma unroll
    for (int jj = 0; jj < W; ++jj) {
        const int j = DIR == 0 ? jj : W - 1 - jj;
        if (j < b) {
            double lij = 0.0;  // off the dependent chain: the address does not depend on r
            if (DIR == 0) {
                if (i > j && i < b) lij = f[j * b - j * (j - 1) / 2 + (i - j)];
            } else {
                if (i < j) lij = f[j * (j + 1) / 2 + i];
            }
            const double vj = __shfl_sync(0xffffffffu, r, j, W);
            r = fma(-lij, vj, r);
        }
    }
    return r;
}

// ---- group-per-block substitution (b = 16, 24, 32): LPB lanes per block, b / LPB rows per lane in registers ----
// Used by solve_group_kernel (bj_solve_kernels.cu).
template <int B, int LPB>
struct GroupGeom {
    static constexpr int P = B * (B + 1) / 2;
    static constexpr int RPL = B / LPB;   // rows per lane
    static constexpr int NBW = 32 / LPB;  // blocks per warp
    // per-block stride in shared memory: packed size padded so that consecutive blocks start LPB * 8 bytes
    // (mod 128) apart -- the groups of a warp then read different banks
    static constexpr int target = (LPB * 8) % 128;
    static constexpr int pad_bytes = ((target - (P * 8) % 128) + 128) % 128;
    static constexpr int STRIDE = P + pad_bytes / 8;
    static_assert(B % LPB == 0 && (P * 8) % 16 == 0 && pad_bytes % 16 == 0, "bulk copies need 16-byte granules");
};

// forward substitution on the staged forward copy (column-major packed lower, rows scaled by 1/l_ii)
template <int B, int LPB>
__device__ __forceinline__ void group_forward(const double* f, int l, double (&r)[B / LPB])
{
    constexpr int RPL = B / LPB;
#pragma unroll
    for (int k = 0; k < RPL; ++k) {
        const int i = k * LPB + l;
        r[k] *= f[i * B - i * (i - 1) / 2];
    }
#pragma unroll
    for (int j = 0; j < B - 1; ++j) {
        const int kj = j / LPB, lj = j % LPB;
        const double vj = __shfl_sync(0xffffffffu, r[kj], lj, LPB);
        const double* col = f + (j * B - j * (j - 1) / 2 - j) + l;  // element (i, j) at col[i - l]
#pragma unroll
        for (int k = kj; k < RPL; ++k) {
            if (k == kj && lj == LPB - 1) continue;  // no row of this register row lies below j
            double lij = col[k * LPB];
            if (k == kj) lij = (l > lj) ? lij : 0.0;
            r[k] = fma(-lij, vj, r[k]);
        }
    }
}

// backward substitution on the FORWARD copy (column-major packed lower, rows scaled: f_ji = l_ji / l_jj, diagonal slot
// 1 / l_jj): with x~_j = l_jj x_j the recurrence is  x~_i = y_i - sum_{j > i} f_ji x~_j,  x_i = x~_i / l_ii.  bj_apply can
// therefore run both substitutions from ONE staged copy: its factor traffic is the algorithmic 4 N (b+1) bytes, not twice
// that.  Lane (row i) walks down its own column: element (j, i) at colbase_i + j.
template <int B, int LPB>
__device__ __forceinline__ void group_backward_fwdcopy(const double* f, int l, double (&r)[B / LPB])
{
    constexpr int RPL = B / LPB;
    int colbase[RPL];  // i B - i (i - 1) / 2 - i: start of column i minus i
#pragma unroll
    for (int k = 0; k < RPL; ++k) {
        const int i = k * LPB + l;
        colbase[k] = i * B - i * (i - 1) / 2 - i;
    }
#pragma unroll
    for (int j = B - 1; j >= 1; --j) {
        const int kj = j / LPB, lj = j % LPB;
        const double vj = __shfl_sync(0xffffffffu, r[kj], lj, LPB);
#pragma unroll
        for (int k = 0; k <= kj; ++k) {
            if (k == kj && lj == 0) continue;
            const double fji = (k < kj || l < lj) ? f[colbase[k] + j] : 0.0;
            r[k] = fma(-fji, vj, r[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < RPL; ++k) {
        const int i = k * LPB + l;
        r[k] *= f[colbase[k] + i];  // the diagonal slot holds 1 / l_ii
    }
}

// Programmatic dependent launch.  Every kernel of the library calls pdl_trigger() first (lets the
// next kernel in the stream start its independent prologue while this grid drains) and pdl_wait()
// before its first access to memory that an earlier kernel in the stream may have written, and
// before its own first global write.  Both are no-ops when the kernel was launched without the
// PDL attribute.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Opt-in to more than 48 KB of dynamic shared memory, once per kernel AND per device (the attribute is per device).
template <typename K>
inline cudaError_t ensure_big_smem(K kernel, std::atomic<bool> (&done)[64])
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (done[dev].load(std::memory_order_acquire)) return cudaSuccess;  // the attribute call is idempotent: a race only repeats it
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 225 * 1024);
    if (e == cudaSuccess) done[dev].store(true, std::memory_order_release);
    return e;
}

// launch with the programmatic-stream-serialization attribute when `pdl` is set
template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                                 bool pdl, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

}  // namespace bj
