// bj_cond_estimate_noalloc: the Lanczos kappa estimate for callers that cannot allocate device memory at call time (code
// under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  It is the single-launch cluster
// kernel of bj_lanczos_cluster.cu with every byte of its global scratch -- the seeded start vector, alpha, beta and the
// status words that bj_cond_estimate_ex keeps in the handle's lazily allocated Lanczos workspace -- in ONE file-scope
// device array of fixed size.  The entry point calls no cudaMalloc / cudaFree / pool routine and no allocating library
// routine; the host side of the read-back lives on the stack.
//
// Limits (beyond them the call returns BJ_ERR_LIMIT): n <= BJ_NOALLOC_MAX_N (16384), iters <= BJ_NOALLOC_MAX_ITERS (1024),
// and a handle the cluster kernel accepts (uniform blocks b <= 8 or b = 0, dense packed factors, no permutation, a CTA's
// share of the basis fits its shared memory).  The array (147 488 bytes) is held by every GPU that loads the library
// until the process exits.
// Sharing: every call on a device uses the same array, and the array keeps the last call's contents -- alpha, beta and
// the status words are cleared on the stream at the start of each call; calls that overlap on the GPU (two handles on two
// streams of one device) race on it.  The call synchronises its stream before it returns.
#include <string.h>

#include <atomic>

#include "bj_internal.cuh"

#define BJ_CHECK_H(h) do { if (!(h) || (h)->failed) return BJ_ERR_INVALID_ARG; } while (0)

namespace bj {

namespace {

struct NoAllocScratch {
    double v0[BJ_NOALLOC_MAX_N];         // seeded start vector (unused when the caller passes one)
    double alpha[BJ_NOALLOC_MAX_ITERS];
    double beta[BJ_NOALLOC_MAX_ITERS];
    int done[8];                         // [0] stop flag, [1] m_eff, [2] invalid start vector
};

// In host code this name is a host-side stand-in, not a device address: only cudaGetSymbolAddress turns it into one.
static __device__ __align__(256) unsigned char g_noalloc_scratch[sizeof(NoAllocScratch)];

// the device address of the array, looked up once per device with that device current
int noalloc_scratch(NoAllocScratch** out)
{
    static NoAllocScratch* ptr[64];
    static std::atomic<bool> have[64];
    int dev = 0;
    BJ_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return BJ_ERR_INVALID_ARG;
    if (!have[dev].load(std::memory_order_acquire)) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            set_cuda_error(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
            return BJ_ERR_CUDA;
        }
        ptr[dev] = static_cast<NoAllocScratch*>(p);  // a race between two threads stores the same address twice
        have[dev].store(true, std::memory_order_release);
    }
    *out = ptr[dev];
    return BJ_OK;
}

}  // namespace

}  // namespace bj

extern "C" int bj_cond_estimate_noalloc(bj_handle_t h, const bj_lanczos_opts_t* o, bj_lanczos_result_t* res)
{
    using namespace bj;
    BJ_CHECK_H(h);
    if (!o || !res || o->iters < 1) return BJ_ERR_INVALID_ARG;
    const int m = o->iters;
    const bool reorth = o->reorth != 0;
    if (h->n > BJ_NOALLOC_MAX_N || m > BJ_NOALLOC_MAX_ITERS || !lanczos_cluster_usable(h, m, reorth)) return BJ_ERR_LIMIT;
    NoAllocScratch* s = nullptr;
    int rc = noalloc_scratch(&s);
    if (rc != BJ_OK) return rc;
    cudaStream_t st = h->stream;
    const double tol = o->breakdown_tol > 0.0 ? o->breakdown_tol : BJ_DEFAULT_BREAKDOWN_TOL;
    // the array keeps the last call's contents: everything the kernel only partly writes starts at zero
    BJ_CUDA(cudaMemsetAsync(s->alpha, 0, sizeof(s->alpha) + sizeof(s->beta) + sizeof(s->done), st));
    const double* v0 = o->v0;
    if (!v0) {
        rc = launch_seeded_vector(h, o->seed, s->v0);
        if (rc != BJ_OK) return rc;
        v0 = s->v0;
    }
    rc = launch_lanczos_cluster(h, m, reorth, tol, v0, s->alpha, s->beta, s->done);
    if (rc != BJ_OK) return rc;
    double a[BJ_NOALLOC_MAX_ITERS], b[BJ_NOALLOC_MAX_ITERS];  // host stack: 16 KB
    int done[8];
    BJ_CUDA(cudaMemcpyAsync(a, s->alpha, sizeof(double) * (size_t)m, cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaMemcpyAsync(b, s->beta, sizeof(double) * (size_t)m, cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaMemcpyAsync(done, s->done, sizeof(done), cudaMemcpyDeviceToHost, st));
    BJ_CUDA(cudaStreamSynchronize(st));
    if (done[2]) return BJ_ERR_INVALID_ARG;  // ||v0|| is zero or not finite
    const int me = done[1];
    if (me < 1) return BJ_ERR_CUDA;
    lanczos_fill_result(me, a, b, res);
    return BJ_OK;
}
