"""Thin Python binding of the C ABI in include/bj.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libbj.so; torch is used for device memory
and streams.  There is no CPU fallback: if the library is missing or no CUDA device is present
the calls raise.  Function names mirror the C entry points.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbj.so")

BJ_B_MAX = 32
BJ_DEFAULT_SEED = 0x241002408
BJ_OK, BJ_ERR_INVALID_ARG, BJ_ERR_NOT_CANONICAL, BJ_ERR_TOO_LARGE, BJ_ERR_NOT_SPD, BJ_ERR_ALLOC, BJ_ERR_CUDA = 0, -1, -2, -3, -4, -5, -6
BJ_ERR_LIMIT = -7
BJ_NOALLOC_MAX_N, BJ_NOALLOC_MAX_ITERS = 16384, 1024
BJ_K_SOLVE_LT, BJ_K_SPMV, BJ_K_SOLVE_L, BJ_K_APPLY, BJ_K_SPMV_SOLVE_L, BJ_K_COUNT = 0, 1, 2, 3, 4, 5
BJ_OPT_SPMV_KERNEL, BJ_OPT_FUSE_FORWARD, BJ_OPT_LANCZOS_FUSE, BJ_OPT_PCG_FUSE, BJ_OPT_LANCZOS_SINGLE_LAUNCH = 1, 2, 3, 4, 5
BJ_OPT_PCG_SINGLE_LAUNCH = 6
KERNEL_KIND_NAMES = ["solve_Lt", "spmv", "solve_L", "apply", "spmv_solve_L"]

EXPORTS = ["bj_setup", "bj_setup_on_stream", "bj_setup_ex", "bj_get_setup_time", "bj_set_stream", "bj_set_option", "bj_destroy", "bj_get_info",
           "bj_strerror", "bj_apply", "bj_spmv", "bj_solve_L", "bj_solve_Lt", "bj_op_apply", "bj_cond_estimate",
           "bj_cond_estimate_ex", "bj_seeded_vector", "bj_op_apply_host", "bj_apply_host", "bj_profile_enable",
           "bj_profile_get", "bj_release_cached_memory", "bj_pcg_solve",
           "bj_cond_estimate_batch", "bj_pcg_solve_batch", "bj_cond_estimate_minv", "bj_setup_blocks", "bj_setup_perm",
           "bj_setup_blocks_perm", "bj_cond_estimate_noalloc"]


class bj_csr_t(C.Structure):
    _fields_ = [("n", C.c_int64), ("nnz", C.c_int64), ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p),
                ("val", C.c_void_p)]


class bj_setup_opts_t(C.Structure):
    _fields_ = [("cuda_stream", C.c_void_p), ("band", C.c_int32), ("col16", C.c_int32), ("bsr", C.c_int32),
                ("serp_keep_mb", C.c_int32), ("reserved", C.c_int32 * 8)]


class bj_lanczos_opts_t(C.Structure):
    _fields_ = [("iters", C.c_int32), ("reorth", C.c_int32), ("seed", C.c_uint64), ("v0", C.c_void_p),
                ("breakdown_tol", C.c_double)]


class bj_lanczos_result_t(C.Structure):
    _fields_ = [("iters_done", C.c_int32), ("lmin", C.c_double), ("lmax", C.c_double), ("res_min", C.c_double),
                ("res_max", C.c_double), ("alpha_host", C.c_void_p), ("beta_host", C.c_void_p)]


class bj_pcg_opts_t(C.Structure):
    _fields_ = [("max_iters", C.c_int32), ("check_every", C.c_int32), ("rtol", C.c_double)]


class bj_pcg_result_t(C.Structure):
    _fields_ = [("iters", C.c_int32), ("converged", C.c_int32), ("relres", C.c_double), ("true_relres", C.c_double),
                ("lmin", C.c_double), ("lmax", C.c_double), ("alpha_host", C.c_void_p), ("beta_host", C.c_void_p),
                ("relres_host", C.c_void_p)]


class bj_info_t(C.Structure):
    _fields_ = [("n", C.c_int64), ("nnz", C.c_int64), ("b", C.c_int32), ("nblocks", C.c_int64),
                ("bad_block", C.c_int64), ("factor_bytes", C.c_int64), ("workspace_bytes", C.c_int64),
                ("kernel_launches", C.c_int64), ("spmv_kernel", C.c_int32), ("spmv_lanes", C.c_int32),
                ("solve_kernel", C.c_int32), ("fused_forward", C.c_int32), ("band_width", C.c_int32), ("col16", C.c_int32),
                ("permuted", C.c_int32)]


class BJError(RuntimeError):
    def __init__(self, code: int, msg: str, bad_block: int = -1):
        super().__init__(f"bj error {code}: {msg}")
        self.code = code
        self.bad_block = bad_block


_lib = None


def lib():
    """Load libbj.so (built in-tree by `python -m paper_2410_02408_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2410_02408_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int, C.c_int64
        L.bj_setup.argtypes = [C.POINTER(bj_csr_t), i32, C.POINTER(vp)]
        L.bj_setup_on_stream.argtypes = [C.POINTER(bj_csr_t), i32, vp, C.POINTER(vp)]
        L.bj_setup_ex.argtypes = [C.POINTER(bj_csr_t), i32, C.POINTER(bj_setup_opts_t), C.POINTER(vp)]
        L.bj_get_setup_time.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i64)]
        L.bj_cond_estimate_minv.argtypes = [vp, C.POINTER(bj_lanczos_opts_t), C.POINTER(bj_lanczos_result_t)]
        L.bj_cond_estimate_noalloc.argtypes = [vp, C.POINTER(bj_lanczos_opts_t), C.POINTER(bj_lanczos_result_t)]
        L.bj_setup_blocks.argtypes = [C.POINTER(bj_csr_t), vp, i64, vp, C.POINTER(vp)]
        L.bj_setup_perm.argtypes = [C.POINTER(bj_csr_t), i32, vp, vp, C.POINTER(vp)]
        L.bj_setup_blocks_perm.argtypes = [C.POINTER(bj_csr_t), vp, i64, vp, vp, C.POINTER(vp)]
        L.bj_set_stream.argtypes = [vp, vp]
        L.bj_set_option.argtypes = [vp, i32, i32]
        L.bj_destroy.argtypes = [vp]
        L.bj_get_info.argtypes = [vp, C.POINTER(bj_info_t)]
        L.bj_strerror.argtypes = [i32]
        L.bj_strerror.restype = C.c_char_p
        for f in ("bj_apply", "bj_spmv", "bj_solve_L", "bj_solve_Lt", "bj_op_apply", "bj_op_apply_host", "bj_apply_host"):
            getattr(L, f).argtypes = [vp, vp, vp]
        L.bj_cond_estimate.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.bj_cond_estimate_ex.argtypes = [vp, C.POINTER(bj_lanczos_opts_t), C.POINTER(bj_lanczos_result_t)]
        L.bj_seeded_vector.argtypes = [vp, C.c_uint64, vp]
        L.bj_pcg_solve.argtypes = [vp, vp, vp, C.POINTER(bj_pcg_opts_t), C.POINTER(bj_pcg_result_t)]
        L.bj_release_cached_memory.argtypes = []
        L.bj_cond_estimate_batch.argtypes = [vp, i64, vp, i32, C.c_uint64, vp, vp, vp]
        L.bj_pcg_solve_batch.argtypes = [vp, i64, vp, vp, vp, i32, C.c_double, vp, vp, vp]
        L.bj_profile_enable.argtypes = [vp, i32]
        L.bj_profile_get.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(i64)]
        for f in EXPORTS:
            if f != "bj_strerror":
                getattr(L, f).restype = i32
        _lib = L
    return _lib


def bj_strerror(code: int) -> str:
    return lib().bj_strerror(code).decode()


def _check(code: int, bad_block: int = -1):
    if code != BJ_OK:
        raise BJError(code, bj_strerror(code), bad_block)


def _dptr(t, dtype, n=None):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"expected a contiguous CUDA tensor of dtype {dtype}")
    if n is not None and t.numel() < n:
        raise ValueError("tensor too short")
    return C.c_void_p(t.data_ptr())


class Handle:
    """Owns a bj_handle_t.  Keeps references to the borrowed CSR tensors so they outlive it."""

    def __init__(self, ptr, keep, n):
        self.ptr, self._keep, self.n = ptr, keep, n

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def destroy(self):
        if self.ptr is not None:
            lib().bj_destroy(self.ptr)
            self.ptr = None


def bj_setup(row_ptr, col_idx, val, b: int, stream=None, band: int = 0, col16: int = 0, bsr: int = 0,
             serp_keep_mb: int = 0) -> Handle:
    """row_ptr/col_idx: int32 CUDA tensors, val: float64 CUDA tensor (borrowed).  stream: a torch stream,
    default the current one.  The keyword options are the fields of bj_setup_opts_t (bj_setup_ex)."""
    import torch
    n = row_ptr.numel() - 1
    nnz = val.numel()
    csr = bj_csr_t(n, nnz, _dptr(row_ptr, torch.int32), _dptr(col_idx, torch.int32, nnz), _dptr(val, torch.float64))
    st = (stream or torch.cuda.current_stream()).cuda_stream
    opts = bj_setup_opts_t(C.c_void_p(st), int(band), int(col16), int(bsr), int(serp_keep_mb))
    out = C.c_void_p()
    code = lib().bj_setup_ex(C.byref(csr), int(b), C.byref(opts), C.byref(out))
    if code == BJ_ERR_NOT_SPD and out.value:
        info = bj_info_t()
        lib().bj_get_info(out, C.byref(info))
        lib().bj_destroy(out)
        _check(code, int(info.bad_block))
    _check(code)
    return Handle(out, (row_ptr, col_idx, val), n)


def bj_get_setup_time(h: Handle) -> dict:
    """Device milliseconds of this handle's setup kernels and the bytes they must move."""
    ms, nb = C.c_double(), C.c_int64()
    _check(lib().bj_get_setup_time(h.ptr, C.byref(ms), C.byref(nb)))
    return {"kernel_ms": ms.value, "algorithmic_bytes": nb.value}


def bj_setup_blocks(row_ptr, col_idx, val, block_ptr, stream=None) -> Handle:
    """Variable-size diagonal blocks: block_ptr = host int64 sequence 0 = p_0 < .. < p_nblocks = n, sizes 1..32."""
    import numpy as np
    import torch
    n = row_ptr.numel() - 1
    nnz = val.numel()
    ptr = np.ascontiguousarray(np.asarray(block_ptr, dtype=np.int64))
    csr = bj_csr_t(n, nnz, _dptr(row_ptr, torch.int32), _dptr(col_idx, torch.int32, nnz), _dptr(val, torch.float64))
    st = (stream or torch.cuda.current_stream()).cuda_stream
    out = C.c_void_p()
    code = lib().bj_setup_blocks(C.byref(csr), ptr.ctypes.data_as(C.c_void_p), C.c_int64(len(ptr) - 1), C.c_void_p(st), C.byref(out))
    if code == BJ_ERR_NOT_SPD and out.value:
        info = bj_info_t()
        lib().bj_get_info(out, C.byref(info))
        lib().bj_destroy(out)
        _check(code, int(info.bad_block))
    _check(code)
    return Handle(out, (row_ptr, col_idx, val), n)


def bj_setup_perm(row_ptr, col_idx, val, b: int, perm, block_ptr=None, stream=None) -> Handle:
    """Block-Jacobi after a symmetric permutation: perm = int32 CUDA tensor, perm[i] = original index of the unknown at
    permuted position i; vectors stay in the original ordering.  block_ptr (host int64 sequence, optional): block sizes
    1..32 in the permuted ordering instead of the uniform b."""
    import numpy as np
    import torch
    n = row_ptr.numel() - 1
    nnz = val.numel()
    csr = bj_csr_t(n, nnz, _dptr(row_ptr, torch.int32), _dptr(col_idx, torch.int32, nnz), _dptr(val, torch.float64))
    st = (stream or torch.cuda.current_stream()).cuda_stream
    out = C.c_void_p()
    pp = _dptr(perm, torch.int32, n)
    if block_ptr is None:
        code = lib().bj_setup_perm(C.byref(csr), int(b), pp, C.c_void_p(st), C.byref(out))
    else:
        ptr = np.ascontiguousarray(np.asarray(block_ptr, dtype=np.int64))
        code = lib().bj_setup_blocks_perm(C.byref(csr), ptr.ctypes.data_as(C.c_void_p), C.c_int64(len(ptr) - 1), pp,
                                          C.c_void_p(st), C.byref(out))
    if code == BJ_ERR_NOT_SPD and out.value:
        info = bj_info_t()
        lib().bj_get_info(out, C.byref(info))
        lib().bj_destroy(out)
        _check(code, int(info.bad_block))
    _check(code)
    return Handle(out, (row_ptr, col_idx, val), n)


def bj_set_stream(h: Handle, stream):
    _check(lib().bj_set_stream(h.ptr, C.c_void_p(stream.cuda_stream)))


def bj_set_option(h: Handle, option: int, value: int):
    _check(lib().bj_set_option(h.ptr, option, value))


def bj_destroy(h: Handle):
    h.destroy()


def bj_get_info(h: Handle) -> dict:
    info = bj_info_t()
    _check(lib().bj_get_info(h.ptr, C.byref(info)))
    return {k: getattr(info, k) for k, _ in bj_info_t._fields_}


def _vec_call(name, h, a, out):
    import torch
    if out is None:
        out = torch.empty_like(a)
    _check(getattr(lib(), name)(h.ptr, _dptr(a, torch.float64, h.n), _dptr(out, torch.float64, h.n)))
    return out


def bj_apply(h, r, z=None):
    return _vec_call("bj_apply", h, r, z)


def bj_spmv(h, x, y=None):
    return _vec_call("bj_spmv", h, x, y)


def bj_solve_L(h, r, y=None):
    return _vec_call("bj_solve_L", h, r, y)


def bj_solve_Lt(h, y, x=None):
    return _vec_call("bj_solve_Lt", h, y, x)


def bj_op_apply(h, x, y=None):
    return _vec_call("bj_op_apply", h, x, y)


def _host_call(name, h, a, out):
    import torch
    for t in (a, out):
        if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or t.numel() < h.n:
            raise TypeError("expected contiguous float64 HOST tensors of length n")
    _check(getattr(lib(), name)(h.ptr, C.c_void_p(a.data_ptr()), C.c_void_p(out.data_ptr())))
    return out


def bj_op_apply_host(h, x_host, y_host):
    return _host_call("bj_op_apply_host", h, x_host, y_host)


def bj_apply_host(h, r_host, z_host):
    return _host_call("bj_apply_host", h, r_host, z_host)


def bj_cond_estimate(h, iters: int):
    lmin, lmax = C.c_double(), C.c_double()
    _check(lib().bj_cond_estimate(h.ptr, int(iters), C.byref(lmin), C.byref(lmax)))
    return lmin.value, lmax.value


def bj_cond_estimate_ex(h, iters: int, reorth: bool = True, seed: int = BJ_DEFAULT_SEED, v0=None,
                        breakdown_tol: float = 0.0) -> dict:
    import numpy as np
    import torch
    alpha = np.zeros(iters)
    beta = np.zeros(iters)
    o = bj_lanczos_opts_t(int(iters), int(bool(reorth)), seed & 0xFFFFFFFFFFFFFFFF,
                          _dptr(v0, torch.float64, h.n) if v0 is not None else None, breakdown_tol)
    r = bj_lanczos_result_t(0, 0.0, 0.0, 0.0, 0.0, alpha.ctypes.data_as(C.c_void_p), beta.ctypes.data_as(C.c_void_p))
    _check(lib().bj_cond_estimate_ex(h.ptr, C.byref(o), C.byref(r)))
    k = r.iters_done
    return {"iters_done": k, "lmin": r.lmin, "lmax": r.lmax, "kappa": r.lmax / r.lmin, "res_min": r.res_min,
            "res_max": r.res_max, "alpha": alpha[:k].copy(), "beta": beta[:k].copy()}


def bj_cond_estimate_noalloc(h, iters: int, reorth: bool = True, seed: int = BJ_DEFAULT_SEED, v0=None,
                             breakdown_tol: float = 0.0) -> dict:
    """bj_cond_estimate_ex without any device allocation at call time (fixed file-scope device scratch; BJ_ERR_LIMIT beyond
    n <= 16384, iters <= 1024, b <= 8).  Calls that overlap on one GPU race on the scratch."""
    import numpy as np
    import torch
    alpha = np.zeros(iters)
    beta = np.zeros(iters)
    o = bj_lanczos_opts_t(int(iters), int(bool(reorth)), seed & 0xFFFFFFFFFFFFFFFF,
                          _dptr(v0, torch.float64, h.n) if v0 is not None else None, breakdown_tol)
    r = bj_lanczos_result_t(0, 0.0, 0.0, 0.0, 0.0, alpha.ctypes.data_as(C.c_void_p), beta.ctypes.data_as(C.c_void_p))
    _check(lib().bj_cond_estimate_noalloc(h.ptr, C.byref(o), C.byref(r)))
    k = r.iters_done
    return {"iters_done": k, "lmin": r.lmin, "lmax": r.lmax, "kappa": r.lmax / r.lmin, "res_min": r.res_min,
            "res_max": r.res_max, "alpha": alpha[:k].copy(), "beta": beta[:k].copy()}


def bj_cond_estimate_minv(h, iters: int, seed: int = BJ_DEFAULT_SEED, r0=None, breakdown_tol: float = 0.0) -> dict:
    """Lanczos on M^-1 A in the M inner product (one factor pass per step); same result fields as bj_cond_estimate_ex."""
    import numpy as np
    import torch
    alpha = np.zeros(iters)
    beta = np.zeros(iters)
    o = bj_lanczos_opts_t(int(iters), 0, seed & 0xFFFFFFFFFFFFFFFF,
                          _dptr(r0, torch.float64, h.n) if r0 is not None else None, breakdown_tol)
    r = bj_lanczos_result_t(0, 0.0, 0.0, 0.0, 0.0, alpha.ctypes.data_as(C.c_void_p), beta.ctypes.data_as(C.c_void_p))
    _check(lib().bj_cond_estimate_minv(h.ptr, C.byref(o), C.byref(r)))
    k = r.iters_done
    return {"iters_done": k, "lmin": r.lmin, "lmax": r.lmax, "kappa": r.lmax / r.lmin, "res_min": r.res_min,
            "res_max": r.res_max, "alpha": alpha[:k].copy(), "beta": beta[:k].copy()}


def bj_pcg_solve(h, b, x=None, max_iters: int = 1000, rtol: float = 1e-3, check_every: int = 0) -> dict:
    """Preconditioned CG for A x = b from x0 = 0 (rtol defaults to the paper's accuracy bar)."""
    import numpy as np
    import torch
    if x is None:
        x = torch.empty(h.n, dtype=torch.float64, device=b.device)
    alpha, beta, rel = np.zeros(max_iters), np.zeros(max_iters), np.zeros(max_iters)
    o = bj_pcg_opts_t(int(max_iters), int(check_every), float(rtol))
    r = bj_pcg_result_t(0, 0, 0.0, 0.0, 0.0, 0.0, alpha.ctypes.data_as(C.c_void_p), beta.ctypes.data_as(C.c_void_p),
                        rel.ctypes.data_as(C.c_void_p))
    _check(lib().bj_pcg_solve(h.ptr, _dptr(b, torch.float64, h.n), _dptr(x, torch.float64, h.n), C.byref(o), C.byref(r)))
    k = r.iters
    nb = k - 1 if (k > 0 and r.converged) else k
    return {"x": x, "iters": k, "converged": bool(r.converged), "relres": r.relres, "true_relres": r.true_relres,
            "lmin": r.lmin, "lmax": r.lmax, "alpha": alpha[:k].copy(), "beta": beta[:max(nb, 0)].copy(),
            "relres_hist": rel[:k].copy()}


def bj_seeded_vector(h, seed: int, v=None):
    import torch
    if v is None:
        v = torch.empty(h.n, dtype=torch.float64, device="cuda")
    _check(lib().bj_seeded_vector(h.ptr, seed & 0xFFFFFFFFFFFFFFFF, _dptr(v, torch.float64, h.n)))
    return v


def _offsets_arg(offsets, nsys):
    import numpy as np
    if offsets is None:
        return None, None
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    if off.shape != (nsys + 1,):
        raise ValueError("offsets must have nsys + 1 entries")
    return off, off.ctypes.data_as(C.c_void_p)


def bj_cond_estimate_batch(h, nsys: int, iters: int, seed: int = BJ_DEFAULT_SEED, offsets=None) -> dict:
    """Per-system Lanczos extremes of a batch of `nsys` systems stored as one block-diagonal CSR (equal sizes, or
    `offsets` = nsys + 1 row offsets)."""
    import numpy as np
    lmin, lmax = np.zeros(nsys), np.zeros(nsys)
    done = np.zeros(nsys, dtype=np.int32)
    keep, offp = _offsets_arg(offsets, nsys)
    _check(lib().bj_cond_estimate_batch(h.ptr, int(nsys), offp, int(iters), seed & 0xFFFFFFFFFFFFFFFF, lmin.ctypes.data_as(C.c_void_p),
                                        lmax.ctypes.data_as(C.c_void_p), done.ctypes.data_as(C.c_void_p)))
    return {"lmin": lmin, "lmax": lmax, "kappa": lmax / lmin, "iters_done": done}


def bj_pcg_solve_batch(h, nsys: int, b, x=None, max_iters: int = 1000, rtol: float = 1e-3, offsets=None) -> dict:
    """PCG on every system of a batch at once (per-system scalars and stopping tests)."""
    import numpy as np
    import torch
    if x is None:
        x = torch.empty(h.n, dtype=torch.float64, device=b.device)
    it = np.zeros(nsys, dtype=np.int32)
    rel, trel = np.zeros(nsys), np.zeros(nsys)
    keep, offp = _offsets_arg(offsets, nsys)
    _check(lib().bj_pcg_solve_batch(h.ptr, int(nsys), offp, _dptr(b, torch.float64, h.n), _dptr(x, torch.float64, h.n), int(max_iters),
                                    float(rtol), it.ctypes.data_as(C.c_void_p), rel.ctypes.data_as(C.c_void_p),
                                    trel.ctypes.data_as(C.c_void_p)))
    return {"x": x, "iters": it, "relres": rel, "true_relres": trel}


def bj_release_cached_memory():
    _check(lib().bj_release_cached_memory())


def bj_profile_enable(h, on: bool):
    _check(lib().bj_profile_enable(h.ptr, int(bool(on))))


def bj_profile_get(h, kind: int):
    ms, cnt = C.c_double(), C.c_int64()
    _check(lib().bj_profile_get(h.ptr, kind, C.byref(ms), C.byref(cnt)))
    return ms.value, cnt.value


def setup_from_host(A, b: int, device="cuda", **opts):
    """Convenience: copy a workloads.CSR to the device and set up (opts: the keyword options of bj_setup).
    Returns (handle, (rp, ci, val))."""
    import torch
    rp = torch.from_numpy(A.row_ptr).to(device)
    ci = torch.from_numpy(A.col_idx).to(device)
    val = torch.from_numpy(A.val).to(device)
    return bj_setup(rp, ci, val, b, **opts), (rp, ci, val)
