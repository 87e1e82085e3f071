"""CPU oracle -- TEST INFRASTRUCTURE, not the product.

ctypes wrapper around `bj_oracle.c` (plain fp64 C written from the paper; see that file's
header for citations, build flags and the list of pins) plus a dense numpy path (`dense.py`).
Nothing here imports, links or shares code with the CUDA path.  Allowed callers: `tests/`,
`__graft_entry__.smoke()`, and `bench.py`'s `cpu_baseline` / `--impl reference` legs.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bj_oracle.c")
_LIB = os.path.join(_HERE, "libbj_oracle.so")
DEFAULT_SEED = 0x2410_02408
TOL_BREAKDOWN = 1e-12

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-fopenmp", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(_LIB)
        i64, i32, dbl, vp = C.c_int64, C.c_int, C.c_double, C.c_void_p
        lib.orc_spmv.argtypes = [i64, vp, vp, vp, vp, vp]
        lib.orc_extract.argtypes = [i64, vp, vp, vp, i64, vp]
        lib.orc_factor.argtypes = [i64, i64, vp, C.POINTER(i64)]
        lib.orc_factor.restype = i32
        lib.orc_solve_L.argtypes = [i64, i64, vp, vp, vp]
        lib.orc_solve_Lt.argtypes = [i64, i64, vp, vp, vp]
        lib.orc_apply.argtypes = [i64, i64, vp, vp, vp, vp]
        lib.orc_op_apply.argtypes = [i64, vp, vp, vp, i64, vp, vp, vp, vp]
        lib.orc_seeded_vector.argtypes = [C.c_uint64, i64, vp]
        lib.orc_lanczos.argtypes = [i64, vp, vp, vp, i64, vp, vp, i32, i32, dbl, vp, vp, C.POINTER(i32)]
        lib.orc_lanczos.restype = i32
        lib.orc_tridiag_extremes.argtypes = [i32, vp, vp] + [C.POINTER(dbl)] * 4
        lib.orc_tridiag_all.argtypes = [i32, vp, vp, vp]
        lib.orc_num_threads.restype = i32
        lib.orc_pcg.argtypes = [i64, vp, vp, vp, i64, vp, vp, vp, i32, dbl, vp, vp, vp, C.POINTER(i32), C.POINTER(dbl)]
        lib.orc_pcg.restype = i32
        for f in ("orc_spmv", "orc_extract", "orc_solve_L", "orc_solve_Lt", "orc_apply", "orc_op_apply",
                  "orc_seeded_vector", "orc_tridiag_extremes", "orc_tridiag_all"):
            getattr(lib, f).restype = None
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(_load().orc_num_threads())


class NotSPD(Exception):
    def __init__(self, bad_block: int):
        super().__init__(f"diagonal block {bad_block} is not positive definite")
        self.bad_block = bad_block


def spmv(A, x):
    x = _f64(x)
    y = np.empty(A.n)
    _load().orc_spmv(A.n, _p(A.row_ptr), _p(A.col_idx), _p(A.val), _p(x), _p(y))
    return y


def extract(A, b: int) -> np.ndarray:
    nblocks = (A.n + b - 1) // b
    D = np.empty((nblocks, b, b))
    _load().orc_extract(A.n, _p(A.row_ptr), _p(A.col_idx), _p(A.val), b, _p(D))
    return D


def factor(n: int, b: int, D: np.ndarray) -> np.ndarray:
    L = _f64(D).copy()
    bad = C.c_int64(-1)
    rc = _load().orc_factor(n, b, _p(L), C.byref(bad))
    if rc != 0:
        raise NotSPD(int(bad.value))
    return L


class Precond:
    """setup(A, b): extract + factor.  b == 0: identity (operator = A)."""

    def __init__(self, A, b: int):
        self.A, self.b, self.n = A, int(b), A.n
        self.L = factor(A.n, b, extract(A, b)) if b > 0 else None
        self._tmp = np.empty(2 * A.n)

    def solve_L(self, r):
        r = _f64(r); y = np.empty(self.n)
        _load().orc_solve_L(self.n, self.b, _p(self.L), _p(r), _p(y))
        return y

    def solve_Lt(self, y):
        y = _f64(y); x = np.empty(self.n)
        _load().orc_solve_Lt(self.n, self.b, _p(self.L), _p(y), _p(x))
        return x

    def apply(self, r):
        r = _f64(r); z = np.empty(self.n)
        _load().orc_apply(self.n, self.b, _p(self.L), _p(r), _p(z), _p(self._tmp))
        return z

    def op_apply(self, x):
        x = _f64(x); y = np.empty(self.n)
        A = self.A
        Lp = _p(self.L) if self.L is not None else None
        _load().orc_op_apply(self.n, _p(A.row_ptr), _p(A.col_idx), _p(A.val), self.b, Lp, _p(x), _p(y), _p(self._tmp))
        return y

    def lanczos(self, m: int, v0=None, reorth: bool = True, seed: int = DEFAULT_SEED, tol_bd: float = TOL_BREAKDOWN):
        v0 = seeded_vector(seed, self.n) if v0 is None else _f64(v0)
        alpha = np.zeros(m); beta = np.zeros(m)
        m_eff = C.c_int(0)
        A = self.A
        Lp = _p(self.L) if self.L is not None else None
        rc = _load().orc_lanczos(self.n, _p(A.row_ptr), _p(A.col_idx), _p(A.val), self.b, Lp, _p(v0), m,
                                 int(bool(reorth)), tol_bd, _p(alpha), _p(beta), C.byref(m_eff))
        if rc != 0:
            raise MemoryError("oracle lanczos allocation failed")
        k = m_eff.value
        return alpha[:k].copy(), beta[:k].copy()

    def pcg(self, rhs, max_iters: int, rtol: float):
        """Preconditioned CG from x0 = 0; returns x and the iteration record."""
        rhs = _f64(rhs)
        x = np.empty(self.n)
        alpha = np.zeros(max_iters); beta = np.zeros(max_iters); relres = np.zeros(max_iters)
        it = C.c_int(0); tr = C.c_double(0.0)
        A = self.A
        Lp = _p(self.L) if self.L is not None else None
        rc = _load().orc_pcg(self.n, _p(A.row_ptr), _p(A.col_idx), _p(A.val), self.b, Lp, _p(rhs), _p(x), int(max_iters),
                             float(rtol), _p(alpha), _p(beta), _p(relres), C.byref(it), C.byref(tr))
        if rc != 0:
            raise MemoryError("oracle pcg allocation failed")
        k = it.value
        nb = k - 1 if (k > 0 and relres[k - 1] <= rtol) else k
        return {"x": x, "iters": k, "alpha": alpha[:k].copy(), "beta": beta[:max(nb, 0)].copy(),
                "relres": relres[:k].copy(), "true_relres": tr.value}

    def lanczos_minv(self, m: int, r0=None, seed: int = DEFAULT_SEED, tol_bd: float = TOL_BREAKDOWN, return_basis: bool = False):
        """Lanczos on M^-1 A in the M inner product ("the M^-1 A formulation (same spectrum)"): ONE pass
        over the factor per step instead of the two of L^-1 A L^-T.  With u_j M-orthonormal and rh_j = M u_j the three-term
        recurrence  M^-1 A u_j = bt_{j+1} u_{j+1} + al_j u_j + bt_j u_{j-1}  reads, multiplied by M,
            r_{j+1} = A u_j - al_j rh_j - bt_j rh_{j-1},   al_j = u_j . A u_j,
            z_{j+1} = M^-1 r_{j+1},   bt_{j+1} = sqrt(r_{j+1} . z_{j+1}),   u_{j+1} = z_{j+1} / bt_{j+1},  rh_{j+1} = r_{j+1} / bt_{j+1},
        started from r_0 (seeded vector), z_0 = M^-1 r_0, bt_0 = sqrt(r_0 . z_0) (a normalisation, not an entry of T).
        T = tridiag(bt_1..; al_0..) is the Lanczos matrix of L^-1 A L^-T started at L^-1 r_0 (same spectrum: A^ = L^-1 A L^-T
        is similar to M^-1 A).  No reorthogonalisation.  Same breakdown rule as lanczos().  b = 0: M = I.
        Returns (alpha[0..k-1], beta[0..k-1]) with beta[j] = bt_{j+1}, like lanczos()."""
        r = seeded_vector(seed, self.n) if r0 is None else _f64(r0).copy()
        minv = (lambda v: self.apply(v)) if self.b > 0 else (lambda v: v.copy())
        z = minv(r)
        bt = float(np.sqrt(np.dot(r, z)))
        rh_prev = np.zeros(self.n)
        bt_j = 0.0
        alpha, beta, U = [], [], []
        amax = 0.0
        for j in range(m):
            u = z / bt
            rh = r / bt
            if return_basis:
                U.append(u)
            p = spmv(self.A, u)
            a = float(np.dot(u, p))
            rn = p - a * rh - bt_j * rh_prev
            zn = minv(rn)
            bn = float(np.sqrt(max(np.dot(rn, zn), 0.0)))
            alpha.append(a); beta.append(bn)
            amax = max(amax, abs(a))
            if not (bn > tol_bd * amax):
                break
            rh_prev, bt_j = rh, bn
            r, z, bt = rn, zn, bn
        out = (np.array(alpha), np.array(beta))
        return out + (np.array(U).T,) if return_basis else out

    def cond_estimate_minv(self, m: int, **kw):
        alpha, beta = self.lanczos_minv(m, **kw)
        tmin, tmax, rmin, rmax = tridiag_extremes(alpha, beta)
        return {"lmin": tmin, "lmax": tmax, "kappa": tmax / tmin, "res_min": rmin, "res_max": rmax,
                "iters_done": len(alpha), "alpha": alpha, "beta": beta}

    def cond_estimate(self, m: int, **kw):
        alpha, beta = self.lanczos(m, **kw)
        tmin, tmax, rmin, rmax = tridiag_extremes(alpha, beta)
        return {"lmin": tmin, "lmax": tmax, "kappa": tmax / tmin, "res_min": rmin, "res_max": rmax,
                "iters_done": len(alpha), "alpha": alpha, "beta": beta}


def cg_tridiag(alpha, beta):
    """Lanczos tridiagonal of M^-1 A implied by k CG steps (CG-Lanczos equivalence): diagonal
    d_0 = 1/a_0, d_j = 1/a_j + bt_{j-1}/a_{j-1}; off-diagonal e_j = sqrt(bt_j)/a_j, j = 0..k-2."""
    a, bt = _f64(alpha), _f64(beta)
    k = len(a)
    d = np.empty(k)
    for j in range(k):
        d[j] = 1.0 / a[j] + (bt[j - 1] / a[j - 1] if j > 0 else 0.0)
    e = np.array([np.sqrt(bt[j]) / a[j] for j in range(k - 1)])
    return d, e


def seeded_vector(seed: int, n: int) -> np.ndarray:
    v = np.empty(n)
    _load().orc_seeded_vector(C.c_uint64(seed & 0xFFFFFFFFFFFFFFFF), n, _p(v))
    return v


def tridiag_extremes(alpha, beta):
    alpha, beta = _f64(alpha), _f64(beta)
    out = [C.c_double() for _ in range(4)]
    _load().orc_tridiag_extremes(len(alpha), _p(alpha), _p(beta), *[C.byref(o) for o in out])
    return tuple(o.value for o in out)


def tridiag_all(alpha, beta) -> np.ndarray:
    alpha, beta = _f64(alpha), _f64(beta)
    out = np.empty(len(alpha))
    _load().orc_tridiag_all(len(alpha), _p(alpha), _p(beta), _p(out))
    return out


class PrecondBlocks:
    """Block-Jacobi with diagonal blocks of DIFFERENT sizes ("variable-size / supervariable blocks").
    block_ptr[0..nblocks] (0 = p_0 < p_1 < .. = n) delimits contiguous index ranges; block k is the dense diagonal slice
    D_k = A[p_k:p_{k+1}, p_k:p_{k+1}] (the listing of PAPER.md:254-263 with a per-block size), factored D_k = L_k L_k^T and
    solved block by block -- every step is the uniform-size routine of bj_oracle.c called on ONE block (n = b = s_k), so
    the arithmetic and its order are exactly those of Precond.  Slow (a Python loop over blocks): small cases only."""

    def __init__(self, A, block_ptr):
        self.A, self.n = A, A.n
        p = np.asarray(block_ptr, dtype=np.int64)
        if p[0] != 0 or p[-1] != A.n or np.any(np.diff(p) <= 0):
            raise ValueError("block_ptr must increase strictly from 0 to n")
        self.ptr = p
        rp, ci, val = A.row_ptr, A.col_idx, A.val
        self.L = []
        for k in range(len(p) - 1):
            lo, hi = int(p[k]), int(p[k + 1])
            D = np.zeros((hi - lo, hi - lo))
            for i in range(lo, hi):
                for e in range(int(rp[i]), int(rp[i + 1])):
                    c = int(ci[e])
                    if lo <= c < hi:
                        D[i - lo, c - lo] = val[e]
            try:
                self.L.append(factor(hi - lo, hi - lo, D.reshape(1, hi - lo, hi - lo)))
            except NotSPD:
                raise NotSPD(k)

    def _blockwise(self, fn, v):
        v = _f64(v); out = np.empty(self.n)
        for k, L in enumerate(self.L):
            lo, hi = int(self.ptr[k]), int(self.ptr[k + 1])
            seg = np.ascontiguousarray(v[lo:hi]); res = np.empty(hi - lo)
            fn(hi - lo, hi - lo, _p(L), _p(seg), _p(res))
            out[lo:hi] = res
        return out

    def solve_L(self, r):
        return self._blockwise(_load().orc_solve_L, r)

    def solve_Lt(self, y):
        return self._blockwise(_load().orc_solve_Lt, y)

    def apply(self, r):
        return self.solve_Lt(self.solve_L(r))

    def op_apply(self, x):
        return self.solve_L(spmv(self.A, self.solve_Lt(x)))

    def lanczos(self, m: int, v0=None, reorth: bool = True, seed: int = DEFAULT_SEED, tol_bd: float = TOL_BREAKDOWN):
        """The recurrence of orc_lanczos (bj_oracle.c), statement by statement, on this operator."""
        v0 = seeded_vector(seed, self.n) if v0 is None else _f64(v0)
        V = [v0 / np.sqrt(np.dot(v0, v0))]
        alpha, beta = [], []
        beta_j, amax = 0.0, 0.0
        for j in range(m):
            w = self.op_apply(V[j])
            if j > 0:
                w = w - beta_j * V[j - 1]
            a = float(np.dot(V[j], w))
            w = w - a * V[j]
            if reorth:
                for _ in range(2):
                    c = [float(np.dot(V[q], w)) for q in range(j + 1)]
                    for q in range(j + 1):
                        w = w - c[q] * V[q]
            bn = float(np.sqrt(np.dot(w, w)))
            alpha.append(a); beta.append(bn)
            amax = max(amax, abs(a))
            if not (bn > tol_bd * amax):
                break
            V.append(w / bn)
            beta_j = bn
        return np.array(alpha), np.array(beta)

    def cond_estimate(self, m: int, **kw):
        alpha, beta = self.lanczos(m, **kw)
        tmin, tmax, rmin, rmax = tridiag_extremes(alpha, beta)
        return {"lmin": tmin, "lmax": tmax, "kappa": tmax / tmin, "res_min": rmin, "res_max": rmax,
                "iters_done": len(alpha), "alpha": alpha, "beta": beta}


class _Csr:
    """The four fields the routines above read from a matrix object."""

    def __init__(self, n, row_ptr, col_idx, val):
        self.n, self.row_ptr, self.col_idx, self.val = int(n), row_ptr, col_idx, val


class PrecondPerm:
    """Block-Jacobi after a symmetric permutation of the unknowns ("a permutation argument (RCM or
    strong-coupling lines)"; the paper's partition into diagonal blocks, presupposes an ordering in which
    contiguous index ranges are the intended blocks -- DESIGN.md reading 8).
    perm[i] = original index of the unknown that sits at permuted position i, so (P v)[i] = v[perm[i]] and
    (P A P^T)[i, j] = A[perm[i], perm[j]].  The diagonal blocks are those of P A P^T:
        M = P^T blockdiag(D_k) P,   D_k = (P A P^T)[kb:(k+1)b, kb:(k+1)b] = L_k L_k^T,
    and EVERY vector argument stays in the ORIGINAL ordering:
        solve_L(r) = P^T L^-1 P r,  solve_Lt(y) = P^T L^-T P y,  apply = M^-1,  op_apply = solve_L . A . solve_Lt
    (= P^T [L^-1 (P A P^T) L^-T] P: orthogonally similar to the split operator of the permuted matrix, same spectrum).
    Written out as the definition: P A P^T is formed EXPLICITLY (scipy fancy indexing, a library primitive) and handed to
    Precond / PrecondBlocks; vectors are permuted on the way in and out.  No arithmetic of its own."""

    def __init__(self, A, perm, b: int | None = None, block_ptr=None):
        import scipy.sparse as sp
        p = np.asarray(perm, dtype=np.int64)
        if p.shape != (A.n,) or not np.array_equal(np.sort(p), np.arange(A.n)):
            raise ValueError("perm must be a permutation of 0..n-1")
        self.A, self.n, self.perm = A, A.n, p
        S = sp.csr_matrix((A.val, A.col_idx, A.row_ptr), shape=(A.n, A.n))
        Sp = S[p][:, p].tocsr()
        Sp.sum_duplicates()
        Sp.sort_indices()
        self.Ap = _Csr(A.n, Sp.indptr.astype(np.int32), Sp.indices.astype(np.int32), Sp.data.astype(np.float64))
        self.P = PrecondBlocks(self.Ap, block_ptr) if block_ptr is not None else Precond(self.Ap, int(b))

    def to_perm(self, v):
        return _f64(v)[self.perm]

    def from_perm(self, vp):
        out = np.empty(self.n)
        out[self.perm] = vp
        return out

    def solve_L(self, r):
        return self.from_perm(self.P.solve_L(self.to_perm(r)))

    def solve_Lt(self, y):
        return self.from_perm(self.P.solve_Lt(self.to_perm(y)))

    def apply(self, r):
        return self.from_perm(self.P.apply(self.to_perm(r)))

    def op_apply(self, x):
        return self.from_perm(self.P.op_apply(self.to_perm(x)))

    def cond_estimate(self, m: int, v0=None, seed: int = DEFAULT_SEED, **kw):
        """Lanczos on the operator in the original ordering started at v0 (default: the seeded vector, original ordering)
        = Lanczos on the split operator of P A P^T started at P v0: the same alpha, beta."""
        v0 = seeded_vector(seed, self.n) if v0 is None else _f64(v0)
        return self.P.cond_estimate(m, v0=self.to_perm(v0), **kw)
