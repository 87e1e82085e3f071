"""Seeded synthetic input generators (host side, numpy only).

This module holds NONE of the method's arithmetic (no SpMV, no Cholesky, no
solves, no Lanczos).  It only manufactures inputs: the five sparse SPD
matrices that stand in for the paper's unspecified "sparse, Hermitian,
positive-definite matrices A of size N" (§4.2
§5.1) and seeded dense vectors.  The same arrays are handed to the CPU oracle
(`oracle/`) and, after a host->device copy, to the CUDA path; neither of those
imports the other.  Constructions follow BASELINE.json `configs` as resolved
in SURVEY.md §8(d) and restated in DESIGN.md §4.

All matrices are canonical CSR: int32 `row_ptr`/`col_idx`, float64 `val`,
columns strictly increasing within a row, both triangles stored.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED = 241002408  # documented base seed


@dataclass
class CSR:
    n: int
    row_ptr: np.ndarray  # int32 [n+1]
    col_idx: np.ndarray  # int32 [nnz]
    val: np.ndarray      # float64 [nnz]
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    def to_scipy(self):
        import scipy.sparse as sp
        return sp.csr_matrix((self.val, self.col_idx, self.row_ptr), shape=(self.n, self.n))

    def to_dense(self) -> np.ndarray:
        return self.to_scipy().toarray()


def _rng(cfg: int, seed: int = SEED) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=seed + cfg))


def _from_masked(cols: np.ndarray, vals: np.ndarray, mask: np.ndarray, meta: dict) -> CSR:
    """cols/vals/mask are (N, K) with columns already ascending along axis 1 where mask is set."""
    n = cols.shape[0]
    cnt = mask.sum(axis=1, dtype=np.int64)
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(cnt, out=row_ptr[1:])
    if row_ptr[-1] >= 2**31:
        raise ValueError("nnz does not fit int32")
    return CSR(n, row_ptr.astype(np.int32), cols[mask].astype(np.int32),
               np.ascontiguousarray(vals[mask], dtype=np.float64), meta)


def from_scipy(a, meta: dict | None = None) -> CSR:
    a = a.tocsr()
    a.sum_duplicates()
    a.sort_indices()
    return CSR(a.shape[0], a.indptr.astype(np.int32), a.indices.astype(np.int32),
               a.data.astype(np.float64), meta or {})


# --------------------------------------------------------------------------------------
# seeded vectors: counter-based 64-bit mixer (splitmix64 finaliser), u in [0,1), v = 2u-1.
# The oracle (C) and the CUDA library each carry their own copy of these integer steps.
# --------------------------------------------------------------------------------------
_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def mix64(seed: int, idx: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + (idx.astype(np.uint64) + np.uint64(1)) * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def seeded_vector(seed: int, n: int) -> np.ndarray:
    """x_i = 2 u_i - 1, u_i = (mix64(seed, i) >> 11) * 2^-53  (exact in fp64)."""
    z = mix64(seed, np.arange(n, dtype=np.uint64))
    u = (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    return 2.0 * u - 1.0


# --------------------------------------------------------------------------------------
# generic stencil helpers
# --------------------------------------------------------------------------------------
def laplacian(dims: tuple[int, ...]) -> CSR:
    """Constant-coefficient Dirichlet Laplacian (2d on the diagonal, -1 neighbours), first
    dimension fastest.  Used only by the closed-form pins."""
    d = len(dims)
    n = int(np.prod(dims))
    idx = np.arange(n, dtype=np.int64)
    coords = []
    rem = idx
    for s in dims:
        coords.append(rem % s)
        rem = rem // s
    strides = [int(np.prod(dims[:k])) for k in range(d)]
    K = 2 * d + 1
    cols = np.zeros((n, K), dtype=np.int64)
    vals = np.zeros((n, K))
    mask = np.zeros((n, K), dtype=bool)
    # ascending column order: -stride_{d-1}, ..., -stride_0, 0, +stride_0, ..., +stride_{d-1}
    slot = 0
    for k in reversed(range(d)):
        cols[:, slot] = idx - strides[k]
        vals[:, slot] = -1.0
        mask[:, slot] = coords[k] > 0
        slot += 1
    cols[:, slot] = idx
    vals[:, slot] = 2.0 * d
    mask[:, slot] = True
    slot += 1
    for k in range(d):
        cols[:, slot] = idx + strides[k]
        vals[:, slot] = -1.0
        mask[:, slot] = coords[k] < dims[k] - 1
        slot += 1
    return _from_masked(cols, vals, mask, {"kind": "laplacian", "dims": dims})


# --------------------------------------------------------------------------------------
# config 1: 2D 5-point Poisson, n x n, plus uniform diagonal term
# --------------------------------------------------------------------------------------
def config1(n: int = 32, seed: int = SEED) -> CSR:
    a = laplacian((n, n))
    u = _rng(1, seed).random(n * n)
    rp = a.row_ptr.astype(np.int64)
    rows = np.repeat(np.arange(a.n), np.diff(rp))
    diag = a.col_idx == rows
    val = a.val.copy()
    val[diag] = 4.0 + u
    return CSR(a.n, a.row_ptr, a.col_idx, val,
               {"cfg": 1, "n": n, "b": [4], "iters": 50, "name": f"poisson2d_{n}x{n}+U[0,1)diag"})


# --------------------------------------------------------------------------------------
# config 2: 3D 7-point variable-coefficient diffusion, harmonic face averages
# --------------------------------------------------------------------------------------
def config2(n: int = 128, seed: int = SEED, sigma: float = 2.3) -> CSR:
    g = _rng(2, seed).normal(0.0, sigma, size=n * n * n)
    k = np.exp(g).reshape(n, n, n)  # index [z, y, x]; row p = x + n*(y + n*z)
    N = n ** 3

    def face(axis):
        """k_f on the '+' face along axis for every cell; boundary face -> k_cell."""
        a = k
        b = np.roll(k, -1, axis=axis)
        kf = 2.0 * a * b / (a + b)
        sl = [slice(None)] * 3
        sl[axis] = n - 1
        kf[tuple(sl)] = a[tuple(sl)]
        return kf

    def minus(kfp, axis):
        """k_f on the '-' face: the neighbour's '+' face, boundary -> k_cell."""
        m = np.roll(kfp, 1, axis=axis)
        sl = [slice(None)] * 3
        sl[axis] = 0
        m[tuple(sl)] = k[tuple(sl)]
        return m

    fxp, fyp, fzp = face(2), face(1), face(0)
    fxm, fym, fzm = minus(fxp, 2), minus(fyp, 1), minus(fzp, 0)
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    idx = (x + n * (y + n * z)).ravel()
    x, y, z = x.ravel(), y.ravel(), z.ravel()
    cols = np.stack([idx - n * n, idx - n, idx - 1, idx, idx + 1, idx + n, idx + n * n], axis=1)
    diag = (fxp + fxm + fyp + fym + fzp + fzm).ravel()
    vals = np.stack([-fzm.ravel(), -fym.ravel(), -fxm.ravel(), diag,
                     -fxp.ravel(), -fyp.ravel(), -fzp.ravel()], axis=1)
    mask = np.stack([z > 0, y > 0, x > 0, np.ones(N, bool), x < n - 1, y < n - 1, z < n - 1], axis=1)
    return _from_masked(cols, vals, mask,
                        {"cfg": 2, "n": n, "b": [8], "iters": 50, "name": f"diffusion3d_{n}^3_sigma{sigma}"})


# --------------------------------------------------------------------------------------
# config 3: random sparse SPD, badly row-scaled
# --------------------------------------------------------------------------------------
def config3(N: int = 1 << 20, seed: int = SEED, per_row: int = 8) -> CSR:
    import scipy.sparse as sp
    rng = _rng(3, seed)
    rows = np.repeat(np.arange(N, dtype=np.int64), per_row)
    c = rng.integers(0, N - 1, size=N * per_row, dtype=np.int64)
    c = c + (c >= rows)  # uniform on the N-1 off-diagonal positions
    v = rng.normal(0.0, 1.0, size=N * per_row)
    delta = rng.uniform(0.01, 0.1, size=N)
    expo = rng.uniform(-3.0, 3.0, size=N)
    B = sp.coo_matrix((v, (rows, c)), shape=(N, N)).tocsr()
    B.sum_duplicates()
    S = ((B + B.T) * 0.5).tocsr()
    S.sum_duplicates()
    S.sort_indices()
    abs_sum = np.asarray(abs(S).sum(axis=1)).ravel()
    d0 = abs_sum * (1.0 + delta)
    A0 = (S + sp.diags(d0, format="csr")).tocsr()
    s = np.sqrt(10.0 ** expo)
    A0.sum_duplicates()
    A0.sort_indices()
    rows_of = np.repeat(np.arange(N, dtype=np.int64), np.diff(A0.indptr))
    A0.data *= s[rows_of] * s[A0.indices]      # a_ij * (s_i s_j): commutative product keeps A exactly symmetric
    return from_scipy(A0, {"cfg": 3, "n": N, "b": [32], "iters": 50, "name": f"random_spd_N{N}_8perrow_scaled"})


def config3_unscaled(N: int, seed: int = SEED, per_row: int = 8) -> CSR:
    """Same draws as config3 but without the 10^U[-3,3] row scale (for the scaling-invariance pin)."""
    import scipy.sparse as sp
    rng = _rng(3, seed)
    rows = np.repeat(np.arange(N, dtype=np.int64), per_row)
    c = rng.integers(0, N - 1, size=N * per_row, dtype=np.int64)
    c = c + (c >= rows)
    v = rng.normal(0.0, 1.0, size=N * per_row)
    delta = rng.uniform(0.01, 0.1, size=N)
    B = sp.coo_matrix((v, (rows, c)), shape=(N, N)).tocsr()
    B.sum_duplicates()
    S = ((B + B.T) * 0.5).tocsr()
    abs_sum = np.asarray(abs(S).sum(axis=1)).ravel()
    A0 = (S + sp.diags(abs_sum * (1.0 + delta), format="csr")).tocsr()
    return from_scipy(A0, {"cfg": 3, "n": N, "name": "random_spd_unscaled"})


# --------------------------------------------------------------------------------------
# config 4: 2D anisotropic 9-point operator, y fastest
# --------------------------------------------------------------------------------------
def config4(n: int = 2048, eps: float = 1e-4, gamma_over_eps: float = 0.1, x_fastest: bool = False) -> CSR:
    """x_fastest = False: row p = y + n x (y fastest: contiguous blocks follow the strong coupling, the BASELINE.json
    ordering).  x_fastest = True: the SAME operator numbered p = x + n y -- contiguous blocks then run along the weak
    direction; `config4_line_permutation` maps it back (the permutation argument)."""
    gam = gamma_over_eps * eps
    N = n * n
    if x_fastest:
        yg, xg = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")  # index [y, x]; row p = x + n*y
        sx, sy = 1, n
    else:
        xg, yg = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")  # index [x, y]; row p = y + n*x
        sx, sy = n, 1
    x, y = xg.ravel(), yg.ravel()
    idx = sy * y + sx * x
    cols, vals, mask = [], [], []
    # the offset along the slow index is the outer loop, so that the columns of a row ascend (canonical CSR)
    for dslow in (-1, 0, 1):
        for dfast in (-1, 0, 1):
            dx, dy = (dfast, dslow) if x_fastest else (dslow, dfast)
            cols.append(idx + sy * dy + sx * dx)
            if dx == 0 and dy == 0:
                v = 2.0 * eps + 2.0
            elif dx == 0:
                v = -1.0
            elif dy == 0:
                v = -eps
            elif dx * dy > 0:
                v = -gam / 2.0
            else:
                v = +gam / 2.0
            vals.append(np.full(N, v))
            mask.append((x + dx >= 0) & (x + dx < n) & (y + dy >= 0) & (y + dy < n))
    return _from_masked(np.stack(cols, 1), np.stack(vals, 1), np.stack(mask, 1),
                        {"cfg": 4, "n": n, "b": [16], "iters": 50, "eps": eps, "gamma": gam,
                         "name": f"aniso9pt_{n}^2_eps{eps:g}" + ("_xfastest" if x_fastest else "")})


def config4_line_permutation(n: int) -> np.ndarray:
    """perm[i] = index in the x-fastest numbering (x + n y) of the unknown that the y-fastest numbering calls i = y + n x:
    P A_xfastest P^T = A_yfastest, where (P A P^T)[i, j] = A[perm[i], perm[j]]."""
    i = np.arange(n * n, dtype=np.int64)
    x, y = i // n, i % n
    return (x + n * y).astype(np.int32)


def random_permutation(n: int, seed: int = SEED) -> np.ndarray:
    """A seeded permutation of 0..n-1 (int32), perm[i] = original index of the unknown at permuted position i."""
    return np.random.Generator(np.random.Philox(key=seed + 977)).permutation(n).astype(np.int32)


def permuted(A: CSR, perm: np.ndarray) -> CSR:
    """P A P^T as canonical CSR, (P A P^T)[i, j] = A[perm[i], perm[j]] (an input generator: indexing only)."""
    S = A.to_scipy()
    p = np.asarray(perm, dtype=np.int64)
    return from_scipy(S[p][:, p].tocsr(), dict(A.meta, name=str(A.meta.get("name")) + "_permuted"))


# --------------------------------------------------------------------------------------
# config 5: 3D elasticity-like 27-point block system, 3 dofs per node, patch-major numbering
# --------------------------------------------------------------------------------------
_POS_OFFSETS = [(dx, dy, dz) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1)
                if (dz, dy, dx) > (0, 0, 0)]  # 13 'positive' offsets, fixed draw order


def _rotations(rng: np.random.Generator, m: int) -> np.ndarray:
    """Haar rotations from normalised 4-vectors of normals (unit quaternions)."""
    q = rng.normal(size=(m, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((m, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def config5(n: int = 96, seed: int = SEED, nu: float = 0.3, sigma: float = 1e-2) -> CSR:
    if n % 2:
        raise ValueError("config5 needs an even number of nodes per side (2x2x2 patches)")
    rng = _rng(5, seed)
    Nn = n ** 3
    g = np.arange(Nn, dtype=np.int64)
    gx, gy, gz = g % n, (g // n) % n, g // (n * n)
    h = n // 2
    perm = 8 * ((gx // 2) + h * ((gy // 2) + h * (gz // 2))) + (gx % 2) + 2 * (gy % 2) + 4 * (gz % 2)
    dvec = np.array([1.0, nu, nu * nu])
    # blocks[g, o] for the 27 offsets in lexicographic (dz,dy,dx) order; slot 13 is the node itself
    off27 = [(dx, dy, dz) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1)]
    blocks = np.zeros((Nn, 27, 3, 3))
    nid = np.full((Nn, 27), np.iinfo(np.int64).max, dtype=np.int64)
    diag = np.zeros((Nn, 3, 3))
    for (dx, dy, dz) in _POS_OFFSETS:
        R = _rotations(rng, Nn)
        Bm = np.einsum("mij,j,mkj->mik", R, dvec, R)  # Q diag(1,nu,nu^2) Q^T, drawn at the lower node
        Bm = 0.5 * (Bm + Bm.transpose(0, 2, 1))        # exactly symmetric
        ok = (gx + dx >= 0) & (gx + dx < n) & (gy + dy >= 0) & (gy + dy < n) & (gz + dz < n)
        src = g[ok]
        dst = src + dx + n * (dy + n * dz)
        sp_ = off27.index((dx, dy, dz))
        sm_ = off27.index((-dx, -dy, -dz))
        blocks[src, sp_] = -Bm[ok]
        nid[src, sp_] = perm[dst]
        blocks[dst, sm_] = -Bm[ok]
        nid[dst, sm_] = perm[src]
        np.add.at(diag, src, Bm[ok])
        np.add.at(diag, dst, Bm[ok])
        del R, Bm
    blocks[:, 13] = diag + sigma * np.eye(3)
    nid[:, 13] = perm
    # reorder node rows to patch-major, then sort each row's neighbours by node id
    inv = np.argsort(perm)
    blocks = blocks[inv]
    nid = nid[inv]
    order = np.argsort(nid, axis=1, kind="stable")
    nid = np.take_along_axis(nid, order, axis=1)
    blocks = np.take_along_axis(blocks, order[:, :, None, None], axis=1)
    valid = nid != np.iinfo(np.int64).max               # (Nn, 27)
    cnt = valid.sum(axis=1)
    row_ptr = np.zeros(3 * Nn + 1, dtype=np.int64)
    np.cumsum(np.repeat(3 * cnt, 3), out=row_ptr[1:])
    if row_ptr[-1] >= 2**31:
        raise ValueError("nnz does not fit int32")
    mask = np.broadcast_to(valid[:, None, :, None], (Nn, 3, 27, 3))
    V = blocks.transpose(0, 2, 1, 3)                     # (Nn, d, k, e)
    val = np.ascontiguousarray(V[mask])
    del V, blocks
    C = (3 * np.where(valid, nid, 0))[:, None, :, None] + np.arange(3)[None, None, None, :]
    C = np.broadcast_to(C, (Nn, 3, 27, 3))
    col = C[mask].astype(np.int32)
    return CSR(3 * Nn, row_ptr.astype(np.int32), col, val,
               {"cfg": 5, "n": n, "b": [3, 24], "iters": 50, "nu": nu, "sigma": sigma,
                "name": f"elasticity27_{n}^3x3_nu{nu}"})


# --------------------------------------------------------------------------------------
# registry
# --------------------------------------------------------------------------------------
FULL = {1: lambda: config1(32), 2: lambda: config2(128), 3: lambda: config3(1 << 20),
        4: lambda: config4(2048), 5: lambda: config5(96)}
# reduced sizes with the same structure: dense brute force / whole-vector oracle parity in seconds
SMALL = {1: lambda: config1(32), 2: lambda: config2(24), 3: lambda: config3(1 << 14),
         4: lambda: config4(96), 5: lambda: config5(8)}
TINY = {1: lambda: config1(16), 2: lambda: config2(8), 3: lambda: config3(512),
        4: lambda: config4(16), 5: lambda: config5(4)}
BLOCK_SIZES = {1: [4], 2: [8], 3: [32], 4: [16], 5: [3, 24]}


def build(cfg: int, scale: str = "full") -> CSR:
    table = {"full": FULL, "small": SMALL, "tiny": TINY}[scale]
    return table[cfg]()


def block_diagonal_spd(nblocks: int, b: int, seed: int = SEED) -> CSR:
    """The paper's literal model A = diag(A_1..A_k): dense random SPD diagonal blocks."""
    rng = _rng(80, seed)
    G = rng.normal(size=(nblocks, b, b))
    blocks = np.einsum("kij,klj->kil", G, G) + b * np.eye(b)
    blocks = 0.5 * (blocks + blocks.transpose(0, 2, 1))
    n = nblocks * b
    row_ptr = (np.arange(n + 1, dtype=np.int64) * b).astype(np.int32)
    col = (np.arange(nblocks)[:, None, None] * b + np.arange(b)[None, None, :] + np.zeros((1, b, 1), dtype=np.int64))
    return CSR(n, row_ptr, col.ravel().astype(np.int32), np.ascontiguousarray(blocks.ravel()),
               {"kind": "block_diagonal", "b": b})


def batch_poisson(nsys: int, n: int = 32, seed: int = SEED) -> CSR:
    """the paper's own problem sizes (N = 2^10, 2^12, 2^14) as a BATCH of `nsys`
    independent systems in one block-diagonal CSR (the paper's "solve each block separately" picture, PAPER.md:76-82,
    126-130).  System s is config 1's construction on an n x n grid (N = n^2 = 1024 for n = 32) with its own diagonal
    draw u ~ U[0,1) from Philox(key = seed + 1, counter offset by s): rows s N .. (s+1) N - 1."""
    a = laplacian((n, n))
    N = a.n
    u = _rng(1, seed).random(nsys * N)
    rp = a.row_ptr.astype(np.int64)
    rows = np.repeat(np.arange(N), np.diff(rp))
    diag = a.col_idx == rows
    nnz = int(rp[-1])
    val = np.tile(a.val, nsys)
    dmask = np.tile(diag, nsys)
    val[dmask] = 4.0 + u
    col = (np.tile(a.col_idx.astype(np.int64), nsys) + np.repeat(np.arange(nsys, dtype=np.int64) * N, nnz)).astype(np.int32)
    row_ptr = (np.tile(rp[:-1], nsys) + np.repeat(np.arange(nsys, dtype=np.int64) * nnz, N))
    row_ptr = np.concatenate([row_ptr, [nsys * nnz]]).astype(np.int32)
    return CSR(nsys * N, row_ptr, col, val, {"kind": "batch", "nsys": nsys, "seg": N, "name": f"batch{nsys}xpoisson2d_{n}x{n}"})


def batch_system(A: CSR, s: int) -> CSR:
    """System s of a batch built by batch_poisson, as a CSR of its own (for the per-system oracle runs)."""
    seg = A.meta["seg"]
    r0, r1 = s * seg, (s + 1) * seg
    p0, p1 = int(A.row_ptr[r0]), int(A.row_ptr[r1])
    return CSR(seg, (A.row_ptr[r0:r1 + 1] - p0).astype(np.int32), (A.col_idx[p0:p1] - r0).astype(np.int32),
               A.val[p0:p1].copy(), {"kind": "batch_member", "s": s})


def batch_poisson_mixed(grids, seed: int = SEED) -> CSR:
    """A batch of systems of DIFFERENT sizes in one block-diagonal CSR: system s is config 1's construction on a
    grids[s] x grids[s] grid (32, 64, 128 -> N = 2^10, 2^12, 2^14: the paper's three sizes), its diagonal draw
    taken from one Philox stream in system order.  meta["offsets"]: row offsets, len(grids) + 1 entries."""
    import scipy.sparse as sp
    rng = _rng(1, seed)
    mats, offsets = [], [0]
    for n in grids:
        a = laplacian((n, n))
        rows = np.repeat(np.arange(a.n), np.diff(a.row_ptr.astype(np.int64)))
        val = a.val.copy()
        val[a.col_idx == rows] = 4.0 + rng.random(a.n)
        mats.append(sp.csr_matrix((val, a.col_idx, a.row_ptr), shape=(a.n, a.n)))
        offsets.append(offsets[-1] + a.n)
    A = from_scipy(sp.block_diag(mats, format="csr"))
    A.meta.update({"kind": "batch_mixed", "nsys": len(grids), "offsets": np.asarray(offsets, dtype=np.int64),
                   "name": "batch_mixed_poisson2d_" + "_".join(str(g) for g in grids)})
    return A


def batch_member(A: CSR, s: int) -> CSR:
    """System s of a batch with meta["offsets"] as a CSR of its own."""
    off = A.meta["offsets"]
    r0, r1 = int(off[s]), int(off[s + 1])
    p0, p1 = int(A.row_ptr[r0]), int(A.row_ptr[r1])
    return CSR(r1 - r0, (A.row_ptr[r0:r1 + 1] - p0).astype(np.int32), (A.col_idx[p0:p1] - r0).astype(np.int32),
               A.val[p0:p1].copy(), {"kind": "batch_member", "s": s})


def random_block_ptr(n: int, seed: int = SEED, smin: int = 1, smax: int = 32) -> np.ndarray:
    """Variable-size Jacobi blocks (NEXT-3): consecutive sizes drawn from the seeded integer mixer, uniform in
    [smin, smax], the last block cut at n.  int64 array p with p[0] = 0 < p[1] < .. < p[-1] = n."""
    cnt = n // smin + 1
    sizes = smin + (mix64(seed, np.arange(cnt, dtype=np.uint64)) % np.uint64(smax - smin + 1)).astype(np.int64)
    ends = np.cumsum(sizes)
    k = int(np.searchsorted(ends, n))          # first block whose end reaches n
    ends = ends[:k + 1].copy()
    ends[k] = n
    return np.concatenate([[0], ends]).astype(np.int64)


def direct_sum_spd(sizes, seed: int = SEED) -> CSR:
    """Block-diagonal SPD matrix whose dense diagonal blocks have the given (different) sizes: the model M = A of
    PAPER.md:76-82 for variable-size blocks.  Block k = G G^T / s + I with G drawn from the config-independent rng."""
    import scipy.sparse as sp
    rng = np.random.default_rng(seed + 77)
    blocks = []
    for s in sizes:
        G = rng.standard_normal((s, s))
        blocks.append(G @ G.T / s + np.eye(s))
    import scipy.linalg as sla
    return from_scipy(sp.csr_matrix(sla.block_diag(*blocks)), {"name": "direct_sum_spd", "sizes": list(map(int, sizes))})
