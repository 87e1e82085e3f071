"""Pins for the CPU oracle (CPU only).  Each test checks the oracle against something OTHER than
itself: closed forms, invariants, library routines on special cases, dense brute force, or the
few things the paper fixes (cited).  A plausible slip anywhere in oracle/bj_oracle.c (dropped
term, wrong sign or index, transposed operand) fails at least one of them."""
import os

import numpy as np
import pytest
import scipy.linalg as sla

import oracle
from oracle import dense as odense
from paper_2410_02408_b200 import workloads as W

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = line[1]


def mu(n):
    k = np.arange(1, n + 1)
    return 2.0 - 2.0 * np.cos(k * np.pi / (n + 1))


def dense_precond_spectrum(A, b):
    """Independent numpy/scipy restatement: L = blockdiag(chol(D_k)), eig(L^-1 A L^-T)."""
    Ad = A.to_dense()
    n = A.n
    Linv = np.zeros((n, n))
    for lo in range(0, n, b):
        hi = min(lo + b, n)
        Lk = np.linalg.cholesky(Ad[lo:hi, lo:hi])
        Linv[lo:hi, lo:hi] = sla.solve_triangular(Lk, np.eye(hi - lo), lower=True)
    M = Linv @ Ad @ Linv.T
    return np.linalg.eigvalsh(0.5 * (M + M.T)), M


# ---------------------------------------------------------------- SpMV ------------------------------
@pytest.mark.parametrize("dims", [(17,), (9, 7), (5, 4, 6)])
def test_spmv_laplacian_eigenvectors(dims):
    """A sin-mode = lambda sin-mode with lambda = sum mu_k(n_d)  (closed form)."""
    A = W.laplacian(dims)
    rng = np.random.default_rng(1)
    for _ in range(3):
        ks = [int(rng.integers(1, s + 1)) for s in dims]
        grids = np.meshgrid(*[np.arange(1, s + 1) for s in dims], indexing="ij")
        v = np.ones(dims)
        lam = 0.0
        for g, k, s in zip(grids, ks, dims):
            v = v * np.sin(g * k * np.pi / (s + 1))
            lam += 2.0 - 2.0 * np.cos(k * np.pi / (s + 1))
        v = v.ravel(order="F")  # first dimension fastest
        y = oracle.spmv(A, v)
        assert np.abs(y - lam * v).max() < 1e-13


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_spmv_matches_scipy_and_is_not_symmetric_blind(cfg):
    """Library routine (scipy CSR matvec) on every config; plus a nonsymmetric matrix so that a
    transposed gather (x[row] / val^T) cannot pass."""
    A = W.build(cfg, "tiny")
    x = W.seeded_vector(7, A.n)
    y = oracle.spmv(A, x)
    assert np.allclose(y, A.to_scipy() @ x, rtol=1e-14, atol=1e-13 * np.abs(y).max())
    S = A.to_scipy().tolil()
    S[0, A.n - 1] = 3.5  # break symmetry
    B = W.from_scipy(S.tocsr())
    assert np.allclose(oracle.spmv(B, x), B.to_dense() @ x, rtol=1e-13, atol=1e-12)


# ---------------------------------------------------------------- extraction ------------------------
@pytest.mark.parametrize("b", [1, 3, 4, 7, 16])
def test_extract_is_dense_slicing_like_the_papers_listing(b):
    """block = A[i:i+bs, j:j+bs]; only the diagonal tiles; ragged last tile."""
    A = W.build(3, "tiny")
    Ad = A.to_dense()
    D = oracle.extract(A, b)
    n = A.n
    for k, lo in enumerate(range(0, n, b)):
        hi = min(lo + b, n)
        ref = np.zeros((b, b))
        ref[: hi - lo, : hi - lo] = Ad[lo:hi, lo:hi]
        assert np.array_equal(D[k], ref)


# ---------------------------------------------------------------- Cholesky / solves vs LAPACK --------
@pytest.mark.parametrize("b", [1, 2, 3, 5, 8, 24, 32])
def test_cholesky_and_solves_match_library_routines(b):
    rng = np.random.default_rng(b)
    nblocks = 5
    n = nblocks * b - (1 if b > 2 else 0)  # ragged last block when b > 2
    G = rng.normal(size=(nblocks, b, b))
    D = np.einsum("kij,klj->kil", G, G) + 0.5 * np.eye(b)
    if b > 2:
        D[-1, b - 1, :] = 0.0
        D[-1, :, b - 1] = 0.0
    L = oracle.factor(n, b, D)
    r = rng.normal(size=n)
    P = oracle.Precond.__new__(oracle.Precond)
    P.A, P.b, P.n, P.L, P._tmp = None, b, n, L, np.empty(2 * n)
    y, x, z = P.solve_L(r), P.solve_Lt(r), P.apply(r)
    for k, lo in enumerate(range(0, n, b)):
        hi = min(lo + b, n)
        nb = hi - lo
        Lref = np.linalg.cholesky(D[k, :nb, :nb])
        assert np.allclose(L[k, :nb, :nb], Lref, rtol=1e-12, atol=1e-13)
        assert np.all(np.triu(L[k], 1) == 0.0)
        assert np.allclose(y[lo:hi], sla.solve_triangular(Lref, r[lo:hi], lower=True), rtol=1e-10, atol=1e-12)
        assert np.allclose(x[lo:hi], sla.solve_triangular(Lref.T, r[lo:hi], lower=False), rtol=1e-10, atol=1e-12)
        assert np.allclose(z[lo:hi], np.linalg.solve(D[k, :nb, :nb], r[lo:hi]), rtol=1e-9, atol=1e-11)


def test_cholesky_reads_only_lower_triangle_and_flags_non_spd():
    D = np.array([[[4.0, 99.0], [2.0, 5.0]]])
    L = oracle.factor(2, 2, D)
    assert np.allclose(L[0], [[2.0, 0.0], [1.0, 2.0]])
    bad = np.stack([np.eye(3), np.diag([1.0, -1.0, 1.0]), np.diag([1.0, 0.0, 1.0])])
    with pytest.raises(oracle.NotSPD) as ei:
        oracle.factor(9, 3, bad)
    assert ei.value.bad_block == 1
    with pytest.raises(oracle.NotSPD):
        oracle.factor(3, 3, np.array([[[1.0, 0, 0], [0, np.nan, 0], [0, 0, 1.0]]]))


# ---------------------------------------------------------------- the paper's own statements ---------
def test_point_jacobi_is_the_papers_kernel():
    """PAPER.md:234  M[idx] = 1/A[idx*N+idx]  ==> bj_apply(b=1) on r = 1 returns 1/a_ii."""
    A = W.build(1, "full")
    P = oracle.Precond(A, 1)
    z = P.apply(np.ones(A.n))
    assert np.allclose(z, 1.0 / A.to_dense().diagonal(), rtol=1e-15)


def test_point_jacobi_operator_explicit_formula():
    """b=1: A^_ij = a_ij / sqrt(a_ii a_jj)  (SURVEY 8(c) reading 1): a SpMV-only restatement."""
    A = W.build(3, "tiny")
    Ad = A.to_dense()
    d = np.sqrt(Ad.diagonal())
    x = W.seeded_vector(3, A.n)
    assert np.allclose(oracle.Precond(A, 1).op_apply(x), (Ad / np.outer(d, d)) @ x, rtol=1e-12)


@pytest.mark.parametrize("b", [2, 5, 8])
def test_block_diagonal_model_gives_identity(b):
    """PAPER.md:80  A = diag(A_1..A_k) with matching b  ==>  L^-1 A L^-T = I, op_apply(x) = x, kappa = 1."""
    A = W.block_diagonal_spd(6, b)
    P = oracle.Precond(A, b)
    x = W.seeded_vector(11, A.n)
    assert np.abs(P.op_apply(x) - x).max() < 1e-13
    r = P.cond_estimate(20)
    assert r["iters_done"] == 1 and abs(r["kappa"] - 1.0) < 1e-13


def test_b_equals_N_gives_identity_and_breakdown_at_one():
    A = W.build(2, "tiny")
    P = oracle.Precond(A, A.n)
    x = W.seeded_vector(5, A.n)
    assert np.linalg.norm(P.op_apply(x) - x) / np.linalg.norm(x) < 1e-10
    r = P.cond_estimate(30)
    assert r["iters_done"] == 1
    assert abs(r["lmin"] - 1.0) < 1e-10 and abs(r["lmax"] - 1.0) < 1e-10


# ---------------------------------------------------------------- closed-form spectra ----------------
def test_laplacian_2d_kappa_closed_form_dense_and_lanczos():
    n = 32
    A = W.laplacian((n, n))
    m = mu(n)
    lmin, lmax = 2 * m[0], 2 * m[-1]
    assert abs(lmin - float(GOLD["lap2d_n32_lmin"])) < 1e-11
    assert abs(lmax - float(GOLD["lap2d_n32_lmax"])) < 1e-11
    assert abs(lmax / lmin - float(GOLD["lap2d_n32_kappa"])) < 1e-7
    assert abs(lmax / lmin - 1.0 / np.tan(np.pi / 66) ** 2) < 1e-9
    P = oracle.Precond(A, 0)
    ev = odense.spectrum(P)
    assert abs(ev[0] - lmin) < 1e-12 and abs(ev[-1] - lmax) < 1e-12
    r = P.cond_estimate(400)  # long run with full reorthogonalisation converges to the true extremes
    assert abs(r["lmin"] - lmin) < 1e-10 and abs(r["lmax"] - lmax) < 1e-10
    # point Jacobi with constant diagonal leaves kappa unchanged
    r1 = oracle.Precond(A, 1).cond_estimate(400)
    assert abs(r1["kappa"] / (lmax / lmin) - 1.0) < 1e-9
    assert abs(r1["lmax"] - lmax / 4.0) < 1e-10


def test_laplacian_1d_full_lanczos_reproduces_every_eigenvalue():
    n = 24
    A = W.laplacian((n,))
    P = oracle.Precond(A, 0)
    alpha, beta = P.lanczos(n, reorth=True)
    assert len(alpha) == n
    ritz = oracle.tridiag_all(alpha, beta)
    assert np.abs(ritz - mu(n)).max() < 1e-12


def test_laplacian_3d_extremes():
    dims = (6, 5, 7)
    A = W.laplacian(dims)
    lmin = sum(mu(s)[0] for s in dims)
    lmax = sum(mu(s)[-1] for s in dims)
    r = oracle.Precond(A, 0).cond_estimate(A.n)
    assert abs(r["lmin"] - lmin) < 1e-11 and abs(r["lmax"] - lmax) < 1e-11


def test_line_block_jacobi_closed_form_2d():
    """b = n on the x-fastest 2D Laplacian: spectrum {(mu_k + mu_l)/(mu_k + 2)}."""
    n = 32
    A = W.laplacian((n, n))
    m = mu(n)
    # k = mode ACROSS lines (block index direction), l = mode ALONG the line: block = T_l + 2I ... derived:
    # A = I (x) T + T (x) I ; M = I (x) (T + 2I) ; M^-1 A has eigenvalues (mu_l + mu_k)/(mu_l + 2)
    spec = np.sort(((m[:, None] + m[None, :]) / (m[:, None] + 2.0)).ravel())
    assert abs(spec[0] - float(GOLD["line2d_n32_lmin"])) < 1e-11
    assert abs(spec[-1] - float(GOLD["line2d_n32_lmax"])) < 1e-11
    assert abs(spec[-1] / spec[0] - float(GOLD["line2d_n32_kappa"])) < 1e-7
    P = oracle.Precond(A, n)
    ev = odense.spectrum(P)
    assert np.abs(ev - spec).max() < 1e-12
    r = P.cond_estimate(300)
    assert abs(r["lmin"] - spec[0]) < 1e-10 and abs(r["lmax"] - spec[-1]) < 1e-10


def test_line_and_plane_block_closed_forms_3d():
    n = 6
    A = W.laplacian((n, n, n))
    m = mu(n)
    a, b_, c = m[:, None, None], m[None, :, None], m[None, None, :]
    line = np.sort(((a + b_ + c) / (a + 4.0)).ravel())
    plane = np.sort(((a + b_ + c) / (a + b_ + 2.0)).ravel())
    assert np.abs(odense.spectrum(oracle.Precond(A, n)) - line).max() < 1e-12
    assert np.abs(odense.spectrum(oracle.Precond(A, n * n)) - plane).max() < 1e-12


def test_anisotropic_closed_forms():
    """cfg 4 with the cross term off, y fastest: lambda(A) = eps mu_k + mu_l; b = n: (eps mu_k + mu_l)/(mu_l + 2 eps)."""
    n, eps = 12, 1e-2
    A = W.config4(n, eps=eps, gamma_over_eps=0.0)
    m = mu(n)
    lamA = np.sort((eps * m[:, None] + m[None, :]).ravel())
    assert np.abs(odense.spectrum(oracle.Precond(A, 0)) - lamA).max() < 1e-12
    lamP = np.sort(((eps * m[:, None] + m[None, :]) / (m[None, :] + 2 * eps)).ravel())
    assert np.abs(odense.spectrum(oracle.Precond(A, n)) - lamP).max() < 1e-12


# ---------------------------------------------------------------- invariants -------------------------
@pytest.mark.parametrize("cfg,b", [(1, 1), (1, 4), (2, 1), (2, 8)])
def test_two_cyclic_spectrum_is_symmetric_about_one(cfg, b):
    """5-/7-point stencils with b=1 or line-segment blocks: theta_min + theta_max = 2."""
    A = W.build(cfg, "tiny")
    ev = odense.spectrum(oracle.Precond(A, b))
    assert abs(ev[0] + ev[-1] - 2.0) < 1e-11
    r = oracle.Precond(A, b).cond_estimate(A.n)
    assert abs(r["lmin"] + r["lmax"] - 2.0) < 1e-9


def test_point_jacobi_is_invariant_under_diagonal_scaling_cfg3():
    N = 512
    ev_s = odense.spectrum(oracle.Precond(W.config3(N), 1))
    ev_u = odense.spectrum(oracle.Precond(W.config3_unscaled(N), 1))
    assert np.abs(ev_s - ev_u).max() < 1e-12
    assert ev_s[0] > 1 - 1 / 1.01 - 1e-12 and ev_s[-1] < 1 + 1 / 1.01 + 1e-12  # strict diagonal dominance


def test_cfg5_smallest_eigenvalue_is_the_shift():
    """lambda_min(A) = sigma exactly, multiplicity 3 (rigid translations); nnz = 9 (3n-2)^3."""
    A = W.config5(4)
    assert A.nnz == 9 * (3 * 4 - 2) ** 3
    ev = odense.spectrum(oracle.Precond(A, 0))
    assert np.abs(ev[:3] - 1e-2).max() < 1e-12 and ev[3] > 1e-2 + 1e-6


# ---------------------------------------------------------------- dense brute force ------------------
@pytest.mark.parametrize("cfg,b", [(1, 4), (2, 8), (3, 32), (4, 16), (5, 3), (5, 24), (3, 7)])
def test_op_apply_and_spectrum_match_dense_numpy(cfg, b, rel):
    A = W.build(cfg, "tiny")
    P = oracle.Precond(A, b)
    ev_ref, M = dense_precond_spectrum(A, b)
    x = W.seeded_vector(13, A.n)
    e2, ei = rel(P.op_apply(x), M @ x)
    assert e2 < 1e-11 and ei < 1e-11
    ev = odense.spectrum(P)
    assert np.abs(ev - ev_ref).max() < 1e-9 * ev_ref[-1]
    # apply = (L L^T)^-1 = blockdiag(D_k)^-1
    Ad = A.to_dense()
    z_ref = np.empty(A.n)
    for lo in range(0, A.n, b):
        hi = min(lo + b, A.n)
        z_ref[lo:hi] = np.linalg.solve(Ad[lo:hi, lo:hi], x[lo:hi])
    e2, _ = rel(P.apply(x), z_ref)
    assert e2 < 1e-10


@pytest.mark.parametrize("cfg,b", [(1, 4), (3, 32), (4, 16)])
def test_lanczos_full_run_equals_dense_spectrum_and_interlaces(cfg, b):
    A = W.build(cfg, "tiny")
    P = oracle.Precond(A, b)
    ev_ref, _ = dense_precond_spectrum(A, b)
    alpha, beta = P.lanczos(A.n, reorth=True)
    if len(alpha) == A.n:
        assert np.abs(oracle.tridiag_all(alpha, beta) - ev_ref).max() < 1e-9 * ev_ref[-1]
    prev_min, prev_max = np.inf, -np.inf
    for m in (2, 5, 10, 20, 40):
        tmin, tmax, rmin, rmax = oracle.tridiag_extremes(alpha[:m], beta[:m])
        assert tmin >= ev_ref[0] - 1e-12 and tmax <= ev_ref[-1] + 1e-12       # interlacing
        assert tmin <= prev_min + 1e-13 and tmax >= prev_max - 1e-13          # monotone in m
        # Ritz residual bound: an eigenvalue lies within res of each Ritz value
        assert np.abs(ev_ref - tmin).min() <= rmin + 1e-12
        assert np.abs(ev_ref - tmax).min() <= rmax + 1e-12
        prev_min, prev_max = tmin, tmax


def test_lanczos_matches_krylov_qr_brute_force():
    """m-step Ritz values = eigenvalues of Q^T A^ Q with Q an orthonormal basis of the Krylov space."""
    A = W.build(1, "tiny")
    b, m = 4, 8
    P = oracle.Precond(A, b)
    _, M = dense_precond_spectrum(A, b)
    v0 = oracle.seeded_vector(oracle.DEFAULT_SEED, A.n)
    K = np.empty((A.n, m), dtype=np.longdouble)
    v = v0.astype(np.longdouble)
    Ml = M.astype(np.longdouble)
    for j in range(m):
        v = v / np.sqrt((v * v).sum())
        K[:, j] = v
        v = Ml @ v
    Q, _ = np.linalg.qr(K.astype(np.float64))
    ritz_ref = np.linalg.eigvalsh(Q.T @ M @ Q)
    alpha, beta = P.lanczos(m, reorth=True)
    ritz = oracle.tridiag_all(alpha, beta)
    assert np.abs(ritz - ritz_ref).max() < 1e-9


def test_no_reorth_equals_full_reorth_for_few_steps():
    A = W.build(2, "tiny")
    P = oracle.Precond(A, 8)
    a1, b1 = P.lanczos(6, reorth=True)
    a0, b0 = P.lanczos(6, reorth=False)
    assert np.allclose(a1, a0, rtol=1e-10) and np.allclose(b1, b0, rtol=1e-10)


def test_tridiag_bisection_matches_lapack():
    rng = np.random.default_rng(5)
    for m in (1, 2, 3, 17, 60):
        d = rng.normal(size=m)
        e = rng.normal(size=m)  # e[m-1] is the residual norm, not part of T
        T = np.diag(d) + np.diag(e[: m - 1], 1) + np.diag(e[: m - 1], -1)
        w, S = np.linalg.eigh(T)
        assert np.abs(oracle.tridiag_all(d, e) - w).max() < 1e-13
        tmin, tmax, rmin, rmax = oracle.tridiag_extremes(d, e)
        assert abs(tmin - w[0]) < 1e-13 and abs(tmax - w[-1]) < 1e-13
        assert abs(rmin - abs(e[m - 1]) * abs(S[-1, 0])) < 1e-10
        assert abs(rmax - abs(e[m - 1]) * abs(S[-1, -1])) < 1e-10


# ---------------------------------------------------------------- seeded vector ----------------------
def test_seeded_vector_matches_published_splitmix64_sequence():
    v = oracle.seeded_vector(0, 3)
    for i in range(3):
        z = int(GOLD[f"splitmix64_seed0_out{i}"], 16)
        assert v[i] == 2.0 * ((z >> 11) / 2.0**53) - 1.0
    big = oracle.seeded_vector(oracle.DEFAULT_SEED, 200000)
    assert big.min() >= -1.0 and big.max() < 1.0
    assert abs(big.mean()) < 5e-3 and abs(big.var() - 1.0 / 3.0) < 5e-3
    # the input-generator module carries its own copy of the same integer steps
    assert np.array_equal(big, W.seeded_vector(oracle.DEFAULT_SEED, 200000))


# ---------------------------------------------------------------- PCG -----------
def _scipy_csr(A):
    import scipy.sparse as sp
    return sp.csr_matrix((A.val, A.col_idx, A.row_ptr), shape=(A.n, A.n))


@pytest.mark.parametrize("cfg,b", [(1, 4), (2, 8), (3, 32), (4, 16), (5, 3), (1, 0)])
def test_pcg_solves_the_system_dense_numpy(cfg, b):
    """x from the oracle PCG = numpy dense solve; reported true residual = ||Ax - b|| / ||b||
    recomputed here with scipy; the recurrence residual agrees with it; A-norm error decreases monotonically."""
    A = W.build(cfg, "tiny")
    P = oracle.Precond(A, b)
    xs = W.seeded_vector(11, A.n)
    S = _scipy_csr(A)
    rhs = S @ xs
    r = P.pcg(rhs, 4 * A.n, 1e-13)
    xd = np.linalg.solve(A.to_dense(), rhs)
    kap = np.linalg.cond(A.to_dense())
    assert np.linalg.norm(r["x"] - xd) <= 1e-12 * kap * np.linalg.norm(xd)
    tr = np.linalg.norm(S @ r["x"] - rhs) / np.linalg.norm(rhs)
    assert abs(tr - r["true_relres"]) <= 1e-14 + 1e-6 * tr
    assert r["relres"][-1] <= 1e-13 and tr <= 1e-11
    # monotone A-norm error (a property of CG, not of the residual norm): re-run with growing iteration caps
    errs = []
    for k in (1, 2, 3, 5, 8):
        xk = P.pcg(rhs, k, 0.0)["x"]
        e = xk - xd
        errs.append(float(e @ (S @ e)))
    assert all(errs[i + 1] <= errs[i] * (1 + 1e-12) for i in range(len(errs) - 1))


@pytest.mark.parametrize("cfg,b", [(1, 4), (2, 8), (4, 16)])
def test_pcg_iterates_match_scipy_cg(cfg, b):
    """Library special case: scipy.sparse.linalg.cg with M = (L L^T)^-1 built from numpy Cholesky factors
    runs the same recurrence; after k steps the iterates agree to rounding."""
    import scipy.sparse.linalg as spla
    A = W.build(cfg, "tiny")
    P = oracle.Precond(A, b)
    S = _scipy_csr(A)
    Ad = A.to_dense()
    blocks = [np.linalg.inv(Ad[lo:min(lo + b, A.n), lo:min(lo + b, A.n)]) for lo in range(0, A.n, b)]

    def minv(r):
        out = np.empty_like(r)
        for q, lo in enumerate(range(0, A.n, b)):
            hi = min(lo + b, A.n)
            out[lo:hi] = blocks[q] @ r[lo:hi]
        return out

    M = spla.LinearOperator((A.n, A.n), matvec=minv, dtype=np.float64)
    rhs = W.seeded_vector(5, A.n)
    for k in (1, 4, 9):
        xs, _ = spla.cg(S, rhs, rtol=0.0, atol=0.0, maxiter=k, M=M)
        xo = P.pcg(rhs, k, 0.0)["x"]
        assert np.linalg.norm(xs - xo) <= 1e-10 * np.linalg.norm(xs), (cfg, b, k)


def test_pcg_with_exact_preconditioner_takes_one_step():
    """b = N: M = A, so x_1 = A^-1 b exactly (alpha_0 = 1) -- the paper's literal block-diagonal model."""
    A = W.build(1, "tiny")
    P = oracle.Precond(A, A.n)
    rhs = W.seeded_vector(2, A.n)
    r = P.pcg(rhs, 10, 1e-12)
    assert r["iters"] == 1 and abs(r["alpha"][0] - 1.0) <= 1e-12 and r["true_relres"] <= 1e-13
    Ab = W.block_diagonal_spd(9, 6)
    r = oracle.Precond(Ab, 6).pcg(W.seeded_vector(3, Ab.n), 10, 1e-12)
    assert r["iters"] == 1


@pytest.mark.parametrize("cfg,b", [(1, 4), (2, 8), (3, 32)])
def test_pcg_coefficients_give_the_lanczos_ritz_values(cfg, b):
    """CG-Lanczos equivalence: the tridiagonal built from (alpha_k, beta_k) has the Ritz values of k-step Lanczos
    on A^ = L^-1 A L^-T started from L^-1 b -- computed by the oracle's separate Lanczos routine."""
    A = W.build(cfg, "tiny")
    P = oracle.Precond(A, b)
    rhs = W.seeded_vector(8, A.n)
    k = 12
    r = P.pcg(rhs, k, 0.0)
    d, e = oracle.cg_tridiag(r["alpha"], r["beta"])
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    ritz_cg = np.linalg.eigvalsh(T)
    al, be = P.lanczos(k, v0=P.solve_L(rhs), reorth=True)
    ritz_lz = oracle.tridiag_all(al, be)
    assert np.allclose(ritz_cg, np.sort(ritz_lz), rtol=1e-9, atol=1e-12)


def test_pcg_zero_rhs_and_residual_threshold():
    A = W.build(2, "tiny")
    P = oracle.Precond(A, 8)
    r = P.pcg(np.zeros(A.n), 5, 1e-3)
    assert r["iters"] == 0 and not r["x"].any()
    rhs = W.seeded_vector(4, A.n)
    r = P.pcg(rhs, 500, 1e-3)          # the paper's accuracy bar
    assert r["true_relres"] <= 1.05e-3 and r["relres"][-1] <= 1e-3
    assert len(r["relres"]) == r["iters"] and (r["iters"] == 1 or r["relres"][-2] > 1e-3)


# ---------------------------------------------------------------- batch workload ----
def test_batch_generator_is_block_diagonal_and_members_match():
    """The batch CSR is exactly the direct sum of its members (input generator, no method arithmetic): dense comparison
    on a tiny batch, and every member is config 1's construction (diagonal 4 + U[0,1), off-diagonals -1)."""
    A = W.batch_poisson(5, 8)
    D = A.to_dense()
    assert np.array_equal(D, D.T)
    seg = A.meta["seg"]
    rebuilt = np.zeros_like(D)
    for s in range(5):
        M = W.batch_system(A, s).to_dense()
        rebuilt[s * seg:(s + 1) * seg, s * seg:(s + 1) * seg] = M
        d = np.diag(M)
        assert (d >= 4.0).all() and (d < 5.0).all()
        off = M - np.diag(d)
        assert set(np.unique(off)) <= {-1.0, 0.0} and (off.sum(axis=1) >= -4).all()
    assert np.array_equal(rebuilt, D)
    assert len({tuple(np.diag(W.batch_system(A, s).to_dense())) for s in range(5)}) == 5   # each system has its own draw


def test_pcg_terminates_in_as_many_steps_as_distinct_eigenvalues():
    """Textbook property of CG: with k distinct eigenvalues of M^-1 A the residual vanishes after k steps.  A diagonal
    matrix with the values {1, 2, 5} (b = 0: M = I) needs exactly 3; with b = 1 (M = diag A) the preconditioned operator
    is the identity and one step is enough.  Pins the recurrence without any library."""
    import scipy.sparse as sp
    n = 60
    d = np.array([1.0, 2.0, 5.0])[np.arange(n) % 3]
    A = W.from_scipy(sp.diags([d], [0], format="csr"))
    rhs = W.seeded_vector(9, n)
    r = oracle.Precond(A, 0).pcg(rhs, 10, 1e-13)
    assert r["iters"] == 3 and r["relres"][1] > 1e-6 and r["true_relres"] <= 1e-13
    assert np.allclose(r["x"], rhs / d, rtol=1e-13, atol=0)
    r1 = oracle.Precond(A, 1).pcg(rhs, 10, 1e-13)
    assert r1["iters"] == 1 and abs(r1["alpha"][0] - 1.0) <= 1e-15
    # 1D Dirichlet Laplacian, n = 12: exact termination in at most n steps, and the CG-Lanczos tridiagonal of the FULL run
    # reproduces the closed-form spectrum mu_k = 2 - 2 cos(k pi / (n + 1))
    L = W.laplacian((12,))
    rl = oracle.Precond(L, 0).pcg(W.seeded_vector(4, 12), 12, 0.0)
    dd, ee = oracle.cg_tridiag(rl["alpha"], rl["beta"][:11])
    ev = np.linalg.eigvalsh(np.diag(dd) + np.diag(ee, 1) + np.diag(ee, -1))
    assert np.allclose(ev, mu(12), rtol=1e-8, atol=0)


def test_oracle_reproduces_its_committed_fixture():
    """Regression guard for the oracle + generator pair: tests/golden/oracle_cfg1_fixture.txt was written by
    tests/golden/write_oracle_fixture.py (oracle only, never the CUDA path); a change of the oracle's arithmetic or of the
    config-1 generator shows up here and must be justified in the commit that rewrites the file."""
    fix = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "oracle_cfg1_fixture.txt")) as fh:
        for line in fh:
            parts = line.split("#")[0].split()
            if len(parts) == 2:
                fix[parts[0]] = float(parts[1])
    A = W.build(1, "full")
    x = W.seeded_vector(12345, A.n)
    for b in (0, 1, 4):
        P = oracle.Precond(A, b)
        y = P.op_apply(x)
        r = P.cond_estimate(50)
        pc = P.pcg(W.seeded_vector(17, A.n), 200, 1e-8)
        got = {f"b{b}_op_apply_norm2": float(np.linalg.norm(y)), f"b{b}_op_apply_y0": float(y[0]), f"b{b}_lmin_m50": r["lmin"],
               f"b{b}_lmax_m50": r["lmax"], f"b{b}_kappa_m50": r["kappa"], f"b{b}_pcg_iters": float(pc["iters"]),
               f"b{b}_pcg_alpha0": float(pc["alpha"][0]), f"b{b}_pcg_x_norm2": float(np.linalg.norm(pc["x"]))}
        for k, v in got.items():
            assert k in fix, k
            assert abs(v - fix[k]) <= 1e-11 * max(1.0, abs(fix[k])), (k, v, fix[k])


# ---------------------------------------------------------------- M-inner-product Lanczos (NEXT-2) ----
def _dense_M(A, b):
    """blockdiag(D_k) from the dense matrix by plain slicing (not through the oracle's extract)."""
    Ad = A.to_dense()
    M = np.zeros_like(Ad)
    for lo in range(0, A.n, b):
        hi = min(lo + b, A.n)
        M[lo:hi, lo:hi] = Ad[lo:hi, lo:hi]
    return Ad, M


@pytest.mark.parametrize("cfg,b", [(1, 4), (2, 8), (4, 16), (5, 3), (3, 7)])
def test_minv_lanczos_basis_is_M_orthonormal_and_projects_A_onto_T(cfg, b):
    """What defines the method: U^T M U = I and U^T A U = T (a dropped term, a wrong sign or a missing 1/bt breaks one),
    and the residual of the three-term relation A U = M U T + r_{m} e_m^T."""
    A = W.build(cfg, "tiny")
    P = oracle.Precond(A, b)
    m = 8
    alpha, beta, U = P.lanczos_minv(m, return_basis=True)
    assert len(alpha) == m and U.shape == (A.n, m)
    Ad, M = _dense_M(A, b)
    T = np.diag(alpha) + np.diag(beta[:-1], 1) + np.diag(beta[:-1], -1)
    scale = np.abs(T).max()
    assert np.abs(U.T @ M @ U - np.eye(m)).max() < 1e-10
    assert np.abs(U.T @ Ad @ U - T).max() < 1e-10 * scale
    Rm = Ad @ U - M @ U @ T                      # only the last column is non-zero: bt_m M u_m
    assert np.abs(Rm[:, :-1]).max() < 1e-10 * scale
    last = Rm[:, -1]
    assert abs(np.sqrt(last @ np.linalg.solve(M, last)) - beta[-1]) < 1e-10 * scale


@pytest.mark.parametrize("cfg,b", [(1, 4), (4, 16)])
def test_minv_lanczos_full_run_gives_the_generalised_eigenvalues(cfg, b):
    """Library routine for the same spectrum: scipy.linalg.eigh(A, M) (A x = lambda M x).  Small n, so the run without
    reorthogonalisation is cut at 12 steps and checked through interlacing + Ritz residual bounds; the extremes it finds
    must be eigenvalues to within the bound."""
    A = W.build(cfg, "tiny")
    P = oracle.Precond(A, b)
    Ad, M = _dense_M(A, b)
    ev = sla.eigh(Ad, M, eigvals_only=True)
    alpha, beta = P.lanczos_minv(12)
    for m in (3, 6, 12):
        tmin, tmax, rmin, rmax = oracle.tridiag_extremes(alpha[:m], beta[:m])
        assert tmin >= ev[0] - 1e-10 and tmax <= ev[-1] + 1e-10
        assert np.abs(ev - tmin).min() <= rmin + 1e-10
        assert np.abs(ev - tmax).min() <= rmax + 1e-10


@pytest.mark.parametrize("cfg,b", [(1, 4), (2, 8), (3, 32), (4, 16), (5, 24)])
def test_minv_lanczos_equals_split_lanczos_started_at_Linv_r0(cfg, b):
    """Same tridiagonal as Lanczos on L^-1 A L^-T from v_1 = L^-1 r_0 / ||.|| (similarity) for as many steps as
    rounding keeps the two recurrences together."""
    A = W.build(cfg, "tiny")
    P = oracle.Precond(A, b)
    r0 = W.seeded_vector(5, A.n)
    a1, b1 = P.lanczos_minv(6, r0=r0)
    a2, b2 = P.lanczos(6, v0=P.solve_L(r0), reorth=False)
    assert np.abs(a1 - a2).max() < 1e-9 * np.abs(a2).max()
    assert np.abs(b1 - b2).max() < 1e-9 * np.abs(a2).max()


def test_minv_lanczos_special_cases():
    A = W.build(1, "tiny")
    # b = 0: M = I, the plain Lanczos recurrence on A from the same start
    P0 = oracle.Precond(A, 0)
    r0 = W.seeded_vector(9, A.n)
    a1, b1 = P0.lanczos_minv(10, r0=r0)
    a2, b2 = P0.lanczos(10, v0=r0, reorth=False)
    assert np.abs(a1 - a2).max() < 1e-11 and np.abs(b1 - b2).max() < 1e-11
    # exact preconditioner (one block = the matrix): M^-1 A = I, alpha_0 = 1 and breakdown after one step
    Pn = oracle.Precond(A, A.n)
    al, be = Pn.lanczos_minv(5)
    assert len(al) == 1 and abs(al[0] - 1.0) < 1e-12 and be[0] < 1e-10
    # first coefficient in closed form: al_0 = (z0 . A z0) / (r0 . z0), z0 = D^-1 r0 for b = 1
    P1 = oracle.Precond(A, 1)
    Ad = A.to_dense()
    z0 = r0 / np.diag(Ad)
    al, _ = P1.lanczos_minv(1, r0=r0)
    assert abs(al[0] - (z0 @ Ad @ z0) / (r0 @ z0)) < 1e-12 * abs(al[0])
    # M-Lanczos and the CG coefficients see the same Krylov space: T from PCG with right-hand side r0 is the same matrix
    pc = P1.pcg(r0, 6, 0.0)
    d, e = oracle.cg_tridiag(pc["alpha"], pc["beta"])
    a6, b6 = P1.lanczos_minv(6, r0=r0)
    assert np.abs(d - a6).max() < 1e-9 * np.abs(a6).max() and np.abs(e - b6[:5]).max() < 1e-9 * np.abs(a6).max()


# ---------------------------------------------------------------- variable-size blocks (NEXT-3) ------
def test_variable_blocks_with_equal_sizes_are_the_uniform_preconditioner():
    A = W.build(2, "tiny")
    for b in (3, 8, 16):
        ptr = np.minimum(np.arange(0, A.n + b, b), A.n)
        ptr = np.unique(ptr)
        Pv, Pu = oracle.PrecondBlocks(A, ptr), oracle.Precond(A, b)
        x = W.seeded_vector(3, A.n)
        for f in ("solve_L", "solve_Lt", "apply", "op_apply"):
            assert np.array_equal(getattr(Pv, f)(x), getattr(Pu, f)(x)), (b, f)
        av, bv = Pv.lanczos(12, reorth=True)
        au, bu = Pu.lanczos(12, reorth=True)
        assert np.abs(av - au).max() < 1e-12 * np.abs(au).max() and np.abs(bv - bu).max() < 1e-12 * np.abs(au).max()


@pytest.mark.parametrize("cfg", [1, 3, 4, 5])
def test_variable_blocks_match_dense_numpy(cfg, rel):
    """Independent restatement: per block np.linalg.solve / np.linalg.cholesky on dense slices."""
    A = W.build(cfg, "tiny")
    ptr = W.random_block_ptr(A.n, seed=cfg, smin=1, smax=32)
    assert ptr[0] == 0 and ptr[-1] == A.n and np.diff(ptr).min() >= 1 and np.diff(ptr).max() <= 32
    assert len(set(np.diff(ptr)[:-1].tolist())) > 3          # sizes really differ
    P = oracle.PrecondBlocks(A, ptr)
    Ad = A.to_dense()
    x = W.seeded_vector(11, A.n)
    z_ref = np.empty(A.n)
    Linv = np.zeros((A.n, A.n))
    for lo, hi in zip(ptr[:-1], ptr[1:]):
        z_ref[lo:hi] = np.linalg.solve(Ad[lo:hi, lo:hi], x[lo:hi])
        Lk = np.linalg.cholesky(Ad[lo:hi, lo:hi])
        Linv[lo:hi, lo:hi] = sla.solve_triangular(Lk, np.eye(hi - lo), lower=True)
    assert rel(P.apply(x), z_ref)[0] < 1e-10
    assert rel(P.solve_L(x), Linv @ x)[0] < 1e-11 and rel(P.solve_Lt(x), Linv.T @ x)[0] < 1e-11
    Mop = Linv @ Ad @ Linv.T
    assert rel(P.op_apply(x), Mop @ x)[0] < 1e-11
    ev = np.linalg.eigvalsh(0.5 * (Mop + Mop.T))
    r = P.cond_estimate(min(A.n, 40), reorth=True)
    assert r["lmin"] >= ev[0] - 1e-10 and r["lmax"] <= ev[-1] + 1e-10          # interlacing
    assert np.abs(ev - r["lmin"]).min() <= r["res_min"] + 1e-10 and np.abs(ev - r["lmax"]).min() <= r["res_max"] + 1e-10


def test_variable_blocks_equal_to_the_matrix_blocks_give_identity():
    """M = A with blocks of different sizes: A^ = I, Lanczos breaks down after one step."""
    sizes = [5, 1, 32, 7, 16, 2, 24]
    A = W.direct_sum_spd(sizes)
    ptr = np.concatenate([[0], np.cumsum(sizes)])
    P = oracle.PrecondBlocks(A, ptr)
    x = W.seeded_vector(2, A.n)
    assert np.abs(P.op_apply(x) - x).max() < 1e-13
    r = P.cond_estimate(10)
    assert r["iters_done"] == 1 and abs(r["kappa"] - 1) < 1e-12
    with pytest.raises(ValueError):
        oracle.PrecondBlocks(A, [0, 5, 5, A.n])


# ---------------------------------------------------------------- permutation argument ------
def _dense_perm_reference(A, perm, b):
    """M = P^T blockdiag(D_k) P built by dense slicing of P A P^T (numpy only)."""
    Ad = A.to_dense()
    p = np.asarray(perm)
    Ap = Ad[np.ix_(p, p)]
    Mp = np.zeros_like(Ap)
    for lo in range(0, A.n, b):
        hi = min(lo + b, A.n)
        Mp[lo:hi, lo:hi] = Ap[lo:hi, lo:hi]
    M = np.zeros_like(Mp)
    M[np.ix_(p, p)] = Mp          # M[perm[i], perm[j]] = Mp[i, j]
    return Ad, M


@pytest.mark.parametrize("cfg,b", [(1, 4), (2, 8), (3, 5), (4, 16), (5, 3)])
def test_perm_apply_and_spectrum_match_dense_numpy(cfg, b, rel):
    """oracle.PrecondPerm against the definition written densely: z = M^-1 r by numpy.linalg.solve with
    M = P^T blockdiag(D_k) P, and the spectrum of the split operator = the generalised spectrum of (A, M)."""
    A = W.build(cfg, "tiny")
    perm = W.random_permutation(A.n, seed=100 + cfg)
    Ad, M = _dense_perm_reference(A, perm, b)
    P = oracle.PrecondPerm(A, perm, b)
    r = W.seeded_vector(3, A.n)
    e2, ei = rel(P.apply(r), np.linalg.solve(M, r))
    assert e2 < 1e-12 and ei < 1e-12
    # solve_Lt(solve_L(r)) is apply; op_apply = solve_L . A . solve_Lt, all in the ORIGINAL ordering
    assert rel(P.solve_Lt(P.solve_L(r)), P.apply(r))[0] < 1e-14
    assert rel(P.op_apply(r), P.solve_L(Ad @ P.solve_Lt(r)))[0] < 1e-13
    cols = np.stack([P.op_apply(e) for e in np.eye(A.n)], axis=1)
    assert np.abs(cols - cols.T).max() <= 1e-12 * np.abs(cols).max()      # symmetric operator
    ev = np.linalg.eigvalsh(0.5 * (cols + cols.T))
    gen = sla.eigh(Ad, M, eigvals_only=True)
    assert np.abs(ev - gen).max() <= 1e-10 * np.abs(gen).max()
    c = P.cond_estimate(A.n, reorth=True)                                    # m = N: Lanczos sees the whole spectrum
    assert abs(c["lmin"] / gen[0] - 1) < 1e-8 and abs(c["lmax"] / gen[-1] - 1) < 1e-8


def test_perm_identity_is_the_unpermuted_preconditioner_bit_for_bit():
    A = W.build(2, "tiny")
    P0, P1 = oracle.Precond(A, 8), oracle.PrecondPerm(A, np.arange(A.n), 8)
    x = W.seeded_vector(5, A.n)
    for name in ("solve_L", "solve_Lt", "apply", "op_apply"):
        assert np.array_equal(getattr(P0, name)(x), getattr(P1, name)(x)), name
    c0, c1 = P0.cond_estimate(20), P1.cond_estimate(20)
    assert np.array_equal(c0["alpha"], c1["alpha"]) and np.array_equal(c0["beta"], c1["beta"])


def test_point_jacobi_is_invariant_under_any_permutation():
    """b = 1: M = diag(A) whatever the ordering, so the operator in the original ordering does not depend on P."""
    A = W.build(3, "tiny")
    x = W.seeded_vector(9, A.n)
    ref = oracle.Precond(A, 1).op_apply(x)
    for seed in (1, 2):
        P = oracle.PrecondPerm(A, W.random_permutation(A.n, seed), 1)
        assert np.abs(P.op_apply(x) - ref).max() <= 1e-14 * np.abs(ref).max()
        k0, k1 = oracle.Precond(A, 1).cond_estimate(A.n)["kappa"], P.cond_estimate(A.n)["kappa"]
        assert abs(k1 / k0 - 1) < 1e-9


def test_line_permutation_turns_xfastest_config4_into_the_yfastest_one():
    """Config 4 numbered x-fastest has its contiguous blocks along the WEAK direction; the line permutation
    (workloads.config4_line_permutation) gives back exactly the y-fastest matrix of BASELINE.json: same factors, same
    operator (in the permuted coordinates bit for bit), same kappa estimate -- and the natural blocks are far worse."""
    n = 24
    Ax, Ay = W.config4(n, x_fastest=True), W.config4(n)
    perm = W.config4_line_permutation(n)
    Pp, Py = oracle.PrecondPerm(Ax, perm, 8), oracle.Precond(Ay, 8)
    assert np.array_equal(Pp.Ap.row_ptr, Ay.row_ptr) and np.array_equal(Pp.Ap.col_idx, Ay.col_idx)
    assert np.array_equal(Pp.Ap.val, Ay.val)
    assert np.array_equal(Pp.P.L, Py.L)
    x = W.seeded_vector(2, Ax.n)
    assert np.array_equal(Pp.op_apply(x)[perm], Py.op_apply(x[perm]))
    kp = Pp.cond_estimate(Ax.n)["kappa"]
    ky = Py.cond_estimate(Ax.n, v0=W.seeded_vector(oracle.DEFAULT_SEED, Ax.n)[perm])["kappa"]
    assert abs(kp / ky - 1) < 1e-10
    k_natural = oracle.Precond(Ax, 8).cond_estimate(Ax.n)["kappa"]
    assert k_natural > 3 * kp          # blocks across the weak coupling barely help


def test_rcm_restores_the_block_diagonal_model_after_a_shuffle():
    """PAPER.md:80 (A = diag(A_1..A_k)) hidden by a random symmetric shuffle: reverse Cuthill-McKee (scipy) makes every
    connected component contiguous again, the blocks match it, M = A and the preconditioned operator is the identity."""
    from scipy.sparse.csgraph import reverse_cuthill_mckee
    b = 6
    A0 = W.block_diagonal_spd(40, b)
    shuffle = W.random_permutation(A0.n, seed=7)
    A = W.permuted(A0, shuffle)
    x = W.seeded_vector(4, A.n)
    assert np.abs(oracle.Precond(A, b).op_apply(x) - x).max() > 1e-3        # natural blocks of the shuffled matrix: not I
    perm = reverse_cuthill_mckee(A.to_scipy(), symmetric_mode=True)
    P = oracle.PrecondPerm(A, perm, b)
    assert np.abs(P.op_apply(x) - x).max() <= 1e-13
    c = P.cond_estimate(10)
    assert c["iters_done"] == 1 and abs(c["kappa"] - 1) < 1e-12


def test_perm_rejects_non_permutations_and_takes_variable_blocks():
    A = W.build(1, "tiny")
    with pytest.raises(ValueError):
        oracle.PrecondPerm(A, np.zeros(A.n, dtype=np.int64), 4)
    with pytest.raises(ValueError):
        oracle.PrecondPerm(A, np.arange(A.n - 1), 4)
    perm = W.random_permutation(A.n, 3)
    ptr = W.random_block_ptr(A.n, seed=5, smin=1, smax=9)
    P = oracle.PrecondPerm(A, perm, block_ptr=ptr)
    Ad = A.to_dense()
    Ap = Ad[np.ix_(perm, perm)]
    Mp = np.zeros_like(Ap)
    for k in range(len(ptr) - 1):
        Mp[ptr[k]:ptr[k + 1], ptr[k]:ptr[k + 1]] = Ap[ptr[k]:ptr[k + 1], ptr[k]:ptr[k + 1]]
    M = np.zeros_like(Mp)
    M[np.ix_(perm, perm)] = Mp
    r = W.seeded_vector(8, A.n)
    assert np.abs(P.apply(r) - np.linalg.solve(M, r)).max() <= 1e-12 * np.abs(r).max()
