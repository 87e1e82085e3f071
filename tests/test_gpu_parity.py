"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle,
element by element on the same seeded inputs.  Tolerances are BASELINE.json's: normwise relative
error <= 1e-12 on apply outputs (2-norm and inf-norm, reading 14) and <= 1e-6 on
kappa estimates, fp64."""
import numpy as np
import pytest

import oracle
from paper_2410_02408_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_APPLY = 1e-12
TOL_KAPPA = 1e-6


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2410_02408_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def torch_():
    import torch
    return torch


_MATS = {}


def mat(cfg, scale):
    key = (cfg, scale)
    if key not in _MATS:
        _MATS[key] = W.build(cfg, scale)
    return _MATS[key]


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check_all_ops(B, torch, A, b, rel, seeds=(101, 202), tol=TOL_APPLY, kernels=(None,), **opts):
    h, keep = B.setup_from_host(A, b, **opts)
    try:
        P = oracle.Precond(A, b)
        for kern in kernels:
            if kern is not None:
                B.bj_set_option(h, B.BJ_OPT_SPMV_KERNEL, kern[0])
                B.bj_set_option(h, B.BJ_OPT_FUSE_FORWARD, kern[1])
            for seed in seeds:
                x = W.seeded_vector(seed, A.n)
                xd = dev(torch, x)
                got = {
                    "spmv": B.bj_spmv(h, xd).cpu().numpy(),
                    "op_apply": B.bj_op_apply(h, xd).cpu().numpy(),
                }
                ref = {"spmv": oracle.spmv(A, x), "op_apply": P.op_apply(x)}
                if b > 0:
                    got.update(solve_L=B.bj_solve_L(h, xd).cpu().numpy(), solve_Lt=B.bj_solve_Lt(h, xd).cpu().numpy(),
                               apply=B.bj_apply(h, xd).cpu().numpy())
                    ref.update(solve_L=P.solve_L(x), solve_Lt=P.solve_Lt(x), apply=P.apply(x))
                for name in got:
                    e2, ei = rel(got[name], ref[name])
                    assert e2 <= tol and ei <= tol, f"{name} b={b} kern={kern}: rel2={e2:.3e} relinf={ei:.3e}"
                # in-place operator apply
                y = xd.clone()
                B.bj_op_apply(h, y, y)
                e2, ei = rel(y.cpu().numpy(), ref["op_apply"])
                assert e2 <= tol and ei <= tol
    finally:
        B.bj_destroy(h)


KERNELS = ((0, 0), (1, 0), (1, 1))


# ------------------------------------------------------------------ small configs, every op -----------
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_ops_match_oracle_on_small_configs(B, torch_, rel, cfg):
    A = mat(cfg, "small")
    for b in W.BLOCK_SIZES[cfg]:
        check_all_ops(B, torch_, A, b, rel, kernels=KERNELS)


@pytest.mark.parametrize("b", [0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 16, 20, 24, 31, 32])
def test_every_block_size_including_ragged_last_block(B, torch_, rel, b):
    A = mat(3, "small") if b % 2 else mat(2, "small")   # 16384 and 13824 rows: ragged for 5,7,9,20,31 / 5,7,..
    check_all_ops(B, torch_, A, b, rel, seeds=(7,), kernels=KERNELS)


def test_ragged_tail_sizes(B, torch_, rel):
    """n not a multiple of anything: 1D Laplacian + diagonal, n = 100003 rows spans many tiles and a tail."""
    n = 100003
    A = W.laplacian((n,))
    for b in (3, 8, 16, 32):
        check_all_ops(B, torch_, A, b, rel, seeds=(5,), kernels=KERNELS)


def test_config1_exact(B, torch_, rel):
    A = mat(1, "full")
    check_all_ops(B, torch_, A, 4, rel, kernels=KERNELS)
    h, keep = B.setup_from_host(A, 4)
    P = oracle.Precond(A, 4)
    r_gpu = B.bj_cond_estimate_ex(h, 50, reorth=True)
    r_cpu = P.cond_estimate(50)
    assert r_gpu["iters_done"] == r_cpu["iters_done"] == 50
    assert abs(r_gpu["kappa"] / r_cpu["kappa"] - 1) <= TOL_KAPPA
    assert abs(r_gpu["lmin"] / r_cpu["lmin"] - 1) <= TOL_KAPPA and abs(r_gpu["lmax"] / r_cpu["lmax"] - 1) <= TOL_KAPPA
    lmin, lmax = B.bj_cond_estimate(h, 50)      # the 4-argument call of the north star
    assert abs((lmax / lmin) / r_cpu["kappa"] - 1) <= TOL_KAPPA
    B.bj_destroy(h)


# ------------------------------------------------------------------ Lanczos ------------------------------
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_kappa_estimates_match_oracle_small(B, torch_, cfg):
    A = mat(cfg, "small")
    for b in [0] + W.BLOCK_SIZES[cfg]:
        h, keep = B.setup_from_host(A, b)
        P = oracle.Precond(A, b)
        g = B.bj_cond_estimate_ex(h, 50, reorth=True)
        c = P.cond_estimate(50, reorth=True)
        assert g["iters_done"] == c["iters_done"]
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (cfg, b, g["kappa"], c["kappa"])
        assert np.allclose(g["alpha"], c["alpha"], rtol=1e-8, atol=1e-10 * abs(c["alpha"]).max())
        assert abs(g["res_min"] - c["res_min"]) <= 1e-6 * c["lmax"] and abs(g["res_max"] - c["res_max"]) <= 1e-6 * c["lmax"]
        if b > 0:
            # fused fast mode (no reorthogonalisation) is safe on the preconditioned operators
            g0 = B.bj_cond_estimate_ex(h, 50, reorth=False)
            c0 = P.cond_estimate(50, reorth=False)
            assert abs(g0["kappa"] / c0["kappa"] - 1) <= TOL_KAPPA
        B.bj_destroy(h)


def test_caller_supplied_start_vector_and_seed(B, torch_):
    A = mat(2, "small")
    h, keep = B.setup_from_host(A, 8)
    P = oracle.Precond(A, 8)
    v0 = W.seeded_vector(999, A.n)
    g = B.bj_cond_estimate_ex(h, 30, reorth=True, v0=dev(torch_, v0))
    c = P.cond_estimate(30, v0=v0)
    assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
    g2 = B.bj_cond_estimate_ex(h, 30, reorth=True, seed=999)
    assert abs(g2["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
    sv = B.bj_seeded_vector(h, 999).cpu().numpy()
    assert np.array_equal(sv, oracle.seeded_vector(999, A.n))   # integer mixer: bit-exact
    B.bj_destroy(h)


def test_breakdown_is_not_an_error(B, torch_, rel):
    """b = N (<= B_MAX) and the paper's block-diagonal model: A^ = I, m_eff = 1, kappa = 1."""
    A = W.block_diagonal_spd(1, 24)
    h, keep = B.setup_from_host(A, 24)
    g = B.bj_cond_estimate_ex(h, 20, reorth=True)
    assert g["iters_done"] == 1 and abs(g["kappa"] - 1) < 1e-12
    B.bj_destroy(h)
    for b in (2, 5, 8, 16, 32):
        A = W.block_diagonal_spd(257, b)
        h, keep = B.setup_from_host(A, b)
        x = W.seeded_vector(3, A.n)
        y = B.bj_op_apply(h, dev(torch_, x)).cpu().numpy()
        e2, ei = rel(y, x)
        assert e2 < 1e-13 and ei < 1e-13
        g = B.bj_cond_estimate_ex(h, 20, reorth=False)
        assert g["iters_done"] == 1 and abs(g["kappa"] - 1) < 1e-12
        B.bj_destroy(h)


@pytest.mark.parametrize("which", ["multi_launch", "single_launch"])
def test_zero_or_nonfinite_start_vector_is_an_invalid_argument(B, torch_, which):
    """beta_1 = ||v0|| = 0 (or NaN / inf) is not a breakdown: every estimator rejects it, fused and unfused alike
    (config 1 takes the single-launch kernel of bj_lanczos_small.cu, the 13 824-row matrix the multi-launch paths)."""
    A = mat(2, "small") if which == "multi_launch" else mat(1, "full")
    z = torch_.zeros(A.n, dtype=torch_.float64, device="cuda")
    nan = z.clone()
    nan[5] = float("nan")
    for b in (0, 8, 16, 12):              # no solve / thread-per-block / group / stream solve (unfused only)
        h, keep = B.setup_from_host(A, b)
        for fuse in (1, 0):
            B.bj_set_option(h, B.BJ_OPT_LANCZOS_FUSE, fuse)
            B.bj_set_option(h, B.BJ_OPT_LANCZOS_SINGLE_LAUNCH, 1 if fuse else 2)   # cluster form / single-CTA form
            for v0 in (z, nan):
                for reorth in (False, True):
                    with pytest.raises(B.BJError) as e:
                        B.bj_cond_estimate_ex(h, 10, reorth=reorth, v0=v0)
                    assert e.value.code == B.BJ_ERR_INVALID_ARG, (b, fuse, reorth)
            g = B.bj_cond_estimate_ex(h, 10, reorth=False)      # the handle is still usable afterwards
            assert g["iters_done"] == 10 and np.isfinite(g["kappa"])
        B.bj_destroy(h)


def test_single_launch_lanczos_for_launch_bound_sizes(B, torch_):
    """Config 1 (N = 1024, the paper's smallest size) and its relatives run the whole Lanczos estimate as ONE single-CTA
    kernel: same recurrence as the multi-launch path and as the oracle, parity and fast mode, every b <= 8 and b = 0,
    ragged last block, breakdown, caller's start vector; bj_set_option can switch it off."""
    cases = [(mat(1, "full"), (0, 1, 3, 4, 7, 8)), (W.laplacian((37, 29)), (4, 5)), (mat(5, "tiny"), (3, 8))]
    for A, blocks in cases:
        for b in blocks:
            h, keep = B.setup_from_host(A, b)
            P = oracle.Precond(A, b)
            c = P.cond_estimate(50, reorth=True)
            c0 = P.cond_estimate(30, reorth=False)
            v0 = W.seeded_vector(77, A.n)
            cv = P.cond_estimate(20, v0=v0)
            for form in (1, 2):      # 1: the eight-CTA cluster kernel where a CTA's share of the basis fits; 2: one CTA
                B.bj_set_option(h, B.BJ_OPT_LANCZOS_SINGLE_LAUNCH, form)
                l0 = B.bj_get_info(h)["kernel_launches"]
                g = B.bj_cond_estimate_ex(h, 50, reorth=True)
                assert B.bj_get_info(h)["kernel_launches"] - l0 <= 2          # seeded vector + the one kernel
                assert g["iters_done"] == c["iters_done"]
                assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (A.n, b, form, g["kappa"], c["kappa"])
                assert np.allclose(g["alpha"], c["alpha"], rtol=1e-8, atol=1e-10 * abs(c["alpha"]).max())
                assert np.allclose(g["beta"], c["beta"], rtol=1e-7, atol=1e-10 * abs(c["alpha"]).max())
                g0 = B.bj_cond_estimate_ex(h, 30, reorth=False)
                assert np.abs(g0["alpha"] - c0["alpha"]).max() <= 1e-8 * abs(c0["alpha"]).max(), (A.n, b, form)
                gv = B.bj_cond_estimate_ex(h, 20, reorth=True, v0=dev(torch_, v0))
                assert abs(gv["kappa"] / cv["kappa"] - 1) <= TOL_KAPPA
            B.bj_set_option(h, B.BJ_OPT_LANCZOS_SINGLE_LAUNCH, 0)           # the multi-launch path on the same handle
            l0 = B.bj_get_info(h)["kernel_launches"]
            gm = B.bj_cond_estimate_ex(h, 50, reorth=True)
            assert B.bj_get_info(h)["kernel_launches"] - l0 > 50
            assert abs(gm["kappa"] / g["kappa"] - 1) <= TOL_KAPPA
            B.bj_destroy(h)
    A = W.block_diagonal_spd(100, 8)          # M = A: breakdown at step 1 inside the single kernel
    h, keep = B.setup_from_host(A, 8)
    for form in (1, 2):
        B.bj_set_option(h, B.BJ_OPT_LANCZOS_SINGLE_LAUNCH, form)
        g = B.bj_cond_estimate_ex(h, 20, reorth=True)
        assert g["iters_done"] == 1 and abs(g["kappa"] - 1) < 1e-12
    B.bj_destroy(h)
    # fewer blocks than CTAs, and a block count that leaves the last CTAs of the cluster without rows
    for A, b in ((W.laplacian((5, 4)), 4), (W.laplacian((9, 9)), 8), (W.laplacian((3, 3)), 0)):
        h, keep = B.setup_from_host(A, b)
        g = B.bj_cond_estimate_ex(h, A.n, reorth=True)
        c = oracle.Precond(A, b).cond_estimate(A.n, reorth=True)
        assert g["iters_done"] == c["iters_done"] and abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (A.n, b)
        B.bj_destroy(h)


def test_single_launch_lanczos_on_the_papers_larger_sizes(B, torch_):
    """N = 2^12: a sixteen-CTA cluster holds what an eight-CTA one cannot -- the basis of N = 4096 at m = 50
    with full reorthogonalisation.  N = 2^14 stays on the multi-launch path (checked against the oracle all the same).
    Same bar as everywhere: kappa to 1e-6, alpha / beta against the oracle."""
    for grid, b, reorth in ((64, 4, True), (64, 8, True), (64, 0, False), (64, 3, False), (128, 4, False), (128, 4, True)):
        A = W.config1(grid)
        h, keep = B.setup_from_host(A, b)
        l0 = B.bj_get_info(h)["kernel_launches"]
        g = B.bj_cond_estimate_ex(h, 50, reorth=reorth)
        if grid == 64:
            assert B.bj_get_info(h)["kernel_launches"] - l0 <= 2, (grid, b, reorth)  # seeded vector + the one kernel
        c = oracle.Precond(A, b).cond_estimate(50, reorth=reorth)
        assert g["iters_done"] == c["iters_done"]
        scale = abs(c["alpha"]).max()
        assert np.abs(g["alpha"] - c["alpha"]).max() <= 1e-8 * scale and np.abs(g["beta"] - c["beta"]).max() <= 1e-7 * scale
        if reorth:
            assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (grid, b, g["kappa"], c["kappa"])
        B.bj_set_option(h, B.BJ_OPT_LANCZOS_SINGLE_LAUNCH, 0)                        # the multi-launch path agrees
        gm = B.bj_cond_estimate_ex(h, 50, reorth=reorth)
        assert np.abs(gm["alpha"] - g["alpha"]).max() <= 1e-8 * scale
        B.bj_destroy(h)


@pytest.mark.parametrize("m", [60, 120, 230])
def test_parity_mode_reorthogonalisation_kernels_beyond_52_vectors(B, torch_, m):
    """Full reorthogonalisation on the multi-launch path: up to 52 basis vectors the fused update + dot pass keeps its tile in
    registers, up to 199 in shared memory (bulk copies), beyond that the four unfused kernels run; odd n takes the unfused
    kernels too.  kappa and the coefficients against the oracle in every regime."""
    for A, b in ((mat(2, "small"), 8), (W.laplacian((113, 97)), 4)):     # n = 13 824 (even), n = 10 961 (odd)
        h, keep = B.setup_from_host(A, b)
        g = B.bj_cond_estimate_ex(h, m, reorth=True)
        c = oracle.Precond(A, b).cond_estimate(m, reorth=True)
        assert g["iters_done"] == c["iters_done"] == m
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (A.n, m, g["kappa"], c["kappa"])
        scale = abs(c["alpha"]).max()
        assert np.abs(g["alpha"] - c["alpha"]).max() <= 1e-8 * scale and np.abs(g["beta"] - c["beta"]).max() <= 1e-7 * scale
        B.bj_destroy(h)


def test_point_jacobi_is_the_papers_kernel(B, torch_):
    """M[idx] = 1/A[idx*N+idx]."""
    A = mat(1, "full")
    h, keep = B.setup_from_host(A, 1)
    z = B.bj_apply(h, torch_.ones(A.n, dtype=torch_.float64, device="cuda")).cpu().numpy()
    assert np.allclose(z, 1.0 / A.to_dense().diagonal(), rtol=1e-15)
    B.bj_destroy(h)


# ------------------------------------------------------------------ errors and edge cases ----------------
def test_error_codes(B, torch_):
    A = mat(1, "full")
    rp, ci, val = dev(torch_, A.row_ptr), dev(torch_, A.col_idx), dev(torch_, A.val)
    with pytest.raises(B.BJError) as e:
        B.bj_setup(rp, ci, val, 33)
    assert e.value.code == B.BJ_ERR_INVALID_ARG
    with pytest.raises(B.BJError) as e:
        B.bj_setup(rp, ci, val, -1)
    assert e.value.code == B.BJ_ERR_INVALID_ARG
    # unsorted columns
    ci2 = A.col_idx.copy()
    s = A.row_ptr[10]
    ci2[s], ci2[s + 1] = ci2[s + 1], ci2[s]
    with pytest.raises(B.BJError) as e:
        B.bj_setup(rp, dev(torch_, ci2), val, 4)
    assert e.value.code == B.BJ_ERR_NOT_CANONICAL
    # column out of range
    ci3 = A.col_idx.copy()
    ci3[-1] = A.n
    with pytest.raises(B.BJError) as e:
        B.bj_setup(rp, dev(torch_, ci3), val, 4)
    assert e.value.code == B.BJ_ERR_NOT_CANONICAL
    # row_ptr not ending at nnz
    rp2 = A.row_ptr.copy()
    rp2[-1] -= 1
    with pytest.raises(B.BJError) as e:
        B.bj_setup(dev(torch_, rp2), ci, val, 4)
    assert e.value.code == B.BJ_ERR_NOT_CANONICAL
    # non-SPD block: first bad block index is reported, same as the oracle
    v2 = A.val.copy()
    rows = np.repeat(np.arange(A.n), np.diff(A.row_ptr))
    for r in (41, 333):
        v2[(rows == r) & (A.col_idx == r)] = -1.0
    A2 = W.CSR(A.n, A.row_ptr, A.col_idx, v2)
    with pytest.raises(B.BJError) as e:
        B.bj_setup(rp, ci, dev(torch_, v2), 4)
    assert e.value.code == B.BJ_ERR_NOT_SPD and e.value.bad_block == 41 // 4
    with pytest.raises(oracle.NotSPD) as eo:
        oracle.Precond(A2, 4)
    assert eo.value.bad_block == e.value.bad_block
    # spmv must not alias
    h = B.bj_setup(rp, ci, val, 4)
    x = torch_.ones(A.n, dtype=torch_.float64, device="cuda")
    with pytest.raises(B.BJError):
        B.bj_spmv(h, x, x)
    info = B.bj_get_info(h)
    assert info["n"] == A.n and info["nnz"] == A.nnz and info["b"] == 4 and info["nblocks"] == 256 and info["bad_block"] == -1
    B.bj_destroy(h)


def test_setup_options_are_per_handle_arguments(B, torch_, rel):
    """bj_setup_ex: storage variants are arguments of the call, not process state -- handles of one process differ."""
    import ctypes as C
    A = mat(4, "small")
    rp, ci, val = dev(torch_, A.row_ptr), dev(torch_, A.col_idx), dev(torch_, A.val)
    hs = {"default": B.bj_setup(rp, ci, val, 16), "band": B.bj_setup(rp, ci, val, 16, band=1),
          "col16": B.bj_setup(rp, ci, val, 16, col16=1), "both": B.bj_setup(rp, ci, val, 16, band=1, col16=1)}
    infos = {k: B.bj_get_info(h) for k, h in hs.items()}
    assert [infos[k]["band_width"] for k in ("default", "band", "col16", "both")] == [-1, 1, -1, 1]
    assert [infos[k]["col16"] for k in ("default", "band", "col16", "both")] == [0, 0, 1, 1]
    assert infos["band"]["factor_bytes"] < infos["default"]["factor_bytes"]
    x = W.seeded_vector(12, A.n)
    ref = oracle.Precond(A, 16).op_apply(x)
    for k, h in hs.items():       # interleaved use of all four
        e2, ei = rel(B.bj_op_apply(h, dev(torch_, x)).cpu().numpy(), ref)
        assert e2 <= TOL_APPLY and ei <= TOL_APPLY, k
        t = B.bj_get_setup_time(h)
        assert t["kernel_ms"] > 0 and t["algorithmic_bytes"] == 12 * A.nnz + 4 * (A.n + 1) + infos[k]["factor_bytes"]
    for h in hs.values():
        B.bj_destroy(h)
    # a non-zero reserved field is rejected; NULL options are the defaults
    csr = B.bj_csr_t(A.n, A.nnz, rp.data_ptr(), ci.data_ptr(), val.data_ptr())
    o = B.bj_setup_opts_t()
    o.reserved[3] = 1
    out = C.c_void_p()
    assert B.lib().bj_setup_ex(C.byref(csr), 16, C.byref(o), C.byref(out)) == B.BJ_ERR_INVALID_ARG and not out.value
    assert B.lib().bj_setup_ex(C.byref(csr), 16, None, C.byref(out)) == B.BJ_OK
    B.lib().bj_destroy(out)


def test_setup_rejects_bad_inputs_in_the_middle_of_a_large_matrix(B, torch_):
    """a1 / a3 on a matrix that spans many CTAs of the validation kernels: a negative pivot deep inside (first bad block
    = the oracle's), swapped columns, a column out of range, row pointers that are not monotone or point far outside."""
    A = mat(2, "small")
    rp, ci, val = A.row_ptr, A.col_idx, A.val
    rows = np.repeat(np.arange(A.n), np.diff(rp))
    bad_val = val.copy()
    for r in (4001, 9000):
        bad_val[(rows == r) & (ci == r)] = -2.0
    swapped = ci.copy()
    s0 = rp[7000]
    swapped[s0], swapped[s0 + 1] = swapped[s0 + 1], swapped[s0]
    big = ci.copy()
    big[12345] = A.n + 5
    rp_bad = rp.copy()
    rp_bad[5000] = rp_bad[5001] + 3          # not monotone in the middle
    rp_wild = rp.copy()
    rp_wild[6000:6100] = 2 ** 30             # far outside the arrays
    for b in (8, 16):
        with pytest.raises(B.BJError) as e:
            B.bj_setup(dev(torch_, rp), dev(torch_, ci), dev(torch_, bad_val), b)
        assert e.value.code == B.BJ_ERR_NOT_SPD and e.value.bad_block == 4001 // b, b
        with pytest.raises(oracle.NotSPD) as eo:
            oracle.Precond(W.CSR(A.n, rp, ci, bad_val), b)
        assert eo.value.bad_block == e.value.bad_block
        for bad_ci in (swapped, big):
            with pytest.raises(B.BJError) as e:
                B.bj_setup(dev(torch_, rp), dev(torch_, bad_ci), dev(torch_, val), b)
            assert e.value.code == B.BJ_ERR_NOT_CANONICAL, b
        for bad_rp in (rp_bad, rp_wild):
            with pytest.raises(B.BJError) as e:
                B.bj_setup(dev(torch_, bad_rp), dev(torch_, ci), dev(torch_, val), b)
            assert e.value.code == B.BJ_ERR_NOT_CANONICAL, b


def test_tiny_and_degenerate_shapes(B, torch_, rel):
    # n = 1
    A = W.CSR(1, np.array([0, 1], np.int32), np.array([0], np.int32), np.array([4.0]))
    for b in (0, 1, 2):
        check_all_ops(B, torch_, A, b, rel, seeds=(1,), kernels=KERNELS)
    # empty rows are fine for SpMV (b = 0); with b >= 1 their zero diagonal is not SPD
    S = mat(3, "tiny").to_scipy().tolil()
    S[5, :] = 0
    S[:, 5] = 0
    A = W.from_scipy(S.tocsr())
    assert A.row_ptr[5] == A.row_ptr[6]
    check_all_ops(B, torch_, A, 0, rel, seeds=(1,), kernels=KERNELS)
    with pytest.raises(B.BJError) as e:
        B.setup_from_host(A, 4)
    assert e.value.code == B.BJ_ERR_NOT_SPD and e.value.bad_block == 1
    # one very long row (arrow matrix): exercises the long-row path of the SpMV kernels
    import scipy.sparse as sp
    n = 5000
    M = sp.lil_matrix((n, n))
    M.setdiag(np.full(n, 10.0 * n))
    M[0, :] = 1.0
    M[:, 0] = 1.0
    M[0, 0] = 10.0 * n
    A = W.from_scipy(M.tocsr())
    check_all_ops(B, torch_, A, 8, rel, seeds=(1,), kernels=KERNELS)


def test_host_buffer_entry_points(B, torch_, rel):
    A = mat(2, "small")
    h, keep = B.setup_from_host(A, 8)
    P = oracle.Precond(A, 8)
    x = W.seeded_vector(77, A.n)
    xh = torch_.from_numpy(x).pin_memory()
    yh = torch_.empty(A.n, dtype=torch_.float64).pin_memory()
    B.bj_op_apply_host(h, xh, yh)
    e2, ei = rel(yh.numpy(), P.op_apply(x))
    assert e2 <= TOL_APPLY and ei <= TOL_APPLY
    B.bj_apply_host(h, xh, yh)
    e2, ei = rel(yh.numpy(), P.apply(x))
    assert e2 <= TOL_APPLY and ei <= TOL_APPLY
    B.bj_destroy(h)


def test_runs_on_a_side_stream_and_profiling_counts(B, torch_, rel):
    A = mat(4, "small")
    s = torch_.cuda.Stream()
    with torch_.cuda.stream(s):
        h, keep = B.setup_from_host(A, 16)
        x = dev(torch_, W.seeded_vector(8, A.n))
        B.bj_profile_enable(h, True)
        for _ in range(5):
            y = B.bj_op_apply(h, x)
        s.synchronize()
        fused = B.bj_get_info(h)["fused_forward"]
        kinds = [B.bj_profile_get(h, k) for k in range(B.BJ_K_COUNT)]
        B.bj_profile_enable(h, False)
    assert kinds[B.BJ_K_SOLVE_LT][1] == 5
    if fused:
        assert kinds[B.BJ_K_SPMV_SOLVE_L][1] == 5
    else:
        assert kinds[B.BJ_K_SPMV][1] == 5 and kinds[B.BJ_K_SOLVE_L][1] == 5
    assert all(ms >= 0 for ms, _ in kinds)
    e2, _ = rel(y.cpu().numpy(), oracle.Precond(A, 16).op_apply(W.seeded_vector(8, A.n)))
    assert e2 <= TOL_APPLY
    B.bj_destroy(h)


def test_operator_apply_replays_from_a_cuda_graph(B, torch_, rel):
    """The library's launches (PDL-chained) can be captured on a side stream and replayed: bitwise the eager result."""
    for cfg, b in ((1, 4), (4, 16)):
        A = mat(cfg, "small")
        h, keep = B.setup_from_host(A, b)
        x = dev(torch_, W.seeded_vector(9, A.n))
        y_eager = B.bj_op_apply(h, x).clone()
        side = torch_.cuda.Stream()
        B.bj_set_stream(h, side)
        y = torch_.zeros_like(x)
        with torch_.cuda.stream(side):
            B.bj_op_apply(h, x, y)
            side.synchronize()
            y.zero_()
            g = torch_.cuda.CUDAGraph()
            with torch_.cuda.graph(g, stream=side):
                B.bj_op_apply(h, x, y)
                B.bj_op_apply(h, x, y)
            side.synchronize()
            assert not y.cpu().numpy().any()      # capture does not execute
            g.replay()
            side.synchronize()
        assert np.array_equal(y.cpu().numpy(), y_eager.cpu().numpy())
        B.bj_set_stream(h, torch_.cuda.current_stream())
        del g
        B.bj_destroy(h)


def test_banded_factor_path(B, torch_, rel):
    """SURVEY 8(f) NEXT-2, opt-in (bj_setup_opts_t.band): when every diagonal block is banded (w <= 2) the factor keeps the band and
    only (w+1) b doubles per block are stored and streamed.  Same parity bar as the dense-packed path; blocks that are
    not banded fall back to it."""
    import scipy.sparse as sp
    n = 5000
    T = sp.diags([-np.ones(n - 1), 2.5 * np.ones(n), -np.ones(n - 1)], [-1, 0, 1], format="csr")
    penta = W.from_scipy((T @ T).tocsr(), {"name": "pentadiagonal"})        # w = 2 inside every block
    cases = [(mat(4, "small"), 16, 1), (mat(2, "small"), 16, 1), (mat(4, "small"), 32, 1), (penta, 24, 2), (penta, 9, 2),
             (W.block_diagonal_spd(2000, 1), 16, 0), (mat(3, "small"), 32, None), (mat(5, "small"), 24, None)]
    for A, b, w in cases:
        h, keep = B.setup_from_host(A, b, band=1)
        info = B.bj_get_info(h)
        if w is None:
            assert info["solve_kernel"] == 2 and info["band_width"] == -1     # not banded: dense packed factors
        else:
            assert info["solve_kernel"] == 3 and info["band_width"] == w, (b, info)
            assert info["factor_bytes"] < 8 * A.n * (w + 1) + 8 * 32 * (w + 1) * b + 1
        B.bj_destroy(h)
        check_all_ops(B, torch_, A, b, rel, seeds=(3,), kernels=((1, 0),), band=1)
        h, keep = B.setup_from_host(A, b, band=1)
        P = oracle.Precond(A, b)
        g = B.bj_cond_estimate_ex(h, 20, reorth=True)
        c = P.cond_estimate(20, reorth=True)
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
        g = B.bj_cond_estimate_ex(h, 20, reorth=False)       # fused Lanczos step: hooks of the band solve kernel
        c = P.cond_estimate(20, reorth=False)
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
        rhs = W.seeded_vector(5, A.n)
        gp = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=8, rtol=0.0)   # fused PCG iteration
        cp = P.pcg(rhs, 8, 0.0)
        if w != 0:   # w = 0 is M = A: one exact step, everything after it is rounding noise
            assert np.allclose(gp["alpha"], cp["alpha"], rtol=1e-9, atol=0)
            assert np.allclose(gp["relres_hist"], cp["relres"], rtol=1e-9, atol=0)
        else:
            assert abs(gp["alpha"][0] - 1.0) <= 1e-12 and gp["relres_hist"][0] <= 1e-14
        B.bj_destroy(h)
    # a banded block that is not positive definite is reported like any other
    bad = sp.diags([-np.ones(n - 1), np.r_[2.5 * np.ones(n - 40), -1.0, 2.5 * np.ones(39)], -np.ones(n - 1)], [-1, 0, 1], format="csr")
    Ab = W.from_scipy(bad, {"name": "indefinite tridiagonal"})
    with pytest.raises(B.BJError) as ei:
        B.setup_from_host(Ab, 16, band=1)
    assert ei.value.code == B.BJ_ERR_NOT_SPD and ei.value.bad_block == (n - 40) // 16


def test_tridiagonal_compact_factors_small_blocks(B, torch_, rel):
    """bj_setup_opts_t.band with b <= 8: tridiagonal blocks keep 2b - 1 factor elements; the same kernels run (thread per block,
    fused SpMV + solve, fused Lanczos and PCG hooks) with a compact index map."""
    import scipy.sparse as sp
    n = 3001
    T = sp.diags([-np.ones(n - 1), 2.5 * np.ones(n), -np.ones(n - 1)], [-1, 0, 1], format="csr")
    penta = W.from_scipy((T @ T).tocsr(), {"name": "pentadiagonal"})
    for A, b, tri in ((mat(2, "small"), 8, True), (mat(4, "small"), 8, True), (mat(1, "small"), 4, True),
                      (mat(2, "small"), 5, True), (penta, 8, False), (mat(5, "small"), 3, False)):
        h, keep = B.setup_from_host(A, b, band=1)
        info = B.bj_get_info(h)
        assert info["solve_kernel"] == 1
        assert (info["band_width"] == 1) == tri, (b, info)
        if tri:
            assert info["factor_bytes"] == ((A.n + b - 1) // b + 31) // 32 * 32 * (2 * b - 1) * 8
        P = oracle.Precond(A, b)
        g = B.bj_cond_estimate_ex(h, 30, reorth=False)      # fused Lanczos step on the compact factors
        c = P.cond_estimate(30, reorth=False)
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
        rhs = W.seeded_vector(5, A.n)
        gp = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=8, rtol=0.0)   # fused PCG iteration
        cp = P.pcg(rhs, 8, 0.0)
        assert np.allclose(gp["alpha"], cp["alpha"], rtol=1e-9, atol=0)
        B.bj_destroy(h)
        check_all_ops(B, torch_, A, b, rel, seeds=(3,), kernels=KERNELS, band=1)


def test_batched_small_systems(B, torch_, rel):
    """a batch of independent N = 1024 systems (the paper's smallest size) in one
    block-diagonal CSR.  Per system the kappa estimate equals the oracle's Lanczos on that system alone with the same
    start-vector slice; the operator apply equals the per-system applies."""
    nsys, m = 12, 30
    A = W.batch_poisson(nsys, 32)
    seg = A.meta["seg"]
    v0 = W.seeded_vector(B.BJ_DEFAULT_SEED, A.n)
    for b in (0, 1, 4, 16):
        h, keep = B.setup_from_host(A, b)
        g = B.bj_cond_estimate_batch(h, nsys, m)
        x = W.seeded_vector(7, A.n)
        y = B.bj_op_apply(h, dev(torch_, x)).cpu().numpy()
        for s in range(nsys):
            As = W.batch_system(A, s)
            P = oracle.Precond(As, b)
            c = P.cond_estimate(m, v0=v0[s * seg:(s + 1) * seg], reorth=False)
            assert g["iters_done"][s] == c["iters_done"]
            assert abs(g["kappa"][s] / c["kappa"] - 1) <= TOL_KAPPA, (b, s, g["kappa"][s], c["kappa"])
            e2, ei = rel(y[s * seg:(s + 1) * seg], P.op_apply(x[s * seg:(s + 1) * seg]))
            assert e2 <= TOL_APPLY and ei <= TOL_APPLY
        assert len(set(np.round(g["kappa"], 6))) == nsys          # every system has its own spectrum
        B.bj_destroy(h)
    # the solve side: per-system PCG, each system with its own stopping iteration
    h, keep = B.setup_from_host(A, 4)
    rhs = W.seeded_vector(17, A.n)
    rhs[3 * seg:4 * seg] = 0.0                                    # one system has nothing to solve
    g = B.bj_pcg_solve_batch(h, nsys, dev(torch_, rhs), max_iters=200, rtol=1e-8)
    xg = g["x"].cpu().numpy()
    for s in range(nsys):
        c = oracle.Precond(W.batch_system(A, s), 4).pcg(rhs[s * seg:(s + 1) * seg], 200, 1e-8)
        assert abs(int(g["iters"][s]) - c["iters"]) <= 1, (s, g["iters"][s], c["iters"])
        if s == 3:
            assert g["iters"][s] == 0 and not xg[s * seg:(s + 1) * seg].any()
            continue
        e2, ei = rel(xg[s * seg:(s + 1) * seg], c["x"])
        assert e2 <= 1e-7 and g["relres"][s] <= 1e-8 and g["true_relres"][s] <= 2e-8, (s, e2)
    assert len(set(g["iters"].tolist())) > 1                      # the systems really stop at different steps
    B.bj_destroy(h)
    # systems of DIFFERENT sizes in one batch: the paper's three sizes N = 2^10, 2^12, 2^14 side by side
    Am = W.batch_poisson_mixed([32, 64, 32, 128, 16])
    off = Am.meta["offsets"]
    ns = len(off) - 1
    v0m = W.seeded_vector(B.BJ_DEFAULT_SEED, Am.n)
    h, keep = B.setup_from_host(Am, 4)
    g = B.bj_cond_estimate_batch(h, ns, 25, offsets=off)
    rhs = W.seeded_vector(21, Am.n)
    gp = B.bj_pcg_solve_batch(h, ns, dev(torch_, rhs), max_iters=300, rtol=1e-8, offsets=off)
    xg = gp["x"].cpu().numpy()
    for s in range(ns):
        P = oracle.Precond(W.batch_member(Am, s), 4)
        lo, hi = int(off[s]), int(off[s + 1])
        c = P.cond_estimate(25, v0=v0m[lo:hi], reorth=False)
        assert abs(g["kappa"][s] / c["kappa"] - 1) <= TOL_KAPPA, (s, g["kappa"][s], c["kappa"])
        cp = P.pcg(rhs[lo:hi], 300, 1e-8)
        assert abs(int(gp["iters"][s]) - cp["iters"]) <= 1
        e2, ei = rel(xg[lo:hi], cp["x"])
        assert e2 <= 1e-7, (s, e2)
    with pytest.raises(B.BJError):
        B.bj_cond_estimate_batch(h, ns, 5, offsets=np.r_[off[:-1], off[-1] - 4])      # offsets must end at n
    with pytest.raises(B.BJError):
        B.bj_cond_estimate_batch(h, ns, 5, offsets=np.r_[0, off[1] + 2, off[2:]])      # ... and fall on block boundaries
    B.bj_destroy(h)
    # a matrix with an entry that couples two systems is rejected (every per-system result would be silently wrong)
    h, keep = B.setup_from_host(mat(1, "full"), 4)
    with pytest.raises(B.BJError) as e:
        B.bj_cond_estimate_batch(h, 2, 5)                  # one 32 x 32 grid cut in two halves: rows 15 | 16 are coupled
    assert e.value.code == B.BJ_ERR_INVALID_ARG
    with pytest.raises(B.BJError) as e:
        B.bj_pcg_solve_batch(h, 2, dev(torch_, W.seeded_vector(3, 1024)), max_iters=5, rtol=0.0)
    assert e.value.code == B.BJ_ERR_INVALID_ARG
    B.bj_destroy(h)
    # a system whose residual becomes EXACTLY zero while the stopping test cannot fire (rtol < 0) is frozen where it stands
    # instead of taking the step length 0 / 0: A = 2 I without preconditioner makes every quantity of step 1 exact
    # (z = r, a = 1/2, r_new = 0)
    nd = 64
    Ad = W.CSR(nd, np.arange(nd + 1, dtype=np.int32), np.arange(nd, dtype=np.int32), np.full(nd, 2.0))
    h, keep = B.setup_from_host(Ad, 0)
    rhs = W.seeded_vector(4, nd)
    g = B.bj_pcg_solve_batch(h, 4, dev(torch_, rhs), max_iters=6, rtol=-1.0)
    assert np.array_equal(g["x"].cpu().numpy(), rhs / 2.0) and (g["iters"] == 1).all() and (g["true_relres"] == 0.0).all()
    B.bj_destroy(h)
    # a system whose preconditioner is exact breaks down at step 1 while the others go on
    Ab = W.block_diagonal_spd(64, 8)
    h, keep = B.setup_from_host(Ab, 8)
    g = B.bj_cond_estimate_batch(h, 4, 10)
    assert (g["iters_done"] == 1).all() and np.allclose(g["kappa"], 1.0, atol=1e-12)
    with pytest.raises(B.BJError):
        B.bj_cond_estimate_batch(h, 5, 10)       # 512 rows do not split into 5 systems
    B.bj_destroy(h)


def test_16_bit_column_deltas(B, torch_, rel):
    """SURVEY 8(f) NEXT-2, opt-in (bj_setup_opts_t.col16): when every |col - row| < 32768 the tile kernel streams the columns as
    int16 deltas (10 bytes per entry instead of 12); bit-identical products (same values, same order)."""
    for cfg, b in ((2, 8), (4, 8), (1, 4), (3, 4), (4, 16), (5, 3)):
        A = mat(cfg, "small")
        x = dev(torch_, W.seeded_vector(6, A.n))
        h_ref, keep_ref = B.setup_from_host(A, b)
        h, keep = B.setup_from_host(A, b, col16=1)          # two handles of one process, different options
        assert B.bj_get_info(h)["col16"] == 1 and B.bj_get_info(h_ref)["col16"] == 0
        ref_spmv, ref_op = B.bj_spmv(h_ref, x).clone(), B.bj_op_apply(h_ref, x).clone()
        B.bj_destroy(h_ref)
        assert np.array_equal(B.bj_spmv(h, x).cpu().numpy(), ref_spmv.cpu().numpy())
        assert np.array_equal(B.bj_op_apply(h, x).cpu().numpy(), ref_op.cpu().numpy())
        P = oracle.Precond(A, b)
        g = B.bj_cond_estimate_ex(h, 15, reorth=False)       # the hooked kernels keep the 32-bit columns
        assert abs(g["kappa"] / P.cond_estimate(15, reorth=False)["kappa"] - 1) <= TOL_KAPPA
        B.bj_destroy(h)
    # a matrix with a far off-diagonal keeps the 32-bit stream
    import scipy.sparse as sp
    n = 70000
    far = sp.diags([np.full(n, 4.0), np.full(n - 40000, -1.0), np.full(n - 40000, -1.0)], [0, 40000, -40000], format="csr")
    h, keep = B.setup_from_host(W.from_scipy(far), 4, col16=1)
    assert B.bj_get_info(h)["col16"] == 0
    B.bj_destroy(h)
    check_all_ops(B, torch_, mat(2, "small"), 8, rel, seeds=(3,), kernels=KERNELS, col16=1)


def test_bsr3_matrix_copy(B, torch_, rel):
    """SURVEY 8(f) NEXT-2, opt-in (bj_setup_opts_t.bsr): a 3x3-blocked matrix (config 5: three dofs per node) is also kept as BSR(3)
    -- 8.44 bytes per entry instead of 12 -- and every product of the path runs from that copy; a matrix without the block
    structure keeps the CSR kernels."""
    A = mat(5, "small")
    for b in (0, 3, 24, 6):
        h, keep = B.setup_from_host(A, b, bsr=1)
        assert B.bj_get_info(h)["spmv_kernel"] == 2
        P = oracle.Precond(A, b)
        for seed in (3, 4):
            x = W.seeded_vector(seed, A.n)
            xd = dev(torch_, x)
            for name, got, ref in (("spmv", B.bj_spmv(h, xd), oracle.spmv(A, x)), ("op_apply", B.bj_op_apply(h, xd), P.op_apply(x))):
                e2, ei = rel(got.cpu().numpy(), ref)
                assert e2 <= TOL_APPLY and ei <= TOL_APPLY, (b, name, e2, ei)
        g = B.bj_cond_estimate_ex(h, 20, reorth=True)
        c = P.cond_estimate(20, reorth=True)
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
        if b:
            g = B.bj_cond_estimate_ex(h, 20, reorth=False)
            c = P.cond_estimate(20, reorth=False)
            assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
        rhs = W.seeded_vector(5, A.n)
        gp = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=8, rtol=0.0)
        cp = P.pcg(rhs, 8, 0.0)
        assert np.allclose(gp["alpha"], cp["alpha"], rtol=1e-9, atol=0)
        B.bj_set_option(h, B.BJ_OPT_SPMV_KERNEL, 1)            # the CSR kernels stay selectable
        assert B.bj_get_info(h)["spmv_kernel"] in (0, 1)
        B.bj_destroy(h)
    for cfg in (2, 3):                                         # no 3x3 block structure: CSR kernels
        h, keep = B.setup_from_host(mat(cfg, "small"), 3, bsr=1)
        assert B.bj_get_info(h)["spmv_kernel"] in (0, 1)
        B.bj_destroy(h)
    # a matrix whose size and entry count are multiples of 3 and 9 but whose pattern is not blocked
    h, keep = B.setup_from_host(W.block_diagonal_spd(27, 9), 3, bsr=1)
    info = B.bj_get_info(h)
    B.bj_destroy(h)
    assert info["spmv_kernel"] == 2                            # 9x9 dense blocks ARE 3x3-blocked
    h, keep = B.setup_from_host(W.laplacian((9, 9, 9)), 3, bsr=1)
    assert B.bj_get_info(h)["spmv_kernel"] in (0, 1)
    B.bj_destroy(h)


def test_block_size_sweep_runs_the_real_path(B, torch_):
    """a11: host-side sweep over b; kappa estimates agree with the oracle at the chosen b; b = N/.. ordering sane."""
    from paper_2410_02408_b200 import sweep
    A = mat(1, "full")
    rp, ci, val = dev(torch_, A.row_ptr), dev(torch_, A.col_idx), dev(torch_, A.val)
    res = sweep.sweep(rp, ci, val, blocks=(1, 4, 32), iters=50, apply_steps=20)
    assert [r["b"] for r in res["rows"]] == [1, 4, 32]
    for r in res["rows"]:
        c = oracle.Precond(A, r["b"]).cond_estimate(50)
        assert abs(r["kappa_est"] / c["kappa"] - 1) <= TOL_KAPPA
        assert r["applies_per_s"] > 0 and r["setup_ms"] > 0
    c0 = oracle.Precond(A, 0).cond_estimate(50)
    assert abs(res["kappa_A"]["kappa_est"] / c0["kappa"] - 1) <= TOL_KAPPA
    assert res["best_b"] == sweep.pick_best(res["rows"])["b"]


# ------------------------------------------------------------------ BASELINE.json full sizes -------------
@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_full_size_configs(B, torch_, rel, cfg):
    """Full-size matrices in the launch configuration bench.py times: whole-vector parity of every op
    (the oracle finishes one apply in well under a second), kappa parity at a reduced step count for
    the preconditioned operator, and the 2-cyclic invariant where it holds."""
    A = mat(cfg, "full")
    for b in W.BLOCK_SIZES[cfg]:
        check_all_ops(B, torch_, A, b, rel, seeds=(31,))
        h, keep = B.setup_from_host(A, b)
        P = oracle.Precond(A, b)
        m = 50 if cfg == 2 else 16
        g = B.bj_cond_estimate_ex(h, m, reorth=True)
        c = P.cond_estimate(m, reorth=True)
        assert g["iters_done"] == c["iters_done"] == m
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (cfg, b, g["kappa"], c["kappa"])
        # The FUSED fast mode on the default kernels -- the path bench.py times (`fast_mode`, `long_run`): at full size the
        # hooked solve / SpMV kernels take several ring passes per warp and close their sums with many-CTA tickets, which the
        # `small` matrices never reach.  Coefficients of the first 12 steps element by element, kappa at m = 50.
        for name, gpu_fn, cpu_fn in (("split", lambda k: B.bj_cond_estimate_ex(h, k, reorth=False),
                                      lambda k: P.cond_estimate(k, reorth=False)),
                                     ("minv", lambda k: B.bj_cond_estimate_minv(h, k), lambda k: P.cond_estimate_minv(k))):
            c50 = cpu_fn(50)
            g12, g50 = gpu_fn(12), gpu_fn(50)
            sc = np.abs(c50["alpha"]).max()
            assert g12["iters_done"] == 12 and g50["iters_done"] == c50["iters_done"] == 50
            assert np.abs(g12["alpha"] - c50["alpha"][:12]).max() <= 1e-9 * sc, (cfg, b, name)
            assert np.abs(g12["beta"] - c50["beta"][:12]).max() <= 1e-9 * sc, (cfg, b, name)
            assert np.abs(g50["alpha"][:12] - c50["alpha"][:12]).max() <= 1e-9 * sc, (cfg, b, name)
            assert abs(g50["kappa"] / c50["kappa"] - 1) <= TOL_KAPPA, (cfg, b, name, g50["kappa"], c50["kappa"])
        if cfg == 2:
            lmin, lmax = B.bj_cond_estimate(h, 50)      # the 4-argument call of the north star, full size
            assert abs((lmax / lmin) / c["kappa"] - 1) <= TOL_KAPPA
        B.bj_destroy(h)
        del h, keep
    if cfg == 2:
        # kappa(A) itself (b = 0, parity mode, m = 50): the value the bench line prints as kappa.A
        h, keep = B.setup_from_host(A, 0)
        g = B.bj_cond_estimate_ex(h, 50, reorth=True)
        c = oracle.Precond(A, 0).cond_estimate(50, reorth=True)
        assert g["iters_done"] == c["iters_done"] == 50
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (g["kappa"], c["kappa"])
        B.bj_destroy(h)
        del h, keep
    _MATS.pop((cfg, "full"), None)
    torch_.cuda.empty_cache()


# ------------------------------------------------------------------ PCG -------------
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_pcg_matches_oracle_small(B, torch_, rel, cfg):
    """Same rhs as the oracle's textbook PCG.  (i) A fixed, short run (rounding has not been amplified yet: CG
    coefficients are as sensitive as unreorthogonalised Lanczos): step lengths, residual history, x and the
    CG-Lanczos spectrum estimate agree tightly.  (ii) A run to the paper's accuracy bar 1e-3: both
    stop within a step or two of each other and meet the bar; the reported true residual is ||Ax - b|| / ||b||
    (PAPER.md:136), checked against scipy."""
    import scipy.sparse as sp
    A = mat(cfg, "small")
    S = sp.csr_matrix((A.val, A.col_idx, A.row_ptr), shape=(A.n, A.n))
    rhs = W.seeded_vector(17, A.n)
    for b in [0] + W.BLOCK_SIZES[cfg]:
        h, keep = B.setup_from_host(A, b)
        P = oracle.Precond(A, b)
        k = 12
        g = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=k, rtol=0.0, check_every=5)
        c = P.pcg(rhs, k, 0.0)
        assert g["iters"] == c["iters"] == k and not g["converged"]
        assert np.allclose(g["alpha"], c["alpha"], rtol=1e-9, atol=0), (cfg, b)
        assert np.allclose(g["beta"], c["beta"], rtol=1e-9, atol=0), (cfg, b)
        assert np.allclose(g["relres_hist"], c["relres"], rtol=1e-9, atol=0)
        xg = g["x"].cpu().numpy()
        e2, ei = rel(xg, c["x"])
        # an iteration, not an apply: the O(eps sqrt N) differences between the GPU's tree sums and the oracle's serial
        # dot products pass through the coefficient formulas (kappa up to 1e6 at b = 0); DESIGN.md section 3
        assert e2 <= 1e-9 and ei <= 1e-7, (cfg, b, e2, ei)
        tr = np.linalg.norm(S @ xg - rhs) / np.linalg.norm(rhs)
        assert abs(g["true_relres"] - tr) <= 1e-10 * tr
        d, e = oracle.cg_tridiag(c["alpha"], c["beta"])
        ev = np.linalg.eigvalsh(np.diag(d) + np.diag(e, 1) + np.diag(e, -1))
        assert abs(g["lmin"] / ev[0] - 1) <= 1e-6 and abs(g["lmax"] / ev[-1] - 1) <= 1e-6
        # to the paper's bar
        cap = 600
        g = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=cap, rtol=1e-3, check_every=7)
        c = P.pcg(rhs, cap, 1e-3)
        assert abs(g["iters"] - c["iters"]) <= max(2, c["iters"] // 50), (cfg, b, g["iters"], c["iters"])
        if c["iters"] < cap - 2:
            assert g["converged"] and g["relres"] <= 1e-3 and g["true_relres"] <= 1.2e-3
            xg = g["x"].cpu().numpy()
            tr = np.linalg.norm(S @ xg - rhs) / np.linalg.norm(rhs)
            assert abs(g["true_relres"] - tr) <= 1e-9 * tr
        B.bj_destroy(h)


@pytest.mark.parametrize("fuse", [0, 1])
def test_pcg_fused_and_unfused_iterations_agree(B, torch_, rel, fuse):
    """BJ_OPT_PCG_FUSE = 0 runs the seven-kernel iteration of bj_pcg.cu, the default rides on the SpMV and solve kernels
    (three kernels per iteration): both follow the oracle, for every solve kernel (b = 3, 8: thread per block; 16, 24, 32:
    group per block; 12: no hook -> unfused either way)."""
    A = mat(2, "small")
    rhs = W.seeded_vector(23, A.n)
    for b in (3, 8, 12, 16, 24, 32):
        h, keep = B.setup_from_host(A, b)
        B.bj_set_option(h, B.BJ_OPT_PCG_FUSE, fuse)
        g = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=10, rtol=0.0, check_every=4)
        c = oracle.Precond(A, b).pcg(rhs, 10, 0.0)
        assert g["iters"] == 10
        assert np.allclose(g["alpha"], c["alpha"], rtol=1e-9, atol=0) and np.allclose(g["beta"], c["beta"], rtol=1e-9, atol=0), b
        assert np.allclose(g["relres_hist"], c["relres"], rtol=1e-9, atol=0)
        e2, ei = rel(g["x"].cpu().numpy(), c["x"])
        assert e2 <= 1e-9, (b, e2)
        g = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=500, rtol=1e-6, check_every=16)
        c = oracle.Precond(A, b).pcg(rhs, 500, 1e-6)
        assert g["converged"] and abs(g["iters"] - c["iters"]) <= max(2, c["iters"] // 50) and g["true_relres"] <= 2e-6
        B.bj_destroy(h)


def test_pcg_single_launch_on_the_papers_sizes(B, torch_, rel):
    """N = 2^10 and 2^12: bj_pcg_solve runs as ONE kernel of one cluster (8 / 16 CTAs).  Against the oracle's
    textbook PCG and against the multi-launch iteration on the same handle: coefficients, residual history, x, the paper's
    residual; zero right-hand side; exact preconditioner; ragged last block."""
    import scipy.sparse as sp
    for A, blocks in ((W.config1(32), (0, 1, 4, 7, 8)), (W.config1(64), (4, 8)), (W.laplacian((37, 29)), (5,))):
        S = sp.csr_matrix((A.val, A.col_idx, A.row_ptr), shape=(A.n, A.n))
        rhs = W.seeded_vector(23, A.n)
        rd = dev(torch_, rhs)
        for b in blocks:
            h, keep = B.setup_from_host(A, b)
            P = oracle.Precond(A, b)
            l0 = B.bj_get_info(h)["kernel_launches"]
            g = B.bj_pcg_solve(h, rd, max_iters=10, rtol=0.0)
            assert B.bj_get_info(h)["kernel_launches"] - l0 == 1, (A.n, b)
            c = P.pcg(rhs, 10, 0.0)
            assert g["iters"] == c["iters"] == 10 and not g["converged"]
            assert np.allclose(g["alpha"], c["alpha"], rtol=1e-9, atol=0) and np.allclose(g["beta"], c["beta"], rtol=1e-9, atol=0)
            assert np.allclose(g["relres_hist"], c["relres"], rtol=1e-9, atol=0)
            xg = g["x"].cpu().numpy()
            e2, ei = rel(xg, c["x"])
            assert e2 <= 1e-10 and ei <= 1e-9, (A.n, b, e2, ei)
            tr = np.linalg.norm(S @ xg - rhs) / np.linalg.norm(rhs)
            assert abs(g["true_relres"] - tr) <= 1e-10 * tr
            g = B.bj_pcg_solve(h, rd, max_iters=400, rtol=1e-8)
            c = P.pcg(rhs, 400, 1e-8)
            assert g["converged"] and abs(g["iters"] - c["iters"]) <= 1 and g["true_relres"] <= 2e-8, (A.n, b, g["iters"], c["iters"])
            B.bj_set_option(h, B.BJ_OPT_PCG_SINGLE_LAUNCH, 0)      # the multi-launch iteration on the same handle
            l0 = B.bj_get_info(h)["kernel_launches"]
            gm = B.bj_pcg_solve(h, rd, max_iters=400, rtol=1e-8)
            assert B.bj_get_info(h)["kernel_launches"] - l0 > 20
            assert gm["iters"] == g["iters"] and rel(g["x"].cpu().numpy(), gm["x"].cpu().numpy())[0] <= 1e-10
            B.bj_set_option(h, B.BJ_OPT_PCG_SINGLE_LAUNCH, 1)
            z = B.bj_pcg_solve(h, torch_.zeros_like(rd), max_iters=5, rtol=1e-3)
            assert z["iters"] == 0 and float(z["x"].abs().max()) == 0.0
            B.bj_destroy(h)
    A = W.block_diagonal_spd(100, 8)          # M = A: one step
    h, keep = B.setup_from_host(A, 8)
    rhs = W.seeded_vector(5, A.n)
    g = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=20, rtol=1e-10)
    assert g["iters"] == 1 and g["converged"] and g["true_relres"] <= 1e-12
    B.bj_destroy(h)


def test_pcg_degenerate_cases(B, torch_, rel):
    A = W.block_diagonal_spd(65, 8)     # M = A: one step
    h, keep = B.setup_from_host(A, 8)
    rhs = W.seeded_vector(5, A.n)
    g = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=10, rtol=1e-12)
    assert g["iters"] == 1 and g["converged"] and abs(g["alpha"][0] - 1) <= 1e-12 and g["true_relres"] <= 1e-13
    z = torch_.zeros(A.n, dtype=torch_.float64, device="cuda")
    g = B.bj_pcg_solve(h, z, max_iters=10, rtol=1e-3)
    assert g["iters"] == 0 and not g["x"].cpu().numpy().any()
    with pytest.raises(B.BJError):
        B.bj_pcg_solve(h, z, x=z, max_iters=10)
    B.bj_destroy(h)


@pytest.mark.parametrize("cfg", [2, 4])
def test_pcg_full_size(B, torch_, rel, cfg):
    """Full-size matrix in the launch configuration the benchmark uses: a short fixed run agrees with the oracle
    (step lengths, x), true residual recomputed on the host."""
    import scipy.sparse as sp
    A = mat(cfg, "full")
    b = W.BLOCK_SIZES[cfg][0]
    S = sp.csr_matrix((A.val, A.col_idx, A.row_ptr), shape=(A.n, A.n))
    rhs = W.seeded_vector(17, A.n)
    h, keep = B.setup_from_host(A, b)
    g = B.bj_pcg_solve(h, dev(torch_, rhs), max_iters=12, rtol=0.0)
    c = oracle.Precond(A, b).pcg(rhs, 12, 0.0)
    assert g["iters"] == c["iters"] == 12
    assert np.allclose(g["alpha"], c["alpha"], rtol=1e-9, atol=0) and np.allclose(g["beta"], c["beta"], rtol=1e-9, atol=0)
    e2, ei = rel(g["x"].cpu().numpy(), c["x"])
    assert e2 <= 1e-9, (cfg, e2)
    tr = np.linalg.norm(S @ g["x"].cpu().numpy() - rhs) / np.linalg.norm(rhs)
    assert abs(g["true_relres"] - tr) <= 1e-9 * tr
    B.bj_destroy(h)
    del h, keep
    _MATS.pop((cfg, "full"), None)
    torch_.cuda.empty_cache()


@pytest.mark.parametrize("cfg,b,env", [(2, 8, {"band": 1, "col16": 1}), (4, 16, {"band": 1, "col16": 1}), (5, 3, {"bsr": 1})])
def test_full_size_opt_in_variants(B, torch_, rel, cfg, b, env):
    """The byte-reducing variants at BASELINE.json's full sizes, in the launch configuration
    `bench.py --band 1 --col16 1` / `--bsr 1` times (options of bj_setup_ex): whole-vector parity of every op with the oracle, and a short kappa run."""
    A = mat(cfg, "full")
    h, keep = B.setup_from_host(A, b, **env)
    info = B.bj_get_info(h)
    if "band" in env:
        assert info["band_width"] == 1 and info["col16"] == 1
    if "bsr" in env:
        assert info["spmv_kernel"] == 2
    P = oracle.Precond(A, b)
    g = B.bj_cond_estimate_ex(h, 12, reorth=False)
    c = P.cond_estimate(12, reorth=False)
    assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
    B.bj_destroy(h)
    del h, keep
    check_all_ops(B, torch_, A, b, rel, seeds=(31,), **env)
    _MATS.pop((cfg, "full"), None)
    torch_.cuda.empty_cache()


def test_handles_release_their_device_memory(B, torch_):
    """Setup / Lanczos / PCG / batch / BSR / 16-bit-column workspaces all belong to the handle: after destroy and
    bj_release_cached_memory the free device memory is back where it started."""
    A = mat(5, "small")
    rp, ci, val = (torch_.from_numpy(a).cuda() for a in (A.row_ptr, A.col_idx, A.val))
    x = dev(torch_, W.seeded_vector(1, A.n))
    Ab = W.batch_poisson(4, 32)
    rpb, cib, valb = (torch_.from_numpy(a).cuda() for a in (Ab.row_ptr, Ab.col_idx, Ab.val))
    xb = dev(torch_, W.seeded_vector(2, Ab.n))
    torch_.cuda.synchronize()
    B.bj_release_cached_memory()
    free0, _ = torch_.cuda.mem_get_info()
    for rep in range(12):
        for b in (0, 3, 8, 24):
            h = B.bj_setup(rp, ci, val, b, band=1, col16=1, bsr=1)
            B.bj_op_apply(h, x)
            B.bj_cond_estimate_ex(h, 6, reorth=bool(rep & 1))
            B.bj_pcg_solve(h, x, max_iters=4, rtol=0.0)
            B.bj_destroy(h)
        hb = B.bj_setup(rpb, cib, valb, 4, band=1)          # batch workspaces (a block-diagonal batch of four systems)
        B.bj_cond_estimate_batch(hb, 4, 4)
        B.bj_pcg_solve_batch(hb, 4, xb, max_iters=3, rtol=0.0)
        B.bj_destroy(hb)
    torch_.cuda.synchronize()
    torch_.cuda.empty_cache()
    B.bj_release_cached_memory()
    free1, _ = torch_.cuda.mem_get_info()
    assert free0 - free1 <= 64 << 20, (free0, free1)


# ------------------------------------------------------------------ Lanczos on M^-1 A (NEXT-2) ----------
@pytest.mark.parametrize("fuse", [1, 0])
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_minv_lanczos_matches_oracle_small(B, torch_, cfg, fuse):
    """bj_cond_estimate_minv (one factor pass per step) against the oracle's M-inner-product Lanczos: the first coefficients
    element by element, kappa at m = 50 to the bar of the north star.  fuse=1: two kernels per step where the solve kernel
    carries the hook; fuse=0: the six-kernel step (also the path of b = 0 and of block sizes without a hooked kernel)."""
    A = mat(cfg, "small")
    for b in ([0] if fuse == 0 else []) + W.BLOCK_SIZES[cfg]:
        h, keep = B.setup_from_host(A, b)
        B.bj_set_option(h, B.BJ_OPT_PCG_FUSE, fuse)
        P = oracle.Precond(A, b)
        g = B.bj_cond_estimate_minv(h, 12)
        c = P.cond_estimate_minv(12)
        assert g["iters_done"] == c["iters_done"] == 12
        sc = np.abs(c["alpha"]).max()
        assert np.abs(g["alpha"] - c["alpha"]).max() <= 1e-9 * sc, (cfg, b)
        assert np.abs(g["beta"] - c["beta"]).max() <= 1e-9 * sc, (cfg, b)
        if b > 0:   # without reorthogonalisation kappa at m = 50 is reproducible on the preconditioned operators only
            g = B.bj_cond_estimate_minv(h, 50)
            c = P.cond_estimate_minv(50)
            assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (cfg, b, g["kappa"], c["kappa"])
            assert abs(g["res_min"] - c["res_min"]) <= 1e-6 * c["lmax"] and abs(g["res_max"] - c["res_max"]) <= 1e-6 * c["lmax"]
        B.bj_destroy(h)


def test_minv_lanczos_is_the_split_lanczos_from_Linv_r0(B, torch_):
    """Both device estimates see one spectrum: T of bj_cond_estimate_minv from r_0 equals T of bj_cond_estimate_ex started at
    v_0 = L^-1 r_0 (bj_solve_L) for the first steps, and a caller-supplied r_0 is honoured."""
    A = mat(4, "small")
    h, keep = B.setup_from_host(A, 16)
    r0 = dev(torch_, W.seeded_vector(31, A.n))
    g1 = B.bj_cond_estimate_minv(h, 8, r0=r0)
    v0 = torch_.empty_like(r0)
    B.bj_solve_L(h, r0, v0)
    g2 = B.bj_cond_estimate_ex(h, 8, reorth=False, v0=v0)
    sc = np.abs(g2["alpha"]).max()
    assert np.abs(g1["alpha"] - g2["alpha"]).max() <= 1e-9 * sc and np.abs(g1["beta"] - g2["beta"]).max() <= 1e-9 * sc
    c = oracle.Precond(A, 16).cond_estimate_minv(8, r0=r0.cpu().numpy())
    assert np.abs(g1["alpha"] - c["alpha"]).max() <= 1e-9 * sc
    B.bj_destroy(h)


def test_minv_lanczos_degenerate_cases(B, torch_):
    A = W.block_diagonal_spd(65, 8)     # M = A: M^-1 A = I, breakdown after one step, kappa = 1
    h, keep = B.setup_from_host(A, 8)
    g = B.bj_cond_estimate_minv(h, 10)
    assert g["iters_done"] == 1 and abs(g["alpha"][0] - 1) <= 1e-12 and abs(g["kappa"] - 1) <= 1e-12
    z = torch_.zeros(A.n, dtype=torch_.float64, device="cuda")
    with pytest.raises(B.BJError):
        B.bj_cond_estimate_minv(h, 10, r0=z)
    B.bj_destroy(h)


def test_minv_lanczos_banded_factors(B, torch_):
    A = mat(4, "small")
    h, keep = B.setup_from_host(A, 16, band=1)
    assert B.bj_get_info(h)["band_width"] >= 1
    g = B.bj_cond_estimate_minv(h, 50)
    c = oracle.Precond(A, 16).cond_estimate_minv(50)
    assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA
    B.bj_destroy(h)


# ------------------------------------------------------------------ variable-size blocks (NEXT-3) --------
def _setup_blocks(B, torch_, A, ptr):
    rp, ci, val = dev(torch_, A.row_ptr), dev(torch_, A.col_idx), dev(torch_, A.val)
    return B.bj_setup_blocks(rp, ci, val, ptr), (rp, ci, val)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_variable_blocks_match_oracle(B, torch_, rel, cfg):
    """bj_setup_blocks with seeded block sizes 1..32 (several hundred blocks, ragged last block): every apply entry point
    element by element against oracle.PrecondBlocks, kappa with full reorthogonalisation to the bar of the north star."""
    A = mat(cfg, "tiny" if cfg != 1 else "full")
    ptr = W.random_block_ptr(A.n, seed=40 + cfg, smin=1, smax=32)
    h, keep = _setup_blocks(B, torch_, A, ptr)
    info = B.bj_get_info(h)
    assert info["b"] == -1 and info["solve_kernel"] == 4 and info["nblocks"] == len(ptr) - 1
    P = oracle.PrecondBlocks(A, ptr)
    for seed in (7, 8):
        x = W.seeded_vector(seed, A.n)
        xd = dev(torch_, x)
        for name in ("bj_solve_L", "bj_solve_Lt", "bj_apply", "bj_op_apply"):
            got = getattr(B, name)(h, xd).cpu().numpy()
            want = getattr(P, name[3:])(x)
            e2, ei = rel(got, want)
            assert e2 <= TOL_APPLY, (cfg, name, e2)
    g = B.bj_cond_estimate_ex(h, 30, reorth=True)
    c = P.cond_estimate(30, reorth=True)
    assert g["iters_done"] == c["iters_done"]
    assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (cfg, g["kappa"], c["kappa"])
    B.bj_destroy(h)


def test_variable_blocks_equal_sizes_reproduce_the_uniform_handle(B, torch_, rel):
    A = mat(2, "small")
    x = dev(torch_, W.seeded_vector(5, A.n))
    for b in (3, 8, 16, 32):
        ptr = np.unique(np.minimum(np.arange(0, A.n + b, b), A.n))
        hv, keep = _setup_blocks(B, torch_, A, ptr)
        hu, keep2 = B.setup_from_host(A, b)
        for name in ("bj_apply", "bj_op_apply"):
            e2, ei = rel(getattr(B, name)(hv, x).cpu().numpy(), getattr(B, name)(hu, x).cpu().numpy())
            assert e2 <= TOL_APPLY, (b, name, e2)
        B.bj_destroy(hv); B.bj_destroy(hu)


def test_variable_blocks_exact_preconditioner_pcg_and_errors(B, torch_, rel):
    sizes = [5, 1, 32, 7, 16, 2, 24] * 9
    A = W.direct_sum_spd(sizes)
    ptr = np.concatenate([[0], np.cumsum(sizes)])
    h, keep = _setup_blocks(B, torch_, A, ptr)
    x = W.seeded_vector(2, A.n)
    y = B.bj_op_apply(h, dev(torch_, x)).cpu().numpy()
    assert np.abs(y - x).max() <= 1e-13                      # M = A: A^ = I
    g = B.bj_cond_estimate_ex(h, 10, reorth=True)
    assert g["iters_done"] == 1 and abs(g["kappa"] - 1) <= 1e-12
    r = B.bj_pcg_solve(h, dev(torch_, x), max_iters=10, rtol=1e-12)
    assert r["iters"] == 1 and r["true_relres"] <= 1e-13
    gm = B.bj_cond_estimate_minv(h, 10)
    assert gm["iters_done"] == 1 and abs(gm["kappa"] - 1) <= 1e-12
    with pytest.raises(B.BJError):
        B.bj_cond_estimate_batch(h, 9, 10, 1)
    B.bj_destroy(h)
    rp, ci, val = keep
    for bad in ([0, 5, 5, A.n], [1, A.n], [0, 40, A.n], [0, A.n - 1]):
        with pytest.raises(B.BJError):
            B.bj_setup_blocks(rp, ci, val, bad)
    # a block that is not positive definite is reported by index
    A2 = W.direct_sum_spd([4, 6, 3])
    v = A2.val.copy()
    Ad = A2.to_dense()
    d_idx = [e for i in range(4, 10) for e in range(A2.row_ptr[i], A2.row_ptr[i + 1]) if A2.col_idx[e] == i]
    v[d_idx[2]] = -1.0
    with pytest.raises(B.BJError) as ei:
        B.bj_setup_blocks(dev(torch_, A2.row_ptr), dev(torch_, A2.col_idx), dev(torch_, v), [0, 4, 10, 13])
    assert ei.value.bad_block == 1


def test_serpentine_walk_of_the_block_solves(B, torch_, rel):
    """bj_setup_opts_t.serp_keep_mb: the plain backward solve visits the blocks from the last to the first and the
    last megabytes of every walk stay ordinary L2 lines.  Only the visiting order and the cache policy change, so every
    output is bit-identical to the forward walk (keep = 0); sizes chosen so that keep = 1 MB covers PART of the factor array
    (both policies and the reversed tail tile in one launch), with a ragged last block / tile.  Oracle parity at keep = 1."""
    cases = ((W.config2(48), 8), (W.config2(47), 8), (W.config4(256), 16), (mat(3, "small"), 32), (W.config5(14), 24),
             (W.config5(14), 3), (W.config4(250), 16))
    for A, b in cases:
        xs = [dev(torch_, W.seeded_vector(s, A.n)) for s in (11, 12)]
        out = {}
        for keep_mb in ("0", "1", "48"):
            h, keep = B.setup_from_host(A, b, serp_keep_mb=int(keep_mb) or -1)     # -1: off, 0 would be the default (48)
            res = []
            for x in xs:   # a chain of applies, so that a walk really starts where the previous one stopped
                y = B.bj_op_apply(h, x).clone()
                y2 = B.bj_op_apply(h, y).clone()
                res += [y.cpu().numpy(), y2.cpu().numpy(), B.bj_solve_Lt(h, x).cpu().numpy(), B.bj_solve_L(h, x).cpu().numpy(),
                        B.bj_apply(h, x).cpu().numpy()]
            out[keep_mb] = res
            if keep_mb == "1":
                P = oracle.Precond(A, b)
                x = W.seeded_vector(11, A.n)
                for got, ref in ((res[0], P.op_apply(x)), (res[2], P.solve_Lt(x)), (res[3], P.solve_L(x))):
                    e2, ei = rel(got, ref)
                    assert e2 <= TOL_APPLY and ei <= TOL_APPLY, f"n={A.n} b={b}: rel2={e2:.3e} relinf={ei:.3e}"
                g = B.bj_cond_estimate_ex(h, 12, reorth=True)
                assert abs(g["kappa"] / P.cond_estimate(12, reorth=True)["kappa"] - 1) <= TOL_KAPPA
            B.bj_destroy(h)
        for keep_mb in ("1", "48"):
            for got, ref in zip(out[keep_mb], out["0"]):
                assert np.array_equal(got, ref), f"n={A.n} b={b} keep={keep_mb}"


# ------------------------------------------------------------------ permutation argument (NEXT-3) --------
def _setup_perm(B, torch_, A, b, perm, block_ptr=None):
    rp, ci, val = dev(torch_, A.row_ptr), dev(torch_, A.col_idx), dev(torch_, A.val)
    pd = dev(torch_, np.asarray(perm, dtype=np.int32))
    return B.bj_setup_perm(rp, ci, val, b, pd, block_ptr=block_ptr), (rp, ci, val, pd)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_permuted_blocks_match_oracle(B, torch_, rel, cfg):
    """bj_setup_perm with a seeded random permutation (the hardest case for the gathers): every apply entry point, in the
    ORIGINAL ordering, element by element against oracle.PrecondPerm (explicit P A P^T); kappa with full
    reorthogonalisation to the bar of the north star; in-place calls; ragged last block."""
    A = mat(cfg, "small" if cfg != 5 else "tiny")
    for b in sorted(set(W.BLOCK_SIZES[cfg] + [7, 12])):   # thread-per-block, group, and stream solve kernels
        perm = W.random_permutation(A.n, seed=60 + cfg + b)
        h, keep = _setup_perm(B, torch_, A, b, perm)
        info = B.bj_get_info(h)
        assert info["permuted"] == 1 and info["b"] == b and info["nblocks"] == (A.n + b - 1) // b
        assert info["solve_kernel"] in (1, 2) and info["fused_forward"] == 0          # the uniform-block kernels
        P = oracle.PrecondPerm(A, perm, b)
        for seed in (7, 8):
            x = W.seeded_vector(seed, A.n)
            xd = dev(torch_, x)
            for name in ("bj_solve_L", "bj_solve_Lt", "bj_apply", "bj_op_apply"):
                got = getattr(B, name)(h, xd).cpu().numpy()
                e2, ei = rel(got, getattr(P, name[3:])(x))
                assert e2 <= TOL_APPLY and ei <= TOL_APPLY, (cfg, b, name, e2, ei)
            y = xd.clone()
            B.bj_op_apply(h, y, y)
            assert rel(y.cpu().numpy(), P.op_apply(x))[0] <= TOL_APPLY
        g = B.bj_cond_estimate_ex(h, 30, reorth=True)
        c = P.cond_estimate(30, reorth=True)
        assert g["iters_done"] == c["iters_done"]
        assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (cfg, b, g["kappa"], c["kappa"])
        B.bj_destroy(h)


def test_line_permutation_gives_xfastest_config4_the_yfastest_preconditioner(B, torch_, rel):
    """Config 4 numbered along the weak direction: natural blocks of 16 are nearly useless; with the line permutation
    (workloads.config4_line_permutation, and the one predict.strong_coupling_lines finds by itself) the handle reproduces
    the y-fastest results: the operator equals the y-fastest handle's in permuted coordinates, kappa equals the oracle's."""
    from paper_2410_02408_b200 import predict
    n, b = 96, 16
    Ax, Ay = W.config4(n, x_fastest=True), W.config4(n)
    perm = W.config4_line_permutation(n)
    hp, keep = _setup_perm(B, torch_, Ax, b, perm)
    hy, keepy = B.setup_from_host(Ay, b)
    x = W.seeded_vector(4, Ax.n)
    yp = B.bj_op_apply(hp, dev(torch_, x)).cpu().numpy()          # original (x-fastest) ordering
    yy = B.bj_op_apply(hy, dev(torch_, x[perm])).cpu().numpy()    # the y-fastest handle sees P x
    e2, ei = rel(yp[perm], yy)
    assert e2 <= TOL_APPLY and ei <= TOL_APPLY
    P = oracle.PrecondPerm(Ax, perm, b)
    g = B.bj_cond_estimate_ex(hp, 40, reorth=True)
    assert abs(g["kappa"] / P.cond_estimate(40)["kappa"] - 1) <= TOL_KAPPA
    hn, keepn = B.setup_from_host(Ax, b)                          # natural blocks of the badly numbered matrix
    k_nat = B.bj_cond_estimate_ex(hn, 200, reorth=True)["kappa"]
    k_perm = B.bj_cond_estimate_ex(hp, 200, reorth=True)["kappa"]
    assert k_nat > 3 * k_perm
    lines = predict.strong_coupling_lines(Ax, b)                   # found from the matrix alone
    hl, keepl = _setup_perm(B, torch_, Ax, b, lines)
    k_lines = B.bj_cond_estimate_ex(hl, 200, reorth=True)["kappa"]
    assert abs(k_lines / k_perm - 1) < 0.05                        # same blocks in another order: same spectrum
    rhs = dev(torch_, W.seeded_vector(17, Ax.n))
    it_nat = B.bj_pcg_solve(hn, rhs, max_iters=3000, rtol=1e-3)["iters"]
    r = B.bj_pcg_solve(hl, rhs, max_iters=3000, rtol=1e-3)
    assert r["converged"] and r["true_relres"] <= 1.2e-3 and r["iters"] < 0.7 * it_nat
    for h in (hp, hy, hn, hl):
        B.bj_destroy(h)


def test_rcm_restores_the_block_diagonal_model_on_the_device(B, torch_, rel):
    """PAPER.md:80 hidden by a shuffle: with the RCM ordering (predict.rcm_permutation) M = A, the operator is the
    identity, Lanczos stops at one step, PCG converges in one step; variable block sizes combine with the permutation;
    a sequence that is not a permutation is rejected."""
    from paper_2410_02408_b200 import predict
    sizes = [5, 1, 32, 7, 16, 2, 24] * 6
    A0 = W.direct_sum_spd(sizes)
    A = W.permuted(A0, W.random_permutation(A0.n, seed=11))
    # RCM keeps components contiguous but in its own order and with its own internal order: recover the component sizes
    perm = predict.rcm_permutation(A)
    import scipy.sparse.csgraph as csg
    ncomp, label = csg.connected_components(A.to_scipy(), directed=False)
    lab = label[perm]
    cuts = np.flatnonzero(np.diff(lab)) + 1
    ptr = np.concatenate([[0], cuts, [A.n]])
    assert len(ptr) - 1 == len(sizes)
    h, keep = _setup_perm(B, torch_, A, 0, perm, block_ptr=ptr)
    x = W.seeded_vector(2, A.n)
    y = B.bj_op_apply(h, dev(torch_, x)).cpu().numpy()
    assert np.abs(y - x).max() <= 1e-13
    g = B.bj_cond_estimate_ex(h, 10, reorth=True)
    assert g["iters_done"] == 1 and abs(g["kappa"] - 1) <= 1e-12
    r = B.bj_pcg_solve(h, dev(torch_, x), max_iters=10, rtol=1e-12)
    assert r["iters"] == 1 and r["true_relres"] <= 1e-13
    P = oracle.PrecondPerm(A, perm, block_ptr=ptr)
    e2, ei = rel(B.bj_apply(h, dev(torch_, x)).cpu().numpy(), P.apply(x))
    assert e2 <= TOL_APPLY
    B.bj_destroy(h)
    rp, ci, val, pd = keep
    bad = perm.copy()
    bad[3] = bad[4]
    for seq in (bad, np.full(A.n, A.n, dtype=np.int32)):
        with pytest.raises(B.BJError) as e:
            B.bj_setup_perm(rp, ci, val, 4, dev(torch_, seq.astype(np.int32)))
        assert e.value.code == B.BJ_ERR_INVALID_ARG
    # identity permutation = bj_setup_blocks with equal sizes = the uniform handle (to the tolerance)
    hi = B.bj_setup_perm(rp, ci, val, 8, dev(torch_, np.arange(A.n, dtype=np.int32)))
    hu = B.bj_setup(rp, ci, val, 8)
    e2, ei = rel(B.bj_op_apply(hi, dev(torch_, x)).cpu().numpy(), B.bj_op_apply(hu, dev(torch_, x)).cpu().numpy())
    assert e2 <= TOL_APPLY
    B.bj_destroy(hi); B.bj_destroy(hu)
