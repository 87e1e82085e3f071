"""bj_cond_estimate_noalloc (include/bj.h): the kappa estimate for callers that cannot allocate device memory at call
time.  Same kernel as bj_cond_estimate_ex on launch-bound sizes, its device scratch in one file-scope device array.
Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_2410_02408_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_KAPPA = 1e-6   # the kappa bar of tests/test_gpu_parity.py (BASELINE.json)


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2410_02408_b200 import binding
    binding.lib()
    return binding


def _same(g, c):
    assert g["iters_done"] == c["iters_done"]
    assert abs(g["kappa"] / c["kappa"] - 1) <= TOL_KAPPA, (g["kappa"], c["kappa"])
    assert abs(g["lmin"] / c["lmin"] - 1) <= TOL_KAPPA and abs(g["lmax"] / c["lmax"] - 1) <= TOL_KAPPA
    scale = np.abs(c["alpha"]).max()
    assert np.abs(g["alpha"] - c["alpha"]).max() <= 1e-8 * scale and np.abs(g["beta"] - c["beta"]).max() <= 1e-8 * scale


def test_noalloc_cond_estimate_matches_the_existing_path_on_two_calls_in_a_row(B):
    import torch
    A = W.build(1, "full")                                  # the paper's N = 1024
    v0 = torch.from_numpy(W.seeded_vector(77, A.n)).cuda()
    for b in (4, 0):
        h, keep = B.setup_from_host(A, b)
        ws0 = B.bj_get_info(h)["workspace_bytes"]
        B.bj_cond_estimate_noalloc(h, 8)                    # loads the kernels (module loading may take device memory once)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        # two calls in a row on the shared scratch: the second is shorter, with another start vector and without
        # reorthogonalisation -- nothing of the first call's alpha / beta / status may leak into it
        g1 = B.bj_cond_estimate_noalloc(h, 50, reorth=True)
        g2 = B.bj_cond_estimate_noalloc(h, 20, reorth=False, v0=v0)
        g3 = B.bj_cond_estimate_noalloc(h, 50, reorth=True)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0, "the no-alloc entry point changed the free device memory"
        assert B.bj_get_info(h)["workspace_bytes"] == ws0   # and the handle's workspace was neither created nor grown
        c1 = B.bj_cond_estimate_ex(h, 50, reorth=True)      # the existing path (allocates its workspace on first use)
        c2 = B.bj_cond_estimate_ex(h, 20, reorth=False, v0=v0)
        _same(g1, c1)
        _same(g2, c2)
        _same(g3, c1)
        assert np.array_equal(g1["alpha"], g3["alpha"]) and np.array_equal(g1["beta"], g3["beta"])
        B.bj_destroy(h)


def test_noalloc_cond_estimate_rejects_what_is_beyond_its_limits(B):
    import torch
    A = W.build(1, "full")
    h, keep = B.setup_from_host(A, 4)
    for iters in (B.BJ_NOALLOC_MAX_ITERS + 1, 4000):
        with pytest.raises(B.BJError) as e:
            B.bj_cond_estimate_noalloc(h, iters)
        assert e.value.code == B.BJ_ERR_LIMIT and "limits" in str(e.value)
    z = torch.zeros(A.n, dtype=torch.float64, device="cuda")
    with pytest.raises(B.BJError) as e:                      # a zero start vector is an invalid argument, as everywhere
        B.bj_cond_estimate_noalloc(h, 10, v0=z)
    assert e.value.code == B.BJ_ERR_INVALID_ARG
    g = B.bj_cond_estimate_noalloc(h, 10)                    # and the scratch is usable afterwards
    assert g["iters_done"] == 10 and np.isfinite(g["kappa"])
    B.bj_destroy(h)
    h, keep = B.setup_from_host(A, 16)                       # group-kernel block size: not a launch-bound layout
    with pytest.raises(B.BJError) as e:
        B.bj_cond_estimate_noalloc(h, 10)
    assert e.value.code == B.BJ_ERR_LIMIT
    B.bj_destroy(h)
    big = W.laplacian((160, 160))                            # n = 25 600 > BJ_NOALLOC_MAX_N
    assert big.n > B.BJ_NOALLOC_MAX_N
    h, keep = B.setup_from_host(big, 4)
    with pytest.raises(B.BJError) as e:
        B.bj_cond_estimate_noalloc(h, 10)
    assert e.value.code == B.BJ_ERR_LIMIT
    B.bj_destroy(h)
