"""Host-side sweep over the block size b.

Stands in for the paper's ML tuner, which predicts a block size from (matrix size, sparsity)
(sec 4.5): for each candidate b it runs the real path -- bj_setup, timed
bj_op_apply, bj_cond_estimate_ex -- and picks the b that minimises the predicted HHL cost
kappa_est(b)^2 (the paper's O(log n_b kappa^2)), ties (kappa within 1 % relative) broken by the
cheaper apply (`pick_best`).
Everything runs through the C ABI; nothing here touches the oracle.

    python -m paper_2410_02408_b200.sweep --config 2 [--scale full] [--iters 50] [--long-iters 0] [--pcg-rtol 1e-3]
"""
from __future__ import annotations

import argparse
import json
import time

DEFAULT_BLOCKS = (1, 2, 3, 4, 8, 16, 24, 32)
TIE_REL = 0.01  # kappa estimates within 1 % of the smallest count as tied


def pick_best(rows, key: str = "kappa_est", tie_rel: float = TIE_REL):
    """a11's selection rule: minimise the predicted HHL cost kappa_est^2; candidates whose
    kappa_est is within a RELATIVE `tie_rel` of the smallest are tied and the cheapest operator apply among them wins
    (then the smaller b).  Rows with an "error" key are ignored.  Returns the winning row, or None."""
    ok = [r for r in rows if "error" not in r]
    if not ok:
        return None
    kmin = min(r[key] for r in ok)
    tied = [r for r in ok if r[key] <= kmin * (1.0 + tie_rel)]
    return min(tied, key=lambda r: (r["op_apply_us"], r["b"]))


def sweep(rp, ci, val, blocks=DEFAULT_BLOCKS, iters: int = 50, reorth: bool = True, apply_steps: int = 200,
          long_iters: int = 0, pcg_rtol: float = 0.0, pcg_max_iters: int = 2000) -> dict:
    """rp/ci/val: CUDA CSR tensors.  Returns {"rows": [...], "kappa_A": ..., "best_b": ...}."""
    import torch
    from . import binding as B

    n = rp.numel() - 1
    out = {"n": n, "nnz": int(val.numel()), "iters": iters, "rows": []}
    h0 = B.bj_setup(rp, ci, val, 0)
    r0 = B.bj_cond_estimate_ex(h0, iters, reorth=reorth)
    out["kappa_A"] = {"kappa_est": r0["kappa"], "lmin": r0["lmin"], "lmax": r0["lmax"], "res_min": r0["res_min"],
                      "res_max": r0["res_max"], "iters": r0["iters_done"]}
    if long_iters:
        rl = B.bj_cond_estimate_ex(h0, long_iters, reorth=False)
        out["kappa_A"]["kappa_est_long"] = rl["kappa"]
    B.bj_destroy(h0)
    x = None
    for b in blocks:
        if b > B.BJ_B_MAX:
            continue
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        try:
            h = B.bj_setup(rp, ci, val, b)
        except B.BJError as e:
            out["rows"].append({"b": b, "error": str(e)})
            continue
        torch.cuda.synchronize()
        setup_ms = 1e3 * (time.perf_counter() - t0)
        if x is None:
            x = B.bj_seeded_vector(h, 31)
            y = torch.empty_like(x)
        for _ in range(5):
            B.bj_op_apply(h, x, y)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(apply_steps):
            B.bj_op_apply(h, x, y)
        e1.record()
        torch.cuda.synchronize()
        us = 1e3 * e0.elapsed_time(e1) / apply_steps
        r = B.bj_cond_estimate_ex(h, iters, reorth=reorth)
        row = {"b": b, "setup_ms": setup_ms, "op_apply_us": us, "applies_per_s": 1e6 / us, "kappa_est": r["kappa"],
               "lmin": r["lmin"], "lmax": r["lmax"], "res_min": r["res_min"], "res_max": r["res_max"],
               "iters": r["iters_done"], "hhl_gain_kappa_sq": (r0["kappa"] / r["kappa"]) ** 2,
               "factor_bytes": B.bj_get_info(h)["factor_bytes"]}
        if long_iters:
            row["kappa_est_long"] = B.bj_cond_estimate_ex(h, long_iters, reorth=False)["kappa"]
        if pcg_rtol > 0.0:
            # the classical stand-in for the solve stage (bj_pcg_solve): iterations and time to the residual bar
            rhs = B.bj_seeded_vector(h, 17)
            B.bj_pcg_solve(h, rhs, max_iters=8, rtol=0.0)  # allocate the workspace outside the timed call
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            pr = B.bj_pcg_solve(h, rhs, max_iters=pcg_max_iters, rtol=pcg_rtol)
            torch.cuda.synchronize()
            row.update({"pcg_iters": pr["iters"], "pcg_ms": 1e3 * (time.perf_counter() - t0), "pcg_converged": pr["converged"],
                        "pcg_true_relres": pr["true_relres"]})
        out["rows"].append(row)
        B.bj_destroy(h)
    key = "kappa_est_long" if long_iters else "kappa_est"
    best = pick_best(out["rows"], key)
    if best is not None:
        out["best_b"] = best["b"]
        out["criterion"] = f"argmin {key}^2, ties (within {TIE_REL:.0%} relative) -> cheaper apply"
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--scale", default="full", choices=["full", "small", "tiny"])
    ap.add_argument("--iters", type=int, default=50)
    ap.add_argument("--long-iters", type=int, default=0)
    ap.add_argument("--blocks", default=",".join(map(str, DEFAULT_BLOCKS)))
    ap.add_argument("--pcg-rtol", type=float, default=0.0, help="> 0: also solve A x = b by PCG to this residual (paper: 1e-3)")
    args = ap.parse_args()
    import torch
    from . import workloads as W
    A = W.build(args.config, args.scale)
    rp, ci, val = (torch.from_numpy(a).cuda() for a in (A.row_ptr, A.col_idx, A.val))
    res = sweep(rp, ci, val, tuple(int(b) for b in args.blocks.split(",")), iters=args.iters, long_iters=args.long_iters,
                pcg_rtol=args.pcg_rtol)
    res["workload"] = A.meta.get("name")
    from . import predict  # NEXT-3: the structural suggestion beside the measured choice
    sug = predict.suggest_block(A, tuple(int(b) for b in args.blocks.split(",")))
    res["suggested_b"] = sug["suggested_b"]
    res["captured_coupling"] = sug["captured"]
    print(json.dumps(res))


if __name__ == "__main__":
    main()
