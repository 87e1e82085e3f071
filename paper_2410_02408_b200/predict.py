"""Feature-based block-size suggestion: the paper's tuner idea without RL.

The paper trains a RandomForestRegressor on three (matrix size, sparsity) rows to predict a block size
(sec 4.5).  Size and sparsity alone cannot say which unknowns are strongly coupled, so this module
uses the one structural feature block-Jacobi actually exploits: the share of the off-diagonal weight that falls INSIDE
the diagonal blocks,

    c(b) = sum_{i != j, floor(i/b) = floor(j/b)} |a_ij| / sum_{i != j} |a_ij|          (0 <= c <= 1, c(1) = 0).

M = blockdiag(D_k) removes exactly that coupling from M^-1 A; what stays outside the blocks is what Lanczos / CG / HHL
still see.  The suggestion is the SMALLEST candidate b that captures (almost) all the coupling any candidate captures:
a larger block costs 4 N (b + 1) factor bytes per solve pass and buys nothing once c(b) has saturated.  Host-side numpy,
O(nnz) per candidate; it never replaces the measured sweep (sweep.py), it orders its candidates.

    python -m paper_2410_02408_b200.predict --config 4 [--scale small]
"""
from __future__ import annotations

import argparse
import json

import numpy as np

DEFAULT_BLOCKS = (1, 2, 3, 4, 8, 16, 24, 32)


def coupling_captured(A, b: int) -> float:
    """c(b): fraction of the off-diagonal absolute weight inside the diagonal b x b blocks (contiguous index ranges,
    DESIGN.md reading 8)."""
    rows = np.repeat(np.arange(A.n, dtype=np.int64), np.diff(A.row_ptr.astype(np.int64)))
    cols = A.col_idx.astype(np.int64)
    w = np.abs(A.val)
    off = rows != cols
    total = float(w[off].sum())
    if total == 0.0:
        return 1.0  # a diagonal matrix: nothing to capture, every b is exact
    inside = off & ((rows // b) == (cols // b))
    return float(w[inside].sum()) / total


def features(A, blocks=DEFAULT_BLOCKS) -> dict:
    """The paper's two features (size, sparsity: PAPER.md:303-318) plus c(b) per candidate."""
    return {"n": int(A.n), "nnz_per_row": float(A.nnz) / float(A.n),
            "captured": {int(b): coupling_captured(A, int(b)) for b in blocks}}


def suggest_block(A, blocks=DEFAULT_BLOCKS, saturation: float = 0.98) -> dict:
    """Smallest candidate whose captured coupling reaches `saturation` x the best any candidate reaches; b = 1 when no
    candidate captures more than 2 % of the coupling (blocks would buy nothing: config 3's random columns)."""
    f = features(A, blocks)
    c = f["captured"]
    best = max(c.values())
    if best < 0.02:
        choice = min(blocks)
    else:
        choice = min(b for b in blocks if c[b] >= saturation * best)
    f.update({"suggested_b": int(choice), "rule": f"smallest b with c(b) >= {saturation} max c; b = min when max c < 0.02"})
    return f


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--scale", default="small", choices=["full", "small", "tiny"])
    ap.add_argument("--blocks", default=",".join(map(str, DEFAULT_BLOCKS)))
    args = ap.parse_args()
    from . import workloads as W
    A = W.build(args.config, args.scale)
    out = suggest_block(A, tuple(int(b) for b in args.blocks.split(",")))
    out["workload"] = A.meta.get("name")
    print(json.dumps(out))


if __name__ == "__main__":
    main()
