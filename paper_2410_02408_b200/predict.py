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


def coupling_captured(A, b: int, perm=None) -> float:
    """c(b): fraction of the off-diagonal absolute weight inside the diagonal b x b blocks (contiguous index ranges,
    DESIGN.md reading 8).  perm (optional, perm[i] = original index at permuted position i): the blocks are contiguous
    ranges of the PERMUTED ordering (bj_setup_perm)."""
    rows = np.repeat(np.arange(A.n, dtype=np.int64), np.diff(A.row_ptr.astype(np.int64)))
    cols = A.col_idx.astype(np.int64)
    if perm is not None:
        pinv = np.empty(A.n, dtype=np.int64)
        pinv[np.asarray(perm, dtype=np.int64)] = np.arange(A.n, dtype=np.int64)
        rows, cols = pinv[rows], pinv[cols]
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


def strong_coupling_lines(A, b: int) -> np.ndarray:
    """An ordering for bj_setup_perm ("a permutation argument (RCM or strong-coupling lines)"): greedy
    chains of up to b unknowns that follow the STRONGEST remaining coupling.  Starting from the lowest unvisited index, a
    chain is extended by the unvisited neighbour with the largest |a_ij| of its last member until it has b members or no
    unvisited neighbour is left; chains are laid out one after the other, so each fills one diagonal block (short chains
    are padded by the start of the next one).  On a grid operator with one strong direction the chains are the grid
    lines along it, whatever the numbering.  Returns perm (int32), perm[i] = original index at permuted position i.
    Host-side, O(nnz) Python steps: meant for matrices up to ~10^6 entries."""
    n = int(A.n)
    rp = A.row_ptr.tolist()
    ci = A.col_idx.tolist()
    w = np.abs(A.val).tolist()
    visited = bytearray(n)
    perm = []
    start = 0
    while len(perm) < n:
        while visited[start]:
            start += 1
        cur = start
        visited[cur] = 1
        perm.append(cur)
        for _ in range(b - 1):
            best, bw = -1, -1.0
            for e in range(rp[cur], rp[cur + 1]):
                c = ci[e]
                if not visited[c] and w[e] > bw:   # ties: the first (lowest column) wins -- deterministic
                    best, bw = c, w[e]
            if best < 0:
                break
            visited[best] = 1
            perm.append(best)
            cur = best
    return np.asarray(perm, dtype=np.int32)


def rcm_permutation(A) -> np.ndarray:
    """Reverse Cuthill-McKee ordering (scipy.sparse.csgraph, a library routine): makes every connected component -- and,
    for banded structure, every neighbourhood -- contiguous.  perm[i] = original index at permuted position i."""
    from scipy.sparse.csgraph import reverse_cuthill_mckee
    return np.asarray(reverse_cuthill_mckee(A.to_scipy(), symmetric_mode=True), dtype=np.int32)


def suggest_ordering(A, b: int) -> dict:
    """Which of {natural, strong-coupling lines, RCM} captures the most coupling inside blocks of size b: the same
    structural feature as suggest_block, applied to the ordering.  Returns the captured shares and the best perm
    (None = keep the natural ordering)."""
    cands = {"natural": None, "lines": strong_coupling_lines(A, b), "rcm": rcm_permutation(A)}
    captured = {k: coupling_captured(A, b, p) for k, p in cands.items()}
    best = max(captured, key=lambda k: (captured[k], k == "natural"))   # ties: keep the natural ordering
    return {"captured": captured, "best": best, "perm": cands[best]}


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
