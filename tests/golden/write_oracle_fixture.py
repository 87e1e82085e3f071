"""Writes tests/golden/oracle_cfg1_fixture.txt from the CPU oracle ONLY (never from the CUDA path).

Run from the repo root:  python tests/golden/write_oracle_fixture.py
The fixture is a regression guard for the oracle + generator pair on BASELINE.json config 1
(2D Poisson 32x32 + U[0,1) diagonal, b = 4, 50 Lanczos steps, full reorthogonalisation).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2410_02408_b200 import workloads as W  # noqa: E402


def main():
    A = W.build(1, "full")
    out = []
    x = W.seeded_vector(12345, A.n)
    for b in (0, 1, 4):
        P = oracle.Precond(A, b)
        y = P.op_apply(x)
        r = P.cond_estimate(50)
        out.append(f"b{b}_op_apply_norm2 {float(np.linalg.norm(y))!r}")
        out.append(f"b{b}_op_apply_y0 {float(y[0])!r}")
        out.append(f"b{b}_lmin_m50 {r['lmin']!r}")
        out.append(f"b{b}_lmax_m50 {r['lmax']!r}")
        out.append(f"b{b}_kappa_m50 {r['kappa']!r}")
        pc = P.pcg(W.seeded_vector(17, A.n), 200, 1e-8)      # NEXT-1: PCG to 1e-8 from x0 = 0
        out.append(f"b{b}_pcg_iters {pc['iters']!r}")
        out.append(f"b{b}_pcg_alpha0 {float(pc['alpha'][0])!r}")
        out.append(f"b{b}_pcg_x_norm2 {float(np.linalg.norm(pc['x']))!r}")
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_cfg1_fixture.txt")
    with open(path, "w") as fh:
        fh.write("# written by tests/golden/write_oracle_fixture.py (oracle only); config 1, seed %d\n" % W.SEED)
        fh.write("\n".join(out) + "\n")
    print(open(path).read())


if __name__ == "__main__":
    main()
