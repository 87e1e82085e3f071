"""Dense path of the oracle for N <= ~1024 -- TEST INFRASTRUCTURE.

Forms A^ = L^-1 A L^-T explicitly, column by column, with the oracle's own op_apply, and
hands the symmetric matrix to numpy's dense eigensolver (a library primitive used as one step).
"""
from __future__ import annotations

import numpy as np

from . import Precond


def dense_operator(P: Precond) -> np.ndarray:
    n = P.n
    M = np.empty((n, n))
    e = np.zeros(n)
    for j in range(n):
        e[j] = 1.0
        M[:, j] = P.op_apply(e)
        e[j] = 0.0
    return M


def spectrum(P: Precond) -> np.ndarray:
    M = dense_operator(P)
    return np.linalg.eigvalsh(0.5 * (M + M.T))


def kappa(P: Precond) -> float:
    ev = spectrum(P)
    return float(ev[-1] / ev[0])
