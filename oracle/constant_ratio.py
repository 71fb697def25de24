"""Oracle for f4 (first variant): the constant-photometric-ratio constraint ("drops the
sum-flux freedom of higher-order terms") -- TEST INFRASTRUCTURE, numpy FP64 on top of oracle.sfft_oracle.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares no
code with the CUDA path.

PAPER.md does not spell the constraint out; the reading (R1): the flux scaling between template
and science image, sum_{u,v} K(u, v; x, y) = sum_t xt^i yt^j sum_{u,v} a_{t,u,v}, must not vary across the frame, i.e.
    sum_{u,v} a_{t,u,v} = 0   for every polynomial term t >= 1,
while t = 0 and the background stay free.  The fit is the same least-squares problem restricted to that subspace.
The oracle writes the restriction out: c = T c' with the centre tap of each term t >= 1 eliminated,
    a_{t,0,0} = - sum_{(u,v) != (0,0)} a_{t,u,v},
solves the reduced normal equations (T^T G T) c' = T^T h with the textbook Cholesky of oracle.solve, and expands.
"""
from __future__ import annotations

import numpy as np

from . import sfft_oracle as _o


def elimination_matrix(L: int, DK: int, DB: int):
    """T (n x (n - NK + 1)): columns are the free unknowns; rows of the eliminated centre taps carry -1."""
    NK, LL = _o.num_poly(DK), L * L
    n = _o.num_unknowns(L, DK, DB)
    centre = (L * L - 1) // 2                  # index of (u, v) = (0, 0) inside a term's block
    elim = {t * LL + centre for t in range(1, NK)}
    free = [k for k in range(n) if k not in elim]
    T = np.zeros((n, len(free)))
    for col, k in enumerate(free):
        T[k, col] = 1.0
        t = k // LL
        if 1 <= t < NK:
            T[t * LL + centre, col] = -1.0
    return T


def solve_constant_ratio(G, h, L: int, DK: int, DB: int):
    """Constrained least-squares coefficients (length n) from the oracle's G, h."""
    G = np.asarray(G, dtype=np.float64)
    h = np.asarray(h, dtype=np.float64)
    T = elimination_matrix(L, DK, DB)
    Gr = T.T @ G @ T
    Gr = 0.5 * (Gr + Gr.T)
    cr = _o.solve(Gr, T.T @ h)
    return T @ cr
