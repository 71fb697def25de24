"""Pins of oracle/constant_ratio.py (f4, constant photometric ratio; reading R1 of DESIGN.md section 15) -- CPU only."""
import numpy as np
import pytest

import oracle
from oracle import constant_ratio as cr
from paper_2509_18544_b200 import starfield


def _case(nx, ny, L, DK, DB, seed):
    S, R = starfield.random_pair(nx, ny, seed=seed)
    G, h = oracle.build_system(S, R, None, L, DK, DB)
    return S, R, G, h


@pytest.mark.parametrize("L,DK,DB", [(3, 1, 0), (5, 2, 1), (3, 3, 0)])
def test_constraint_holds_and_free_terms_stay_free(L, DK, DB):
    S, R, G, h = _case(40, 36, L, DK, DB, 7)
    c = cr.solve_constant_ratio(G, h, L, DK, DB)
    LL, NK = L * L, oracle.num_poly(DK)
    scale = np.abs(c[:NK * LL]).sum()
    for t in range(1, NK):
        assert abs(c[t * LL:(t + 1) * LL].sum()) < 1e-13 * scale
    assert abs(c[:LL].sum()) > 1e-3                      # the flux scale itself is not constrained


def test_equals_lstsq_on_the_reduced_design_matrix():
    """Brute force: least squares with the explicit design matrix A restricted to the constrained subspace (A T),
    solved by numpy's SVD-based lstsq -- no normal equations, no Cholesky."""
    nx, ny, L, DK, DB = 24, 20, 3, 1, 1
    S, R = starfield.random_pair(nx, ny, seed=3)
    A = oracle.design_matrix(R, None, L, DK, DB)
    T = cr.elimination_matrix(L, DK, DB)
    cref = T @ np.linalg.lstsq(A @ T, S.ravel(), rcond=None)[0]
    G, h = oracle.build_system(S, R, None, L, DK, DB)
    c = cr.solve_constant_ratio(G, h, L, DK, DB)
    assert np.max(np.abs(c - cref)) < 1e-9 * np.max(np.abs(cref))


def test_kkt_conditions():
    """Optimality on the subspace: the gradient G c - h is a combination of the constraint normals only, i.e. it is
    constant over each constrained block and zero on the free ones."""
    L, DK, DB = 5, 2, 1
    S, R, G, h = _case(48, 40, L, DK, DB, 11)
    c = cr.solve_constant_ratio(G, h, L, DK, DB)
    g = G @ c - h
    LL, NK = L * L, oracle.num_poly(DK)
    tol = 1e-9 * np.max(np.abs(h))
    assert np.max(np.abs(g[:LL])) < tol and np.max(np.abs(g[NK * LL:])) < tol
    for t in range(1, NK):
        blk = g[t * LL:(t + 1) * LL]
        assert np.max(np.abs(blk - blk.mean())) < tol


def test_dk0_is_the_unconstrained_solution():
    L, DK, DB = 5, 0, 1
    S, R, G, h = _case(40, 36, L, DK, DB, 5)
    assert np.max(np.abs(cr.solve_constant_ratio(G, h, L, DK, DB) - oracle.solve(G, h))) < 1e-12


def test_inactive_constraint_changes_nothing():
    """S = R (*) K0 with a constant kernel: the unconstrained optimum already satisfies the constraint."""
    nx, ny, L, DK, DB = 40, 36, 3, 1, 0
    _, R = starfield.random_pair(nx, ny, seed=9)
    K0 = np.array([[0.0, 0.1, 0.0], [0.2, 0.5, 0.1], [0.0, 0.1, 0.0]])
    S = oracle.convolve_stamp(R, K0)
    G, h = oracle.build_system(S, R, None, L, DK, DB)
    c = cr.solve_constant_ratio(G, h, L, DK, DB)
    assert np.max(np.abs(c[:9] - K0.ravel())) < 1e-9 and np.max(np.abs(c[9:])) < 1e-9
