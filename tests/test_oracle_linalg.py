"""Pins for the oracle's textbook Cholesky and substitutions."""
import numpy as np
import pytest

import oracle


@pytest.mark.parametrize("p", [1, 2, 7, 64, 150])
def test_cholesky_and_solves_match_numpy(p):
    rng = np.random.default_rng(p)
    A = rng.standard_normal((3 * p + 2, p))
    Q = A.T @ A + np.diag(rng.uniform(0.1, 5.0, p))
    rc, L = oracle.cholesky_lower(Q)
    assert rc == 0
    Lref = np.linalg.cholesky(Q)
    assert np.max(np.abs(L - Lref)) <= 1e-12 * np.max(np.abs(Lref))
    assert np.linalg.norm(L @ L.T - Q) <= 1e-13 * np.linalg.norm(Q)
    b = rng.standard_normal(p)
    y = oracle.solve_lower(L, b)
    assert np.allclose(L @ y, b, rtol=0, atol=1e-11 * np.abs(b).max())
    x = oracle.solve_lower(L, b, transpose=True)
    assert np.allclose(L.T @ x, b, rtol=0, atol=1e-11 * np.abs(b).max())
    assert np.allclose(x, np.linalg.solve(Lref.T, b), rtol=1e-9, atol=1e-12)


def test_cholesky_reads_only_lower_triangle_and_flags_non_pd():
    Q = np.array([[4.0, 99.0], [2.0, 3.0]])          # upper entry is garbage on purpose
    rc, L = oracle.cholesky_lower(Q)
    assert rc == 0 and np.allclose(L, [[2.0, 0.0], [1.0, np.sqrt(2.0)]])
    rc, _ = oracle.cholesky_lower(np.array([[1.0, 0.0], [2.0, 1.0]]))   # 1 - 4 < 0
    assert rc == 2
