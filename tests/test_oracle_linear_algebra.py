"""Pins for the oracle's own Gaussian elimination and for the structure of the assembled cell matrix.

- GEPP vs numpy.linalg.solve (a library routine the special case reduces to) and P A = L U reconstruction.
- Matrix structure vs Eq. 41 / Fig. 4: occupancy (N+2)/(4N) for one group.
- Matrix entries vs Eq. 3a-d assembled independently for a single cell (tests/pins.py).
"""
import numpy as np
import pytest

import oracle
import workloads as W
from pins import global_system


@pytest.mark.parametrize("n", [1, 4, 16, 33, 64])
def test_gepp_matches_numpy_solve(n):
    rng = np.random.default_rng(n)
    A = rng.standard_normal((n, n))
    b = rng.standard_normal(n)
    LU, piv, info = oracle.gepp_factor(A)
    assert info == 0
    x = oracle.gepp_solve(LU, piv, b)
    np.testing.assert_allclose(x, np.linalg.solve(A, b), rtol=0, atol=1e-10 * np.abs(x).max())


def test_gepp_pa_equals_lu_and_pivots_first_max():
    rng = np.random.default_rng(5)
    n = 24
    A = rng.standard_normal((n, n))
    A[0, 0] = 0.0                       # forces an exchange at the first step
    A[3, 0] = A[7, 0] = 9.0             # tie: first maximal entry (row 3) must be chosen
    LU, piv, info = oracle.gepp_factor(A)
    assert info == 0 and piv[0] == 3
    L = np.tril(LU, -1) + np.eye(n)
    U = np.triu(LU)
    PA = A.copy()
    for k in range(n):
        PA[[k, piv[k]]] = PA[[piv[k], k]]
    np.testing.assert_allclose(L @ U, PA, atol=1e-13)
    assert np.abs(L).max() <= 1.0 + 1e-15      # partial pivoting bounds the multipliers


def test_gepp_flags_singular():
    A = np.ones((3, 3))
    _, _, info = oracle.gepp_factor(A)
    assert info == 2
    A = np.zeros((2, 2))
    assert oracle.gepp_factor(A)[2] == 1


def test_gepp_needs_pivoting_case():
    # without row exchanges this system loses all accuracy; with them it is exact to rounding
    A = np.array([[1e-20, 1.0], [1.0, 1.0]])
    LU, piv, _ = oracle.gepp_factor(A)
    x = oracle.gepp_solve(LU, piv, np.array([1.0, 2.0]))
    np.testing.assert_allclose(x, [1.0, 1.0], atol=1e-15)


@pytest.mark.parametrize("N", [4, 8, 16])
def test_occupancy_one_group_eq41(N):
    """Eq. 41: O_c = G(N+2)/(4NG); per row N+2 non-zeros (Fig. 4)."""
    p = W.homogeneous(J=1, N=N, sigma_t=1.3, c=0.7, dx=0.2, v=2.0, dt=0.1)
    A = oracle.Oracle(p).assemble_cell(0)
    nnz_per_row = (A != 0).sum(axis=1)
    assert (nnz_per_row == N + 2).all()
    assert (A != 0).mean() == pytest.approx((N + 2) / (4 * N))


def test_occupancy_multigroup_dense_transfer():
    p = W.random_problem(3, J=1, N=4, G=3)
    A = oracle.Oracle(p).assemble_cell(0)
    assert ((A != 0).sum(axis=1) == p.N * p.G + 2).all()
    # triangular (down-scatter only) transfer: group g couples to g' <= g only -> block lower triangular
    p = W.random_problem(3, J=1, N=4, G=3, upscatter=False)
    A = oracle.Oracle(p).assemble_cell(0)
    nb = 4 * p.N
    for g in range(p.G):
        for gp in range(g + 1, p.G):
            assert not A[g * nb:(g + 1) * nb, gp * nb:(gp + 1) * nb].any()


@pytest.mark.parametrize("seed,N,G", [(1, 2, 1), (2, 4, 2), (3, 6, 3)])
def test_cell_matrix_equals_eq3_single_cell(seed, N, G):
    """For J = 1 with vacuum boundaries the global system of Eq. 3 IS the cell matrix A_j (no incident terms)."""
    p = W.random_problem(seed, J=1, N=N, G=G)
    A = oracle.Oracle(p).assemble_cell(0)
    M, _ = global_system(p, p.q, p.psi0)
    np.testing.assert_allclose(A, M, rtol=0, atol=1e-14 * np.abs(M).max())


def test_diagonal_block_is_eq8b_as_printed():
    """Eq. 8b PAPER.md:132 spelled out entry by entry for one negative and one positive ordinate (no scattering)."""
    p = W.homogeneous(J=1, N=2, sigma_t=1.7, c=0.0, dx=0.3, v=2.0, dt=0.25)
    A = oracle.Oracle(p).assemble_cell(0)
    dx, sig, v, dt = 0.3, 1.7, 2.0, 0.25
    for m, mu in enumerate(p.mu):
        a = (abs(mu) + dx * sig) / 2
        gam = dx / (v * dt)
        want = np.array([[a, mu / 2, gam / 2, 0],
                         [-mu / 2, a, 0, gam / 2],
                         [-gam, 0, gam + a, mu / 2],
                         [0, -gam, -mu / 2, gam + a]])
        np.testing.assert_allclose(A[4 * m:4 * m + 4, 4 * m:4 * m + 4], want, rtol=1e-15)
    assert not A[0:4, 4:8].any() and not A[4:8, 0:4].any()
