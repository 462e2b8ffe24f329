"""CPU pins for (i) the block-diagonal-plus-low-rank structure of the cell matrix that the structured cell solve
(csrc/structured.cu) rests on, checked on the ORACLE's assembled matrix with numpy only, and
(ii) the seeded workload recipes of DESIGN.md section 4 (shapes and value ranges of BASELINE.json's configs)."""
import numpy as np
import pytest

import workloads as W
from oracle import Oracle


def _structure(p, j):
    """D (4x4 blocks of the oracle's own matrix), U, V^T of A_j = D - U V^T as read from Eq. 8a-b, 10, 40b."""
    N, G, n = p.N, p.G, p.n
    A = Oracle(p).assemble_cell(j)
    dx = np.broadcast_to(np.asarray(p.dx, dtype=float), (p.J,))[j]
    K = np.broadcast_to(np.asarray(p.transfer, dtype=float), (p.J, G, G))[j]
    U = np.zeros((n, 4 * G))
    Vt = np.zeros((4 * G, n))
    for g in range(G):
        for m in range(N):
            for q in range(4):
                r = (g * N + m) * 4 + q
                Vt[g * 4 + q, r] = p.w[m]                       # V^T psi = phi (Eq. 44)
                for gp in range(G):
                    U[r, gp * 4 + q] = dx * K[g, gp] / 4.0      # (U phi)[g][m][q] = dx/4 sum_g' K[g][g'] phi[g'][q]
    D = A + U @ Vt
    return A, D, U, Vt


@pytest.mark.parametrize("seed,N,G", [(1, 4, 1), (2, 8, 2), (3, 6, 3), (4, 2, 4)])
def test_cell_matrix_is_block_diagonal_minus_rank_4G(seed, N, G):
    p = W.random_problem(seed, 5, N, G, bc_left=1, bc_right=2)
    A, D, U, Vt = _structure(p, 2)
    n = p.n
    mask = np.kron(np.eye(N * G), np.ones((4, 4))) > 0
    assert np.max(np.abs(D[~mask])) < 1e-15 * np.max(np.abs(A))          # D is block diagonal, 4x4 blocks (Eq. 8a)
    assert np.linalg.matrix_rank(U @ Vt) <= 4 * G
    # Sherman-Morrison-Woodbury in the form the kernel applies it: z = D^-1 b; y = C^-1 V^T z; x = z + D^-1 U y
    rng = np.random.default_rng(seed)
    b = rng.standard_normal(n)
    Dinv = np.linalg.inv(D)
    C = np.eye(4 * G) - Vt @ Dinv @ U
    z = Dinv @ b
    y = np.linalg.solve(C, Vt @ z)
    x = z + Dinv @ (U @ y)
    x_ref = np.linalg.solve(A, b)
    np.testing.assert_allclose(x, x_ref, rtol=0, atol=1e-12 * np.abs(x_ref).max())
    np.testing.assert_allclose(y, Vt @ x_ref, rtol=0, atol=1e-12 * np.abs(x_ref).max())   # y IS the new scalar flux


def test_config_recipes():
    p1 = W.config1()
    assert (p1.J, p1.N, p1.G, p1.n) == (16, 4, 1, 16) and p1.dt == 0.1 and p1.n_steps == 5
    p2 = W.config2(dt=0.01)
    q2 = np.broadcast_to(p2.q, (p2.J, p2.G, 4))
    assert (p2.J, p2.N, p2.n) == (1024, 8, 32) and np.all(q2[:512] == 1.0) and np.all(q2[512:] == 0.0)
    p3 = W.config3(J=512)
    assert (p3.N, p3.G, p3.n) == (8, 4, 128)
    K, sig = np.asarray(p3.transfer), np.asarray(p3.sigma_t)
    assert np.all(sig >= 0.5) and np.all(sig <= 5.0)
    ids = p3.meta["material_id"]
    for j in (0, 100, 511):
        Kj = K[j].copy()
        if ids[j] == 1:                       # material index 1 carries chi_1 nu Sigma_f = 0.1 Sigma_t into group 1
            Kj[0] -= 0.1 * sig[j]
        assert np.allclose(np.triu(Kj, 1), 0.0)                      # down-scatter only: [to][from], to >= from
        c = Kj.sum(axis=0) / sig[j]                                   # ratio of group g' = sum over destinations
        assert np.all(c > 0.3 - 1e-12) and np.all(c < 0.95 + 1e-12)
    assert np.allclose(p3.v, 1e9 / 10.0 ** np.arange(1, 5))
    p4 = W.config4()
    assert (p4.J, p4.n) == (2048, 256) and p4.bc_left == W.BC_REFLECTIVE and p4.bc_right == W.BC_VACUUM
    K4, s4 = np.broadcast_to(p4.transfer, (p4.J, 8, 8))[0], np.broadcast_to(p4.sigma_t, (p4.J, 8))[0]
    np.testing.assert_allclose(K4.sum(axis=0) / s4, 0.99)
    assert np.all(p4.source_at_step(0) == 1.0) and np.all(p4.source_at_step(1) == 0.0)
    p5 = W.config5(J=4096)
    s5 = np.asarray(p5.sigma_t)[:, 0]
    c5 = np.asarray(p5.transfer)[:, 0, 0] / s5
    assert p5.n == 64 and s5.min() >= 0.01 and s5.max() <= 100.0 and c5.min() >= 0.5 and c5.max() <= 0.999
    assert abs(np.log10(s5).mean()) < 0.1                               # log-uniform over [1e-2, 1e2]
    # seeded: the same call gives the same bits
    assert np.array_equal(W.config5(J=64).sigma_t, W.config5(J=64).sigma_t)
