"""Pins (a) and (b) of BASELINE.json north_star / SURVEY.md section 8(c):

(a) the fixed point of the oracle's OCI iteration and of its SI iteration equals a brute-force dense solve of the
    whole space-angle-group-time system of one step, assembled independently from Eq. 3a-d (tests/pins.py);
(b) OCI and SI converge to the same solution.
Run with a tight tolerance (1e-13) because the BASELINE stopping rule at 1e-8 leaves an error ~ tol*rho/(1-rho)
(SURVEY hazard H1).
"""
import numpy as np
import pytest

import oracle
import workloads as W
from pins import global_solve

CASES = {
    "cfg1": lambda: W.config1(),
    "rand_vac_2g": lambda: W.random_problem(11, J=6, N=4, G=2),
    "rand_reflL_3g": lambda: W.random_problem(12, J=5, N=4, G=3, bc_left=W.BC_REFLECTIVE),
    "rand_reflR_prescL": lambda: W.random_problem(13, J=7, N=2, G=2, bc_left=W.BC_PRESCRIBED,
                                                  bc_right=W.BC_REFLECTIVE),
    "rand_presc_both_1g": lambda: W.random_problem(14, J=9, N=6, G=1, bc_left=W.BC_PRESCRIBED,
                                                   bc_right=W.BC_PRESCRIBED),
    "table2_tiny": lambda: W.table2(J=7, N=4, dt=0.1, L=3.5),
}


@pytest.mark.parametrize("name", list(CASES))
def test_oci_and_si_fixed_points_equal_global_solve(name):
    p = CASES[name]()
    oci, si = oracle.Oracle(p), oracle.Oracle(p)
    psi_prev = p.psi0.copy()
    for step in range(2):
        q = p.source_at_step(step)
        oci.set_source(q)
        si.set_source(q)
        exact = global_solve(p, q, psi_prev)
        it_o, _ = oci.oci_step(tol=1e-13, max_iters=20000)
        it_s, _ = si.si_step(tol=1e-13, max_iters=20000)
        scale = np.abs(exact).max()
        assert it_o < 20000 and it_s < 20000
        np.testing.assert_allclose(oci.psi, exact, rtol=0, atol=1e-11 * scale)   # (a) OCI
        np.testing.assert_allclose(si.psi, exact, rtol=0, atol=1e-11 * scale)    # (a) SI
        np.testing.assert_allclose(oci.phi, si.phi, rtol=0, atol=1e-11 * scale)  # (b)
        psi_prev = exact[..., 2:4].copy()
        np.testing.assert_allclose(oci.psi_prev, psi_prev, rtol=0, atol=1e-11 * scale)


def test_one_oci_iteration_is_block_jacobi_of_the_global_system():
    """One iteration = solve the block-diagonal part with the off-diagonal (incident) part at the old iterate."""
    from pins import global_system
    p = W.random_problem(21, J=5, N=4, G=2, bc_left=W.BC_REFLECTIVE)
    M, rhs = global_system(p, p.q, p.psi0)
    n = p.n
    D = np.zeros_like(M)
    for j in range(p.J):
        D[j * n:(j + 1) * n, j * n:(j + 1) * n] = M[j * n:(j + 1) * n, j * n:(j + 1) * n]
    # the lagged reflective term couples cell 0 to itself but is NOT part of A_0: move it off-diagonal
    o = oracle.Oracle(p)
    for j in range(p.J):
        D[j * n:(j + 1) * n, j * n:(j + 1) * n] = o.assemble_cell(j)
    Off = M - D
    rng = np.random.default_rng(0)
    x0 = rng.uniform(0, 1, size=M.shape[0])
    want = np.linalg.solve(D, rhs - Off @ x0)
    o.set_iterate(x0)
    o.factor()
    o.const_rhs()
    got = o.oci_iterate(1).reshape(-1)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13 * np.abs(want).max())


def test_rule1_controls_false_convergence():
    """Eq. 12-13: with rho close to 1, rule 1 ends closer to the fixed point than rule 0."""
    p = W.config2(dt=1.0, J=96)       # thin cells, c = 0.9: slow OCI convergence
    exact = global_solve(p, p.q, p.psi0) if p.J * p.n <= 4096 else None
    o0, o1 = oracle.Oracle(p), oracle.Oracle(p)
    it0, _ = o0.oci_step(tol=1e-8, rule=0)
    it1, r1 = o1.oci_step(tol=1e-8, rule=1)
    assert it1 > it0
    ref = oracle.Oracle(p)
    ref.oci_step(tol=1e-14, max_iters=200000)
    err0 = np.abs(o0.psi - ref.psi).max()
    err1 = np.abs(o1.psi - ref.psi).max()
    assert err1 < err0
    if exact is not None:
        assert np.abs(ref.psi - exact).max() < 1e-11


# ---------------------------------------------------------------------------------------------------------------
# Red-black ordering of the cell solves: pins of oracle.oci_iterate(ordering=1)
# ---------------------------------------------------------------------------------------------------------------
def test_one_redblack_iteration_is_block_gauss_seidel_of_the_global_system():
    """Even cells from the old iterate, then odd cells from the new even cells: two half-steps on the global matrix,
    done here with numpy on the independently assembled global system."""
    from pins import global_system
    p = W.random_problem(22, J=7, N=4, G=2, bc_left=W.BC_REFLECTIVE, bc_right=W.BC_PRESCRIBED)
    M, rhs = global_system(p, p.q, p.psi0)
    n = p.n
    o = oracle.Oracle(p)
    D = np.zeros_like(M)
    for j in range(p.J):
        D[j * n:(j + 1) * n, j * n:(j + 1) * n] = o.assemble_cell(j)   # the lagged reflective term is NOT in A_0 (A12)
    Off = M - D
    rng = np.random.default_rng(1)
    x = rng.uniform(0, 1, size=M.shape[0])
    want = x.copy()
    for colour in (0, 1):
        r = rhs - Off @ want
        for j in range(colour, p.J, 2):
            want[j * n:(j + 1) * n] = np.linalg.solve(D[j * n:(j + 1) * n, j * n:(j + 1) * n], r[j * n:(j + 1) * n])
    o.set_iterate(x)
    o.factor()
    o.const_rhs()
    got = o.oci_iterate(1, ordering=1).reshape(-1)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13 * np.abs(want).max())


def test_redblack_reaches_the_same_fixed_point_in_about_half_the_iterations():
    """Same fixed point as the global solve; for this consistently ordered block-tridiagonal system the Gauss-Seidel
    rate is the square of the Jacobi rate, so about half the iterations."""
    p = W.config2(dt=1.0, J=96)       # thin cells, c = 0.9: slow convergence, several hundred Jacobi iterations
    exact = global_solve(p, p.q, p.psi0)
    jac, rb = oracle.Oracle(p), oracle.Oracle(p)
    it_j, _ = jac.oci_step(tol=1e-12, max_iters=20000, rule=0, advance=False)
    it_r, hist = rb.oci_step(tol=1e-12, max_iters=20000, rule=0, advance=False, ordering=1)
    scale = max(np.abs(exact).max(), 1e-300)
    np.testing.assert_allclose(rb.psi, exact, rtol=0, atol=1e-10 * scale + 1e-12)
    np.testing.assert_allclose(jac.psi, exact, rtol=0, atol=1e-10 * scale + 1e-12)
    assert 0.4 * it_j <= it_r <= 0.65 * it_j, (it_j, it_r)
