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


@pytest.mark.parametrize("bc_left,bc_right", [(W.BC_REFLECTIVE, W.BC_VACUUM), (W.BC_PRESCRIBED, W.BC_REFLECTIVE)])
def test_one_si_iteration_is_a_sweep_with_every_group_lagged(bc_left, bc_right):
    """The SI twin of the pin above (Eq. 42-45; Alg. 1): ONE iteration solves the streaming + removal
    operator L_c + L_b for every (g, m) with the whole scattering source -- all groups, the group's own included -- and
    the mirror ordinate of a reflective face taken from the OLD iterate (readings A12 and "group-Jacobi").
    A group-Gauss-Seidel sweep or a mirror from the current sweep reaches the same fixed point but fails this test.
    Built from Eq. 3 only: M(transfer) - M(0) is the scattering operator; in M(0) the only coupling between two
    different ordinates is the reflective mirror term."""
    import copy
    from pins import global_system, idx
    p = W.random_problem(31, J=4, N=4, G=3, bc_left=bc_left, bc_right=bc_right)
    M, rhs = global_system(p, p.q, p.psi0)
    p0 = copy.copy(p)
    p0.transfer = np.zeros_like(p.transfer)
    M0, rhs0 = global_system(p0, p.q, p.psi0)
    assert np.array_equal(rhs, rhs0)
    S = M0 - M                                   # scattering (+ fission) moved to the right-hand side
    assert np.abs(S).max() > 0
    ordinate = (np.arange(M.shape[0]) // 4) % p.N
    mirror = np.where(ordinate[:, None] != ordinate[None, :], M0, 0.0)
    assert np.count_nonzero(mirror) == 2 * p.G * (p.N // 2)   # one face: N/2 incoming ordinates x 2 time levels x G
    L = M0 - mirror                              # L_c + L_b: what the sweep inverts, ordinate by ordinate
    rng = np.random.default_rng(1)
    x0 = rng.uniform(0, 1, size=M.shape[0])
    want = np.linalg.solve(L, S @ x0 + rhs - mirror @ x0)
    o = oracle.Oracle(p)
    o.set_iterate(x0)
    got = o.si_iterate(1).reshape(-1)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13 * np.abs(want).max())
    # and the variants this pin is there to exclude are really different iterations on this problem
    scale = np.abs(want).max()
    assert np.abs(np.linalg.solve(M0, S @ x0 + rhs) - want).max() > 1e-6 * scale   # mirror from the new sweep
    group = (np.arange(M.shape[0]) // (4 * p.N)) % p.G
    x = x0.copy()                                                                  # group Gauss-Seidel
    for g in range(p.G):
        rows = np.flatnonzero(group == g)
        x[rows] = np.linalg.solve(L[np.ix_(rows, rows)], (S @ x + rhs - mirror @ x0)[rows])
    assert np.abs(x - want).max() > 1e-6 * scale


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


# ---------------------------------------------------------------------------------------------------------------
# The stopping arithmetic itself (Eq. 12-13; Alg. 2; Eq. 46 for SI), pinned hard:
# the tested quantity of every iteration and the iteration at which the loop stops are re-evaluated in numpy from
# iterates obtained one iteration at a time, never from the loop under test.
# ---------------------------------------------------------------------------------------------------------------
def _stop_index(e, tol, rule):
    """First 0-based l at which the rule holds for the tested quantities e[0], e[1], ...: rule 0: e_l < tol; rule 1:
    e_l < tol (1 - e_l / e_{l-1}), tested from l >= 1 (Alg. 2 computes e only in its else-branch)."""
    for l in range(len(e)):
        if rule == 0 and e[l] < tol:
            return l
        if rule == 1 and l >= 1 and e[l] < tol * (1.0 - e[l] / e[l - 1]):
            return l
    return None


@pytest.mark.parametrize("scheme", ["oci", "si"])
@pytest.mark.parametrize("rule", [0, 1])
def test_stop_rules_tested_quantity_and_stop_iteration(scheme, rule):
    p = W.random_problem(91, J=23, N=4, G=2, bc_left=W.BC_REFLECTIVE, bc_right=W.BC_PRESCRIBED, dt=0.4, c_max=0.9)
    tol = 1e-7
    # the loop under test
    o = oracle.Oracle(p)
    it, hist = (o.oci_step if scheme == "oci" else o.si_step)(tol=tol, rule=rule, advance=False)
    # the same iterates, one iteration at a time, norms taken by numpy
    s = oracle.Oracle(p)
    if scheme == "oci":
        s.factor()
        s.const_rhs()
    e = []
    for l in range(it + 3):
        psi_old, phi_old = s.psi.copy(), s.phi.copy()
        s.oci_iterate(1) if scheme == "oci" else s.si_iterate(1)
        if rule == 0:
            e.append(np.max(np.abs(s.phi - phi_old)))                       # BASELINE.json: |dphi|_inf
        elif scheme == "oci":
            e.append(np.linalg.norm((s.psi - psi_old).reshape(-1)))         # Eq. 12: ||Psi^(l+1) - Psi^(l)||_2
        else:
            e.append(np.linalg.norm((s.phi - phi_old).reshape(-1)))         # Eq. 46: ||phi^(l+1) - phi^(l)||_2
    e = np.array(e)
    np.testing.assert_allclose(hist, e[:it], rtol=1e-12, atol=0)
    stop = _stop_index(e, tol, rule)
    assert stop is not None and it == stop + 1, (it, stop)
    if rule == 1:
        # a max-norm in place of the 2-norm, or a test that starts at l = 0, would stop elsewhere on this problem
        e_inf = []
        s2 = oracle.Oracle(p)
        if scheme == "oci":
            s2.factor()
            s2.const_rhs()
        for l in range(it + 3):
            old = (s2.psi if scheme == "oci" else s2.phi).copy()
            s2.oci_iterate(1) if scheme == "oci" else s2.si_iterate(1)
            e_inf.append(np.max(np.abs((s2.psi if scheme == "oci" else s2.phi) - old)))
        assert _stop_index(np.array(e_inf), tol, 1) != stop
        assert hist[0] > tol                                                 # l = 0 is recorded but never tested


def test_rule1_counts_on_config2_first_step():
    """SURVEY 8(c) H1, re-derived here: config 2 at dt = 1, J = 1024, first step. Rule 0 (|dphi|_inf < 1e-8) stops after
    725 iterations with a true error of ~5e-7; the paper's rule 1 (eps = 1e-8) needs 1145 (rho_e ~ 0.974) and ends
    ~1e-10 from the fixed point: the (1 - rho_e) factor does what PAPER.md:441-442 says."""
    p = W.config2(dt=1.0)
    o0, o1, ref = oracle.Oracle(p), oracle.Oracle(p), oracle.Oracle(p)
    it0, _ = o0.oci_step(tol=1e-8, rule=0, advance=False)
    it1, h1 = o1.oci_step(tol=1e-8, rule=1, advance=False)
    assert (it0, it1) == (725, 1145)
    assert abs(h1[-1] / h1[-2] - 0.974) < 2e-3
    ref.oci_step(tol=1e-14, max_iters=200000, advance=False)
    err0, err1 = np.abs(o0.phi - ref.phi).max(), np.abs(o1.phi - ref.phi).max()
    assert 2e-7 < err0 < 1e-6 and err1 < 5e-10
