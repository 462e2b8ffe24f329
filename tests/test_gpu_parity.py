"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle, element by
element on the same seeded inputs. Tolerances (BASELINE.json north_star):
  * assembled A_j: bit-exact (every rounding in the kernel is explicit);
  * per-iteration angular flux: max|psi_gpu - psi_orc| / max|psi_orc| <= 1e-11 after the same number of iterations;
  * converged scalar flux: <= 1e-9 relative, GPU and oracle run for the same number of iterations.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL_ITER = 1e-11
TOL_PHI = 1e-9


def _solver(p, **kw):
    from paper_2503_00264_b200 import OCISolver
    return OCISolver(p, **kw)


def _oracle(p):
    from oracle import Oracle
    return Oracle(p)


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


SMALL_CASES = [
    # seed, J, N, G, bc_left, bc_right   (n = 4NG: 8, 16, 24, 32, 48, 64, 96, 128, 160, 200, 256; ragged J everywhere)
    (1, 5, 2, 1, 0, 0),
    (2, 37, 4, 1, 0, 0),
    (3, 19, 2, 3, 1, 0),
    (4, 67, 8, 1, 2, 2),
    (5, 23, 6, 2, 0, 1),
    (6, 301, 16, 1, 1, 1),
    (7, 9, 8, 3, 2, 0),
    (8, 150, 8, 4, 0, 0),
    (9, 7, 10, 4, 0, 2),
    (10, 11, 8, 8, 1, 0),
    (11, 1, 4, 2, 0, 0),      # a single cell: both neighbours are boundaries
    (12, 2, 2, 1, 1, 1),
    (18, 300, 2, 1, 0, 2),    # S2 with J G > 64: 128 (j, g) pairs per block of si_finish_kernel (the round-1 bug)
    (19, 200, 2, 3, 1, 0),    # S2, three groups
    (20, 6, 10, 5, 0, 0),     # n = 200: not a multiple of 64 and too large for shared memory (global-scratch factor path)
]


@pytest.mark.parametrize("seed,J,N,G,bl,br", SMALL_CASES)
def test_assembly_bit_exact(seed, J, N, G, bl, br):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br)
    s, o = _solver(p), _oracle(p)
    for j in sorted({0, J // 2, J - 1}):
        A_gpu = s.debug_matrix(j)
        A_orc = o.assemble_cell(j)
        assert np.array_equal(A_gpu, A_orc), f"cell {j}: max diff {np.max(np.abs(A_gpu - A_orc))}"


@pytest.mark.parametrize("seed,J,N,G,bl,br", SMALL_CASES)
def test_factor_gives_inverse(seed, J, N, G, bl, br):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br, dt=10.0 ** (-(seed % 4)))
    s, o = _solver(p), _oracle(p)
    assert s.factor() == 0
    for j in sorted({0, J // 3, J - 1}):
        A = o.assemble_cell(j)
        Ainv = s.debug_inverse(j)
        n = A.shape[0]
        assert np.max(np.abs(A @ Ainv - np.eye(n))) < 1e-12 * np.linalg.cond(A)


def test_factor_flags_singular_cell():
    p = W.random_problem(21, 12, 4, 1)
    p.sigma_t = p.sigma_t.copy()
    p.sigma_t[7] = np.nan
    s = _solver(p)
    assert s.factor() == 8  # 1-based index of the first bad cell


def test_flagged_factors_are_dropped_with_the_dt_they_belong_to():
    """After an oci_factor that reported a singular cell the debug getter may read the other cells' inverses; once dt
    (or the factor kernel) changes, those belong to a matrix that no longer exists: OCI_E_STATE until the next factor."""
    from paper_2503_00264_b200 import OCIError
    p = W.random_problem(21, 12, 4, 1)
    p.sigma_t = p.sigma_t.copy()
    p.sigma_t[7] = np.nan
    s = _solver(p)
    assert s.factor() == 8
    assert np.all(np.isfinite(s.debug_inverse(3)))
    s.set_dt(p.dt * 0.5)
    with pytest.raises(OCIError) as e:
        s.debug_inverse(3)
    assert e.value.code == -103
    assert s.factor() == 8
    s.set_option("factor_kernel", 0)
    with pytest.raises(OCIError) as e:
        s.debug_inverse(3)
    assert e.value.code == -103


def test_step_that_meets_a_singular_cell_leaves_a_defined_state():
    """oci_step enqueues the factor with its first batch of iterations; when the factor flags a cell the call must not
    hand back whatever those iterations wrote: iterate = both time levels of psi_{k-1/2}, its phi, empty history."""
    from paper_2503_00264_b200 import OCIError
    p = W.random_problem(23, 40, 4, 2, bc_left=W.BC_REFLECTIVE)
    p.sigma_t = p.sigma_t.copy()
    p.sigma_t[17] = np.nan
    s = _solver(p)
    edge = s.get_state().cpu().numpy()
    for _ in range(2):  # the same answer and the same state on a retry
        with pytest.raises(OCIError) as e:
            s.step(tol=1e-9, max_iters=50, check_every=5)
        assert e.value.code == 18
        psi = s.angular_flux().cpu().numpy()
        assert np.array_equal(psi[..., 0:2], edge) and np.array_equal(psi[..., 2:4], edge)
        phi = s.scalar_flux().cpu().numpy()
        assert np.allclose(phi, np.einsum("m,jgmp->jgp", p.w, psi), rtol=0, atol=1e-13 * max(np.abs(psi).max(), 1.0))
        assert np.array_equal(s.get_state().cpu().numpy(), edge)
        assert len(s.residual_history(0)) == 0


def test_option_values_outside_their_range_are_refused():
    from paper_2503_00264_b200 import OCIError
    s = _solver(W.random_problem(22, 9, 4, 1))
    bad = {"factor_kernel": [2, 3, 5, -1], "factor_update": [3, -1], "factor_cluster": [2],
           "refactor_every_step": [2], "persistent": [2, -2], "iterate_kernel": [2], "si_lanes": [3, 32],
           "solve_mode": [2], "ordering": [2], "si_sweep": [2], "iterate_stages": [-1]}
    for key, values in bad.items():
        for v in values:
            with pytest.raises(OCIError) as e:
                s.set_option(key, v)
            assert e.value.code == -3, (key, v)
    # unknown keys, among them the tuning probes that left the public header after round 2
    for key in ("no_such_key", "st_warp_local", "st_consumer_threads", "st_fused_setup", "iterate_ctas_per_sm"):
        with pytest.raises(OCIError) as e:
            s.set_option(key, 0)
        assert e.value.code == -2, key
    for key, v in [("factor_kernel", 4), ("factor_update", 0), ("si_lanes", 16), ("persistent", -1), ("iterate_stages", 0)]:
        s.set_option(key, v)  # the documented values still pass


@pytest.mark.parametrize("kernel", [1, 0])
@pytest.mark.parametrize("seed,J,N,G,bl,br", SMALL_CASES)
def test_oci_per_iteration_parity(seed, J, N, G, bl, br, kernel):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br)
    s, o = _solver(p, options={"iterate_kernel": kernel}), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    o.const_rhs()
    assert rel(s.debug_const_rhs().cpu().numpy(), o.c) < 1e-14
    for l in range(6):
        s.iterate(1)
        o.oci_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"iteration {l + 1}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER
    s.iterate(7)
    o.oci_iterate(7)
    assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER


@pytest.mark.parametrize("seed,J,N,G,bl,br", SMALL_CASES)
def test_si_per_iteration_parity(seed, J, N, G, bl, br):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br)
    s, o = _solver(p), _oracle(p)
    for l in range(5):
        s.si_iterate(1)
        o.si_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"iteration {l + 1}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_step_loop_matches_oracle(scheme, rule):
    """Several time steps: iteration counts (check_every = 1 -> natural count), residual history, converged phi."""
    p = W.random_problem(31, 40, 4, 2, bc_left=1, bc_right=2, dt=0.05)
    s, o = _solver(p), _oracle(p)
    for step in range(3):
        if scheme == "oci":
            it_g, conv_g, res_g = s.step(tol=1e-9, max_iters=500, check_every=1, stop_rule=rule)
            it_o, hist_o = o.oci_step(tol=1e-9, max_iters=500, rule=rule)
        else:
            it_g, conv_g, res_g = s.si_step(tol=1e-9, max_iters=500, check_every=1, stop_rule=rule)
            it_o, hist_o = o.si_step(tol=1e-9, max_iters=500, rule=rule)
        assert it_g == it_o == conv_g, f"step {step}"
        hist_g = s.residual_history(kind=rule)
        assert len(hist_g) == it_o
        np.testing.assert_allclose(hist_g, hist_o, rtol=1e-6, atol=1e-15)
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
        assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI


def test_check_every_overshoot_is_bounded_and_same_iterations_agree():
    """with check_every = k the GPU may run < k extra iterations; the oracle run for exactly that many
    iterations agrees to 1e-9."""
    p = W.config2(dt=0.1, J=256)
    s, o = _solver(p), _oracle(p)
    it_g, conv_g, _ = s.step(tol=1e-8, max_iters=4000, check_every=8, advance=False)
    o2 = _oracle(p)
    it_nat, _ = o2.oci_step(tol=1e-8, max_iters=4000, advance=False)
    assert conv_g == it_nat
    assert 0 <= it_g - it_nat < 8
    o.factor()
    o.const_rhs()
    o.oci_iterate(it_g)
    assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI


def test_config1_full_run_both_schemes():
    p = W.config1()
    s, o = _solver(p), _oracle(p)
    s2, o2 = _solver(p), _oracle(p)
    for step in range(p.n_steps):
        it_g, conv_g, _ = s.step(tol=p.tol, check_every=1)
        it_o, _ = o.oci_step(tol=p.tol)
        assert it_g == it_o
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
        it_g2, _, _ = s2.si_step(tol=p.tol, check_every=1)
        it_o2, _ = o2.si_step(tol=p.tol)
        assert it_g2 == it_o2
        assert rel(s2.scalar_flux().cpu().numpy(), o2.phi) < TOL_PHI


def test_set_iterate_worked_example_head():
    """Random initial iterate (PAPER.md:479 verification run), no source: the iterate itself is the error."""
    p = W.worked_example(J=200)
    s, o = _solver(p), _oracle(p)
    s.set_iterate(p.meta["psi_guess"])
    o.set_iterate(p.meta["psi_guess"])
    s.factor(); o.factor(); o.const_rhs()
    s.iterate(25)
    o.oci_iterate(25)
    assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER


def test_set_dt_refactors():
    p = W.random_problem(41, 30, 4, 2)
    s = _solver(p)
    s.factor()
    s.iterate(3)
    s.set_dt(p.dt / 10)
    with pytest.raises(Exception):
        s.iterate(1)  # factors are stale: OCI_E_STATE
    s.factor()
    o = _oracle(p.with_dt(p.dt / 10))
    o.set_iterate(s.angular_flux().cpu().numpy())
    o.factor(); o.const_rhs()
    s.iterate(2)
    o.oci_iterate(2)
    assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("scheme", ["oci", "si"])
@pytest.mark.parametrize("k", [2, 5, 8])
def test_device_side_stop_runs_the_natural_iteration_count(scheme, rule, k):
    """DESIGN.md section 5 "device-side stop": with check_every = k the launches after the iteration at which the
    rule first held skip themselves, so the iterations that ran, the converged iterate (whichever Jacobi buffer
    it ended in) and the state handed to the next step equal the oracle's natural run."""
    p = W.random_problem(33, 61, 4, 2, bc_left=1, bc_right=2, dt=0.05)
    s, o = _solver(p), _oracle(p)
    for step in range(3):
        if scheme == "oci":
            it_g, conv_g, _ = s.step(tol=1e-9, max_iters=500, check_every=k, stop_rule=rule)
            it_o, hist_o = o.oci_step(tol=1e-9, max_iters=500, rule=rule)
        else:
            it_g, conv_g, _ = s.si_step(tol=1e-9, max_iters=500, check_every=k, stop_rule=rule)
            it_o, hist_o = o.si_step(tol=1e-9, max_iters=500, rule=rule)
        assert it_g == conv_g == it_o, f"step {step}"
        hist_g = s.residual_history(kind=rule)
        assert len(hist_g) == it_o
        np.testing.assert_allclose(hist_g, hist_o, rtol=1e-6, atol=1e-15)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_PHI
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
        assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI


def test_max_iters_reached_without_convergence():
    p = W.config2(dt=1.0, J=128)
    s, o = _solver(p), _oracle(p)
    it_g, conv_g, res = s.step(tol=1e-14, max_iters=13, check_every=4, advance=False)
    assert (it_g, conv_g) == (13, 0)
    o.factor(); o.const_rhs(); o.oci_iterate(13)
    assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER


# ---------------------------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times (production kernels, check_every = 8).
# The oracle runs the whole problem (factor + a few iterations: tens of seconds of host time in total), so every
# cell of every iterate is compared element by element; nothing is sampled from the CUDA path.
# ---------------------------------------------------------------------------------------------------------------
FULL_CASES = [
    ("cfg2", lambda: W.config2(dt=0.01), 4),
    ("cfg3", lambda: W.config3(), 3),
    ("cfg4", lambda: W.config4(), 3),
    ("cfg4b", lambda: W.config4(v=1000.0), 3),
    ("cfg5@1e-2", lambda: W.config5(dt=1e-2), 3),
    ("cfg5@1e-4", lambda: W.config5(dt=1e-4), 2),
]


@pytest.mark.parametrize("name,make,n_it", FULL_CASES, ids=[c[0] for c in FULL_CASES])
def test_full_size_per_iteration_parity(name, make, n_it):
    p = make()
    s, o = _solver(p), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    o.const_rhs()
    for l in range(n_it):
        s.iterate(1)
        o.oci_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"{name}: OCI iteration {l + 1}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER
    # the factors themselves, on cells spread over the slab (first, last, tile boundaries, random)
    rng = np.random.default_rng(7)
    for j in sorted({0, 1, p.J // 2, p.J - 2, p.J - 1, *rng.integers(0, p.J, 3).tolist()}):
        A = o.assemble_cell(j)
        assert np.array_equal(s.debug_matrix(j), A)
        assert np.max(np.abs(A @ s.debug_inverse(j) - np.eye(p.n))) < 1e-12 * np.linalg.cond(A)


@pytest.mark.parametrize("name,make", [("cfg2", lambda: W.config2(dt=0.01)), ("cfg5@1e-3", lambda: W.config5(dt=1e-3)),
                                        ("cfg4", lambda: W.config4())], ids=["cfg2", "cfg5@1e-3", "cfg4"])
def test_full_size_converged_step_parity(name, make):
    """One converged time step exactly as bench.py runs it (check_every = 8, device-side stop): iteration count equal
    to the oracle's natural count, converged phi and the state handed to the next step within 1e-9; same for SI."""
    p = make()
    s, o = _solver(p), _oracle(p)
    it_g, conv_g, _ = s.step(tol=p.tol, max_iters=4000, check_every=8)
    it_o, _ = o.oci_step(tol=p.tol, max_iters=4000)
    assert it_g == conv_g == it_o
    assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
    assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI
    s2, o2 = _solver(p), _oracle(p)
    it_g2, conv_g2, _ = s2.si_step(tol=p.tol, max_iters=4000, check_every=8)
    it_o2, _ = o2.si_step(tol=p.tol, max_iters=4000)
    assert it_g2 == conv_g2 == it_o2
    assert rel(s2.scalar_flux().cpu().numpy(), o2.phi) < TOL_PHI


def test_full_size_si_per_iteration_parity_cfg5():
    p = W.config5(dt=1e-2)
    s, o = _solver(p), _oracle(p)
    for l in range(3):
        s.si_iterate(1)
        o.si_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"SI iteration {l + 1}"


@pytest.mark.parametrize("lanes", [4, 16])
def test_si_lane_groupings_agree(lanes):
    p = W.random_problem(8, 150, 8, 4, bc_left=1, bc_right=2)
    s, o = _solver(p, options={"si_lanes": lanes}), _oracle(p)
    for l in range(3):
        s.si_iterate(1)
        o.si_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER


def test_factor_kernels_agree_n64():
    """n = 64: the two-warp kernel (default) and the generic shared-memory kernel give the same inverse to rounding."""
    p = W.config5(J=300, dt=1e-3)
    a, b = _solver(p), _solver(p, options={"factor_kernel": 0})
    assert a.factor() == 0 and b.factor() == 0
    for j in (0, 149, 299):
        A = _oracle(p).assemble_cell(j)
        for s in (a, b):
            assert np.max(np.abs(A @ s.debug_inverse(j) - np.eye(64))) < 1e-12 * np.linalg.cond(A)


# ---------------------------------------------------------------------------------------------------------------
# structured cell solve ("solve_mode" = 1). Same oracle, same tolerances.
# ---------------------------------------------------------------------------------------------------------------
ST = {"solve_mode": 1}


@pytest.mark.parametrize("kernel", [1, 0])   # 1: persistent bulk-copy pipeline (default); 0: one batch of cells per CTA
@pytest.mark.parametrize("seed,J,N,G,bl,br", SMALL_CASES)
def test_structured_per_iteration_parity(seed, J, N, G, bl, br, kernel):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br)
    s, o = _solver(p, options={"solve_mode": 1, "iterate_kernel": kernel}), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    o.const_rhs()
    for l in range(6):
        s.iterate(1)
        o.oci_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"iteration {l + 1}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER
    s.iterate(7)
    o.oci_iterate(7)
    assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER


@pytest.mark.parametrize("name,make,n_it", FULL_CASES, ids=[c[0] for c in FULL_CASES])
def test_structured_full_size_parity(name, make, n_it):
    p = make()
    s, o = _solver(p, options=ST), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    o.const_rhs()
    for l in range(n_it):
        s.iterate(1)
        o.oci_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"{name}: iteration {l + 1}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER


@pytest.mark.parametrize("kernel", [1, 0])
@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("k", [1, 5])
def test_structured_step_loop_matches_oracle(rule, k, kernel):
    p = W.random_problem(33, 61, 4, 2, bc_left=1, bc_right=2, dt=0.05)
    s, o = _solver(p, options={"solve_mode": 1, "iterate_kernel": kernel}), _oracle(p)
    for step in range(3):
        it_g, conv_g, _ = s.step(tol=1e-9, max_iters=500, check_every=k, stop_rule=rule)
        it_o, hist_o = o.oci_step(tol=1e-9, max_iters=500, rule=rule)
        assert it_g == conv_g == it_o, f"step {step}"
        np.testing.assert_allclose(s.residual_history(kind=rule), hist_o, rtol=1e-6, atol=1e-15)
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
        assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI


def test_structured_and_dense_paths_agree_on_a_converged_config5_step():
    p = W.config5(dt=1e-1)
    a, b = _solver(p, options=ST), _solver(p)
    ia, _, _ = a.step(tol=p.tol, max_iters=4000, check_every=8)
    ib, _, _ = b.step(tol=p.tol, max_iters=4000, check_every=8)
    assert ia == ib
    assert rel(a.scalar_flux().cpu().numpy(), b.scalar_flux().cpu().numpy()) < 1e-12


def test_structured_mode_switch_refactors_and_flags_singular():
    p = W.random_problem(21, 12, 4, 1)
    s = _solver(p)
    s.factor()
    s.set_option("solve_mode", 1)
    with pytest.raises(Exception):
        s.iterate(1)                 # factors of the other mode: OCI_E_STATE
    assert s.factor() == 0
    s.iterate(2)
    p.sigma_t = p.sigma_t.copy()
    p.sigma_t[7] = np.nan
    assert _solver(p, options=ST).factor() == 8


# ---------------------------------------------------------------------------------------------------------------
# the SI sweep evaluated as a parallel scan ("si_sweep" = 1). Same oracle (serial sweep).
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,J,N,G,bl,br", SMALL_CASES + [(13, 2500, 4, 2, 1, 2), (14, 1024, 8, 1, 0, 0)])
def test_si_scan_per_iteration_parity(seed, J, N, G, bl, br):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br)
    s, o = _solver(p, options={"si_sweep": 1}), _oracle(p)
    for l in range(4):
        s.si_iterate(1)
        o.si_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"iteration {l + 1}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER


def test_si_scan_full_size_step_cfg5():
    p = W.config5(dt=1e-2)
    s, o = _solver(p, options={"si_sweep": 1}), _oracle(p)
    it_g, conv_g, _ = s.si_step(tol=p.tol, max_iters=4000, check_every=8)
    it_o, _ = o.si_step(tol=p.tol, max_iters=4000)
    assert it_g == conv_g == it_o
    assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
    assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI


# ---------------------------------------------------------------------------------------------------------------
# a batch of structured iterations as ONE cooperative launch with grid-wide barriers.
# ---------------------------------------------------------------------------------------------------------------
PERSIST = {"solve_mode": 1, "persistent": 1}


@pytest.mark.parametrize("seed,J,N,G,bl,br", SMALL_CASES + [(15, 3000, 4, 2, 1, 2)])
def test_persistent_multi_iteration_parity(seed, J, N, G, bl, br):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br)
    s, o = _solver(p, options=PERSIST), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    o.const_rhs()
    for k in (2, 5, 8):          # even and odd batch lengths: the two Psi buffers alternate inside the launch
        s.iterate(k)
        o.oci_iterate(k)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"after a batch of {k}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("k", [2, 5, 8])
def test_persistent_step_loop_stops_at_the_natural_iteration(rule, k):
    p = W.random_problem(33, 61, 4, 2, bc_left=1, bc_right=2, dt=0.05)
    s, o = _solver(p, options=PERSIST), _oracle(p)
    for step in range(3):
        it_g, conv_g, _ = s.step(tol=1e-9, max_iters=500, check_every=k, stop_rule=rule)
        it_o, hist_o = o.oci_step(tol=1e-9, max_iters=500, rule=rule)
        assert it_g == conv_g == it_o, f"step {step}"
        np.testing.assert_allclose(s.residual_history(kind=rule), hist_o, rtol=1e-6, atol=1e-15)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_PHI
        assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI


def test_persistent_auto_applies_to_config2_and_matches():
    p = W.config2(dt=0.1)
    a, b = _solver(p, options={"solve_mode": 1}), _solver(p, options={"solve_mode": 1, "persistent": 0})
    ia, _, _ = a.step(tol=p.tol, max_iters=4000, check_every=8)
    ib, _, _ = b.step(tol=p.tol, max_iters=4000, check_every=8)
    assert ia == ib
    assert a.last_timing(1)[1] < b.last_timing(1)[1]          # fewer launches: one per batch instead of one per iteration
    assert rel(a.scalar_flux().cpu().numpy(), b.scalar_flux().cpu().numpy()) < 1e-13


# ---------------------------------------------------------------------------------------------------------------
# SURVEY 8(f) row f4 (first half): red-black ordering of the cell solves ("ordering" = 1, structured path).
# ---------------------------------------------------------------------------------------------------------------
RB = {"solve_mode": 1, "ordering": 1}


@pytest.mark.parametrize("seed,J,N,G,bl,br", SMALL_CASES + [(16, 1001, 8, 2, 1, 2), (17, 1000, 16, 1, 0, 1)])
def test_redblack_per_iteration_parity(seed, J, N, G, bl, br):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br)
    s, o = _solver(p, options=RB), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    o.const_rhs()
    for l in range(5):
        s.iterate(1)
        o.oci_iterate(1, ordering=1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"iteration {l + 1}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER
    s.iterate(6)
    o.oci_iterate(6, ordering=1)
    assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("k", [1, 5])
def test_redblack_step_loop_matches_oracle(rule, k):
    p = W.random_problem(33, 61, 4, 2, bc_left=1, bc_right=2, dt=0.05)
    s, o = _solver(p, options=RB), _oracle(p)
    for step in range(3):
        it_g, conv_g, _ = s.step(tol=1e-9, max_iters=500, check_every=k, stop_rule=rule)
        it_o, hist_o = o.oci_step(tol=1e-9, max_iters=500, rule=rule, ordering=1)
        assert it_g == conv_g == it_o, f"step {step}"
        np.testing.assert_allclose(s.residual_history(kind=rule), hist_o, rtol=1e-6, atol=1e-15)
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
        assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI


def test_redblack_config5_full_size_halves_the_iterations():
    p = W.config5(dt=1.0)
    rb, jac, o = _solver(p, options=RB), _solver(p, options={"solve_mode": 1}), _oracle(p)
    it_r, conv_r, _ = rb.step(tol=p.tol, max_iters=4000, check_every=8)
    it_j, _, _ = jac.step(tol=p.tol, max_iters=4000, check_every=8)
    it_o, _ = o.oci_step(tol=p.tol, max_iters=4000, ordering=1)
    assert it_r == conv_r == it_o
    assert it_r < 0.65 * it_j
    assert rel(rb.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
    assert float((rb.scalar_flux() - jac.scalar_flux()).abs().max()) < 1e-6     # both stopped at tol 1e-8


def test_redblack_needs_the_structured_path():
    p = W.random_problem(2, 9, 4, 1)
    s = _solver(p, options={"ordering": 1})
    s.factor()
    with pytest.raises(Exception):
        s.iterate(1)


# ---------------------------------------------------------------------------------------------------------------
# SURVEY 8(f) row f2, dense path: a batch of iterations as ONE cooperative launch with the inverses resident in shared
# memory (automatic when they fit: BASELINE.json configs 1-2). Mirrors the test_persistent_* tests of the structured path.
# ---------------------------------------------------------------------------------------------------------------
def _fits_resident(J, N, G, sms=148, smem=200 * 1024):
    """the inverses of ceil(J / SMs) cells fit in one CTA's shared memory (launch_dense_multi's condition, with margin)"""
    n = 4 * N * G
    return -(-J // sms) * n * n * 8 <= smem


@pytest.mark.parametrize("seed,J,N,G,bl,br", [c for c in SMALL_CASES if _fits_resident(c[1], c[2], c[3])] + [(21, 1200, 8, 1, 1, 2)])
def test_dense_resident_multi_iteration_parity(seed, J, N, G, bl, br):
    p = W.random_problem(seed, J, N, G, bc_left=bl, bc_right=br)
    s, o = _solver(p), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    o.const_rhs()
    for k in (2, 5, 8):          # even and odd batch lengths: the two Psi buffers alternate inside the launch
        s.iterate(k)
        assert s.last_timing(1)[1] <= 2, "the batch should have been ONE launch (+ the constant right-hand side the first time)"
        o.oci_iterate(k)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"after a batch of {k}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("k", [2, 5, 8])
def test_dense_resident_step_loop_stops_at_the_natural_iteration(rule, k):
    p = W.random_problem(33, 61, 4, 2, bc_left=1, bc_right=2, dt=0.05)
    s, o = _solver(p), _oracle(p)
    for step in range(3):
        it_g, conv_g, _ = s.step(tol=1e-9, max_iters=500, check_every=k, stop_rule=rule)
        it_o, hist_o = o.oci_step(tol=1e-9, max_iters=500, rule=rule)
        assert it_g == conv_g == it_o, f"step {step}"
        np.testing.assert_allclose(s.residual_history(kind=rule), hist_o, rtol=1e-6, atol=1e-15)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_PHI
        assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI


def test_dense_resident_auto_applies_to_config2_and_matches_the_per_iteration_kernel():
    p = W.config2(dt=0.1)
    a, b = _solver(p), _solver(p, options={"persistent": 0})
    ia, _, _ = a.step(tol=p.tol, max_iters=4000, check_every=8)
    ib, _, _ = b.step(tol=p.tol, max_iters=4000, check_every=8)
    assert ia == ib
    assert a.last_timing(1)[1] < b.last_timing(1)[1]          # one launch per batch instead of one per iteration
    assert rel(a.scalar_flux().cpu().numpy(), b.scalar_flux().cpu().numpy()) < 1e-13


@pytest.mark.parametrize("opts", [{}, {"solve_mode": 1}], ids=["dense", "structured"])
@pytest.mark.parametrize("J,N,G", [(1201, 16, 1), (333, 8, 4), (150, 8, 8)])   # n = 64, 128, 256: the warp-per-cell kernels
def test_walk_direction_does_not_change_an_iteration(J, N, G, opts):
    """The streaming iterate kernels walk every CTA's range of cells upwards or downwards depending on the parity of the
    history slot (the tail of one iteration is still in the L2 when the next one asks for it). A Jacobi iteration does
    not depend on the order of its cells, so the iterates must be BIT-identical whichever way they were produced: one
    solver iterates from slot 0 (down, up, down), the other burns one slot first and starts again from the same iterate
    at slot 1 (up, down, up). Ragged J: the CTAs' ranges and the last group of four cells are ragged in both directions."""
    p = W.random_problem(400 + J, J, N, G, bc_left=1, bc_right=2)
    a, b = _solver(p, options=opts), _solver(p, options=opts)
    assert a.factor() == 0 and b.factor() == 0
    psi0 = b.angular_flux().clone()
    b.iterate(1)
    b.set_iterate(psi0)
    for l in range(3):
        a.iterate(1)
        b.iterate(1)
        assert np.array_equal(a.angular_flux().cpu().numpy(), b.angular_flux().cpu().numpy()), f"iteration {l + 1}"
        assert np.array_equal(a.scalar_flux().cpu().numpy(), b.scalar_flux().cpu().numpy()), f"iteration {l + 1}"
    o = _oracle(p)
    assert o.factor() == 0
    o.const_rhs()
    o.oci_iterate(3)
    assert rel(a.angular_flux().cpu().numpy(), o.psi) < TOL_ITER
