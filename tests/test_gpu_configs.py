"""GPU parity on BASELINE.json's five configurations run as CONFIGURED (the dt sequences, the step counts, the pulsed
source), on the paper's Table-2 workload, and on the launch paths and shapes the small-case file does not reach.

north_star: "OCI on one B200 matches the oracle within 1e-9 on all five configs". Every step of every sequence is
compared: iterations performed (device-side stop, check_every = 8 as in bench.py) == the oracle's natural count,
converged scalar flux and the state handed to the next step within 1e-9 (max-norm, and per cell at CELL_TOL), for OCI
and for the SI comparator. Nothing here is sampled from the CUDA path: the oracle runs the same sequence in full.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL_ITER = 1e-11
TOL_PHI = 1e-9
# Per-cell metric: max over cells of max|diff in the cell| / max|reference in the cell|. On
# config 5 sigma_t spans four decades, so a cell can sit 1e4 below the global maximum; the global max-norm bound
# 1e-11 (per iteration) / 1e-9 (converged) then only guarantees 1e-7 / 1e-5 there. Measured per-cell differences are
# ~1e-13; the bound asserted is 1e-9 per iteration and 1e-8 converged -- two to three decades tighter than what the
# global norm implies, and loose enough for cond(A_j) <= ~1e3 times a few ulp accumulated over a step.
CELL_TOL_ITER = 1e-9
CELL_TOL_PHI = 1e-8


def _solver(p, **kw):
    from paper_2503_00264_b200 import OCISolver
    return OCISolver(p, **kw)


def _oracle(p, **kw):
    from oracle import Oracle
    return Oracle(p, **kw)


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def rel_cell(a, b):
    """max_j ( max|a_j - b_j| / max|b_j| ) over cells j (axis 0); cells whose reference is exactly 0 are compared
    absolutely against the global scale."""
    a, b = np.asarray(a), np.asarray(b)
    J = b.shape[0]
    d = np.max(np.abs(a - b).reshape(J, -1), axis=1)
    s = np.max(np.abs(b).reshape(J, -1), axis=1)
    g = max(float(np.max(s)), 1e-300)
    s = np.where(s > 0.0, s, g)
    return float(np.max(d / s))


def _run_sequence(p, schedule, scheme, solver_options=None, check_every=8, max_iters=4000):
    """schedule: list of (dt, n_steps). One oracle walks through the whole sequence and with it one solver per entry of
    `solver_options` (a dict, or a list of dicts: e.g. the dense and the structured path side by side, each compared
    with the ORACLE step by step, never with each other); set_dt between the blocks goes through oci_step / si_step
    (which refactors when the factors are stale). The source of step s is p.source_at_step(s) (config 4's pulse).
    Returns the per-step iteration counts."""
    option_sets = solver_options if isinstance(solver_options, list) else [solver_options or {}]
    solvers = [_solver(p, dt=schedule[0][0], options=opts) for opts in option_sets]
    o = _oracle(p, dt=schedule[0][0])
    step = 0
    counts = []
    for dt, n_steps in schedule:
        for s in solvers:
            s.set_dt(dt)
        o.set_dt(dt)
        for _ in range(n_steps):
            q = p.source_at_step(step)
            o.set_source(q)
            if scheme == "oci":
                it_o, _ = o.oci_step(tol=p.tol, max_iters=max_iters)
            else:
                it_o, _ = o.si_step(tol=p.tol, max_iters=max_iters)
            for s, opts in zip(solvers, option_sets):
                s.set_source(q)
                if scheme == "oci":
                    it_g, conv_g, _ = s.step(tol=p.tol, max_iters=max_iters, check_every=check_every)
                else:
                    it_g, conv_g, _ = s.si_step(tol=p.tol, max_iters=max_iters, check_every=check_every)
                where = f"{p.name} {scheme} {opts} dt={dt:g} step {step}"
                assert it_g == conv_g == it_o, f"{where}: iterations gpu {it_g} (rule held at {conv_g}), oracle {it_o}"
                phi_g, st_g = s.scalar_flux().cpu().numpy(), s.get_state().cpu().numpy()
                assert rel(phi_g, o.phi) < TOL_PHI, where
                assert rel(st_g, o.psi_prev) < TOL_PHI, where
                assert rel_cell(phi_g, o.phi) < CELL_TOL_PHI, where
            counts.append(it_o)
            step += 1
    return counts


# the dense path (the paper's method) and the structured cell solve, each against the oracle
BOTH_PATHS = [{}, {"solve_mode": 1}]


def _paths(scheme):
    return BOTH_PATHS if scheme == "oci" else None


# ---------------------------------------------------------------------------------------------------------------
# config 1: 5 steps (also in test_gpu_parity.py with check_every = 1); here as bench.py's per_config runs it
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_config1_as_configured(scheme):
    p = W.config1()
    counts = _run_sequence(p, [(p.dt, p.n_steps)], scheme, solver_options=_paths(scheme))
    # 17,17,16,16,16 OCI iterations, 6 SI iterations per step (the oracle's own counts are pinned on the CPU)
    assert counts == ([17, 17, 16, 16, 16] if scheme == "oci" else [6] * 5)


# ---------------------------------------------------------------------------------------------------------------
# config 2: dt in {1, 0.1, 0.01}, 20 steps each, J = 1024. dt = 1 is the rho ~ 0.99 stress case:
# ~700 iterations in the first step.
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", ["oci", "si"])
@pytest.mark.parametrize("dt", [1.0, 0.1, 0.01])
def test_config2_as_configured(dt, scheme):
    p = W.config2(dt=dt)
    counts = _run_sequence(p, [(dt, p.n_steps)], scheme, solver_options=_paths(scheme), max_iters=20000)
    if scheme == "oci" and dt == 1.0:
        assert counts[0] > 500          # the slowly converging regime really is exercised


def test_config2_dt_changes_mid_run_through_oci_step():
    """set_dt between blocks of steps of ONE run: oci_step must refactor, the state carries over."""
    p = W.config2(dt=1.0, J=256)
    _run_sequence(p, [(1.0, 2), (0.1, 3), (0.01, 3), (0.1, 2)], "oci", solver_options=BOTH_PATHS, max_iters=20000)


# ---------------------------------------------------------------------------------------------------------------
# config 3: ten steps, 4 groups, n = 128 (cluster factor kernel, warp-per-cell iterate kernel with RPL = 4)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_config3_as_configured(scheme):
    p = W.config3()
    _run_sequence(p, [(p.dt, p.n_steps)], scheme, solver_options=_paths(scheme))


# ---------------------------------------------------------------------------------------------------------------
# config 4: n = 256, reflective left, source on during step 0 only. v = 1 (literal reading): all 50 steps (3-4
# iterations each). Variant 4b (v = 1000, where c = 0.99 bites, ~90 iterations per step): the first 3 steps, which
# include two with the source off.
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_config4_as_configured_pulsed_source(scheme):
    p = W.config4()
    counts = _run_sequence(p, [(p.dt, p.n_steps)], scheme, solver_options=_paths(scheme))
    assert len(counts) == 50


@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_config4b_first_steps_pulsed_source(scheme):
    p = W.config4(v=1000.0)
    _run_sequence(p, [(p.dt, 3)], scheme, solver_options=_paths(scheme))


# ---------------------------------------------------------------------------------------------------------------
# config 5 as BASELINE.json configs[4] writes it: dt in {1, 0.1, 0.01, 1e-3, 1e-4}, 10 steps each, J = 65536, one run,
# dt changed between the blocks through oci_step (factors re-used inside a block, as bench.py times it). OCI: the
# dense path (the headline) and the structured cell solve walk the full 50 steps beside one oracle (half a minute of
# host time); the SI comparator walks the same 50 steps (100-350 sweeps per step at dt = 1 and 0.1).
# ---------------------------------------------------------------------------------------------------------------
def test_config5_oci_dt_sweep_as_configured_dense_and_structured():
    p = W.config5()
    counts = _run_sequence(p, [(dt, p.n_steps) for dt in p.meta["dt_sweep"]], "oci", solver_options=BOTH_PATHS)
    assert len(counts) == 50


def test_config5_si_dt_sweep_as_configured():
    p = W.config5()
    counts = _run_sequence(p, [(dt, p.n_steps) for dt in p.meta["dt_sweep"]], "si")
    assert len(counts) == 50


def test_config5_per_cell_scaled_error_of_an_iterate():
    """sigma_t spans four decades: compare iterates cell by cell, each cell on its own scale."""
    p = W.config5(dt=1e-2)
    s, o = _solver(p), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    o.const_rhs()
    for l in range(3):
        s.iterate(1)
        o.oci_iterate(1)
        psi = s.angular_flux().cpu().numpy()
        assert rel(psi, o.psi) < TOL_ITER
        assert rel_cell(psi, o.psi) < CELL_TOL_ITER, f"iteration {l + 1}"
        assert rel_cell(s.scalar_flux().cpu().numpy(), o.phi) < CELL_TOL_ITER


# ---------------------------------------------------------------------------------------------------------------
# oci_step_host: the call bench.py's e2e leg is timed through (H2D of q from pinned memory, the step, D2H of phi)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", [0, 1])
def test_step_host_matches_the_oracle_and_the_device_getters(scheme):
    import torch
    p = W.random_problem(61, 211, 8, 2, bc_left=W.BC_PRESCRIBED, bc_right=W.BC_REFLECTIVE, dt=0.03)
    s, o = _solver(p), _oracle(p)
    q_host = torch.empty((p.J, p.G, 4), dtype=torch.float64).pin_memory()
    phi_host = torch.full((p.J, p.G, 4), float("nan"), dtype=torch.float64).pin_memory()
    rng = np.random.default_rng(7)
    for step in range(3):  # a new source every step: the H2D copy must be the one the step uses
        q = rng.uniform(0.0, 2.0, size=(p.J, p.G, 4))
        q_host.copy_(torch.from_numpy(q))
        it_g, conv_g, _ = s.step_host(scheme, q_host, phi_host, tol=1e-9, max_iters=4000, check_every=8)
        o.set_source(q)
        it_o, _ = (o.oci_step if scheme == 0 else o.si_step)(tol=1e-9, max_iters=4000)
        assert it_g == conv_g == it_o, (step, it_g, conv_g, it_o)
        assert rel(phi_host.numpy(), o.phi) < TOL_PHI
        assert np.array_equal(phi_host.numpy(), s.scalar_flux().cpu().numpy())  # the same array, copied out
        assert rel(s.get_state().cpu().numpy(), o.psi_prev) < TOL_PHI
    # q_host = NULL keeps the source of the last call; phi_host = NULL skips the read-back
    it_g, _, _ = s.step_host(scheme, None, None, tol=1e-9, max_iters=4000, check_every=8)
    it_o, _ = (o.oci_step if scheme == 0 else o.si_step)(tol=1e-9, max_iters=4000)
    assert it_g == it_o
    assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI


# ---------------------------------------------------------------------------------------------------------------
# refactor_every_step = 1 (Alg. 2 as printed: `_gesv` at the start of every step) runs to the same answers
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_refactor_every_step(scheme):
    p = W.random_problem(51, 83, 8, 2, bc_left=1, bc_right=2, dt=0.02)
    counts = _run_sequence(p, [(0.02, 3), (0.2, 2)], scheme, solver_options={"refactor_every_step": 1})
    assert len(counts) == 5


# ---------------------------------------------------------------------------------------------------------------
# the paper's Table-2 two-group problem, the shapes bench.py --table2 times:
# S16 (n = 128) and S32 (n = 256), small J and J ~ 455 (delta = 0.1). Dense, structured and SI, per iteration.
# ---------------------------------------------------------------------------------------------------------------
TABLE2_CASES = [(16, 7, 10.0), (16, 455, 0.1), (32, 5, 0.1), (32, 455, 10.0)]


@pytest.mark.parametrize("N,J,dt", TABLE2_CASES)
@pytest.mark.parametrize("path", ["dense", "structured", "si"])
def test_table2_per_iteration_parity(N, J, dt, path):
    p = W.table2(J, N, dt)
    opts = {"solve_mode": 1} if path == "structured" else {}
    s, o = _solver(p, options=opts), _oracle(p)
    if path != "si":
        assert s.factor() == 0 and o.factor() == 0
        o.const_rhs()
    for l in range(5):
        if path == "si":
            s.si_iterate(1)
            o.si_iterate(1)
        else:
            s.iterate(1)
            o.oci_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"iteration {l + 1}"
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_ITER
    if path == "dense":
        for j in sorted({0, J // 2, J - 1}):
            A = o.assemble_cell(j)
            assert np.array_equal(s.debug_matrix(j), A)
            assert np.max(np.abs(A @ s.debug_inverse(j) - np.eye(p.n))) < 1e-12 * np.linalg.cond(A)


@pytest.mark.parametrize("N", [16, 32])
def test_table2_converged_step_paper_stop_rule(N):
    """One time step as bench.py --table2 runs it: Eq. 12-13 stop rule, eps = 1e-8, OCI dense + structured and SI."""
    p = W.table2(455, N, 0.1)
    for opts, scheme in (({}, "oci"), ({"solve_mode": 1}, "oci"), ({}, "si")):
        s, o = _solver(p, options=opts), _oracle(p)
        if scheme == "oci":
            it_g, conv_g, _ = s.step(tol=1e-8, max_iters=60000, check_every=16, stop_rule=1, advance=False)
            it_o, _ = o.oci_step(tol=1e-8, max_iters=60000, rule=1, advance=False)
        else:
            it_g, conv_g, _ = s.si_step(tol=1e-8, max_iters=60000, check_every=16, stop_rule=1, advance=False)
            it_o, _ = o.si_step(tol=1e-8, max_iters=60000, rule=1, advance=False)
        assert it_g == conv_g == it_o, (opts, scheme)
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI


# ---------------------------------------------------------------------------------------------------------------
# The assembly the PRODUCTION factor kernels do on chip (their own inline a1), dumped before the elimination
# ---------------------------------------------------------------------------------------------------------------
PRODUCTION_ASSEMBLY_CASES = [
    ("cfg5", lambda: W.config5(J=4096, dt=1e-3)),
    ("cfg5@dt=1", lambda: W.config5(J=512, dt=1.0)),
    ("n64 N8 G2", lambda: W.random_problem(61, 33, 8, 2, bc_left=1)),
    ("n64 N4 G4", lambda: W.random_problem(62, 17, 4, 4)),
    ("n64 N2 G8", lambda: W.random_problem(63, 9, 2, 8)),
    ("cfg3", lambda: W.config3(J=512)),
    ("cfg4", lambda: W.config4(J=64)),
    ("n192 N6 G8", lambda: W.random_problem(64, 5, 6, 8)),
    ("table2 S32", lambda: W.table2(9, 32, 0.1)),
]


@pytest.mark.parametrize("name,make", PRODUCTION_ASSEMBLY_CASES, ids=[c[0] for c in PRODUCTION_ASSEMBLY_CASES])
def test_production_assembly_bit_exact(name, make):
    p = make()
    s, o = _solver(p), _oracle(p)
    rng = np.random.default_rng(3)
    for j in sorted({0, 1, p.J // 2, p.J - 1, *rng.integers(0, p.J, 3).tolist()}):
        A_gpu = s.debug_factor_input(j)
        A_orc = o.assemble_cell(j)
        assert np.array_equal(A_gpu, A_orc), f"{name} cell {j}: max diff {np.max(np.abs(A_gpu - A_orc))}"


# ---------------------------------------------------------------------------------------------------------------
# Factor paths the default options do not take
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,G,opts", [
    (6, 8, {"factor_kernel": 0}),      # n = 192, generic kernel with its working array in global scratch
    (8, 8, {"factor_kernel": 0}),      # n = 256, same
    (10, 5, {}),                       # n = 200: not a multiple of 64 -> the generic kernel by default, global scratch
    (16, 1, {"factor_kernel": 0}),     # n = 64, generic kernel, working array in shared memory
    (16, 1, {"factor_update": 1}),     # n = 64, production kernel with one rank-8 pass per panel (default: panels paired)
    (16, 1, {"factor_kernel": 4}),     # n = 64, one warp per cell (DMMA update)
    (16, 1, {"factor_kernel": 4, "factor_update": 0}),   # n = 64, one warp per cell (DFMA update)
    (8, 4, {"factor_kernel": 0}),      # n = 128, generic kernel
    (6, 8, {"factor_cluster": 1}),     # n = 192, clusters of three CTAs with eight column blocks each (default: two x 12)
    (8, 8, {"factor_cluster": 1}),     # n = 256, clusters of four CTAs (default: three, 10 + 11 + 11 blocks)
])
def test_alternative_factor_paths(N, G, opts):
    p = W.random_problem(70 + N + G, 21, N, G, bc_left=2, bc_right=1, dt=0.03)
    s, o = _solver(p, options=opts), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    for j in (0, 10, 20):
        A = o.assemble_cell(j)
        assert np.max(np.abs(A @ s.debug_inverse(j) - np.eye(p.n))) < 1e-12 * np.linalg.cond(A)
    o.const_rhs()
    for l in range(3):
        s.iterate(1)
        o.oci_iterate(1)
        assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER, f"iteration {l + 1}"


def test_pivot_ties_take_the_first_maximal_row():
    """Scattering-dominated cells (c >> 1, unphysical but a legitimate matrix): the entries -dx K w_m'/4 of a column are
    IDENTICAL in every row of the same p (Eq. 10) and exceed the diagonal, so the pivot search meets exact ties in
    both key words; LAPACK's and the oracle's choice is the first maximal row. The production kernel records the tie
    in its optimistic pass and repeats the panel with exact tie resolution."""
    p = W.config5(J=200, dt=1.0)
    p.sigma_t = np.full_like(p.sigma_t, 50.0)
    p.transfer = np.full_like(p.transfer, 3000.0)
    p.transfer[::2] *= 1.5                            # two kinds of cells
    s, o = _solver(p), _oracle(p)
    assert s.factor() == 0 and o.factor() == 0
    for j in (0, 57, 199):
        A = o.assemble_cell(j)
        col = np.abs(A[:, 0])
        assert (col == col.max()).sum() >= 2 and col[0] < col.max()   # the first pivot search already meets an exact tie
        assert np.array_equal(s.debug_factor_input(j), A)
        Ainv = s.debug_inverse(j)
        assert np.max(np.abs(A @ Ainv - np.eye(p.n))) < 1e-12 * np.linalg.cond(A)
    o.const_rhs()
    s.iterate(1)
    o.oci_iterate(1)
    assert rel(s.angular_flux().cpu().numpy(), o.psi) < TOL_ITER


# ---------------------------------------------------------------------------------------------------------------
# Library robustness
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,G", [(16, 1), (8, 4), (6, 8), (8, 8)])   # n = 64, 128, 192, 256: the production factor kernels
def test_production_kernels_flag_singular_cells_and_go_on(N, G):
    """A singular cell in the middle of the batch: oci_factor returns the 1-based index of the FIRST bad cell, and the
    CTA / cluster that met it carries on with its next cells (in the cluster kernel the panel buffers and their
    mbarrier parities must survive a cell that stops at an arbitrary panel). G = 1: sigma_t is NaN, caught in the first
    panel; G > 1: one column group of the transfer matrix is NaN, which the pivot search only meets when it reaches
    that group's columns -- panel 20 of 32 at n = 256, in the third CTA of the cluster."""
    J, bad = 161, (7, 55, 140)
    p = W.random_problem(300 + N + G, J, N, G, dt=0.02)
    p.sigma_t = p.sigma_t.copy()
    p.transfer = p.transfer.copy()
    for j in bad:
        if G == 1:
            p.sigma_t[j] = np.nan
        else:
            p.transfer[j, :, (5 * G) // 8] = np.nan
    s = _solver(p)
    assert s.factor() == bad[0] + 1
    o = _oracle(p)
    good = [j for j in (0, 6, 8, 40, 54, 56, 73, 106, 139, 141, 160)]
    for j in good:
        A = o.assemble_cell(j)
        assert np.max(np.abs(A @ s.debug_inverse(j) - np.eye(p.n))) < 1e-12 * np.linalg.cond(A), f"cell {j}"
    for j in bad:
        assert np.all(s.debug_inverse(j) == 0.0)
    s.set_dt(0.03)                       # and the next elimination on the same context is sound
    assert s.factor() == bad[0] + 1
    A = _oracle(p.with_dt(0.03)).assemble_cell(73)
    assert np.max(np.abs(A @ s.debug_inverse(73) - np.eye(p.n))) < 1e-12 * np.linalg.cond(A)


def test_two_contexts_with_different_shapes_in_one_process():
    import torch
    pa, pb = W.config5(J=600, dt=1e-2), W.config3(J=300)
    a, b = _solver(pa), _solver(pb)                  # n = 64 and n = 128: different kernel instantiations / smem sizes
    oa, ob = _oracle(pa), _oracle(pb)
    for s, o in ((a, oa), (b, ob), (a, oa)):
        it_g, _, _ = s.step(tol=1e-9, max_iters=2000, check_every=4)
        it_o, _ = o.oci_step(tol=1e-9, max_iters=2000)
        assert it_g == it_o
        assert rel(s.scalar_flux().cpu().numpy(), o.phi) < TOL_PHI
    if torch.cuda.device_count() > 1:
        c = _solver(pa, device="cuda:1")
        oc = _oracle(pa)
        it_g, _, _ = c.step(tol=1e-9, max_iters=2000, check_every=4)
        it_o, _ = oc.oci_step(tol=1e-9, max_iters=2000)
        assert it_g == it_o
        assert rel(c.scalar_flux().cpu().numpy(), oc.phi) < TOL_PHI
        # a call on the first context while another device is current
        torch.cuda.set_device(1)
        a.iterate(1)
        torch.cuda.set_device(0)


def test_failed_create_reports_its_reason():
    from paper_2503_00264_b200 import OCIError, create_error
    p = W.random_problem(5, 4, 4, 1)
    p.mu = p.mu.copy()
    p.mu[1] = 0.0
    with pytest.raises(OCIError):
        _solver(p)
    assert isinstance(create_error(), int)
