"""Pins (e), (e'), (e'') of SURVEY.md section 8(c): convergence rates of the oracle's OCI and SI iterations against
the Fourier analysis of PAPER.md Section 2.3 (Eq. 27-38), and the trends the paper states.

The Fourier matrices are built in tests/pins.py from the cell matrix the ORACLE assembles (L_c - S) and from the
boundary operators of Eq. 36-37; the measured rate comes from running the oracle's iteration on a long homogeneous
slab with zero source and a random initial iterate (the error is then the iterate itself).
"""
from pathlib import Path

import numpy as np
import pytest

import oracle
import workloads as W
from pins import spectral_radius

GOLDEN = Path(__file__).parent / "golden"


def _rho(delta, tau, c, N=8, scheme="oci", return_eig=False, sig=1.0, v=1.0):
    dx = delta / sig
    dt = tau / (sig * v) if np.isfinite(tau) else 1e30
    p = W.homogeneous(1, N, sig, c, dx, v, dt)
    A = oracle.Oracle(p).assemble_cell(0)
    Lc = oracle.Oracle(W.homogeneous(1, N, sig, 0.0, dx, v, dt)).assemble_cell(0)
    return spectral_radius(A, Lc, p.mu, scheme, return_eig=return_eig)


def _measured_rate(p, solver, psi_guess, lo, hi):
    o = oracle.Oracle(p)
    o.set_iterate(psi_guess)
    if solver == "oci":
        o.factor()
        o.const_rhs()
    norms = []
    for _ in range(hi + 1):
        getattr(o, solver + "_iterate")(1)
        norms.append(np.linalg.norm(o.phi if solver == "si" else o.psi))
    return (norms[hi] / norms[lo]) ** (1.0 / (hi - lo))


def test_worked_example_rate_matches_fourier():
    """PAPER.md:479 inputs as stated: Fourier rho (own script) vs geometric-mean measured rate, within 5 %."""
    p = W.worked_example(J=400)
    pred = _rho(0.25, 1.0, 0.9)
    rate = _measured_rate(p, "oci", p.meta["psi_guess"], lo=20, hi=60)
    assert pred == pytest.approx(0.6403, abs=5e-4)            # 0.6403, not the printed 0.4831
    assert rate == pytest.approx(pred, rel=0.05)


def test_worked_example_printed_eigenvalue_at_half_dt():
    """The printed lambda_max = 0.429 + 0.216i (tests/golden/paper_worked_example.txt) is what Eq. 32 gives at
    dt = 0.05; the oracle's measured rate at that dt oscillates about |lambda|."""
    g = dict(l.split() for l in (GOLDEN / "paper_worked_example.txt").read_text().splitlines()
             if l and not l.startswith("#"))
    sig, dx, c, v = float(g["sigma_t"]), float(g["dx"]), float(g["c"]), float(g["v"])
    dt = float(g["dt_reproducing"])
    rho, lam = _rho(sig * dx, sig * v * dt, c, return_eig=True, sig=sig, v=v)
    assert lam.real == pytest.approx(float(g["lambda_re"]), abs=1e-3)
    assert abs(lam.imag) == pytest.approx(float(g["lambda_im"]), abs=1e-3)
    assert rho == pytest.approx(float(g["rho"]), abs=5e-3)
    p = W.worked_example(J=400, dt=dt)
    rate = _measured_rate(p, "oci", p.meta["psi_guess"], lo=15, hi=45)
    assert rate == pytest.approx(rho, rel=0.05)


@pytest.mark.parametrize("tau", [1.0, 0.1, 0.01])
def test_si_rate_closed_form(tau):
    """(e') rho_SI = c / sqrt(1 + 2/tau + 2/tau^2), independent of delta (flat mode of Eq. 2a-b + Eq. 38);
    PAPER.md:39: 'independent of delta for the homogeneous infinite-medium problem'."""
    c = 0.9
    want = c / np.sqrt(1 + 2 / tau + 2 / tau ** 2)
    for delta in (10.0, 1.0, 0.1):
        assert _rho(delta, tau, c, scheme="si") == pytest.approx(want, rel=1e-9)
    # measured on the oracle's SI at the centre of a 150-mean-free-path slab (boundary layers never reach it)
    p = W.homogeneous(J=300, N=8, sigma_t=1.0, c=c, dx=0.5, v=1.0, dt=tau)
    guess = np.ones((p.J, 1, p.N, 4))
    guess[..., 2:4] = 0.3                      # flat in space and angle, the two time levels differ
    o = oracle.Oracle(p)
    o.set_iterate(guess)
    x = [o.phi[150, 0, [0, 2]].copy()]
    for _ in range(2):
        o.si_iterate(1)
        x.append(o.phi[150, 0, [0, 2]].copy())
        assert np.ptp(o.phi[140:160, 0, 0]) < 1e-12 * abs(x[-1][0])  # the mode stays flat there
    # the flat mode evolves by a 2x2 matrix T: T [x0 x1] = [x1 x2]  ->  |eig T| is the rate (complex pair)
    T = np.column_stack([x[1], x[2]]) @ np.linalg.inv(np.column_stack([x[0], x[1]]))
    assert np.abs(np.linalg.eigvals(T)).max() == pytest.approx(want, rel=1e-8)


def test_si_steady_state_rate_is_c():
    assert _rho(1.0, np.inf, 0.7, scheme="si") == pytest.approx(0.7, rel=1e-6)


def test_oci_trends_of_the_paper():
    """rho_OCI -> 0 as tau -> 0; -> 1 as delta -> 0 at steady state whatever c;
    = 1 at steady state for c = 1 (Table 1 row SS); < 1 when time-dependent."""
    taus = [10, 1, 0.1, 0.01, 0.001]
    r = [_rho(0.1, t, 0.9) for t in taus]
    assert all(a > b for a, b in zip(r, r[1:])) and r[-1] < 1e-3
    ss = [_rho(d, np.inf, 0.9) for d in (10, 1, 0.1, 0.01)]
    assert all(a < b for a, b in zip(ss, ss[1:])) and ss[-1] > 0.995
    for c in (0.1, 0.5):
        assert _rho(0.001, np.inf, c) > 0.99
    for d in (10, 1.0, 0.1):
        assert _rho(d, np.inf, 1.0) == pytest.approx(1.0, abs=1e-6)
        assert _rho(d, 10.0, 1.0) < 1.0


def test_table1_trends():
    """Orderings of the paper's Table 1 (golden fixture) hold for the spectral radii of the oracle's matrices."""
    rows = [l.split() for l in (GOLDEN / "paper_table1_rho_oci.txt").read_text().splitlines()
            if l and not l.startswith("#")]
    deltas = [10.0, 1.0, 0.1]
    paper = {r[0]: [float(x) for x in r[1:]] for r in rows}
    ours = {k: [_rho(d, np.inf if k == "SS" else float(k), 1.0) for d in deltas] for k in paper}
    order = ["SS", "10", "1", "0.1", "0.01"]
    for tab in (paper, ours):
        for a, b in zip(order, order[1:]):                 # smaller tau -> smaller rho, for every delta
            assert all(x >= y for x, y in zip(tab[a], tab[b]))
        for k in order[1:]:                                # thinner cells -> larger rho
            assert tab[k][0] < tab[k][1] < tab[k][2]
    assert ours["SS"] == pytest.approx([1.0, 1.0, 1.0], abs=1e-6)


def test_config_predictions_and_iteration_counts():
    """(e'') cfg 1: Fourier rho_OCI ~ 0.446 > rho_SI ~ 0.034, so OCI needs more iterations than SI (17 vs 6)."""
    assert _rho(1 / 16, 0.1, 0.5, N=4) == pytest.approx(0.446, abs=2e-3)
    assert _rho(1 / 16, 0.1, 0.5, N=4, scheme="si") == pytest.approx(0.5 / np.sqrt(1 + 20 + 200), rel=1e-6)
    p = W.config1()
    o, s = oracle.Oracle(p), oracle.Oracle(p)
    its_o = [o.oci_step(1e-8)[0] for _ in range(p.n_steps)]
    its_s = [s.si_step(1e-8)[0] for _ in range(p.n_steps)]
    assert its_o == [17, 17, 16, 16, 16] and its_s == [6] * 5
    np.testing.assert_allclose(o.phi, s.phi, atol=2e-8)
    # smaller time step -> fewer OCI iterations, and the gap to SI closes
    p2 = W.config2(J=128)
    its = {}
    for dt in (1.0, 0.1, 0.01):
        a, b = oracle.Oracle(p2, dt=dt), oracle.Oracle(p2, dt=dt)
        its[dt] = (a.oci_step(1e-8)[0], b.si_step(1e-8)[0])
    assert its[1.0][0] > its[0.1][0] > its[0.01][0]
    assert its[1.0][0] / its[1.0][1] > its[0.01][0] / its[0.01][1]
