"""Pins (c), (c') and (d) of SURVEY.md section 8(c).

(c)  one group, homogeneous, reflective both ends, isotropic flat initial flux: every psi = phi/2 and phi follows
     the two-level recursion obtained from Eq. 2a-b with all spatial terms gone:
        tau_a = Sigma (1-c) v dt
        phi_{k+1/2} = [phi_{k-1/2} + v dt Q (1 + tau_a/2)] / (1 + tau_a + tau_a^2/2)
        phi_k       = phi_{k+1/2} (1 + tau_a/2) - v dt Q / 2
     and tends to the infinite-medium steady state Q / Sigma_a.
(c') G groups: [[R, D], [-2D, 2D + R]] [phi_k; phi_{k+1/2}] = [Q + D phi_{k-1/2}; Q], R = diag(Sigma_t) - K,
     D = diag(1/(v_g dt)).
(d)  per-group particle balance of the converged step: sum over cells and ordinates of Eq. 3a + 3b (and of
     Eq. 3c + 3d) weighted by w_m -- rate of change + net leakage + removal = in-scatter + source.
"""
import numpy as np
import pytest

import oracle
import workloads as W


@pytest.mark.parametrize("dt,c", [(0.1, 0.5), (2.0, 0.9), (0.01, 0.0)])
def test_infinite_medium_one_group(dt, c):
    sig, v, Q, phi0 = 1.3, 2.0, 0.7, 0.4
    J, N = 6, 4
    rng = np.random.default_rng(1)
    p = W.homogeneous(J=J, N=N, sigma_t=sig, c=c, dx=1.0, v=v, dt=dt, q=Q, bc=W.BC_REFLECTIVE, psi0=phi0 / 2)
    p.dx[:] = rng.uniform(0.05, 1.5, size=J)             # unequal cells: the closed form does not care
    tau_a = sig * (1 - c) * v * dt
    for solver in ("oci", "si"):
        o = oracle.Oracle(p)
        phi_edge = phi0
        for _ in range(4):
            getattr(o, solver + "_step")(tol=1e-14, max_iters=100000)
            phi_edge = (phi_edge + v * dt * Q * (1 + tau_a / 2)) / (1 + tau_a + tau_a ** 2 / 2)
            phi_avg = phi_edge * (1 + tau_a / 2) - v * dt * Q / 2
            np.testing.assert_allclose(o.phi[..., 2:4], phi_edge, rtol=1e-11)
            np.testing.assert_allclose(o.phi[..., 0:2], phi_avg, rtol=1e-11)
            np.testing.assert_allclose(o.psi[..., 2:4], phi_edge / 2, rtol=1e-11)   # isotropic: psi = phi / 2
    # steady limit Q / Sigma_a
    o = oracle.Oracle(p)
    o.set_dt(1e6)
    o.oci_step(tol=1e-14, max_iters=100000)
    np.testing.assert_allclose(o.phi, Q / (sig * (1 - c)), rtol=1e-5)


def test_infinite_medium_multigroup_table2():
    p = W.table2(J=4, N=4, dt=0.3, L=2.0)
    p.bc_left = p.bc_right = W.BC_REFLECTIVE
    G = p.G
    phi_prev = np.array([0.3, 1.1])
    p.psi0[:] = (phi_prev / 2)[None, :, None, None]
    R = np.diag(p.sigma_t[0]) - p.transfer[0]
    D = np.diag(1.0 / (p.v * p.dt))
    Qv = p.q[0, :, 0]
    M = np.block([[R, D], [-2 * D, 2 * D + R]])
    for solver in ("oci", "si"):
        o = oracle.Oracle(p)
        prev = phi_prev.copy()
        for _ in range(3):
            getattr(o, solver + "_step")(tol=1e-14, max_iters=200000)
            sol = np.linalg.solve(M, np.concatenate([Qv + D @ prev, Qv]))
            phi_k, phi_e = sol[:G], sol[G:]
            for g in range(G):
                np.testing.assert_allclose(o.phi[:, g, 0:2], phi_k[g], rtol=1e-10)
                np.testing.assert_allclose(o.phi[:, g, 2:4], phi_e[g], rtol=1e-10)
            prev = phi_e


def _edge_currents(p, psi, lev):
    """Net current sum_m w_m mu_m psi_edge at x = 0 and x = X for every group, upstream closure Eq. 5."""
    JL = np.zeros(p.G)
    JR = np.zeros(p.G)
    for g in range(p.G):
        for m in range(p.N):
            mu, w = p.mu[m], p.w[m]
            if mu > 0:
                right = psi[p.J - 1, g, m, 2 * lev + 1]
                left = (psi[0, g, p.N - 1 - m, 2 * lev] if p.bc_left == W.BC_REFLECTIVE
                        else p.inc_left[g, m, lev] if p.bc_left == W.BC_PRESCRIBED else 0.0)
            else:
                left = psi[0, g, m, 2 * lev]
                right = (psi[p.J - 1, g, p.N - 1 - m, 2 * lev + 1] if p.bc_right == W.BC_REFLECTIVE
                         else p.inc_right[g, m, lev] if p.bc_right == W.BC_PRESCRIBED else 0.0)
            JL[g] += w * mu * left
            JR[g] += w * mu * right
    return JL, JR


@pytest.mark.parametrize("bcl,bcr", [(0, 0), (1, 0), (2, 2), (0, 1)])
@pytest.mark.parametrize("solver", ["oci", "si"])
def test_particle_balance(bcl, bcr, solver):
    p = W.random_problem(31 + bcl + 3 * bcr, J=8, N=4, G=2, bc_left=bcl, bc_right=bcr)
    o = oracle.Oracle(p)
    phi_prev = np.einsum("m,jgme->jge", p.w, p.psi0)           # phi_{k-1/2} at (L,R)
    getattr(o, solver + "_step")(tol=1e-14, max_iters=100000, advance=False)
    phi, psi = o.phi, o.psi
    dx = p.dx[:, None]
    Kphi = np.einsum("jab,jbp->jap", p.transfer, phi)
    inv_vdt = 1.0 / (p.v * p.dt)
    # Eq. 3a + 3b
    JL, JR = _edge_currents(p, psi, 0)
    rate = (dx / 2 * ((phi[..., 2] - phi_prev[..., 0]) + (phi[..., 3] - phi_prev[..., 1]))).sum(0) * inv_vdt
    removal = (dx / 2 * (p.sigma_t * (phi[..., 0] + phi[..., 1]) - Kphi[..., 0] - Kphi[..., 1])).sum(0)
    source = (dx / 2 * (p.q[..., 0] + p.q[..., 1])).sum(0)
    np.testing.assert_allclose(rate + removal + JR - JL, source, rtol=0, atol=1e-12 * max(1.0, np.abs(source).max()))
    # Eq. 3c + 3d
    JL, JR = _edge_currents(p, psi, 1)
    rate = (dx / 2 * ((phi[..., 2] - phi[..., 0]) + (phi[..., 3] - phi[..., 1]))).sum(0) * 2 * inv_vdt
    removal = (dx / 2 * (p.sigma_t * (phi[..., 2] + phi[..., 3]) - Kphi[..., 2] - Kphi[..., 3])).sum(0)
    source = (dx / 2 * (p.q[..., 2] + p.q[..., 3])).sum(0)
    np.testing.assert_allclose(rate + removal + JR - JL, source, rtol=0, atol=1e-12 * max(1.0, np.abs(source).max()))
