"""Test-side reference constructions that are INDEPENDENT of the oracle's own formulas.

Nothing here is imported by oracle/ or by the product. Each function restates a passage of PAPER.md in the
most direct way (one equation -> one block of code), so that the oracle's condensed matrices (Eq. 8b, 10, 40b)
are checked against the un-condensed balance equations (Eq. 3a-d with closures 4-5) they were derived from.
"""
from __future__ import annotations

import numpy as np

BC_VACUUM, BC_REFLECTIVE, BC_PRESCRIBED = 0, 1, 2


def idx(p, j, g, m, pos):
    return ((j * p.G + g) * p.N + m) * 4 + pos


def global_system(p, q, psi_prev, dt=None):
    """Dense matrix and RHS of ONE time step over all unknowns psi[j][g][m][pos], from Eq. 3a-d PAPER.md:85-93.

    Every term of Eq. 3 is added where it stands: time difference, mu * [midpoint average (Eq. 4) - upstream
    edge (Eq. 5)], removal, scattering (+ source) on the right-hand side, moved to the left. Boundary edges use
    PAPER.md:67-71 (prescribed / vacuum) or the mirror ordinate (reflective).
    """
    dt = p.dt if dt is None else dt
    J, G, N = p.J, p.G, p.N
    n_tot = J * G * N * 4
    M = np.zeros((n_tot, n_tot))
    rhs = np.zeros(n_tot)

    def edge(row, coef, j_edge_left_of, g, m, lev):
        """Add coef * psi_{m,lev,(j-1/2)} where the edge is the LEFT edge of cell j_edge_left_of (0..J)."""
        je = j_edge_left_of
        pos_L, pos_R = 2 * lev + 0, 2 * lev + 1
        if p.mu[m] > 0:                        # upstream = cell to the left, its R value (Eq. 5)
            if je > 0:
                M[row, idx(p, je - 1, g, m, pos_R)] += coef
            elif p.bc_left == BC_REFLECTIVE:
                M[row, idx(p, 0, g, N - 1 - m, pos_L)] += coef
            elif p.bc_left == BC_PRESCRIBED:
                rhs[row] -= coef * p.inc_left[g, m, lev]
        else:                                  # upstream = cell to the right, its L value
            if je < J:
                M[row, idx(p, je, g, m, pos_L)] += coef
            elif p.bc_right == BC_REFLECTIVE:
                M[row, idx(p, J - 1, g, N - 1 - m, pos_R)] += coef
            elif p.bc_right == BC_PRESCRIBED:
                rhs[row] -= coef * p.inc_right[g, m, lev]

    for j in range(J):
        dx = p.dx[j]
        for g in range(G):
            sig, v = p.sigma_t[j, g], p.v[g]
            for m in range(N):
                mu = p.mu[m]
                for lev in (0, 1):                       # lev 0: Eq. 3a/3b (time average k); 1: Eq. 3c/3d (k+1/2)
                    L, R = idx(p, j, g, m, 2 * lev), idx(p, j, g, m, 2 * lev + 1)
                    for half, row in (("L", L), ("R", R)):
                        me = L if half == "L" else R
                        # --- time term
                        if lev == 0:   # (dx/2)(1/v)(psi_{k+1/2} - psi_{k-1/2})/dt
                            M[row, idx(p, j, g, m, 2 + (0 if half == "L" else 1))] += dx / 2 / v / dt
                            rhs[row] += dx / 2 / v / dt * psi_prev[j, g, m, 0 if half == "L" else 1]
                        else:          # (dx/2)(1/v)(psi_{k+1/2} - psi_k)/(dt/2)
                            M[row, me] += dx / 2 / v / (dt / 2)
                            M[row, idx(p, j, g, m, 0 if half == "L" else 1)] -= dx / 2 / v / (dt / 2)
                        # --- streaming term
                        if half == "L":   # mu [ (psi_L + psi_R)/2 - psi_{j-1/2} ]
                            M[row, L] += mu / 2
                            M[row, R] += mu / 2
                            edge(row, -mu, j, g, m, lev)
                        else:             # mu [ psi_{j+1/2} - (psi_L + psi_R)/2 ]
                            edge(row, +mu, j + 1, g, m, lev)
                            M[row, L] -= mu / 2
                            M[row, R] -= mu / 2
                        # --- removal
                        M[row, me] += dx / 2 * sig
                        # --- scattering (+fission) and source: (dx/2)(1/2)(sum_g' K[g][g'] sum_n w_n psi_n + Q)
                        pos = 2 * lev + (0 if half == "L" else 1)
                        for gp in range(G):
                            for mp in range(N):
                                M[row, idx(p, j, gp, mp, pos)] -= dx / 4 * p.transfer[j, g, gp] * p.w[mp]
                        rhs[row] += dx / 4 * q[j, g, pos]
    return M, rhs


def global_solve(p, q, psi_prev, dt=None):
    M, rhs = global_system(p, q, psi_prev, dt)
    return np.linalg.solve(M, rhs).reshape(p.J, p.G, p.N, 4)


# ---------------------------------------------------------------------------------------------------------------
# Fourier analysis of one iteration, Section 2.3 (Eq. 27-38)
# ---------------------------------------------------------------------------------------------------------------

def fourier_matrices(A_cell, Lc_cell, mu):
    """Returns (A, S, Bfun): A = L_c - S and S = L_c - A as assembled by the code under test for one homogeneous
    cell; Bfun(theta) = -diag(L_b^-, L_b^+) of Eq. 36-37 in the unknown order of Eq. 11b."""
    n = A_cell.shape[0]
    S = Lc_cell - A_cell

    def B(theta):
        Bm = np.zeros((n, n), dtype=complex)
        for m, mu_m in enumerate(mu):
            r = 4 * m
            if mu_m > 0:      # rows (k,L), (k+1/2,L) receive mu * psi_{j-1,R}: phase exp(-i theta)
                Bm[r + 0, r + 1] = mu_m * np.exp(-1j * theta)
                Bm[r + 2, r + 3] = mu_m * np.exp(-1j * theta)
            else:             # rows (k,R), (k+1/2,R) receive |mu| * psi_{j+1,L}: phase exp(+i theta)
                Bm[r + 1, r + 0] = -mu_m * np.exp(1j * theta)
                Bm[r + 3, r + 2] = -mu_m * np.exp(1j * theta)
        return Bm

    return A_cell, S, B


def spectral_radius(A_cell, Lc_cell, mu, scheme="oci", n_theta=250, return_eig=False):
    """rho = sup_theta max |eig T(theta)| with T_OCI = (L_c - S)^-1 B (Eq. 32), T_SI = (L_c - B)^-1 S (Eq. 38)."""
    A, S, B = fourier_matrices(A_cell, Lc_cell, mu)
    best, best_eig = 0.0, 0j
    for theta in np.linspace(0.0, 2 * np.pi, n_theta):
        Bm = B(theta)
        T = np.linalg.solve(A, Bm) if scheme == "oci" else np.linalg.solve(Lc_cell - Bm, S.astype(complex))
        ev = np.linalg.eigvals(T)
        k = int(np.argmax(np.abs(ev)))
        if abs(ev[k]) > best:
            best, best_eig = abs(ev[k]), ev[k]
    return (best, best_eig) if return_eig else best
