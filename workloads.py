"""Seeded synthetic input generators shared by the oracle tests, the GPU tests and bench.py.

This module holds NO arithmetic of the method (no matrix assembly, no solves, no sweeps):
it only draws cross-sections, meshes, quadrature sets, sources and initial conditions.
Both `oracle/` and `paper_2503_00264_b200/` are driven with the arrays produced here;
neither of them imports this module.

Recipes follow SURVEY.md section 8(d) (BASELINE.json `configs` with the fill-ins listed
there) and PAPER.md: Table 2 and the verification run of Section 3.1
(PAPER.md:479). Everything is fp64 and C-contiguous.

Array conventions (Eq. 11, 40d):
  dx        [J]          cell widths, cm
  sigma_t   [J][G]       total cross-section per cell and group, 1/cm
  transfer  [J][G][G]    transfer[j][g_to][g_from] = Sigma_s(g_from -> g_to) (+ chi_g nuSigma_f,g_from)
  v         [G]          speeds, cm/s
  mu, w     [N]          Gauss-Legendre nodes (ascending, negatives first) and weights, sum(w) = 2
  q         [J][G][4]    isotropic source at (k,L) (k,R) (k+1/2,L) (k+1/2,R)
  psi0      [J][G][N][2] initial time-edge angular flux psi_{-1/2} at (L, R)
  inc_left  [G][N][2]    prescribed incident flux at x=0 for mu_m>0, (k, k+1/2) levels (bc == 2 only)
  inc_right [G][N][2]    same at x=X for mu_m<0
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Callable, Optional

import numpy as np

BC_VACUUM = 0
BC_REFLECTIVE = 1
BC_PRESCRIBED = 2


def gauss_legendre(N: int):
    """Gauss-Legendre set on [-1, 1] (PAPER.md:49 footnote), ascending mu, sum(w) = 2."""
    if N < 2 or N % 2:
        raise ValueError("N must be even and >= 2")
    mu, w = np.polynomial.legendre.leggauss(N)
    return np.ascontiguousarray(mu, dtype=np.float64), np.ascontiguousarray(w, dtype=np.float64)


@dataclass
class Problem:
    name: str
    J: int
    N: int
    G: int
    dx: np.ndarray
    sigma_t: np.ndarray
    transfer: np.ndarray
    v: np.ndarray
    mu: np.ndarray
    w: np.ndarray
    dt: float
    bc_left: int = BC_VACUUM
    bc_right: int = BC_VACUUM
    q: Optional[np.ndarray] = None
    psi0: Optional[np.ndarray] = None
    inc_left: Optional[np.ndarray] = None
    inc_right: Optional[np.ndarray] = None
    n_steps: int = 1
    tol: float = 1e-8
    # steps (0-based) on which the source q is switched on; None = every step
    source_steps: Optional[int] = None
    meta: dict = field(default_factory=dict)

    def __post_init__(self):
        J, N, G = self.J, self.N, self.G
        f = lambda a, shape: np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), shape))
        self.dx = f(self.dx, (J,))
        self.sigma_t = f(self.sigma_t, (J, G))
        self.transfer = f(self.transfer, (J, G, G))
        self.v = f(self.v, (G,))
        self.mu = f(self.mu, (N,))
        self.w = f(self.w, (N,))
        self.q = f(0.0 if self.q is None else self.q, (J, G, 4))
        self.psi0 = f(0.0 if self.psi0 is None else self.psi0, (J, G, N, 2))
        self.inc_left = f(0.0 if self.inc_left is None else self.inc_left, (G, N, 2))
        self.inc_right = f(0.0 if self.inc_right is None else self.inc_right, (G, N, 2))

    @property
    def n(self) -> int:
        """Order of the per-cell system, 4*N*G."""
        return 4 * self.N * self.G

    def source_at_step(self, step: int) -> np.ndarray:
        """Piece-wise constant source per step: q while step < source_steps, else 0."""
        if self.source_steps is None or step < self.source_steps:
            return self.q
        return np.zeros_like(self.q)

    def with_dt(self, dt: float) -> "Problem":
        return replace(self, dt=float(dt), name=f"{self.name.split('@')[0]}@dt={dt:g}")

    def head(self, J: int) -> "Problem":
        """First J cells of the same slab (bounded samples for CPU timing)."""
        J = min(J, self.J)
        return replace(self, J=J, dx=self.dx[:J].copy(), sigma_t=self.sigma_t[:J].copy(),
                       transfer=self.transfer[:J].copy(), q=self.q[:J].copy(), psi0=self.psi0[:J].copy(),
                       name=f"{self.name}[head {J}]")


# ----------------------------------------------------------------------------------------------
# BASELINE.json configs (0-based index i <-> "config i+1" of SURVEY.md section 8d)
# ----------------------------------------------------------------------------------------------

def config1(dt: float = 0.1) -> Problem:
    """Single group, S4, 16 uniform cells on 1 cm, sigma_t=1, c=0.5, q=1, vacuum, v=1, 5 steps."""
    J, N, G = 16, 4, 1
    mu, w = gauss_legendre(N)
    return Problem("cfg1", J, N, G, dx=1.0 / J, sigma_t=1.0, transfer=0.5, v=1.0, mu=mu, w=w, dt=dt,
                   q=1.0, n_steps=5, tol=1e-8)


def config2(dt: float = 0.1, J: int = 1024) -> Problem:
    """Single group, S8, 1024 uniform cells on 10 cm (thin cells), c=0.9, q=1 in the left half."""
    N, G = 8, 1
    mu, w = gauss_legendre(N)
    q = np.zeros((J, G, 4))
    q[: J // 2] = 1.0
    return Problem("cfg2", J, N, G, dx=10.0 / J, sigma_t=1.0, transfer=0.9, v=1.0, mu=mu, w=w, dt=dt,
                   q=q, n_steps=20, tol=1e-8, meta={"dt_sweep": [1.0, 0.1, 0.01]})


def _regions(rng: np.random.Generator, J: int, n_regions: int, n_mat: int) -> np.ndarray:
    """Material id per cell: n_regions contiguous regions with seeded cut points; neighbouring regions differ."""
    cuts = np.sort(rng.choice(np.arange(1, J), size=n_regions - 1, replace=False))
    bounds = np.concatenate(([0], cuts, [J]))
    ids = np.empty(J, dtype=np.int64)
    prev = -1
    for r in range(n_regions):
        choices = [m for m in range(n_mat) if m != prev]
        prev = int(rng.choice(choices))
        ids[bounds[r]:bounds[r + 1]] = prev
    return ids


def config3(J: int = 8192, dt: float = 1e-8, seed: int = 1003) -> Problem:
    """4 groups, S8, 3 materials in seeded contiguous regions, down-scatter + fission in material index 1."""
    N, G, n_mat = 8, 4, 3
    rng = np.random.default_rng(seed)
    mu, w = gauss_legendre(N)
    sig = rng.uniform(0.5, 5.0, size=(n_mat, G))
    c = rng.uniform(0.3, 0.95, size=(n_mat, G))
    K = np.zeros((n_mat, G, G))
    for m in range(n_mat):
        raw = np.tril(rng.uniform(0.0, 1.0, size=(G, G)))        # [to][from], to >= from: down-scatter
        raw *= (c[m] * sig[m]) / raw.sum(axis=0)                  # column (over destinations) sums = c_g' sigma_t,g'
        K[m] = raw
    chi = np.zeros(G)
    chi[0] = 1.0
    K[1] += np.outer(chi, 0.1 * sig[1])                           # chi_g * nuSigma_f,g'
    ids = _regions(rng, J, n_regions=min(12, max(1, J // 4)), n_mat=n_mat)
    v = 1e9 / 10.0 ** np.arange(1, G + 1)
    return Problem("cfg3", J, N, G, dx=0.1, sigma_t=sig[ids], transfer=K[ids], v=v, mu=mu, w=w, dt=dt,
                   q=1.0, n_steps=10, tol=1e-8, meta={"material_id": ids})


def config4(J: int = 2048, dt: float = 1e-3, v: float = 1.0, seed: int = 1004, N: int = 8, G: int = 8) -> Problem:
    """8 groups, S8 (n=256), dense scattering normalised to c=0.99, reflective left / vacuum right, pulsed source."""
    rng = np.random.default_rng(seed)
    mu, w = gauss_legendre(N)
    sig = rng.uniform(0.1, 10.0, size=G)
    K = rng.uniform(0.0, 1.0, size=(G, G))
    K *= (0.99 * sig) / K.sum(axis=0)
    return Problem("cfg4" if v == 1.0 else "cfg4b", J, N, G, dx=0.1, sigma_t=sig, transfer=K, v=v, mu=mu, w=w,
                   dt=dt, bc_left=BC_REFLECTIVE, bc_right=BC_VACUUM, q=1.0, n_steps=50, tol=1e-8, source_steps=1)


def config5(J: int = 65536, dt: float = 0.1, seed: int = 1005, N: int = 16) -> Problem:
    """Single group, S16 (n=64), every cell its own sigma_t (log-uniform) and c."""
    G = 1
    rng = np.random.default_rng(seed)
    mu, w = gauss_legendre(N)
    sig = 10.0 ** rng.uniform(-2.0, 2.0, size=J)
    c = rng.uniform(0.5, 0.999, size=J)
    return Problem("cfg5", J, N, G, dx=0.1, sigma_t=sig[:, None], transfer=(c * sig)[:, None, None], v=1.0,
                   mu=mu, w=w, dt=dt, q=1.0, n_steps=10, tol=1e-8,
                   meta={"dt_sweep": [1.0, 1e-1, 1e-2, 1e-3, 1e-4]})


CONFIGS: list[Callable[..., Problem]] = [config1, config2, config3, config4, config5]


# ----------------------------------------------------------------------------------------------
# The paper's own two workloads
# ----------------------------------------------------------------------------------------------

def table2(J: int, N: int, dt: float, L: float = 100.0) -> Problem:
    """Two-group problem of Table 2: L=100 cm, vacuum, psi0=0, Q=1, v=(1, 0.5)."""
    G = 2
    mu, w = gauss_legendre(N)
    sig = np.array([1.5454, 0.45468])
    # Table 2 lists, under "Group g", the within-group value and the transfer INTO g from the other group; the
    # printed ratio 0.99997 of group 1 = (0.61789 + 0.92747)/1.5454 confirms 0.92747 leaves group 1.
    K = np.array([[0.61789, 0.38211],      # into group 1: from 1 (within), from 2
                  [0.92747, 0.0072534]])   # into group 2: from 1, from 2 (within)
    return Problem("table2", J, N, G, dx=L / J, sigma_t=sig, transfer=K, v=np.array([1.0, 0.5]), mu=mu, w=w,
                   dt=dt, q=1.0, n_steps=1, tol=1e-8)


def worked_example(J: int = 1000, dt: float = 0.1, seed: int = 7) -> Problem:
    """Verification run of PAPER.md:479: Sigma=2.5, dx=0.1, c=0.9, v=4, S8, no source, random initial guess.

    The random initial *iterate* is returned in meta["psi_guess"] ([J][G][N][4], uniform [0,1]); psi0 = 0 so the
    converged solution is 0 and the iterate itself is the error.
    """
    N, G = 8, 1
    rng = np.random.default_rng(seed)
    mu, w = gauss_legendre(N)
    return Problem("worked", J, N, G, dx=0.1, sigma_t=2.5, transfer=0.9 * 2.5, v=4.0, mu=mu, w=w, dt=dt,
                   q=0.0, n_steps=1, tol=1e-13, meta={"psi_guess": rng.uniform(0.0, 1.0, size=(J, G, N, 4))})


# ----------------------------------------------------------------------------------------------
# Small seeded problems for parity / pin tests
# ----------------------------------------------------------------------------------------------

def random_problem(seed: int, J: int, N: int, G: int, dt: float = 0.05, bc_left: int = BC_VACUUM,
                   bc_right: int = BC_VACUUM, c_max: float = 0.95, upscatter: bool = True,
                   sig_range=(0.2, 4.0), dx_range=(0.05, 0.6), v_range=(0.5, 3.0)) -> Problem:
    """Heterogeneous multigroup slab: every cell its own widths, cross-sections and sources; random psi0, inflow."""
    rng = np.random.default_rng(seed)
    mu, w = gauss_legendre(N)
    dx = rng.uniform(*dx_range, size=J)
    sig = rng.uniform(*sig_range, size=(J, G))
    K = rng.uniform(0.0, 1.0, size=(J, G, G))
    if not upscatter:
        K = np.tril(K)
    c = rng.uniform(0.2, c_max, size=(J, G))
    K *= (c * sig)[:, None, :] / K.sum(axis=1, keepdims=True)
    v = rng.uniform(*v_range, size=G)
    q = rng.uniform(0.0, 2.0, size=(J, G, 4))
    psi0 = rng.uniform(0.0, 1.0, size=(J, G, N, 2))
    inc_l = rng.uniform(0.0, 1.0, size=(G, N, 2)) if bc_left == BC_PRESCRIBED else None
    inc_r = rng.uniform(0.0, 1.0, size=(G, N, 2)) if bc_right == BC_PRESCRIBED else None
    return Problem(f"rand{seed}", J, N, G, dx, sig, K, v, mu, w, dt, bc_left, bc_right, q, psi0, inc_l, inc_r,
                   n_steps=3, tol=1e-10)


def homogeneous(J: int, N: int, sigma_t: float, c: float, dx: float, v: float, dt: float, q: float = 0.0,
                bc: int = BC_VACUUM, psi0: float = 0.0) -> Problem:
    """One-group homogeneous slab (model problem of the Fourier analysis)."""
    mu, w = gauss_legendre(N)
    return Problem("homog", J, N, 1, dx, sigma_t, c * sigma_t, v, mu, w, dt, bc, bc, q=q, psi0=psi0)
