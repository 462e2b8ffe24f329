"""ctypes binding of the CPU fp64 oracle (oracle/oci_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs. The product (paper_2503_00264_b200) never imports this package and this package
never imports the product. All arithmetic of the method lives in the C file; this module only compiles
it (gcc, -ffp-contract=off), marshals numpy arrays and sequences the per-time-step calls
(Alg. 2; advance psi_{k+1/2} -> psi_{k-1/2}).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "oci_oracle.c"
_LIB = _HERE / "liboci_oracle.so"

_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_i, _d, _l = C.c_int, C.c_double, C.c_long


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc if the shared object is missing or older than its source."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall",
               "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        L.orc_num_threads.restype = _i
        L.orc_assemble_cell.argtypes = [_i, _i, _d, _dp, _dp, _dp, _dp, _dp, _d, _dp]
        L.orc_gepp_factor.argtypes = [_i, _dp, _ip]
        L.orc_gepp_factor.restype = _i
        L.orc_gepp_solve.argtypes = [_i, _dp, _ip, _dp]
        L.orc_factor_all.argtypes = [_i, _i, _i, _dp, _dp, _dp, _dp, _dp, _dp, _d, _dp, _ip]
        L.orc_factor_all.restype = _i
        L.orc_const_rhs.argtypes = [_i, _i, _i, _dp, _dp, _d, _dp, _dp, _dp]
        L.orc_oci_iterate.argtypes = [_i, _i, _i, _dp, _i, _i, _dp, _dp, _dp, _ip, _dp, _dp, _dp]
        L.orc_scalar_flux.argtypes = [_i, _i, _i, _dp, _dp, _dp]
        L.orc_max_abs_diff.argtypes = [_l, _dp, _dp]
        L.orc_max_abs_diff.restype = _d
        L.orc_l2_diff.argtypes = [_l, _dp, _dp]
        L.orc_l2_diff.restype = _d
        L.orc_si_iterate.argtypes = [_i, _i, _i, _dp, _dp, _dp, _dp, _dp, _dp, _d, _i, _i, _dp, _dp, _dp, _dp,
                                     _dp, _dp, _dp, _dp]
        L.orc_oci_converge.argtypes = [_i, _i, _i, _dp, _dp, _i, _i, _dp, _dp, _dp, _ip, _dp, _d, _i, _i, _dp,
                                       _dp, _dp, _dp]
        L.orc_oci_converge.restype = _i
        L.orc_oci_iterate_redblack.argtypes = [_i, _i, _i, _dp, _i, _i, _dp, _dp, _dp, _ip, _dp, _dp]
        L.orc_oci_converge_redblack.argtypes = L.orc_oci_converge.argtypes
        L.orc_oci_converge_redblack.restype = _i
        L.orc_si_converge.argtypes = [_i, _i, _i, _dp, _dp, _dp, _dp, _dp, _dp, _d, _i, _i, _dp, _dp, _dp, _dp,
                                      _d, _i, _i, _dp, _dp, _dp, _dp]
        L.orc_si_converge.restype = _i
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def gepp_factor(A: np.ndarray):
    """Own Gaussian elimination with partial pivoting; returns (LU, piv, info)."""
    LU = np.array(A, dtype=np.float64, order="C")
    n = LU.shape[0]
    piv = np.zeros(n, dtype=np.int32)
    info = lib().orc_gepp_factor(n, LU, piv)
    return LU, piv, info


def gepp_solve(LU: np.ndarray, piv: np.ndarray, b: np.ndarray) -> np.ndarray:
    x = np.array(b, dtype=np.float64, order="C")
    lib().orc_gepp_solve(LU.shape[0], LU, piv, x)
    return x


class Oracle:
    """Holds one problem (plain numpy arrays) and its state; every numerical step is a call into the C oracle.

    `p` is any object with the attributes of workloads.Problem (duck-typed; this package does not import it).
    State: psi [J][G][N][4] current iterate, phi [J][G][4], psi_prev [J][G][N][2] = psi_{k-1/2}.
    """

    def __init__(self, p, dt: float | None = None):
        self.J, self.N, self.G = int(p.J), int(p.N), int(p.G)
        self.n = 4 * self.N * self.G
        a = lambda x: np.ascontiguousarray(x, dtype=np.float64)
        self.dx, self.sigma_t, self.transfer, self.v = a(p.dx), a(p.sigma_t), a(p.transfer), a(p.v)
        self.mu, self.w = a(p.mu), a(p.w)
        self.dt = float(p.dt if dt is None else dt)
        self.bc_left, self.bc_right = int(p.bc_left), int(p.bc_right)
        self.inc_left, self.inc_right = a(p.inc_left), a(p.inc_right)
        self.q = a(p.q).copy()
        self.LU = None
        self.piv = None
        self.c = np.zeros((self.J, self.n))
        self.set_state(a(p.psi0))

    # -- state ---------------------------------------------------------------------------------
    def set_state(self, psi_edge: np.ndarray):
        """psi_{k-1/2} [J][G][N][2]; also seeds the iterate with both time levels = psi_edge."""
        self.psi_prev = np.ascontiguousarray(psi_edge, dtype=np.float64).reshape(self.J, self.G, self.N, 2).copy()
        self.psi = np.ascontiguousarray(np.concatenate([self.psi_prev, self.psi_prev], axis=-1))
        self.phi = self.scalar_flux(self.psi)

    def set_iterate(self, psi: np.ndarray):
        self.psi = np.ascontiguousarray(psi, dtype=np.float64).reshape(self.J, self.G, self.N, 4).copy()
        self.phi = self.scalar_flux(self.psi)

    def set_source(self, q: np.ndarray):
        self.q = np.ascontiguousarray(np.broadcast_to(q, (self.J, self.G, 4)), dtype=np.float64).copy()

    def set_dt(self, dt: float):
        self.dt = float(dt)
        self.LU = None

    # -- pieces of the path ---------------------------------------------------------------------
    def assemble_cell(self, j: int) -> np.ndarray:
        A = np.zeros((self.n, self.n))
        lib().orc_assemble_cell(self.N, self.G, float(self.dx[j]), self.sigma_t[j], self.transfer[j], self.v,
                                self.mu, self.w, self.dt, A)
        return A

    def factor(self) -> int:
        self.LU = np.empty((self.J, self.n, self.n))
        self.piv = np.empty((self.J, self.n), dtype=np.int32)
        return lib().orc_factor_all(self.J, self.N, self.G, self.dx, self.sigma_t, self.transfer, self.v, self.mu,
                                    self.w, self.dt, self.LU, self.piv)

    def const_rhs(self):
        lib().orc_const_rhs(self.J, self.N, self.G, self.dx, self.v, self.dt, self.q, self.psi_prev, self.c)
        return self.c

    def scalar_flux(self, psi: np.ndarray) -> np.ndarray:
        phi = np.empty((self.J, self.G, 4))
        lib().orc_scalar_flux(self.J, self.N, self.G, self.w, np.ascontiguousarray(psi), phi)
        return phi

    def oci_iterate(self, n_iters: int = 1, ordering: int = 0):
        """n_iters block-Jacobi (ordering 0, the paper's OCI) or red-black (ordering 1) iterations
        on the current iterate (requires factor() and const_rhs())."""
        if self.LU is None:
            raise RuntimeError("factor() first")
        if ordering == 1:
            self.psi = np.ascontiguousarray(self.psi).copy()
            for _ in range(n_iters):
                lib().orc_oci_iterate_redblack(self.J, self.N, self.G, self.mu, self.bc_left, self.bc_right,
                                               self.inc_left, self.inc_right, self.LU, self.piv, self.c, self.psi)
            self.phi = self.scalar_flux(self.psi)
            return self.psi
        for _ in range(n_iters):
            new = np.empty_like(self.psi)
            lib().orc_oci_iterate(self.J, self.N, self.G, self.mu, self.bc_left, self.bc_right, self.inc_left,
                                  self.inc_right, self.LU, self.piv, self.c, self.psi, new)
            self.psi = new
        self.phi = self.scalar_flux(self.psi)
        return self.psi

    def si_iterate(self, n_iters: int = 1):
        for _ in range(n_iters):
            psi_new, phi_new = np.empty_like(self.psi), np.empty_like(self.phi)
            lib().orc_si_iterate(self.J, self.N, self.G, self.dx, self.sigma_t, self.transfer, self.v, self.mu,
                                 self.w, self.dt, self.bc_left, self.bc_right, self.inc_left, self.inc_right,
                                 self.q, self.psi_prev, self.phi, self.psi, psi_new, phi_new)
            self.psi, self.phi = psi_new, phi_new
        return self.psi

    # -- one time step ---------------------------------------------------------------------------
    def _advance(self):
        self.psi_prev = np.ascontiguousarray(self.psi[..., 2:4]).copy()

    def oci_step(self, tol: float = 1e-8, max_iters: int = 100000, rule: int = 0, advance: bool = True,
                 ordering: int = 0):
        """Converge one time step with OCI; returns (iterations, residual history)."""
        if self.LU is None:
            self.factor()
        self.const_rhs()
        work = np.empty(self.J * self.n)
        resid = np.zeros(max_iters)
        fn = lib().orc_oci_converge_redblack if ordering == 1 else lib().orc_oci_converge
        self.psi = np.ascontiguousarray(self.psi)
        it = fn(self.J, self.N, self.G, self.mu, self.w, self.bc_left, self.bc_right, self.inc_left, self.inc_right,
                self.LU, self.piv, self.c, tol, max_iters, rule, self.psi.reshape(-1), self.phi.reshape(-1), work, resid)
        if advance:
            self._advance()
        return it, resid[:it].copy()

    def si_step(self, tol: float = 1e-8, max_iters: int = 100000, rule: int = 0, advance: bool = True):
        work = np.empty(self.J * self.n + self.J * self.G * 4)
        resid = np.zeros(max_iters)
        it = lib().orc_si_converge(self.J, self.N, self.G, self.dx, self.sigma_t, self.transfer, self.v, self.mu,
                                   self.w, self.dt, self.bc_left, self.bc_right, self.inc_left, self.inc_right,
                                   self.q, self.psi_prev, tol, max_iters, rule, self.psi.reshape(-1),
                                   self.phi.reshape(-1), work, resid)
        if advance:
            self._advance()
        return it, resid[:it].copy()
