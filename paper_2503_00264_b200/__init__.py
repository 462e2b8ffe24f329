"""paper_2503_00264_b200 -- thin Python binding of liboci_b200.so (include/oci.h).

Argument marshalling only: every numerical step of the OCI / SI hot path runs in the hand-written CUDA
kernels behind the C ABI. PyTorch is used for device memory (the caller-owned workspace and the arrays
passed in and out) and for the CUDA stream; nothing in this package computes, and there is no CPU fallback:
constructing a solver without the compiled library or without a CUDA device raises.

The function names mirror the C entry points (oci_create -> OCISolver(...), oci_factor -> .factor(), ...).
This package never imports oracle/ (test infrastructure) and oracle/ never imports it.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

from . import build as _build

__all__ = ["OCISolver", "OCIError", "load_library", "declared_symbols", "create_error", "flux_residual_static",
           "STATIC_MAX_PAIRS", "BC_VACUUM", "BC_REFLECTIVE", "BC_PRESCRIBED", "STOP_DPHI_INF", "STOP_PAPER"]

BC_VACUUM, BC_REFLECTIVE, BC_PRESCRIBED = 0, 1, 2
STOP_DPHI_INF, STOP_PAPER = 0, 1
RESID_CAP = 65536
STATIC_MAX_PAIRS = 1 << 20  # OCI_STATIC_MAX_PAIRS: largest J * G flux_residual_static takes

_dptr = C.c_void_p
_i32, _i64, _f64 = C.c_int32, C.c_int64, C.c_double


class _Problem(C.Structure):
    _fields_ = [("J", _i32), ("N", _i32), ("G", _i32),
                ("dx", _dptr), ("sigma_t", _dptr), ("transfer", _dptr), ("v", _dptr), ("mu", _dptr), ("w", _dptr),
                ("dt", _f64), ("bc_left", _i32), ("bc_right", _i32)]


_SIGNATURES = {
    "oci_workspace_bytes": (C.c_size_t, [C.POINTER(_Problem)]),
    "oci_create": (C.c_int, [C.POINTER(_Problem), _dptr, C.c_size_t, _dptr, C.POINTER(_dptr)]),
    "oci_destroy": (None, [_dptr]),
    "oci_strerror": (C.c_char_p, [C.c_int]),
    "oci_last_cuda_error": (C.c_int, [_dptr]),
    "oci_last_create_error": (C.c_int, []),
    "oci_set_option": (C.c_int, [_dptr, C.c_char_p, _i64]),
    "oci_set_dt": (C.c_int, [_dptr, _f64]),
    "oci_set_source": (C.c_int, [_dptr, _dptr]),
    "oci_set_incident": (C.c_int, [_dptr, _dptr, _dptr]),
    "oci_set_state": (C.c_int, [_dptr, _dptr]),
    "oci_get_state": (C.c_int, [_dptr, _dptr]),
    "oci_set_iterate": (C.c_int, [_dptr, _dptr]),
    "oci_factor": (C.c_int, [_dptr]),
    "oci_iterate": (C.c_int, [_dptr, _i32]),
    "oci_step": (C.c_int, [_dptr, _f64, _i32, _i32, _i32, _i32, C.POINTER(_i32), C.POINTER(_f64)]),
    "si_iterate": (C.c_int, [_dptr, _i32]),
    "si_step": (C.c_int, [_dptr, _f64, _i32, _i32, _i32, _i32, C.POINTER(_i32), C.POINTER(_f64)]),
    "oci_advance": (C.c_int, [_dptr]),
    "oci_scalar_flux": (C.c_int, [_dptr, _dptr]),
    "oci_angular_flux": (C.c_int, [_dptr, _dptr]),
    "oci_residual_history": (C.c_int, [_dptr, _i32, _dptr, _i32, C.POINTER(_i32)]),
    "oci_step_host": (C.c_int, [_dptr, _i32, _dptr, _f64, _i32, _i32, _i32, _i32, C.POINTER(_i32), C.POINTER(_f64),
                                _dptr]),
    "oci_debug_get_matrix": (C.c_int, [_dptr, _i32, _dptr]),
    "oci_debug_get_inverse": (C.c_int, [_dptr, _i32, _dptr]),
    "oci_debug_get_factor_input": (C.c_int, [_dptr, _i32, _dptr]),
    "oci_debug_get_const_rhs": (C.c_int, [_dptr, _dptr]),
    "oci_debug_empty_launches": (C.c_int, [_dptr, _i32]),
    "oci_last_timing": (C.c_int, [_dptr, _i32, C.POINTER(_f64), C.POINTER(_i64)]),
    "oci_flux_residual_static": (C.c_int, [_i32, _i32, _i32, _dptr, _dptr, _dptr, _dptr, _dptr, _dptr]),
    "oci_static_last_cuda_error": (C.c_int, []),
}


def declared_symbols() -> list[str]:
    """Every entry point include/oci.h declares (kept in step with the header by tests/test_abi.py)."""
    return sorted(_SIGNATURES)


_lib = None


def load_library(rebuild: bool = False):
    """dlopen liboci_b200.so, building it with nvcc first if it is missing or stale. Raises if it cannot."""
    global _lib
    if _lib is None or rebuild:
        path = _build.build(force=rebuild)
        lib = C.CDLL(str(path))
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)  # AttributeError = symbol missing: fail loudly
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def create_error() -> int:
    """oci_last_create_error: the cudaError_t behind this thread's most recent failed oci_create (0 if none)."""
    return int(load_library().oci_last_create_error())


class OCIError(RuntimeError):
    def __init__(self, fn: str, code: int, cuda: int = 0):
        msg = load_library().oci_strerror(code).decode()
        super().__init__(f"{fn} failed: {code} ({msg})" + (f", cudaError {cuda}" if cuda else ""))
        self.code, self.cuda = code, cuda


def flux_residual_static(psi, w, phi_prev, phi_out, resid_out, stream=None) -> None:
    """oci_flux_residual_static: phi = sum_m w_m psi_m and the residuals max |phi - phi_prev|, ||phi - phi_prev||_2 for
    arrays the caller holds, without a solver object and without a workspace.

    This is the library's one call for users who cannot allocate device memory: a module living inside an application
    whose memory pool owns the GPU, or code that must not call cudaMalloc / cudaFree because those stall every stream
    of the process. The kernel's scratch is a fixed array inside liboci_b200.so (about 256 KB per GPU), so the call --
    and this wrapper, which only passes pointers -- allocates nothing: `phi_out` [J][G][4] and `resid_out` [2] are the
    caller's, fp64, contiguous, on the GPU of `psi` [J][G][N][4]; `phi_out` may be `phi_prev`. J * G is limited to
    STATIC_MAX_PAIRS (OCIError -105 beyond it). The first call on a GPU fetches the array's address; make it before
    any stream capture. Calls on one GPU share the array: keep them ordered (one stream), never concurrent.
    Asynchronous on `stream` (default: torch's current stream on that GPU)."""
    import torch

    lib = load_library()
    if psi.dim() != 4 or psi.shape[3] != 4:
        raise ValueError("psi must be [J][G][N][4]")
    J, G, N = int(psi.shape[0]), int(psi.shape[1]), int(psi.shape[2])
    for name, t, numel in (("psi", psi, J * G * N * 4), ("w", w, N), ("phi_prev", phi_prev, J * G * 4),
                           ("phi_out", phi_out, J * G * 4), ("resid_out", resid_out, 2)):
        if t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != numel or t.device != psi.device:
            raise ValueError(f"{name}: expected a contiguous fp64 tensor of {numel} elements on {psi.device}")
    if stream is None:
        stream = torch.cuda.current_stream(psi.device)
    code = lib.oci_flux_residual_static(J, N, G, w.data_ptr(), psi.data_ptr(), phi_prev.data_ptr(), phi_out.data_ptr(),
                                        resid_out.data_ptr(), stream.cuda_stream)
    if code != 0:
        raise OCIError("oci_flux_residual_static", code, int(lib.oci_static_last_cuda_error()))


class OCISolver:
    """One transport problem on one GPU. `p` is any object with the attributes J, N, G, dx, sigma_t, transfer,
    v, mu, w, dt, bc_left, bc_right (+ optionally q, psi0, inc_left, inc_right), e.g. workloads.Problem."""

    def __init__(self, p, dt: float | None = None, device: str | int = "cuda:0", stream=None, options=None):
        import numpy as np
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_00264_b200 needs a CUDA device: there is no CPU fallback")
        self._torch, self._np = torch, np
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.J, self.N, self.G = int(p.J), int(p.N), int(p.G)
        self.n = 4 * self.N * self.G
        f = lambda a, shape: np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), shape))
        host = dict(dx=f(p.dx, (self.J,)), sigma_t=f(p.sigma_t, (self.J, self.G)),
                    transfer=f(p.transfer, (self.J, self.G, self.G)), v=f(p.v, (self.G,)),
                    mu=f(p.mu, (self.N,)), w=f(p.w, (self.N,)))
        prob = _Problem(self.J, self.N, self.G, *(host[k].ctypes.data for k in
                                                   ("dx", "sigma_t", "transfer", "v", "mu", "w")),
                        float(p.dt if dt is None else dt), int(p.bc_left), int(p.bc_right))
        nbytes = int(self.lib.oci_workspace_bytes(C.byref(prob)))
        if nbytes == 0:
            raise OCIError("oci_workspace_bytes", -102)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._ctx = _dptr()
        self._check("oci_create", self.lib.oci_create(C.byref(prob), self.workspace.data_ptr(), nbytes,
                                                      self.stream.cuda_stream, C.byref(self._ctx)))
        for k, v in (options or {}).items():
            self.set_option(k, v)
        if getattr(p, "inc_left", None) is not None or getattr(p, "inc_right", None) is not None:
            self.set_incident(getattr(p, "inc_left", None), getattr(p, "inc_right", None))
        if getattr(p, "q", None) is not None:
            self.set_source(p.q)
        if getattr(p, "psi0", None) is not None:
            self.set_state(p.psi0)

    # -- plumbing ------------------------------------------------------------------------------------------
    def _check(self, fn: str, code: int, allow_positive: bool = False) -> int:
        if code < 0 or (code > 0 and not allow_positive):
            cuda = self.lib.oci_last_cuda_error(self._ctx) if self._ctx else self.lib.oci_last_create_error()
            raise OCIError(fn, code, cuda)
        return code

    def _dev(self, a, shape):
        """numpy / torch -> contiguous fp64 device tensor of `shape` (a view if it already is one)."""
        torch = self._torch
        if a is None:
            return None
        if not isinstance(a, torch.Tensor):
            a = torch.from_numpy(self._np.ascontiguousarray(
                self._np.broadcast_to(self._np.asarray(a, dtype=self._np.float64), shape)))
        return a.to(device=self.device, dtype=torch.float64).reshape(shape).contiguous()

    def _new(self, *shape):
        return self._torch.empty(shape, dtype=self._torch.float64, device=self.device)

    def close(self):
        if getattr(self, "_ctx", None):
            self.lib.oci_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def synchronize(self):
        self.stream.synchronize()

    # -- the C entry points, same names ----------------------------------------------------------------------
    def set_option(self, key: str, value: int):
        self._check("oci_set_option", self.lib.oci_set_option(self._ctx, key.encode(), int(value)))

    def set_dt(self, dt: float):
        self._check("oci_set_dt", self.lib.oci_set_dt(self._ctx, float(dt)))

    def set_source(self, q):
        t = self._dev(q, (self.J, self.G, 4))
        self._check("oci_set_source", self.lib.oci_set_source(self._ctx, t.data_ptr() if t is not None else None))
        self.synchronize()  # the library reads t during the stream work; keep it alive until then

    def set_incident(self, left, right):
        lt, rt = self._dev(left, (self.G, self.N, 2)), self._dev(right, (self.G, self.N, 2))
        self._check("oci_set_incident", self.lib.oci_set_incident(
            self._ctx, lt.data_ptr() if lt is not None else None, rt.data_ptr() if rt is not None else None))
        self.synchronize()

    def set_state(self, psi_edge):
        t = self._dev(psi_edge, (self.J, self.G, self.N, 2))
        self._check("oci_set_state", self.lib.oci_set_state(self._ctx, t.data_ptr()))
        self.synchronize()

    def get_state(self):
        out = self._new(self.J, self.G, self.N, 2)
        self._check("oci_get_state", self.lib.oci_get_state(self._ctx, out.data_ptr()))
        return out

    def set_iterate(self, psi):
        t = self._dev(psi, (self.J, self.G, self.N, 4))
        self._check("oci_set_iterate", self.lib.oci_set_iterate(self._ctx, t.data_ptr()))
        self.synchronize()

    def factor(self) -> int:
        """Returns 0, or the 1-based index of the first singular cell."""
        return self._check("oci_factor", self.lib.oci_factor(self._ctx), allow_positive=True)

    def iterate(self, n_iters: int = 1):
        self._check("oci_iterate", self.lib.oci_iterate(self._ctx, int(n_iters)))

    def si_iterate(self, n_iters: int = 1):
        self._check("si_iterate", self.lib.si_iterate(self._ctx, int(n_iters)))

    def _step(self, name, tol, max_iters, check_every, stop_rule, advance):
        its = (_i32 * 2)()
        res = _f64()
        fn = getattr(self.lib, name)
        self._check(name, fn(self._ctx, float(tol), int(max_iters), int(check_every), int(stop_rule),
                             int(bool(advance)), its, C.byref(res)))
        return int(its[0]), int(its[1]), float(res.value)

    def step(self, tol=1e-8, max_iters=RESID_CAP, check_every=8, stop_rule=STOP_DPHI_INF, advance=True):
        """oci_step: returns (iterations performed, iterations after which the rule first held, last residual)."""
        return self._step("oci_step", tol, max_iters, check_every, stop_rule, advance)

    def si_step(self, tol=1e-8, max_iters=RESID_CAP, check_every=8, stop_rule=STOP_DPHI_INF, advance=True):
        return self._step("si_step", tol, max_iters, check_every, stop_rule, advance)

    def advance(self):
        self._check("oci_advance", self.lib.oci_advance(self._ctx))

    def scalar_flux(self):
        out = self._new(self.J, self.G, 4)
        self._check("oci_scalar_flux", self.lib.oci_scalar_flux(self._ctx, out.data_ptr()))
        return out

    def angular_flux(self):
        out = self._new(self.J, self.G, self.N, 4)
        self._check("oci_angular_flux", self.lib.oci_angular_flux(self._ctx, out.data_ptr()))
        return out

    def residual_history(self, kind: int = 0):
        np = self._np
        n = _i32()
        self._check("oci_residual_history", self.lib.oci_residual_history(self._ctx, kind, None, 0, C.byref(n)))
        out = np.zeros(max(int(n.value), 1))
        self._check("oci_residual_history", self.lib.oci_residual_history(self._ctx, kind, out.ctypes.data,
                                                                          int(n.value), C.byref(n)))
        return out[: int(n.value)]

    def step_host(self, scheme, q_host, phi_host, tol=1e-8, max_iters=RESID_CAP, check_every=8,
                  stop_rule=STOP_DPHI_INF, advance=True):
        """oci_step_host: q_host / phi_host are pinned CPU tensors (or None) of shape [J][G][4]."""
        its = (_i32 * 2)()
        res = _f64()
        self._check("oci_step_host", self.lib.oci_step_host(
            self._ctx, int(scheme), q_host.data_ptr() if q_host is not None else None, float(tol), int(max_iters),
            int(check_every), int(stop_rule), int(bool(advance)), its, C.byref(res),
            phi_host.data_ptr() if phi_host is not None else None))
        return int(its[0]), int(its[1]), float(res.value)

    def debug_matrix(self, cell: int):
        out = self._np.empty((self.n, self.n))
        self._check("oci_debug_get_matrix", self.lib.oci_debug_get_matrix(self._ctx, int(cell), out.ctypes.data))
        return out

    def debug_factor_input(self, cell: int):
        """The tile the production factor kernel assembles on chip for `cell`, dumped before the elimination."""
        out = self._np.empty((self.n, self.n))
        self._check("oci_debug_get_factor_input",
                    self.lib.oci_debug_get_factor_input(self._ctx, int(cell), out.ctypes.data))
        return out

    def debug_inverse(self, cell: int):
        out = self._np.empty((self.n, self.n))
        self._check("oci_debug_get_inverse", self.lib.oci_debug_get_inverse(self._ctx, int(cell), out.ctypes.data))
        return out

    def debug_const_rhs(self):
        out = self._new(self.J, self.n)
        self._check("oci_debug_get_const_rhs", self.lib.oci_debug_get_const_rhs(self._ctx, out.data_ptr()))
        return out

    def debug_empty_launches(self, count: int):
        self._check("oci_debug_empty_launches", self.lib.oci_debug_empty_launches(self._ctx, int(count)))

    def last_timing(self, which: int):
        """(ms, launches) of the most recent factor (0) / OCI iterations (1) / SI iterations (2)."""
        ms, ln = _f64(), _i64()
        self._check("oci_last_timing", self.lib.oci_last_timing(self._ctx, int(which), C.byref(ms), C.byref(ln)))
        return float(ms.value), int(ln.value)
