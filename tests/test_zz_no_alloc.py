"""oci_flux_residual_static, the library's one entry point that allocates nothing (include/oci.h, csrc/noalloc.cu).

It exists for users who cannot hand the library a workspace: a transport module inside an application whose memory
pool owns the GPU, or code that may not call cudaMalloc / cudaFree because those stall every stream of the process.
Its scratch is a fixed array inside liboci_b200.so that every call on a GPU shares and that keeps whatever the last
call left in it, so the GPU test below makes two calls in a row of different sizes (the second, smaller one finds the
first one's partial results still lying beyond its own) and a third that repeats the first, and compares each with what
the ordinary, workspace-based path (OCISolver: oci_iterate / si_step + oci_scalar_flux + oci_residual_history) gives
for the same arrays, to the per-iteration tolerance of tests/test_gpu_parity.py.

This file is named to be collected last: it must pass alone in a fresh process (where its first call does the one-time
address look-up) and after all other tests (where other kernels of the library have run before)."""
import ctypes as C

import numpy as np
import pytest

import workloads as W

TOL_ITER = 1e-11  # same per-iteration bound as tests/test_gpu_parity.py


def test_size_beyond_the_fixed_scratch_is_rejected_without_a_device():
    """The size check comes before any CUDA call, so it is testable here: J * G one past the limit, null pointers --
    the answer must be OCI_E_TOO_LARGE (-105) with a message naming the limit, not a launch and not a null-pointer code."""
    import paper_2503_00264_b200 as pkg
    lib = pkg.load_library()
    J = pkg.STATIC_MAX_PAIRS // 2 + 1
    assert lib.oci_flux_residual_static(J, 4, 2, None, None, None, None, None, None) == -105
    assert b"OCI_STATIC_MAX_PAIRS" in lib.oci_strerror(-105)
    # at the limit the size is accepted and the next check (null w_dev) answers instead
    assert lib.oci_flux_residual_static(pkg.STATIC_MAX_PAIRS // 2, 4, 2, None, None, None, None, None, None) == -4
    assert lib.oci_flux_residual_static(0, 4, 2, None, None, None, None, None, None) == -1


def _close(a, b, scale):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b)))) <= TOL_ITER * scale


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_the_workspace_path_on_calls_in_a_row():
    import torch
    import paper_2503_00264_b200 as pkg
    from paper_2503_00264_b200 import OCISolver, flux_residual_static

    dev = torch.device("cuda:0")
    # outputs are the caller's: made once here, reused by every call below
    phi_big = torch.empty((4099, 2, 4), dtype=torch.float64, device=dev)
    phi_small = torch.empty((61, 3, 4), dtype=torch.float64, device=dev)
    resid = torch.empty(2, dtype=torch.float64, device=dev)

    # -- call 1: one OCI iteration of a ragged two-group problem (129 CTAs, the last one partly empty) ----------------
    p = W.random_problem(seed=41, J=4099, N=8, G=2, bc_left=W.BC_REFLECTIVE, bc_right=W.BC_PRESCRIBED)
    s = OCISolver(p, device=dev)
    rng = np.random.default_rng(5)
    s.set_iterate(rng.standard_normal((p.J, p.G, p.N, 4)))
    phi0 = s.scalar_flux().clone()
    assert s.factor() == 0
    s.iterate(1)
    psi1, phi1 = s.angular_flux(), s.scalar_flux()
    r_inf = s.residual_history(0)[-1]
    w = torch.from_numpy(np.ascontiguousarray(p.w, dtype=np.float64)).to(dev)
    flux_residual_static(psi1, w, phi0, phi_big, resid)
    torch.cuda.synchronize()
    scale = float(phi1.abs().max())
    assert _close(phi_big.cpu(), phi1.cpu(), scale)
    first = resid.cpu().numpy().copy()
    assert abs(first[0] - r_inf) <= TOL_ITER * scale
    d = (phi1 - phi0).cpu().numpy()
    assert abs(first[1] - np.sqrt(np.sum(d * d))) <= TOL_ITER * scale * np.sqrt(d.size)

    # -- call 2, straight after: a smaller problem, SI under the paper's rule (which records ||dphi||_2) ------------
    p2 = W.random_problem(seed=42, J=61, N=4, G=3, bc_left=W.BC_VACUUM, bc_right=W.BC_REFLECTIVE)
    s2 = OCISolver(p2, device=dev)
    s2.set_iterate(rng.standard_normal((p2.J, p2.G, p2.N, 4)))
    phi0_2 = s2.scalar_flux().clone()
    s2.si_step(tol=0.0, max_iters=1, check_every=1, stop_rule=pkg.STOP_PAPER, advance=False)
    psi1_2, phi1_2 = s2.angular_flux(), s2.scalar_flux()
    r_inf2, r_l2 = s2.residual_history(0)[-1], s2.residual_history(1)[-1]
    w2 = torch.from_numpy(np.ascontiguousarray(p2.w, dtype=np.float64)).to(dev)
    flux_residual_static(psi1_2, w2, phi0_2, phi_small, resid)
    torch.cuda.synchronize()
    scale2 = float(phi1_2.abs().max())
    assert _close(phi_small.cpu(), phi1_2.cpu(), scale2)
    second = resid.cpu().numpy().copy()
    assert abs(second[0] - r_inf2) <= TOL_ITER * scale2
    assert abs(second[1] - r_l2) <= TOL_ITER * scale2 * np.sqrt(phi1_2.numel())

    # -- call 3: the first one again, this time updating phi in place: the same bits as before ----------------------
    phi_inplace = phi0.clone()
    flux_residual_static(psi1, w, phi_inplace, phi_inplace, resid)
    torch.cuda.synchronize()
    assert torch.equal(phi_inplace, phi_big)
    assert np.array_equal(resid.cpu().numpy(), first)

    # -- arguments the call must refuse: a host pointer, a size beyond the scratch ------------------------------------
    lib = pkg.load_library()
    host = np.zeros(8)
    assert lib.oci_flux_residual_static(1, 2, 1, w.data_ptr(), host.ctypes.data, phi0.data_ptr(), phi_big.data_ptr(),
                                        resid.data_ptr(), None) == -5
    with pytest.raises(pkg.OCIError):
        lib_J = pkg.STATIC_MAX_PAIRS + 1
        big = torch.empty((lib_J, 1, 1, 4), dtype=torch.float64, device=dev)  # the test may allocate; the call may not
        flux_residual_static(big, w[:1].contiguous(), torch.empty((lib_J, 1, 4), dtype=torch.float64, device=dev),
                             torch.empty((lib_J, 1, 4), dtype=torch.float64, device=dev), resid)
