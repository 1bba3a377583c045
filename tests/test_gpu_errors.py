"""Boundary behaviour of the C ABI (include/gs.h "Errors", SURVEY.md section 8(c) test `gpu_errors`):
every argument error is returned synchronously as a status, nothing is launched, nothing hangs.

The calls go through raw ctypes on purpose (the Plan methods of gs.py would reject a bad tensor before the
library sees it): what is tested is the library's own checking of plain pointers and sizes.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu

OK, INVALID, NOT_POSDEF, SINGULAR, CUDA, WORKSPACE = 0, 1, 2, 3, 4, 5


def _gs():
    from paper_2502_02460_b200 import gs
    return gs


def _stream():
    return int(torch.cuda.current_stream().cuda_stream)


def _dev(a):
    return wl.to_colmajor(torch.from_numpy(np.ascontiguousarray(a)).cuda())


def test_singular_u_is_reported_and_later_calls_are_noops():
    """A zero on the diagonal of U: gs_invert_triangular sets the flag, gs_last_info returns GS_ERR_SINGULAR with the
    1-based index of the FIRST zero, later calls are no-ops until the flag is cleared."""
    gs = _gs()
    N = 300
    rng = np.random.default_rng(1)
    U = np.triu(rng.standard_normal((N, N))) + 4.0 * np.eye(N)
    U[140, 140] = 0.0          # block 1
    U[270, 270] = 0.0          # block 2: the first one must be reported
    plan = gs.Plan(N, N)
    V = wl.colmajor_empty(N, N, device="cuda")
    V.fill_(7.0)
    plan.invert_triangular(_dev(U), V)
    with pytest.raises(gs.GsError) as e:
        plan.last_info()
    assert e.value.status == SINGULAR and e.value.info == 141
    # while the flag is set: no-ops (outputs untouched)
    Ht = wl.colmajor_empty(N, N, device="cuda")
    Ht.fill_(-1.0)
    H = _dev(np.eye(N))
    plan.to_standard(H, V, Ht)
    C = wl.colmajor_empty(N, N, device="cuda")
    C.fill_(-2.0)
    plan.backtransform(V, H, C)
    assert plan.last_info(raise_on_failure=False) == 141
    assert torch.all(Ht == -1.0) and torch.all(C == -2.0)
    # gs_plan_clear_info is the way back for a plan that never calls gs_cholesky
    plan.clear_info()
    assert plan.last_info() == 0
    U[140, 140] = 3.0
    U[270, 270] = 3.0
    plan.invert_triangular(_dev(U), V)
    assert plan.last_info() == 0
    R = torch.from_numpy(U).cuda() @ V
    R.diagonal().sub_(1.0)
    assert R.abs().max().item() < 1e-10
    plan.close()


def test_singular_complex():
    gs = _gs()
    N = 130
    rng = np.random.default_rng(2)
    U = np.triu(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))) + 4.0 * np.eye(N)
    U[70, 70] = 0.0
    plan = gs.Plan(N, 0, dtype=gs.GS_COMPLEX128)
    V = wl.colmajor_empty(N, N, dtype=torch.complex128, device="cuda")
    plan.invert_triangular(_dev(U), V)
    with pytest.raises(gs.GsError) as e:
        plan.last_info()
    assert e.value.status == SINGULAR and e.value.info == 71
    plan.close()


def test_null_and_misaligned_pointers():
    gs = _gs()
    L = gs.lib()
    N, nev = 200, 64
    plan = gs.Plan(N, nev)
    h = plan._h
    A, B, C3 = (wl.colmajor_zeros(N, N, device="cuda") for _ in range(3))
    X, Y = (wl.colmajor_zeros(N, nev, device="cuda") for _ in range(2))
    a, b, c, x, y = (t.data_ptr() for t in (A, B, C3, X, Y))
    st = _stream()
    # NULL
    assert L.gs_cholesky(h, None, st) == INVALID
    assert L.gs_invert_triangular(h, None, b, st) == INVALID
    assert L.gs_invert_triangular(h, a, None, st) == INVALID
    assert L.gs_to_standard(h, None, b, c, st) == INVALID
    assert L.gs_to_standard(h, a, None, c, st) == INVALID
    assert L.gs_to_standard(h, a, b, None, st) == INVALID
    assert L.gs_backtransform(h, None, x, y, st) == INVALID
    assert L.gs_backtransform(h, a, None, y, st) == INVALID
    assert L.gs_backtransform(h, a, x, None, st) == INVALID
    assert L.gs_density_matrix(h, x, None, a, st) == INVALID
    assert L.gs_density_matrix(h, x, y, None, st) == INVALID
    assert L.gs_cholesky(None, a, st) == INVALID
    assert L.gs_last_info(h, st, None) == INVALID
    assert L.gs_plan_workspace_bytes(h, None) == INVALID
    assert L.gs_plan_create(None, N, 0, nev) == INVALID
    # 8-byte aligned but not 16-byte aligned
    assert L.gs_cholesky(h, a + 8, st) == INVALID
    assert L.gs_invert_triangular(h, a + 8, b, st) == INVALID
    assert L.gs_invert_triangular(h, a, b + 8, st) == INVALID
    assert L.gs_to_standard(h, a, b, c + 8, st) == INVALID
    assert L.gs_backtransform(h, a, x + 8, y, st) == INVALID
    assert L.gs_invert_triangular_cols(h, a + 8, b, 0, 128, st) == INVALID
    # column ranges off the block grid
    assert L.gs_invert_triangular_cols(h, a, b, 64, 64, st) == INVALID
    assert L.gs_to_standard_cols(h, a, b, c, 0, 100, st) == INVALID
    assert L.gs_backtransform_cols(h, a, x, y, 0, nev + 1, st) == INVALID
    assert L.gs_cholesky_leading(h, a, 100, st) == INVALID
    # nothing was launched, the plan is still fine
    torch.cuda.synchronize()
    assert plan.last_info() == 0 and plan.launch_count() == 0
    plan.close()


def test_outputs_overlapping_inputs_by_a_subrange():
    """The aliasing rule is about byte ranges: an output that starts INSIDE an input is rejected too."""
    gs = _gs()
    L = gs.lib()
    N, nev = 256, 128
    plan = gs.Plan(N, nev)
    h, st = plan._h, _stream()
    big = torch.zeros(3 * N * N, dtype=torch.float64, device="cuda")
    base = big.data_ptr()
    half = (N * N // 2) * 8             # 16-byte aligned offset into a matrix
    other = torch.zeros(N * N, dtype=torch.float64, device="cuda").data_ptr()
    assert L.gs_invert_triangular(h, base, base, st) == INVALID
    assert L.gs_invert_triangular(h, base, base + half, st) == INVALID
    assert L.gs_invert_triangular(h, base + half, base, st) == INVALID
    assert L.gs_to_standard(h, base, other, base + half, st) == INVALID           # H~ inside H
    assert L.gs_to_standard(h, other, base, base + half, st) == INVALID           # H~ inside Uinv
    assert L.gs_backtransform(h, base, other, base + N * N * 8 - 16, st) == INVALID   # C starts in the last bytes of Uinv
    assert L.gs_backtransform(h, other, base, base + 16, st) == INVALID           # C inside C~
    assert L.gs_to_standard_g_cols(h, base, other, base + half, 0, 128, st) == INVALID
    # adjacent (touching, not overlapping) buffers are fine
    assert L.gs_invert_triangular(h, base, base + N * N * 8, st) == OK
    plan.clear_info()                   # (zeros are singular: the flag was set by the call above)
    torch.cuda.synchronize()
    plan.close()


def test_workspace_errors():
    gs = _gs()
    L = gs.lib()
    N = 200
    h = ctypes.c_void_p()
    assert L.gs_plan_create(ctypes.byref(h), N, 0, N) == OK
    n = ctypes.c_size_t(0)
    assert L.gs_plan_workspace_bytes(h, ctypes.byref(n)) == OK and n.value >= N * N * 8
    A = wl.colmajor_zeros(N, N, device="cuda")
    B = wl.colmajor_zeros(N, N, device="cuda")
    st = _stream()
    # no workspace yet: every compute call and gs_last_info say so
    assert L.gs_cholesky(h, A.data_ptr(), st) == WORKSPACE
    assert L.gs_invert_triangular(h, A.data_ptr(), B.data_ptr(), st) == WORKSPACE
    assert L.gs_to_standard(h, A.data_ptr(), B.data_ptr(), A.data_ptr(), st) == WORKSPACE
    info = ctypes.c_int64(0)
    assert L.gs_last_info(h, st, ctypes.byref(info)) == WORKSPACE
    assert L.gs_plan_clear_info(h, st) == WORKSPACE
    ws = torch.empty(n.value + 512, dtype=torch.uint8, device="cuda")
    assert L.gs_plan_set_workspace(h, None, n.value) == WORKSPACE                     # NULL
    assert L.gs_plan_set_workspace(h, ws.data_ptr(), n.value - 1) == WORKSPACE        # too small
    assert L.gs_plan_set_workspace(h, ws.data_ptr() + 16, n.value) == WORKSPACE       # not 256-byte aligned
    assert L.gs_cholesky(h, A.data_ptr(), st) == WORKSPACE                            # still none
    assert L.gs_plan_set_workspace(h, ws.data_ptr(), n.value) == OK
    A.copy_(torch.eye(N, dtype=torch.float64, device="cuda") * 4.0)
    assert L.gs_cholesky(h, A.data_ptr(), st) == OK
    assert L.gs_last_info(h, st, ctypes.byref(info)) == OK and info.value == 0
    assert torch.equal(A, torch.eye(N, dtype=torch.float64, device="cuda") * 2.0)
    assert L.gs_plan_destroy(h) == OK


def test_reduce_host_scratch_errors():
    gs = _gs()
    L = gs.lib()
    N, nev = 200, 50
    plan = gs.Plan(N, nev)
    h, st = plan._h, _stream()
    need = plan.host_scratch_bytes()
    hH = torch.eye(N, dtype=torch.float64).pin_memory()
    hS = torch.eye(N, dtype=torch.float64).pin_memory()
    hHt = torch.empty((N, N), dtype=torch.float64).pin_memory()
    hCt = torch.zeros((nev, N), dtype=torch.float64).pin_memory()
    hC = torch.empty((nev, N), dtype=torch.float64).pin_memory()
    scratch = torch.empty(need + 512, dtype=torch.uint8, device="cuda")
    sp = scratch.data_ptr()
    args = (hH.data_ptr(), hS.data_ptr(), None, None, hHt.data_ptr())
    assert L.gs_reduce_host(h, *args, None, need, st) == WORKSPACE
    assert L.gs_reduce_host(h, *args, sp, need - 1, st) == WORKSPACE                  # undersized
    assert L.gs_reduce_host(h, *args, sp + 16, need, st) == WORKSPACE                 # misaligned
    assert L.gs_reduce_host(h, None, hS.data_ptr(), None, None, hHt.data_ptr(), sp, need, st) == INVALID
    assert L.gs_reduce_host(h, hH.data_ptr(), hS.data_ptr(), None, None, None, sp, need, st) == INVALID
    assert L.gs_backtransform_host(h, hCt.data_ptr(), hC.data_ptr(), sp, need - 1, st) == WORKSPACE
    assert L.gs_backtransform_host(h, None, hC.data_ptr(), sp, need, st) == INVALID
    # and the good call still works afterwards (S = H = I: H~ = I)
    assert L.gs_reduce_host(h, *args, sp, need, st) == OK
    assert torch.equal(torch.triu(hHt.t()), torch.eye(N, dtype=torch.float64))     # the buffer is the column-major image
    plan.close()


def test_second_device_or_reconfiguration_after_set_device():
    """The opt-in to large dynamic shared memory is per device: plans on every visible device work;
    with one device, a plan created after an explicit cudaSetDevice round trip still launches its leaf kernels."""
    gs = _gs()
    N = 260
    p = wl.small_pencil(N, seed=5)
    for d in range(torch.cuda.device_count()):
        with torch.cuda.device(d):
            dev = torch.device("cuda", d)
            plan = gs.Plan(N, 0, device=dev)
            U = wl.to_colmajor(p.S.to(dev))
            plan.cholesky(U, stream=torch.cuda.current_stream(dev))
            assert plan.last_info(stream=torch.cuda.current_stream(dev)) == 0
            R = torch.triu(U).t() @ torch.triu(U) - p.S.to(dev)
            assert (R.norm() / p.S.norm()).item() < 1e-13
            plan.close()


def test_evp_and_truncated_argument_errors():
    """NEXT-4 / (5) entry points: workspace and pointer errors come back as statuses, nothing is launched."""
    gs = _gs()
    L = gs.lib()
    N, nev = 200, 64
    plan = gs.Plan(N, nev)
    h, st = plan._h, _stream()
    A = wl.colmajor_zeros(N, N, device="cuda")
    B = wl.colmajor_zeros(N, N, device="cuda")
    X = wl.colmajor_zeros(N, nev, device="cuda")
    v = torch.zeros(N, dtype=torch.float64, device="cuda")
    a, b, x, vp = A.data_ptr(), B.data_ptr(), X.data_ptr(), v.data_ptr()
    # no eigensolver workspace yet
    assert L.gs_evp_tridiagonalize(h, a, vp, vp, vp, st) == WORKSPACE
    assert L.gs_standard_eigh(h, a, vp, x, st) == WORKSPACE
    assert L.gs_truncated_to_standard(h, a, b, 1e-5, a, b, vp, st) == WORKSPACE
    n = ctypes.c_size_t(0)
    assert L.gs_evp_workspace_bytes(h, ctypes.byref(n)) == OK and n.value > 3 * N * N * 8
    nt = ctypes.c_size_t(0)
    assert L.gs_truncated_workspace_bytes(h, ctypes.byref(nt)) == OK and nt.value > n.value      # all N eigenvectors of S
    ws = torch.empty(nt.value + 512, dtype=torch.uint8, device="cuda")
    assert L.gs_evp_set_workspace(h, None, n.value) == WORKSPACE
    assert L.gs_evp_set_workspace(h, ws.data_ptr(), n.value - 1) == WORKSPACE
    assert L.gs_evp_set_workspace(h, ws.data_ptr() + 16, n.value) == WORKSPACE
    assert L.gs_evp_set_workspace(h, ws.data_ptr(), n.value) == OK
    assert L.gs_truncated_to_standard(h, a, b, 1e-5, x, b, vp, st) == WORKSPACE                # sized for nev only: too small
    assert L.gs_evp_set_workspace(h, ws.data_ptr(), nt.value) == OK
    # pointers
    assert L.gs_evp_tridiagonalize(h, None, vp, vp, vp, st) == INVALID
    assert L.gs_evp_tridiagonalize(h, a + 8, vp, vp, vp, st) == INVALID
    assert L.gs_evp_tridiagonalize(h, a, None, vp, vp, st) == INVALID
    assert L.gs_evp_tridiag_solve(h, vp, vp, None, x, st) == INVALID
    assert L.gs_evp_backtransform(h, a, vp, a + 64, st) == INVALID                              # C~ inside the reflector matrix
    assert L.gs_standard_eigh(h, a, vp, a + 16, st) == INVALID
    assert L.gs_standard_eigh(h, a, None, x, st) == INVALID
    assert L.gs_truncated_to_standard(h, a, b, -1.0, A.data_ptr(), b, vp, st) == INVALID        # delta < 0, X aliases H
    assert L.gs_truncated_to_standard(h, a, b, float("nan"), x, b, vp, st) == INVALID
    assert L.gs_backtransform_dense(h, a, x, x, st) == INVALID
    assert L.gs_truncated_rank(h, st, None) == INVALID
    torch.cuda.synchronize()
    assert plan.last_info() == 0 and plan.launch_count() == 0
    plan.close()


@pytest.mark.parametrize("cplx,N", [(False, 300), (True, 200), (False, 129)])
def test_eigensolver_stages_are_noops_while_the_flag_is_set(cplx, N):
    """include/gs.h, "Errors": all later compute calls on the plan are no-ops while the flag is set.  The step kernels of
    the tridiagonalisation read the flag late (csrc/evp_tridiag.cuh: off the critical path) and must still leave the
    matrix and d, e, tau alone; so must the eigenvalues-only calls.  Even N: the TMA loader, several panels."""
    gs = _gs()
    L = gs.lib()
    dt = torch.complex128 if cplx else torch.float64
    plan = gs.Plan(N, N, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    plan.ensure_evp_workspace()
    bad = np.eye(N) * (1.0 + 0j if cplx else 1.0)
    bad[N // 2, N // 2] = -1.0
    S = wl.to_colmajor(torch.from_numpy(bad).to(dt).cuda())
    plan.cholesky(S)
    assert plan.last_info(raise_on_failure=False) == N // 2 + 1
    g = torch.Generator(device="cpu")
    g.manual_seed(N)
    A0 = torch.randn(N, N, dtype=dt, generator=g)
    A0 = wl.to_colmajor((A0 + A0.conj().t()).cuda())
    A = A0.clone()
    d = torch.full((N,), 5.0, dtype=torch.float64, device="cuda")
    e = torch.full((N,), 6.0, dtype=torch.float64, device="cuda")
    tau = torch.full((N,), 7.0, dtype=dt, device="cuda")
    assert L.gs_evp_tridiagonalize(plan._h, A.data_ptr(), d.data_ptr(), e.data_ptr(), tau.data_ptr(), None) == gs.GS_OK
    lam = torch.full((N,), 8.0, dtype=torch.float64, device="cuda")
    assert L.gs_evp_tridiag_eigenvalues(plan._h, d.data_ptr(), e.data_ptr(), N, lam.data_ptr(), None) == gs.GS_OK
    assert L.gs_standard_eigenvalues(plan._h, A.data_ptr(), N, lam.data_ptr(), None) == gs.GS_OK
    assert plan.last_info(raise_on_failure=False) == N // 2 + 1
    assert torch.equal(A, A0)
    assert torch.all(d == 5.0) and torch.all(e == 6.0) and torch.all(tau == 7.0) and torch.all(lam == 8.0)
    # and the same plan works again once the flag is cleared
    plan.clear_info()
    d2, e2, _ = plan.evp_tridiagonalize(A)
    assert plan.last_info() == 0
    ref = torch.linalg.eigvalsh(A0.cpu() if not cplx else A0.cpu())          # (a check of the recovery only; parity is in test_gpu_evp.py)
    got = plan.evp_tridiag_eigenvalues(d2, e2).cpu()
    assert (got - ref).abs().max().item() <= 1e-11 * max(1.0, ref.abs().max().item())
    plan.close()
