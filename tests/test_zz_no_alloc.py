"""gs_density_matrix_static (include/gs.h): the density matrix P_ij = sum_l f_l c*_li c_lj with its
scratch in libgs's static device array -- for callers that cannot call cudaMalloc.  Checked against the existing
entry point (gs_density_matrix, itself checked against the oracle in tests/test_gpu_density.py) on calls in a row that
share the array.  Collected last on purpose (the suite runs with pytest -x); passes alone and after the others."""
import ctypes

import numpy as np
import pytest
import torch

from paper_2502_02460_b200 import metrics as M
from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _inputs(N, nev, cplx, seed):
    C = wl.to_colmajor(wl.dense_rhs(N, nev, seed=seed, complex=cplx).cuda())
    f = torch.from_numpy(np.random.default_rng(seed).uniform(0.0, 2.0, nev)).cuda()
    return C, f


def _both(gs, N, nev, cplx, seed):
    """P from the existing path (plan workspace) and from the static-scratch entry point, same inputs."""
    dt = torch.complex128 if cplx else torch.float64
    C, f = _inputs(N, nev, cplx, seed)
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    P_ref = wl.colmajor_empty(N, N, dtype=dt, device="cuda")
    P_new = wl.colmajor_empty(N, N, dtype=dt, device="cuda")
    P_ref.fill_(-3.0)
    P_new.fill_(-3.0)
    plan.density_matrix(C, f, P_ref)
    plan.density_matrix_static(C, f, P_new)
    assert plan.last_info() == 0
    plan.close()
    return P_ref, P_new


# consecutive calls share the one array: a large real block first, then smaller / complex / ragged ones that find the
# previous call's contents both inside and beyond their own extent, then the largest size the array admits
CASES = [(700, 333, False), (257, 100, True), (129, 64, False), (5, 3, True), (2048, 1024, False), (1024, 1024, True)]


def test_static_scratch_matches_the_workspace_path_on_calls_in_a_row():
    from paper_2502_02460_b200 import gs
    for rnd in range(2):
        for i, (N, nev, cplx) in enumerate(CASES):
            P_ref, P_new = _both(gs, N, nev, cplx, seed=1000 * rnd + 17 * i + N)
            assert torch.isfinite(torch.view_as_real(P_ref) if cplx else P_ref).all()
            assert M.rel_frob_upper(P_new.cpu(), P_ref.cpu().numpy()) <= M.TOL_FROB, (rnd, N, nev, cplx)
            assert torch.equal(P_new, P_ref), (rnd, N, nev, cplx)      # same kernels, same order: the same bits
                                                                       # (incl. the untouched strictly-lower -3.0)


def test_static_scratch_needs_no_workspace_and_allocates_nothing():
    """A bare plan through the C ABI, no gs_plan_set_workspace; device memory in use does not move across the calls."""
    from paper_2502_02460_b200 import gs
    L = gs.lib()
    N, nev = 300, 100
    C, f = _inputs(N, nev, False, 5)
    ref = gs.Plan(N, nev)
    P_ref = wl.colmajor_zeros(N, N, device="cuda")
    ref.density_matrix(C, f, P_ref)
    assert ref.last_info() == 0
    ref.close()
    h = ctypes.c_void_p()
    assert L.gs_plan_create(ctypes.byref(h), N, gs.GS_REAL64, nev) == gs.GS_OK
    try:
        P = wl.colmajor_zeros(N, N, device="cuda")
        assert L.gs_density_matrix(h, C.data_ptr(), f.data_ptr(), P.data_ptr(), None) == 5      # GS_ERR_WORKSPACE: none set
        assert L.gs_density_matrix_static(h, C.data_ptr(), f.data_ptr(), P.data_ptr(), None) == gs.GS_OK   # warm-up: module and kernels loaded
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        for _ in range(2):
            P.zero_()
            assert L.gs_density_matrix_static(h, C.data_ptr(), f.data_ptr(), P.data_ptr(), None) == gs.GS_OK
            torch.cuda.synchronize()
            assert torch.equal(P, P_ref)
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0
    finally:
        L.gs_plan_destroy(h)


def test_static_scratch_rejects_sizes_beyond_the_array():
    from paper_2502_02460_b200 import gs
    for N, nev, cplx in [(2048, 1026, False), (1024 + 64, 1024, True), (4096, 1024, False)]:
        plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
        dt = torch.complex128 if cplx else torch.float64
        C, f = _inputs(N, nev, cplx, 3)
        P = wl.colmajor_empty(N, N, dtype=dt, device="cuda")
        P.fill_(9.0)
        before = plan.launch_count()
        with pytest.raises(gs.GsError) as e:
            plan.density_matrix_static(C, f, P)
        assert e.value.status == 5 and "GS_STATIC_SCRATCH_BYTES" in str(e.value)     # GS_ERR_WORKSPACE, sizes named
        assert plan.launch_count() == before and torch.all(P == 9.0)                 # nothing was enqueued
        plan.density_matrix(C, f, P)                                                 # the workspace path still takes it
        assert plan.last_info() == 0
        plan.close()


def test_static_scratch_argument_errors_and_nev_zero():
    from paper_2502_02460_b200 import gs
    L = gs.lib()
    plan = gs.Plan(200, 0)
    P = wl.colmajor_empty(200, 200, device="cuda")
    P.fill_(7.0)
    plan.density_matrix_static(None, None, P)
    torch.cuda.synchronize()
    low = torch.tril(torch.ones(200, 200, dtype=torch.bool, device="cuda"), -1)
    assert torch.all(torch.triu(P) == 0) and torch.all(P[low] == 7.0)
    plan.close()
    plan = gs.Plan(64, 8)
    C, f = _inputs(64, 8, False, 1)
    P = wl.colmajor_empty(64, 64, device="cuda")
    assert L.gs_density_matrix_static(None, C.data_ptr(), f.data_ptr(), P.data_ptr(), None) == 1
    assert L.gs_density_matrix_static(plan._h, C.data_ptr(), f.data_ptr(), None, None) == 1
    assert L.gs_density_matrix_static(plan._h, None, f.data_ptr(), P.data_ptr(), None) == 1
    assert L.gs_density_matrix_static(plan._h, C.data_ptr(), f.data_ptr(), P.data_ptr() + 8, None) == 1
    assert L.gs_density_matrix_static(plan._h, P.data_ptr() + 64, f.data_ptr(), P.data_ptr(), None) == 1   # overlap
    plan.close()
