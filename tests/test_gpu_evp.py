"""NEXT-4: the standard eigenproblem H~ C~ = C~ eps on the GPU (gs_evp_tridiagonalize / gs_evp_tridiag_solve /
gs_evp_backtransform / gs_standard_eigh; Table 1 "Tridiag. / Solve / Back") against
the CPU oracle.

What is unique is compared element by element: the eigenvalues (oracle: cyclic Jacobi, O5) and the eigenvalues of the
intermediate tridiagonal matrix (oracle: Sturm bisection, O8/O9).  C~ is unique only up to a phase per column and up
to rotations inside clusters, so it is checked for VALIDITY, completely:
  * residual      ||H~ C~ - C~ eps||_F <= 10 N u ||H~||_F
  * orthonormal   ||C~^H C~ - I||_max <= 1e-12
  * lowest nev, none missing: the inertia of H~ - sigma I (oracle O10: LDL^H without pivoting, independent of every
    tridiagonalisation) just above eps_nev counts exactly nev eigenvalues below sigma.
Inputs: H~ of the BASELINE recipe (workloads.py) as the ORACLE forms it, handed over as an upper triangle with a
NaN-poisoned strictly-lower part (the GPU path must not read it); plus special tridiagonal matrices for the solve
stage (closed-form spectrum, close pairs, exact multiplicities, decoupled blocks).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2502_02460_b200 import metrics as M
from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu
U_ROUND = 2.0 ** -53


def _gs():
    from paper_2502_02460_b200 import gs
    return gs


def _dev(a):
    return wl.to_colmajor(torch.from_numpy(np.ascontiguousarray(a)).cuda())


def _htilde(N, cplx, seed):
    p = wl.small_pencil(N, seed=seed, complex=cplx)
    V = oracle.invert_upper(oracle.cholesky(p.S.numpy()))
    Ht = oracle.hermitian_from_upper(oracle.to_standard(p.H.numpy(), V))
    return p, V, Ht


def _upper_poisoned(Ht):
    A = np.array(Ht, copy=True)
    A[np.tril_indices(A.shape[0], -1)] = np.nan
    return _dev(A)


def _validity(Ht, eps, Ct, nev):
    """residual, orthonormality and the inertia count: returns nothing, asserts."""
    N = Ht.shape[0]
    Ct = Ct.cpu().numpy()
    eps = eps.cpu().numpy()
    assert np.all(np.diff(eps) >= 0)
    R = Ht @ Ct - Ct * eps[None, :]
    assert np.linalg.norm(R) <= 10.0 * N * U_ROUND * np.linalg.norm(Ht) + 1e-300
    G = Ct.conj().T @ Ct - np.eye(nev)
    assert np.abs(G).max() <= 1e-12 if nev else True


def _sigma_above(eps_all, nev):
    """a shift strictly between eigenvalue nev-1 and eigenvalue nev of the full spectrum (or above the top)"""
    N = len(eps_all)
    if nev >= N:
        return eps_all[-1] + 1.0 + abs(eps_all[-1])
    gap = eps_all[nev] - eps_all[nev - 1]
    assert gap > 1e-9 * max(1.0, np.abs(eps_all).max()), "test input has a (near) degenerate pair at the cut"
    return eps_all[nev - 1] + 0.5 * gap


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N", [1, 2, 3, 17, 100, 257, 512])
def test_standard_eigh_against_jacobi_with_inertia_count(N, cplx):
    gs = _gs()
    _, _, Ht = _htilde(N, cplx, seed=300 + N)
    eps_o, _, _ = oracle.jacobi(Ht)
    scale = max(1.0, np.abs(eps_o).max())
    for nev in sorted({N, max(1, N // 3)}):
        plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
        # the intermediate tridiagonal matrix has the spectrum of H~ (oracle: Sturm bisection on the GPU's d, e)
        A = _upper_poisoned(Ht)
        d, e, tau = plan.evp_tridiagonalize(A)
        assert plan.last_info() == 0
        t_eigs = oracle.tridiag_eigenvalues(d.cpu().numpy(), e.cpu().numpy())
        assert np.abs(t_eigs - eps_o).max() <= 1e-12 * scale
        # reflector matrix: zeros on and below the first superdiagonal's unit entries
        if N > 1:
            Ar = A.cpu().numpy()
            assert np.all(Ar[np.tril_indices(N, 0)] == 0) and np.all(np.diag(Ar, 1)[np.abs(tau.cpu().numpy()[1:]) > 0] == 1)
        # the three stages in a row
        eps, Ct = plan.standard_eigh(_upper_poisoned(Ht))
        assert plan.last_info() == 0
        assert np.abs(eps.cpu().numpy() - eps_o[:nev]).max() <= 1e-12 * scale
        _validity(Ht, eps, Ct, nev)
        if N > 1:
            sigma = _sigma_above(eps_o, nev)
            assert oracle.inertia_count(Ht, sigma) == nev                  # they are the LOWEST nev, none missing
            assert int((eps.cpu().numpy() < sigma).sum()) == nev
        plan.close()


def _solve(d, e, nev=None):
    gs = _gs()
    N = len(d)
    nev = N if nev is None else nev
    plan = gs.Plan(N, nev)
    eps, Z = plan.evp_tridiag_solve(torch.from_numpy(np.asarray(d, dtype=np.float64)).cuda(),
                                    torch.from_numpy(np.asarray(e, dtype=np.float64)).cuda())
    assert plan.last_info() == 0
    plan.close()
    return eps.cpu().numpy(), Z.cpu().numpy()


def _check_tridiag_pairs(d, e, eps, Z, tol_eig=1e-13):
    N, nev = len(d), len(eps)
    T = np.diag(d) + (np.diag(e, 1) + np.diag(e, -1) if N > 1 else 0.0)
    ref = oracle.tridiag_eigenvalues(d, e, nev)
    scale = max(np.abs(d).max(), np.abs(e).max() if N > 1 else 0.0, 1e-300)
    assert np.abs(eps - ref).max() <= tol_eig * scale * max(1.0, np.log2(N + 1))
    assert np.linalg.norm(T @ Z - Z * eps[None, :]) <= 10.0 * N * U_ROUND * max(np.linalg.norm(T), 1e-300)
    assert np.abs(Z.T @ Z - np.eye(nev)).max() <= 1e-12


@pytest.mark.parametrize("N", [5, 128, 129, 300, 1000])
def test_solve_closed_form_spectrum(N):
    d, e = 2.0 * np.ones(N), -np.ones(N - 1)
    eps, Z = _solve(d, e)
    ref = 2.0 - 2.0 * np.cos(np.arange(1, N + 1) * np.pi / (N + 1))
    assert np.abs(eps - ref).max() <= 1e-13 * 4.0 * np.log2(N + 1)
    _check_tridiag_pairs(d, e, eps, Z)
    k = max(1, N // 4)
    eps_k, Z_k = _solve(d, e, k)                       # lowest-nev form returns the same lowest pairs
    assert np.abs(eps_k - ref[:k]).max() <= 1e-13 * 4.0 * np.log2(N + 1)
    _check_tridiag_pairs(d, e, eps_k, Z_k)


def test_solve_wilkinson_close_pairs():
    m = 200                                             # W(401)+: the top eigenvalues agree pairwise to rounding
    d = np.abs(np.arange(-m, m + 1)).astype(float)
    e = np.ones(2 * m)
    eps, Z = _solve(d, e)
    _check_tridiag_pairs(d, e, eps, Z)


def test_solve_exact_multiplicities_and_decoupled_blocks():
    rng = np.random.default_rng(3)
    N = 700
    # (a) a multiple of the identity: everything deflates at every level
    eps, Z = _solve(3.0 * np.ones(N), np.zeros(N - 1))
    assert np.array_equal(eps, 3.0 * np.ones(N)) and np.abs(Z.T @ Z - np.eye(N)).max() <= 1e-14
    # (b) zero couplings exactly at the cut points (rho = 0) and tiny ones elsewhere
    d = rng.standard_normal(N)
    e = rng.standard_normal(N - 1)
    e[63::64] = 0.0                                     # (the leaves are 64 wide: every cut of every level)
    e[300] = 1e-200
    eps, Z = _solve(d, e)
    _check_tridiag_pairs(d, e, eps, Z)
    # (c) repeated diagonal blocks: the same 2 x 2 block glued by weak couplings -> clusters of nearly equal eigenvalues
    d = np.tile([1.0, 2.0], N // 2)
    e = np.tile([0.5, 1e-9], N // 2)[:N - 1]
    eps, Z = _solve(d, e)
    _check_tridiag_pairs(d, e, eps, Z)
    # (d) graded
    d = 10.0 ** rng.uniform(-8, 4, N) * rng.choice([-1.0, 1.0], N)
    e = 10.0 ** rng.uniform(-10, 2, N - 1)
    eps, Z = _solve(d, e, N // 2)
    _check_tridiag_pairs(d, e, eps, Z)


@pytest.mark.parametrize("glue", [1e-4, 1e-8, 1e-14])
def test_solve_glued_wilkinson(glue):
    """Copies of W21+ glued by a small coupling: clusters of nearly equal eigenvalues whose secular equations have roots
    next to their poles and nearly coincident poles -- the hard case for the root finder (regula falsi on f |mu| with a
    bisection safeguard, csrc/evp_dc.cuh) and for the deflation test."""
    copies, m = 24, 10
    d = np.tile(np.abs(np.arange(-m, m + 1)).astype(float), copies)
    e = np.ones(len(d) - 1)
    e[2 * m::2 * m + 1] = glue
    eps, Z = _solve(d, e)
    _check_tridiag_pairs(d, e, eps, Z)
    eps_k, Z_k = _solve(d, e, len(d) // 3)
    _check_tridiag_pairs(d, e, eps_k, Z_k)


def test_stage_calls_chain_like_standard_eigh():
    """The three stage calls one by one give what gs_standard_eigh gives (same kernels, same order: bit for bit)."""
    gs = _gs()
    N, nev = 400, 130
    _, _, Ht = _htilde(N, False, seed=9)
    plan = gs.Plan(N, nev)
    A = _upper_poisoned(Ht)
    d, e, tau = plan.evp_tridiagonalize(A)
    eps, Z = plan.evp_tridiag_solve(d, e)
    Ct = plan.evp_backtransform(A, Z)
    eps2, Ct2 = plan.standard_eigh(_upper_poisoned(Ht))
    assert plan.last_info() == 0
    assert torch.equal(eps, eps2) and torch.equal(Ct, Ct2)
    plan.close()


def test_nev_zero_and_single_eigenpair():
    """nev = 0: the stages run (tridiagonalisation, eigenvalue-free solve) and return nothing; nev = 1: the lowest pair."""
    gs = _gs()
    N = 200
    _, _, Ht = _htilde(N, False, seed=12)
    eps_o, _, _ = oracle.jacobi(Ht)
    plan0 = gs.Plan(N, 0)
    eps, Ct = plan0.standard_eigh(_upper_poisoned(Ht))
    assert plan0.last_info() == 0 and eps.numel() == 0 and Ct.shape == (N, 0)
    plan0.close()
    plan1 = gs.Plan(N, 1)
    eps, Ct = plan1.standard_eigh(_upper_poisoned(Ht))
    assert plan1.last_info() == 0
    assert abs(eps.item() - eps_o[0]) <= 1e-12 * np.abs(eps_o).max()
    _validity(Ht, eps, Ct, 1)
    plan1.close()


def test_config0_end_to_end_without_any_library_eigensolver():
    """BASELINE config 0 through the GPU path ONLY -- reduction, standard eigensolver, back-transformation -- against
    the three acceptance tolerances and the oracle's eigenvalues (no torch.linalg anywhere)."""
    gs = _gs()
    cfg = wl.CONFIGS[0]
    p = wl.make_config(0)
    H, S = p.H.numpy(), p.S.numpy()
    ref = oracle.generalized_eigh(H, S, cfg.nev)
    plan, U, Uinv, Ht = gs.generalized_to_standard(_dev(H), _dev(S), cfg.nev)
    eps, Ct = plan.standard_eigh(Ht)
    C = wl.colmajor_empty(cfg.N, cfg.nev, device="cuda")
    plan.backtransform(Uinv, Ct, C)
    assert plan.last_info() == 0
    Cn, en = C.cpu().numpy(), eps.cpu().numpy()
    assert M.eig_residual(H, S, Cn, en) <= M.TOL_RESIDUAL
    assert M.s_orthonormality(S, Cn) <= M.TOL_SORTH
    np.testing.assert_allclose(en, ref["eps"], rtol=0, atol=1e-9 * np.abs(ref["eps"]).max())
    plan.close()


def _generalized_on_gpu(cfg):
    gs = _gs()
    p = wl.make_pencil(cfg.N, cfg.box, cfg.seed, complex=cfg.complex, device="cuda")
    plan, U, V, Ht = gs.generalized_to_standard(p.H, p.S, cfg.nev)
    Hs = torch.triu(Ht) + torch.triu(Ht, 1).conj().t()           # kept for the checks (standard_eigh destroys Ht)
    Hs.diagonal().copy_(Ht.diagonal().real.to(Hs.dtype))
    eps, Ct = plan.standard_eigh(Ht)
    C = wl.colmajor_empty(cfg.N, cfg.nev, dtype=p.H.dtype, device="cuda")
    plan.backtransform(V, Ct, C)
    assert plan.last_info() == 0
    return plan, p, Hs, eps, Ct, C


@pytest.mark.slow
def test_config1_generalized_solve_with_oracle_inertia():
    cfg = wl.CONFIGS[1]
    plan, p, Hs, eps, Ct, C = _generalized_on_gpu(cfg)
    assert M.eig_residual(p.H, p.S, C, eps) <= M.TOL_RESIDUAL
    assert M.s_orthonormality(p.S, C) <= M.TOL_SORTH
    R = Hs @ Ct - Ct * eps.unsqueeze(0)
    assert R.norm().item() <= 10.0 * cfg.N * U_ROUND * Hs.norm().item()
    en = eps.cpu().numpy()
    sigma = en[-1] + 1e-6 * max(1.0, abs(en[-1]))
    # lowest nev, none missing: LDL^T inertia of H~ - sigma I on the CPU (oracle O10), ~20 s at N = 4096
    assert oracle.inertia_count(Hs.cpu().numpy(), sigma) == cfg.nev
    plan.close()


@pytest.mark.slow
@pytest.mark.parametrize("index", [2, 3])
def test_configs_2_and_3_generalized_solve(index):
    """Headline size (N = 16384 real) and the Hermitian config (N = 8192 complex): the acceptance metrics on the
    ORIGINAL pencil, and -- the oracle's O(N^3) inertia count takes too long here -- the count of eigenvalues below
    sigma from an off-path library eigenvalue routine (torch.linalg.eigvalsh, never part of the path)."""
    cfg = wl.CONFIGS[index]
    plan, p, Hs, eps, Ct, C = _generalized_on_gpu(cfg)
    assert M.eig_residual(p.H, p.S, C, eps) <= M.TOL_RESIDUAL
    assert M.s_orthonormality(p.S, C) <= M.TOL_SORTH
    R = Hs @ Ct - Ct * eps.to(Ct.dtype).unsqueeze(0)
    assert R.norm().item() <= 10.0 * cfg.N * U_ROUND * Hs.norm().item()
    del R, Ct, C
    torch.cuda.empty_cache()
    lam = torch.linalg.eigvalsh(Hs)
    assert (lam[:cfg.nev] - eps).abs().max().item() <= 1e-9 * lam.abs().max().item()
    sigma = 0.5 * (lam[cfg.nev - 1] + lam[cfg.nev]).item()
    assert int((eps < sigma).sum().item()) == cfg.nev and int((lam < sigma).sum().item()) == cfg.nev
    plan.close()


@pytest.mark.parametrize("cplx,N,nev", [(False, 256, 256), (False, 300, 77), (True, 150, 150), (False, 1, 1)])
def test_generalized_eigh_one_call(cplx, N, nev):
    """gs_generalized_eigh = the five calls in a row: eigenvalues against the oracle's chain (unblocked
    Cholesky, substitution, triple loops, Jacobi), eigenvectors by the residual of the ORIGINAL pencil and S-orthonormality."""
    gs = _gs()
    p = wl.small_pencil(N, seed=900 + N, complex=cplx)
    H, S = p.H.numpy(), p.S.numpy()
    V_o = oracle.invert_upper(oracle.cholesky(S))
    eps_o, _, _ = oracle.jacobi(oracle.to_standard(H, V_o))
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    Hd, Sd = wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda())
    S_before = Sd.clone()
    eps, C, U, Uinv = plan.generalized_eigh(Hd, Sd)
    assert plan.last_info() == 0
    assert torch.equal(Sd, S_before)
    scale = max(1.0, np.abs(eps_o).max())
    assert np.abs(eps.cpu().numpy() - eps_o[:nev]).max() <= 1e-11 * scale
    assert M.eig_residual(H, S, C.cpu().numpy(), eps.cpu().numpy()) <= M.TOL_RESIDUAL
    assert M.s_orthonormality(S, C.cpu().numpy()) <= M.TOL_SORTH
    assert M.rel_frob_upper(U.cpu(), oracle.cholesky(S)) <= M.TOL_FROB and M.rel_frob_upper(Uinv.cpu(), V_o) <= M.TOL_FROB
    # argument errors come back before anything is enqueued
    L = gs.lib()
    assert L.gs_generalized_eigh(None, Hd.data_ptr(), U.data_ptr(), Uinv.data_ptr(), Hd.data_ptr(), C.data_ptr(), eps.data_ptr(), C.data_ptr(), None) == 1
    assert L.gs_generalized_eigh(plan._h, Hd.data_ptr(), U.data_ptr(), Uinv.data_ptr(), Hd.data_ptr(), C.data_ptr(), eps.data_ptr(), C.data_ptr(), None) == 1   # C~ = C
    plan.close()


@pytest.mark.parametrize("N", [1, 2, 17, 257, 1000])
def test_tridiag_eigenvalues_by_bisection_against_the_oracle(N):
    """gs_evp_tridiag_eigenvalues (eigenvalues only: PAPER.md:67) against the oracle's Sturm bisection (O8/O9, pinned by the
    closed-form spectrum of tridiag(-1, 2, -1)) and, for that matrix, against the closed form itself; partial counts."""
    gs = _gs()
    rng = np.random.default_rng(N)
    cases = {"toeplitz": (np.full(N, 2.0), np.full(max(N - 1, 0), -1.0)),
             "random": (rng.standard_normal(N), rng.standard_normal(max(N - 1, 0))),
             "wilkinson": (np.abs(np.arange(N) - (N - 1) / 2.0), np.ones(max(N - 1, 0))),
             "graded": (10.0 ** -np.linspace(0, 8, N), 1e-3 * 10.0 ** -np.linspace(0, 8, max(N - 1, 1))[:max(N - 1, 0)]),
             "decoupled": (rng.standard_normal(N), np.where(np.arange(max(N - 1, 0)) % 5 == 4, 0.0, 0.3))}
    plan = gs.Plan(N, N)
    for name, (d, e) in cases.items():
        ref = oracle.tridiag_eigenvalues(d, e)
        dd, ee = torch.from_numpy(np.ascontiguousarray(d)).cuda(), torch.from_numpy(np.ascontiguousarray(e)).cuda()
        lam = plan.evp_tridiag_eigenvalues(dd, ee).cpu().numpy()
        assert plan.last_info() == 0
        scale = max(1.0, np.abs(ref).max())
        assert np.abs(lam - ref).max() <= 1e-13 * scale, name
        assert np.all(np.diff(lam) >= 0)
        if name == "toeplitz":
            exact = 2.0 - 2.0 * np.cos(np.arange(1, N + 1) * np.pi / (N + 1))
            assert np.abs(lam - exact).max() <= 1e-13 * 4.0
        k = max(1, N // 3)
        part = plan.evp_tridiag_eigenvalues(dd, ee, count=k).cpu().numpy()
        assert np.array_equal(part, lam[:k])
    assert plan.evp_tridiag_eigenvalues(dd, ee, count=0).numel() == 0
    L = gs.lib()
    assert L.gs_evp_tridiag_eigenvalues(plan._h, dd.data_ptr(), ee.data_ptr() if N > 1 else None, N + 1, dd.data_ptr(), None) == 1
    assert L.gs_evp_tridiag_eigenvalues(plan._h, None, None, 1, dd.data_ptr(), None) == 1
    plan.close()


@pytest.mark.parametrize("cplx,N", [(False, 257), (True, 150), (False, 512)])
def test_standard_eigenvalues_only(cplx, N):
    """gs_standard_eigenvalues = tridiagonalisation + bisection: against the oracle's Jacobi on the same H~ and against the
    eigenvalues gs_standard_eigh (divide and conquer) returns."""
    gs = _gs()
    _, _, Ht = _htilde(N, cplx, seed=700 + N)
    eps_o, _, _ = oracle.jacobi(Ht)
    scale = max(1.0, np.abs(eps_o).max())
    plan = gs.Plan(N, N, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    lam = plan.standard_eigenvalues(_upper_poisoned(Ht)).cpu().numpy()
    assert plan.last_info() == 0
    assert np.abs(lam - eps_o).max() <= 1e-12 * scale
    eps_dc, _ = plan.standard_eigh(_upper_poisoned(Ht))
    assert np.abs(lam - eps_dc.cpu().numpy()).max() <= 1e-12 * scale
    few = plan.standard_eigenvalues(_upper_poisoned(Ht), count=7).cpu().numpy()
    assert np.abs(few - eps_o[:7]).max() <= 1e-12 * scale
    plan.close()
