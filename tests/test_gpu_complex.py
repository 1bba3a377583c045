"""Parity of the complex128 (Hermitian) CUDA path against the CPU oracle and against the real path.

"A^T corresponds to the transpose or conjugate-transpose of a real- or complex-valued matrix"
(PAPER.md:67): S = U^H U, H~ = U^-H H U^-1, C = U^-1 C~ (no conjugation).  Inputs: BASELINE.json
config 3's recipe (real pencil times the phase exp(i k (x_i - x_j)), k = 0.7) at sizes the oracle
finishes in seconds, and at config 3's full size (N = 8192) with the leading-block pin, invariants
and the phase identity U' = U o P, V' = V o P, H~' = H~ o P against the REAL GPU path.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2502_02460_b200 import metrics as M
from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SIZES = [1, 2, 3, 5, 17, 63, 64, 65, 100, 128, 130, 200, 257, 384, 520]


def _gs():
    from paper_2502_02460_b200 import gs
    return gs


def _dev(a):
    return wl.to_colmajor(torch.from_numpy(np.ascontiguousarray(a)).cuda())


def _z(N, M_=None):
    return wl.colmajor_empty(N, N if M_ is None else M_, dtype=torch.complex128, device="cuda")


@pytest.mark.parametrize("N", SIZES)
def test_complex_stages_against_oracle(N):
    gs = _gs()
    p = wl.small_pencil(N, seed=N, complex=True)
    nev = max(1, (2 * N) // 3)
    H, S = p.H.numpy(), p.S.numpy()
    U_o = oracle.cholesky(S)
    V_o = oracle.invert_upper(U_o)
    Ht_o = oracle.to_standard(H, V_o)
    plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128)

    garbage = np.tril(np.full((N, N), 123.0 - 7.0j), -1)
    U_g = _dev(np.triu(S) + garbage)               # strictly-lower part must never be read
    plan.cholesky(U_g)
    assert plan.last_info() == 0
    assert M.rel_frob_upper(U_g.cpu(), U_o) <= M.TOL_FROB
    assert M.strictly_lower_max(U_g.cpu()) == 0.0
    assert torch.all(torch.diagonal(U_g).imag == 0) and torch.all(torch.diagonal(U_g).real > 0)

    V_g = _z(N)
    V_g.fill_(99.0)
    plan.invert_triangular(_dev(U_o + garbage), V_g)
    assert plan.last_info() == 0
    assert M.rel_frob_upper(V_g.cpu(), V_o) <= M.TOL_FROB
    assert M.strictly_lower_max(V_g.cpu()) == 0.0

    Ht_g = _z(N)
    Ht_g.fill_(-3.0)
    plan.to_standard(_dev(H), _dev(V_o + garbage), Ht_g)
    assert plan.last_info() == 0
    assert M.rel_frob_upper(Ht_g.cpu(), Ht_o) <= M.TOL_FROB
    assert torch.all(torch.diagonal(Ht_g).imag == 0)          # Hermitian result: exactly real diagonal
    if N > 1:
        low = Ht_g.cpu()[torch.tril(torch.ones(N, N, dtype=torch.bool), -1)]
        assert torch.all(low == -3.0)

    Ct = wl.dense_rhs(N, nev, seed=N, complex=True)
    C_o = oracle.backtransform(V_o, Ct.numpy())
    C_g = _z(N, nev)
    plan.backtransform(_dev(V_o + garbage), wl.to_colmajor(Ct.cuda()), C_g)
    assert plan.last_info() == 0
    assert M.rel_frob(C_g.cpu(), C_o) <= M.TOL_FROB
    plan.close()


@pytest.mark.parametrize("N", [64, 256, 700])
def test_complex_chained_path_and_eigen_metrics(N):
    gs = _gs()
    p = wl.small_pencil(N, seed=2000 + N, complex=True)
    H, S = p.H.numpy(), p.S.numpy()
    U_o = oracle.cholesky(S)
    V_o = oracle.invert_upper(U_o)
    Ht_o = oracle.to_standard(H, V_o)
    plan, U, Uinv, Ht = gs.generalized_to_standard(wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda()), N)
    assert M.rel_frob_upper(U.cpu(), U_o) <= M.TOL_FROB
    assert M.rel_frob_upper(Uinv.cpu(), V_o) <= M.TOL_FROB
    assert M.rel_frob_upper(Ht.cpu(), Ht_o) <= M.TOL_FROB
    if N <= 256:
        eps, Q, _ = oracle.jacobi(oracle.hermitian_from_upper(Ht.cpu().numpy()))
        C = _z(N)
        plan.backtransform(Uinv, _dev(np.asfortranarray(Q)), C)
        plan.last_info()
        assert M.eig_residual(H, S, C.cpu().numpy(), eps) <= M.TOL_RESIDUAL
        assert M.s_orthonormality(S, C.cpu().numpy()) <= M.TOL_SORTH
    plan.close()


def test_complex_not_positive_definite():
    gs = _gs()
    N = 200
    p = wl.small_pencil(N, seed=4, complex=True)
    S = p.S.numpy().copy()
    S[150, 150] = -1.0
    plan = gs.Plan(N, N, dtype=gs.GS_COMPLEX128)
    plan.cholesky(_dev(S))
    with pytest.raises(gs.GsError) as e:
        plan.last_info()
    assert e.value.status == 2 and e.value.info == 151
    plan.close()


@pytest.mark.slow
def test_complex_n4160_all_three_potrf_tiers_full_oracle():
    """65 complex blocks of 64: every panel tier of the POTRF schedule at its default width, look-ahead on
    two streams, long-k inversion levels and HER2K -- against the WHOLE complex oracle, element by element."""
    gs = _gs()
    N, nev = 4160, 1040
    p = wl.make_pencil(N, wl.scaled_box(N), wl.BASE_SEED + 78, complex=True, device="cuda")
    plan, U, V, Ht = gs.generalized_to_standard(p.H, p.S, nev)
    H, S = p.H.cpu().numpy(), p.S.cpu().numpy()
    U_o = oracle.cholesky(S)
    V_o = oracle.invert_upper(U_o)
    Ht_o = oracle.to_standard(H, V_o)
    for name, X, X_o in (("U", U, U_o), ("Uinv", V, V_o), ("Htilde", Ht, Ht_o)):
        assert M.rel_frob_upper(X.cpu(), X_o) <= M.TOL_FROB, name
        d = torch.triu(X.cpu() - torch.from_numpy(X_o)).abs().max().item()
        assert d <= 1e-11 * np.abs(X_o).max(), name
    Ct = wl.dense_rhs(N, nev, seed=13, complex=True, device="cuda")
    Cg = _z(N, nev)
    plan.backtransform(_dev(V_o), Ct, Cg)
    plan.last_info()
    assert M.rel_frob(Cg.cpu(), oracle.backtransform(V_o, Ct.cpu().numpy())) <= M.TOL_FROB
    plan.close()


def test_config3_full_size_leading_block_phase_identity_and_invariants():
    """BASELINE config 3 (N = 8192 complex Hermitian, nev = 2048), in the configuration bench.py times."""
    gs = _gs()
    cfg = wl.CONFIGS[3]
    N, nev, k = cfg.N, cfg.nev, 2048      # 32 complex blocks: first panel + look-ahead iterations
    dev = "cuda"
    pz = wl.make_pencil(N, cfg.box, cfg.seed, complex=True, device=dev)
    plan, U, V, Ht = gs.generalized_to_standard(pz.H, pz.S, nev)
    Ct = wl.dense_rhs(N, nev, seed=3, complex=True, device=dev)
    C = _z(N, nev)
    plan.backtransform(V, Ct, C)
    assert plan.last_info() == 0

    # leading-block pin against the complex oracle
    U_o = oracle.cholesky(pz.S[:k, :k].cpu().numpy())
    V_o = oracle.invert_upper(U_o)
    Ht_o = oracle.to_standard(pz.H[:k, :k].cpu().numpy(), V_o)
    assert M.rel_frob_upper(U[:k, :k].cpu(), U_o) <= M.TOL_FROB
    assert M.rel_frob_upper(V[:k, :k].cpu(), V_o) <= M.TOL_FROB
    assert M.rel_frob_upper(Ht[:k, :k].cpu(), Ht_o) <= M.TOL_FROB
    # trailing rows of C nest
    C_o = oracle.backtransform(V[N - 512:, N - 512:].cpu().numpy(), Ct[N - 512:, :32].cpu().numpy())
    assert M.rel_frob(C[N - 512:, :32].cpu(), C_o) <= M.TOL_FROB
    # far corner of step 2: trailing blocks of an upper inverse nest
    Vf_o = oracle.invert_upper(U[N - 1024:, N - 1024:].cpu().numpy())
    assert M.rel_frob_upper(V[N - 1024:, N - 1024:].cpu(), Vf_o) <= M.TOL_FROB
    # sampled entries H~_ij = v_i^H H v_j from the definition (CPU, extended precision), far half of the matrix
    rng = np.random.default_rng(21)
    Hh = pz.H.cpu().numpy()
    for _ in range(4):
        j = int(rng.integers(N // 2, N))
        vj = V[:j + 1, j].cpu().numpy().astype(np.clongdouble)
        t = np.concatenate([Hh[r0:min(j + 1, r0 + 1024), :j + 1].astype(np.clongdouble) @ vj for r0 in range(0, j + 1, 1024)])
        for _ in range(8):
            i = int(rng.integers(max(0, j - N // 2), j + 1))
            vi = V[:i + 1, i].cpu().numpy().astype(np.clongdouble)
            ref = complex(np.dot(np.conj(vi), t[:i + 1]))
            scale = float(np.linalg.norm(vi.astype(np.complex128)) * np.linalg.norm(t[:i + 1].astype(np.complex128)))
            assert abs(Ht[i, j].item() - ref) <= 1e-11 * scale, (i, j)

    # invariants at full size (plain torch complex128 on the device, off the hot path)
    assert torch.tril(U, -1).abs().max().item() == 0.0 and torch.tril(V, -1).abs().max().item() == 0.0
    assert ((U.conj().t() @ U - pz.S).norm() / pz.S.norm()).item() <= 1e-13
    R = U @ V
    R.diagonal().sub_(1.0)
    assert R.norm().item() / N ** 0.5 <= 1e-11
    Hs = torch.triu(Ht) + torch.triu(Ht, 1).conj().t()
    assert ((U.conj().t() @ (Hs @ U) - pz.H).norm() / pz.H.norm()).item() <= 1e-10
    assert ((C - V @ Ct).norm() / C.norm()).item() <= 1e-12
    del R, Hs

    # phase identity (SURVEY 8(c) P-phase): the complex pencil is D S D^H, D H D^H with D = diag(exp(i k x)),
    # hence U' = U o P, V' = V o P, H~' = H~ o P where unprimed = the REAL path on the same points / seed.
    pr = wl.make_pencil(N, cfg.box, cfg.seed, complex=False, device=dev)
    plan_r, Ur, Vr, Htr = gs.generalized_to_standard(pr.H, pr.S, nev)
    P = wl.phase_factor(pr.r[:, 0])
    for Z, X in ((U, Ur), (V, Vr), (Ht, Htr)):
        ref = torch.triu(X.to(torch.complex128) * P)
        assert (torch.triu(Z) - ref).norm().item() / ref.norm().item() <= 1e-11
    plan.close()
    plan_r.close()
