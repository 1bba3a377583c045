"""Pins for the CPU oracle (oracle/gs_oracle.c) against what the paper and mathematics fix.

The paper prints no worked numerical example and no error bound, so every pin is
mathematical: closed forms, special cases that reduce to library routines, brute force on tiny N,
and invariants.  Each test is chosen so that a plausible slip in the oracle (dropped term, wrong
sign or index, transposed operand, missing conjugate) fails it.  None of these tests touches the
CUDA path.
"""
import math

import numpy as np
import pytest
import scipy.linalg as sla

import oracle
from paper_2502_02460_b200 import workloads as wl

U52 = 2.0 ** -52


def _rand_spd_pencil(N, seed, cplx):
    rng = np.random.default_rng(seed)
    if cplx:
        A = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
        B = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    else:
        A = rng.standard_normal((N, N))
        B = rng.standard_normal((N, N))
    S = A.conj().T @ A + N * np.eye(N)
    H = B + B.conj().T
    return H, S


# ---------------------------------------------------------------------------------------------
# P-diag: diagonal H, S  =>  U = diag(sqrt S_ii), V = diag(1/sqrt S_ii), H~ = diag(H_ii/S_ii),
# eps_i = H_ii / S_ii (sorted), C = e_i / sqrt(S_ii)      (BASELINE.json north_star)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [1, 7, 64])
@pytest.mark.parametrize("cplx", [False, True])
def test_diagonal_pencil(N, cplx):
    rng = np.random.default_rng(N)
    s = rng.uniform(0.5, 3.0, N)
    h = rng.uniform(-2.0, 2.0, N)
    dt = np.complex128 if cplx else np.float64
    out = oracle.generalized_eigh(np.diag(h).astype(dt), np.diag(s).astype(dt))
    np.testing.assert_allclose(out["U"], np.diag(np.sqrt(s)), rtol=1e-15, atol=0)
    np.testing.assert_allclose(out["V"], np.diag(1 / np.sqrt(s)), rtol=2e-15, atol=0)
    np.testing.assert_allclose(out["Ht"], np.diag(h / s), rtol=4e-15, atol=0)
    order = np.argsort(h / s, kind="stable")
    np.testing.assert_allclose(out["eps"], (h / s)[order], rtol=4e-15, atol=0)
    Cexp = np.zeros((N, N))
    Cexp[order, np.arange(N)] = 1 / np.sqrt(s[order])
    np.testing.assert_allclose(np.abs(out["C"]), Cexp, rtol=4e-15, atol=0)


# ---------------------------------------------------------------------------------------------
# P-ident: S = I reduces to the standard problem: U = V = I, H~ = H exactly, C = C~.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cplx", [False, True])
def test_identity_overlap(cplx):
    N = 50
    H, _ = _rand_spd_pencil(N, 3, cplx)
    out = oracle.generalized_eigh(H, np.eye(N, dtype=H.dtype))
    assert np.array_equal(out["U"], np.eye(N))
    assert np.array_equal(out["V"], np.eye(N))
    assert np.array_equal(out["Ht"], H)
    assert np.array_equal(out["C"], out["Ct"])
    np.testing.assert_allclose(out["eps"], np.linalg.eigvalsh(H), rtol=0, atol=1e-13 * np.abs(H).sum())


# ---------------------------------------------------------------------------------------------
# P-tridiag: S = tridiag(-1, 2, -1) has closed forms for everything with a DENSE U^-1 (1-based):
#   U_ii = sqrt((i+1)/i), U_{i,i+1} = -sqrt(i/(i+1));   V_ij = i / sqrt(j (j+1)),  i <= j
#   H = c S + d I  =>  H~ = c I + d V^T V,  (V^T V)_ij = m(m+1)(2m+1)/6 / sqrt(i(i+1) j(j+1)), m = min(i,j)
#   eps_k = c + d / sigma_k,  sigma_k = 2 - 2 cos(k pi / (N+1));  C_k = v_k / sqrt(sigma_k),
#   v_k(i) = sqrt(2/(N+1)) sin(i k pi/(N+1)).
# A transposed operand, a wrong loop bound or a sign error anywhere in O1-O4 breaks these.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [2, 10, 100, 150])
def test_tridiagonal_closed_forms(N):
    c, d = -0.5, 0.3
    S = 2 * np.eye(N) - np.eye(N, k=1) - np.eye(N, k=-1)
    H = c * S + d * np.eye(N)
    i = np.arange(1, N + 1, dtype=np.float64)
    U_cf = np.diag(np.sqrt((i + 1) / i)) + np.diag(-np.sqrt(i[:-1] / (i[:-1] + 1)), k=1)
    V_cf = np.triu(i[:, None] / np.sqrt(i * (i + 1))[None, :])
    m = np.minimum(i[:, None], i[None, :])
    VtV = m * (m + 1) * (2 * m + 1) / 6 / np.sqrt((i * (i + 1))[:, None] * (i * (i + 1))[None, :])
    Ht_cf = c * np.eye(N) + d * VtV
    k = np.arange(1, N + 1)
    sigma = 2 - 2 * np.cos(k * math.pi / (N + 1))
    eps_cf = np.sort(c + d / sigma)

    U = oracle.cholesky(S)
    V = oracle.invert_upper(U)
    Ht = oracle.to_standard(H, V)
    assert np.abs(U - U_cf).max() <= 1e-14
    assert np.abs(V - V_cf).max() / np.abs(V_cf).max() <= 1e-13
    assert np.linalg.norm(Ht - Ht_cf) / np.linalg.norm(Ht_cf) <= 1e-12
    eps, Q, _ = oracle.jacobi(oracle.hermitian_from_upper(Ht))
    np.testing.assert_allclose(eps, eps_cf, rtol=1e-10, atol=0)
    C = oracle.backtransform(V, Q)
    # every column of C is +- v_k / sqrt(sigma_k) for the matching k (eigenvalues are simple)
    order = np.argsort(c + d / sigma, kind="stable")
    vk = np.sqrt(2 / (N + 1)) * np.sin(np.outer(i, k[order]) * math.pi / (N + 1)) / np.sqrt(sigma[order])
    sign = np.sign(np.sum(C * vk, axis=0))
    assert np.abs(C * sign - vk).max() <= 1e-8 * np.abs(vk).max()


# ---------------------------------------------------------------------------------------------
# P-2x2 / N=1: eps are the roots of det(S) e^2 - (h11 s22 + h22 s11 - 2 h12 s12) e + det(H) = 0.
# ---------------------------------------------------------------------------------------------
def test_two_by_two_quadratic_and_scalar():
    out = oracle.generalized_eigh(np.array([[-3.0]]), np.array([[4.0]]))
    assert out["eps"][0] == -0.75 and out["C"][0, 0] == 0.5
    H = np.array([[1.0, 0.4], [0.4, -2.0]])
    S = np.array([[2.0, 0.3], [0.3, 1.5]])
    a = np.linalg.det(S)
    b = -(H[0, 0] * S[1, 1] + H[1, 1] * S[0, 0] - 2 * H[0, 1] * S[0, 1])
    cc = np.linalg.det(H)
    roots = np.sort(np.roots([a, b, cc]).real)
    out = oracle.generalized_eigh(H, S)
    np.testing.assert_allclose(out["eps"], roots, rtol=1e-14)


# ---------------------------------------------------------------------------------------------
# P-brute: tiny N, independent of Cholesky and Jacobi.  Sylvester's law of inertia: since S is
# positive definite, #{eps_k < sigma} = number of negative pivots in the symmetric elimination
# (LDL^H, no pivoting) of H - sigma S.  Bisect each eps_k.  Written out in pure Python here.
# ---------------------------------------------------------------------------------------------
def _negative_pivots(A):
    A = np.array(A, dtype=np.complex128)
    n = A.shape[0]
    neg = 0
    for k in range(n):
        p = A[k, k].real
        if p == 0.0:
            p = 1e-300
        if p < 0:
            neg += 1
        for i in range(k + 1, n):
            f = A[i, k] / p
            for j in range(k + 1, n):
                A[i, j] -= f * A[k, j]
    return neg


def _bisect_eigs(H, S):
    n = H.shape[0]
    bound = np.abs(H).sum() / np.linalg.eigvalsh(S)[0] * 2 + 1
    out = []
    for k in range(n):
        lo, hi = -bound, bound
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if _negative_pivots(H - mid * S) > k:
                hi = mid
            else:
                lo = mid
            if hi - lo <= 1e-14 * max(1.0, abs(mid)):
                break
        out.append(0.5 * (lo + hi))
    return np.array(out)


@pytest.mark.parametrize("N", [1, 2, 3, 4, 6, 8])
@pytest.mark.parametrize("cplx", [False, True])
def test_bruteforce_inertia(N, cplx):
    H, S = _rand_spd_pencil(N, 100 + N, cplx)
    out = oracle.generalized_eigh(H, S)
    eps_bf = _bisect_eigs(H, S)
    np.testing.assert_allclose(out["eps"], eps_bf, rtol=1e-11, atol=1e-11)
    # and the defining equation H C = S C eps, C^H S C = I   (Eq. 2)
    C = out["C"]
    assert np.abs(H @ C - S @ C * out["eps"]).max() <= 1e-12 * np.abs(H).sum()
    assert np.abs(C.conj().T @ S @ C - np.eye(N)).max() <= 1e-13


# ---------------------------------------------------------------------------------------------
# Library special cases: each oracle routine against LAPACK/BLAS on random well-conditioned input.
# Non-symmetric-looking inputs (random complex upper factors, rectangular C~) catch a transposed
# operand or a missing/extra conjugate.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [5, 64, 193])
@pytest.mark.parametrize("cplx", [False, True])
def test_against_lapack(N, cplx):
    H, S = _rand_spd_pencil(N, 7 * N, cplx)
    U = oracle.cholesky(S)
    U_l = sla.cholesky(S, lower=False)
    assert np.linalg.norm(U - U_l) / np.linalg.norm(U_l) <= 1e-14
    assert np.all(np.diag(U).imag == 0) and np.all(np.diag(U).real > 0)
    assert np.all(np.tril(U, -1) == 0)
    # inversion of an arbitrary (not Cholesky-derived) upper factor, garbage below the diagonal
    rng = np.random.default_rng(N)
    T = np.triu(rng.standard_normal((N, N)) + (1j * rng.standard_normal((N, N)) if cplx else 0)) \
        + 4 * np.sqrt(N) * np.eye(N)
    T_dirty = T + np.tril(np.full((N, N), 7.0), -1)
    V = oracle.invert_upper(T_dirty)
    V_l = sla.solve_triangular(T, np.eye(N), lower=False)
    assert np.linalg.norm(V - V_l) / np.linalg.norm(V_l) <= 1e-13
    assert np.all(np.tril(V, -1) == 0)
    # two-sided transform with a general upper V and a non-Hermitian-looking check of the formula
    Ht = oracle.to_standard(H, V)
    Ht_l = V.conj().T @ H @ V
    assert np.linalg.norm(Ht - Ht_l) / np.linalg.norm(Ht_l) <= 1e-13
    # back-transform, rectangular C~, no conjugation
    nev = max(1, N // 3)
    Ct = rng.standard_normal((N, nev)) + (1j * rng.standard_normal((N, nev)) if cplx else 0)
    C = oracle.backtransform(V, Ct)
    assert np.linalg.norm(C - V @ Ct) / np.linalg.norm(V @ Ct) <= 1e-13
    # full generalized solve vs LAPACK's generalized driver
    out = oracle.generalized_eigh(H, S)
    eps_l = sla.eigh(H, S, eigvals_only=True)
    np.testing.assert_allclose(out["eps"], eps_l, rtol=0, atol=1e-12 * np.abs(eps_l).max())


@pytest.mark.parametrize("cplx", [False, True])
def test_to_standard_is_not_symmetrised(cplx):
    """O3 computes both triangles independently; with a NON-Hermitian H the result must equal
    V^H H V (not its symmetrisation, not V^T H V, not V H V^H)."""
    N = 23
    rng = np.random.default_rng(5)
    H = rng.standard_normal((N, N)) + (1j * rng.standard_normal((N, N)) if cplx else 0)
    V = np.triu(rng.standard_normal((N, N)) + (1j * rng.standard_normal((N, N)) if cplx else 0))
    Ht = oracle.to_standard(H, V)
    ref = V.conj().T @ H @ V
    assert np.linalg.norm(Ht - ref) / np.linalg.norm(ref) <= 1e-14


# ---------------------------------------------------------------------------------------------
# P-jacobi: residual, orthonormality, trace and Frobenius invariants, agreement with LAPACK.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [1, 2, 33, 120])
@pytest.mark.parametrize("cplx", [False, True])
def test_jacobi(N, cplx):
    A, _ = _rand_spd_pencil(N, 11 + N, cplx)
    eps, Q, sweeps = oracle.jacobi(A)
    assert 1 <= sweeps <= 15
    assert np.all(np.diff(eps) >= 0)
    nA = np.linalg.norm(A)
    assert np.linalg.norm(A @ Q - Q * eps) <= 20 * N * U52 * nA
    assert np.abs(Q.conj().T @ Q - np.eye(N)).max() <= 1e-13
    assert abs(eps.sum() - np.trace(A).real) <= 1e-12 * nA
    assert abs((eps ** 2).sum() - nA ** 2) <= 1e-12 * nA ** 2
    np.testing.assert_allclose(eps, np.linalg.eigvalsh(A), rtol=0, atol=1e-13 * nA)


# ---------------------------------------------------------------------------------------------
# P-planted: S := U0^H U0 formed in extended precision from a known factor  =>  chol(S) ~ U0.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cplx", [False, True])
def test_planted_factor(cplx):
    N = 40
    rng = np.random.default_rng(9)
    U0 = np.triu(0.05 * rng.standard_normal((N, N)), 1).astype(np.longdouble)
    U0 = U0 + np.diag(rng.uniform(1, 2, N)).astype(np.longdouble)
    if cplx:
        Ui = np.triu(0.05 * rng.standard_normal((N, N)), 1).astype(np.longdouble)
        Sre = U0.T @ U0 + Ui.T @ Ui
        Sim = U0.T @ Ui - Ui.T @ U0
        S = np.asarray(Sre, dtype=np.float64) + 1j * np.asarray(Sim, dtype=np.float64)
        U0 = np.asarray(U0, dtype=np.float64) + 1j * np.asarray(Ui, dtype=np.float64)
    else:
        S = np.asarray(U0.T @ U0, dtype=np.float64)
        U0 = np.asarray(U0, dtype=np.float64)
    U = oracle.cholesky(S)
    assert np.abs(U - U0).max() <= 1e-13


# ---------------------------------------------------------------------------------------------
# P-invariants on the BASELINE recipe (real and complex), incl. Hermitian symmetry of H~ (Q5).
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [17, 100, 256])
@pytest.mark.parametrize("cplx", [False, True])
def test_recipe_invariants(N, cplx):
    p = wl.small_pencil(N, seed=N, complex=cplx)
    H, S = p.H.numpy(), p.S.numpy()
    U = oracle.cholesky(S)
    V = oracle.invert_upper(U)
    Ht = oracle.to_standard(H, V)
    assert np.linalg.norm(U.conj().T @ U - S) / np.linalg.norm(S) <= 8 * N * U52
    assert np.linalg.norm(U @ V - np.eye(N)) / math.sqrt(N) <= 1e-12
    assert np.abs(Ht - Ht.conj().T).max() <= 1e-12 * np.linalg.norm(Ht)
    assert np.linalg.norm(U.conj().T @ Ht @ U - H) / np.linalg.norm(H) <= 1e-10
    assert abs(np.trace(Ht) - np.trace(np.linalg.solve(S, H))) <= 1e-9 * abs(np.trace(Ht))
    if cplx:
        assert np.abs(np.diag(Ht).imag).max() <= 1e-12 * np.linalg.norm(Ht)


# ---------------------------------------------------------------------------------------------
# P-phase: config 3's S' = S o P, H' = H o P with P_ij = exp(ik(x_i - x_j)) is D S D^H, D H D^H
# with D = diag(exp(i k x_i)) unitary; hence U' = U o P, V' = V o P, H~' = H~ o P, eps' = eps,
# C' = D C (up to a phase per column).  Pins the complex oracle to the real one.
# ---------------------------------------------------------------------------------------------
def test_phase_identity_pins_complex_to_real():
    N = 100
    pr = wl.small_pencil(N, seed=77, complex=False)
    pc = wl.small_pencil(N, seed=77, complex=True)
    x = pr.r[:, 0].numpy()
    P = np.exp(1j * wl.PHASE_K * (x[:, None] - x[None, :]))
    np.testing.assert_allclose(pc.S.numpy(), pr.S.numpy() * P, rtol=0, atol=1e-15)
    real = oracle.generalized_eigh(pr.H.numpy(), pr.S.numpy())
    cplx = oracle.generalized_eigh(pc.H.numpy(), pc.S.numpy())
    for key, tol in (("U", 1e-13), ("V", 1e-12), ("Ht", 1e-12)):
        ref = real[key] * P
        assert np.linalg.norm(cplx[key] - ref) / np.linalg.norm(ref) <= tol, key
    np.testing.assert_allclose(cplx["eps"], real["eps"], rtol=0, atol=1e-10 * np.abs(real["eps"]).max())


# ---------------------------------------------------------------------------------------------
# Q6: non-positive-definite S is reported with the 1-based index of the first bad pivot.
# ---------------------------------------------------------------------------------------------
def test_not_positive_definite_reports_pivot():
    N = 12
    S = np.eye(N)
    S[4, 4] = -1.0
    with pytest.raises(oracle.NotPositiveDefinite) as e:
        oracle.cholesky(S)
    assert e.value.info == 5
    S = np.eye(N)
    S[0, 7] = S[7, 0] = np.nan
    with pytest.raises(oracle.NotPositiveDefinite) as e:
        oracle.cholesky(S)
    assert e.value.info == 8
    # leading 2x2 minor indefinite: [[1,2],[2,1]] -> pivot 2
    S = np.eye(N)
    S[0, 1] = S[1, 0] = 2.0
    with pytest.raises(oracle.NotPositiveDefinite) as e:
        oracle.cholesky(S.astype(np.complex128))
    assert e.value.info == 2


# ---------------------------------------------------------------------------------------------
# End-to-end acceptance metrics on BASELINE config 0 for the oracle itself (reading Q7-Q9).
# ---------------------------------------------------------------------------------------------
def test_config0_end_to_end_metrics():
    from paper_2502_02460_b200 import metrics as M

    p = wl.make_config(0)
    H, S = p.H.numpy(), p.S.numpy()
    out = oracle.generalized_eigh(H, S, nev=wl.CONFIGS[0].nev)
    assert M.eig_residual(H, S, out["C"], out["eps"]) <= M.TOL_RESIDUAL
    assert M.s_orthonormality(S, out["C"]) <= M.TOL_SORTH
    eps_l = sla.eigh(H, S, eigvals_only=True)
    np.testing.assert_allclose(out["eps"], eps_l, rtol=0, atol=1e-9 * np.abs(eps_l).max())
