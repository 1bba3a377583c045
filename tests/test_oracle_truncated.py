"""Pins of the oracle's truncated-basis route for an ill-conditioned overlap matrix (oracle.truncated_eigh, O11;
PAPER.md:73: transform to the basis of eigenvectors D_i of S, omitting every D_i with sigma_i < delta).

The paper prints no worked example of this route, so the pins are mathematical: a commuting pencil with a planted
spectrum (closed form on the kept directions), delta = 0 reproducing the Cholesky route of PAPER.md:61-67, the
Galerkin identities of the reduced problem, and numpy for the plain products.
"""
import numpy as np
import pytest

import oracle


def _unitary(n, cplx, rng):
    A = rng.standard_normal((n, n)) + (1j * rng.standard_normal((n, n)) if cplx else 0.0)
    Q, _ = np.linalg.qr(A)
    return Q


@pytest.mark.parametrize("cplx", [False, True])
def test_plain_products_against_numpy_and_a_hand_case(cplx):
    rng = np.random.default_rng(0)
    A = rng.standard_normal((7, 4)) + (1j * rng.standard_normal((7, 4)) if cplx else 0.0)
    B = rng.standard_normal((7, 5)) + (1j * rng.standard_normal((7, 5)) if cplx else 0.0)
    np.testing.assert_allclose(oracle.matmul_hn(A, B), A.conj().T @ B, rtol=0, atol=1e-14)
    C = rng.standard_normal((4, 6))
    np.testing.assert_allclose(oracle.matmul_nn(A, C), A @ C, rtol=0, atol=1e-14)
    # hand case that fixes where the conjugate sits: [i]^H [1] = -i
    assert oracle.matmul_hn(np.array([[1j]]), np.array([[1.0 + 0j]]))[0, 0] == -1j


@pytest.mark.parametrize("cplx", [False, True])
def test_commuting_pencil_with_planted_near_null_directions(cplx):
    """S = D diag(sigma) D^H, H = D diag(h) D^H: on the kept directions the reduced problem is diagonal,
    eps = h_i / sigma_i, and the dropped directions (sigma < delta) contribute nothing -- whatever their h."""
    rng = np.random.default_rng(5)
    n = 40
    D = _unitary(n, cplx, rng)
    sigma = np.concatenate([[1e-12, 3e-9, 2e-7], rng.uniform(0.5, 3.0, n - 3)])      # three near-null directions
    h = np.concatenate([[50.0, -50.0, 7.0], rng.uniform(-2.0, 1.0, n - 3)])          # other values on them: h / sigma ~ 1e13
    S = (D * sigma) @ D.conj().T
    H = (D * h) @ D.conj().T
    S, H = 0.5 * (S + S.conj().T), 0.5 * (H + H.conj().T)
    out = oracle.truncated_eigh(H, S, 1e-5)
    assert out["kept"] == n - 3
    ref = np.sort(h[3:] / sigma[3:])
    np.testing.assert_allclose(out["eps"], ref, rtol=0, atol=1e-12 * 50.0)      # (H carries rounding of size u * max|h|)
    C = out["C"]
    np.testing.assert_allclose(C.conj().T @ S @ C, np.eye(n - 3), rtol=0, atol=1e-12)
    # C has no component along the dropped eigenvectors of S
    assert np.abs(D[:, :3].conj().T @ C).max() <= 1e-10
    # with delta below every sigma nothing is dropped and the wild directions come back
    assert oracle.truncated_eigh(H, S, 1e-13)["kept"] == n


@pytest.mark.parametrize("cplx", [False, True])
def test_delta_zero_reproduces_the_cholesky_route(cplx):
    rng = np.random.default_rng(8)
    n = 30
    A = rng.standard_normal((n, n)) + (1j * rng.standard_normal((n, n)) if cplx else 0.0)
    S = A @ A.conj().T + n * np.eye(n)
    H = rng.standard_normal((n, n)) + (1j * rng.standard_normal((n, n)) if cplx else 0.0)
    H = H + H.conj().T
    ref = oracle.generalized_eigh(H, S)            # PAPER.md:61-67 (pinned elsewhere)
    out = oracle.truncated_eigh(H, S, 0.0)
    assert out["kept"] == n
    np.testing.assert_allclose(out["eps"], ref["eps"], rtol=0, atol=1e-11 * np.abs(ref["eps"]).max())
    C = out["C"]
    assert np.linalg.norm(H @ C - S @ C * out["eps"][None, :]) <= 1e-10 * np.linalg.norm(H)


def test_galerkin_identities_on_a_truly_ill_conditioned_overlap():
    """Gaussian overlap of nearly coincident centres: cond(S) ~ 1e14.  The reduced problem must satisfy
    X^H S X = I, X^H (H C - S C eps) = 0 and C^H S C = I although the Cholesky route is hopeless here."""
    rng = np.random.default_rng(2)
    n = 24
    r = np.concatenate([rng.uniform(0, 3, (n - 6, 3)), rng.uniform(0, 3, (3, 3)).repeat(2, axis=0) + 1e-5 * rng.standard_normal((6, 3))])
    d2 = ((r[:, None, :] - r[None, :, :]) ** 2).sum(-1)
    S = np.exp(-0.5 * d2)
    H = -S * (1.0 + 0.1 * np.cos(d2)) - np.diag(rng.uniform(0, 2, n))
    H = 0.5 * (H + H.T)
    out = oracle.truncated_eigh(H, S, 1e-6)
    assert 0 < out["kept"] < n
    X, C, eps = out["X"], out["C"], out["eps"]
    np.testing.assert_allclose(X.T @ S @ X, np.eye(out["kept"]), rtol=0, atol=1e-9)
    np.testing.assert_allclose(C.T @ S @ C, np.eye(len(eps)), rtol=0, atol=1e-9)
    assert np.abs(X.T @ (H @ C - S @ C * eps[None, :])).max() <= 1e-8 * np.abs(eps).max()
