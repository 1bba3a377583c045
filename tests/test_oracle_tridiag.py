"""Pins of the oracle's NEXT-4 helpers (oracle/gs_oracle.c O8-O10): Sturm count / bisection on a symmetric
tridiagonal matrix and the LDL^H inertia count.  None of the expected values comes from the oracle itself:
closed forms, a hand-computed factorisation, brute force, LAPACK (scipy) and the oracle's already pinned Jacobi.

The paper gives no worked example of its "Standard EVP" stages (its only numbers are the timings of Table 1,
PAPER.md:126-133), so every pin is mathematical.
"""
import numpy as np
import pytest
import scipy.linalg

import oracle


def _toeplitz(n):
    return 2.0 * np.ones(n), -np.ones(n - 1)


@pytest.mark.parametrize("n", [1, 2, 3, 10, 100, 257])
def test_bisection_reproduces_the_closed_form_spectrum_of_tridiag_m1_2_m1(n):
    d, e = _toeplitz(n)
    ref = 2.0 - 2.0 * np.cos(np.arange(1, n + 1) * np.pi / (n + 1))      # textbook closed form
    got = oracle.tridiag_eigenvalues(d, e)
    assert np.max(np.abs(got - ref)) <= 8e-16 * 4.0 * max(1, np.log2(n + 1))
    # lowest-nev form returns the lowest ones, ascending
    k = max(1, n // 3)
    assert np.array_equal(oracle.tridiag_eigenvalues(d, e, k), got[:k])


def test_sturm_count_is_the_index_between_eigenvalues():
    n = 40
    d, e = _toeplitz(n)
    lam = 2.0 - 2.0 * np.cos(np.arange(1, n + 1) * np.pi / (n + 1))
    assert oracle.sturm_count(d, e, lam[0] - 1e-3) == 0
    assert oracle.sturm_count(d, e, lam[-1] + 1e-3) == n
    for k in range(n - 1):
        assert oracle.sturm_count(d, e, 0.5 * (lam[k] + lam[k + 1])) == k + 1


def test_sturm_hand_computed_3x3():
    # T = [[2,1,0],[1,2,1],[0,1,2]], x = 1: q0 = 1, q1 = 2-1-1/1 = 0 -> -tiny (counts), q2 = 1 - 1/(-tiny) = +huge
    # eigenvalues 2 - sqrt2, 2, 2 + sqrt2: exactly one is < 1
    d, e = np.array([2.0, 2.0, 2.0]), np.array([1.0, 1.0])
    assert oracle.sturm_count(d, e, 1.0) == 1
    # x = 3: q0 = -1 (1), q1 = -1 + 1 = 0 -> -tiny (2), q2 = -1 + 1/tiny = +huge: two eigenvalues < 3
    assert oracle.sturm_count(d, e, 3.0) == 2
    np.testing.assert_allclose(oracle.tridiag_eigenvalues(d, e), [2 - 2 ** 0.5, 2.0, 2 + 2 ** 0.5], rtol=0, atol=4e-16)


def test_diagonal_and_2x2_cases():
    d = np.array([3.0, -1.0, 7.0, 0.5])
    assert np.array_equal(oracle.tridiag_eigenvalues(d, np.zeros(3)), np.sort(d))
    a, b, c = 1.5, -0.25, 2.0              # [[a, c], [c, b]]: roots of the quadratic
    disc = np.sqrt((a - b) ** 2 / 4 + c * c)
    ref = np.array([(a + b) / 2 - disc, (a + b) / 2 + disc])
    np.testing.assert_allclose(oracle.tridiag_eigenvalues(np.array([a, b]), np.array([c])), ref, rtol=0, atol=5e-16)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_bisection_against_lapack_and_jacobi_on_random_and_graded_matrices(seed):
    rng = np.random.default_rng(seed)
    n = 120
    d = rng.standard_normal(n) * 10.0 ** rng.uniform(-3, 3, n)       # graded: widely varying scales
    e = rng.standard_normal(n - 1) * 10.0 ** rng.uniform(-6, 2, n - 1)
    got = oracle.tridiag_eigenvalues(d, e)
    ref = scipy.linalg.eigvalsh_tridiagonal(d, e)                       # LAPACK
    scale = np.abs(ref).max()
    assert np.max(np.abs(got - ref)) <= 1e-13 * scale
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    eps, _, _ = oracle.jacobi(T)
    assert np.max(np.abs(got - eps)) <= 1e-13 * scale


def test_wilkinson_close_pairs_are_both_found():
    # W21+: eigenvalues come in pairs that agree to ~1e-14 at the top; bisection by index must return both
    m = 10
    d = np.abs(np.arange(-m, m + 1)).astype(float)
    e = np.ones(2 * m)
    got = oracle.tridiag_eigenvalues(d, e)
    ref = scipy.linalg.eigvalsh_tridiagonal(d, e)
    assert np.max(np.abs(got - ref)) <= 2e-14
    assert oracle.sturm_count(d, e, got[-1] + 1e-9) == 2 * m + 1
    assert oracle.sturm_count(d, e, 0.5 * (got[-3] + got[-2])) == 2 * m - 1


def test_inertia_hand_computed_ldlt():
    # A = [[4,2,0],[2,-3,1],[0,1,1]] : pivots 4, -3 - 1 = -4, 1 + 1/4 = 1.25 -> one negative eigenvalue
    A = np.array([[4.0, 2.0, 0.0], [2.0, -3.0, 1.0], [0.0, 1.0, 1.0]])
    assert oracle.inertia_count(A, 0.0) == 1
    assert np.sum(np.linalg.eigvalsh(A) < 0) == 1
    with pytest.raises(ZeroDivisionError):
        oracle.inertia_count(np.array([[1.0, 1.0], [1.0, 1.0]]), 1.0)      # first pivot 1 - 1 = 0


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("n", [1, 2, 5, 33, 150])
def test_inertia_equals_brute_force_eigenvalue_count(n, cplx):
    rng = np.random.default_rng(100 + n)
    A = rng.standard_normal((n, n))
    if cplx:
        A = A + 1j * rng.standard_normal((n, n))
    A = A + A.conj().T
    lam = np.linalg.eigvalsh(A)
    # the upper triangle is what is read: garbage below must not matter
    dirty = np.triu(A) + np.tril(np.full((n, n), 99.0), -1)
    for sigma in list(0.5 * (lam[:-1] + lam[1:])[:: max(1, n // 7)]) + [lam[0] - 1.0, lam[-1] + 1.0]:
        assert oracle.inertia_count(dirty, float(sigma)) == int(np.sum(lam < sigma))
    # and against the pinned Jacobi
    eps, _, _ = oracle.jacobi(A)
    mid = 0.5 * (eps[n // 2 - 1] + eps[n // 2]) if n > 1 else eps[0] + 1.0
    assert oracle.inertia_count(A, float(mid)) == int(np.sum(eps < mid))


def test_inertia_matches_sturm_on_a_tridiagonal_matrix():
    n = 80
    d, e = _toeplitz(n)
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    for x in (0.013, 0.77, 1.9, 3.31):
        assert oracle.inertia_count(T, x) == oracle.sturm_count(d, e, x)
