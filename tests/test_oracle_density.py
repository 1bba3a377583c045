"""Pins of the oracle's density matrix (O7, P_ij = sum_l f_l c*_li c_lj with c_li = C(i,l)).

None of these re-types the oracle's loop: a hand-computed 2 x 1 case that fixes WHERE the conjugate sits
(a transposed / mis-conjugated implementation fails it), the electron count that Eqs. (3)-(4) of the
paper imply for S-orthonormal eigenvectors (sum_ij P_ij S_ij = sum_l f_l), the projector identity for
0/1 occupations, Hermitian symmetry with a real non-negative diagonal, and numpy's einsum."""
import numpy as np
import pytest

import oracle
from paper_2502_02460_b200 import workloads as wl


def test_hand_case_fixes_the_conjugate():
    # N = 2, one state c = (1, i), f = 2:  P_12 = f conj(c_1) c_2 = 2i,  P_21 = f conj(c_2) c_1 = -2i
    C = np.array([[1.0], [1.0j]])
    P = oracle.density_matrix(C, [2.0])
    np.testing.assert_allclose(P, np.array([[2.0, 2.0j], [-2.0j, 2.0]]), rtol=0, atol=0)
    # N = 1: P = f |c|^2
    np.testing.assert_allclose(oracle.density_matrix(np.array([[3.0 - 4.0j]]), [0.5]), [[12.5]], rtol=1e-15)


def test_real_two_states_by_hand():
    C = np.array([[1.0, 2.0], [3.0, -1.0], [0.5, 0.0]])
    f = [2.0, 1.0]
    P = oracle.density_matrix(C, f)
    expect = 2.0 * np.outer(C[:, 0], C[:, 0]) + 1.0 * np.outer(C[:, 1], C[:, 1])
    np.testing.assert_allclose(P, expect, rtol=1e-15)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N", [7, 64, 150])
def test_electron_count_projector_and_symmetry(N, cplx):
    p = wl.small_pencil(N, seed=31 + N, complex=cplx)
    H, S = p.H.numpy(), p.S.numpy()
    nev = max(1, N // 2)
    ref = oracle.generalized_eigh(H, S, nev)          # C is S-orthonormal (pinned in test_oracle_pins)
    C = ref["C"]
    rng = np.random.default_rng(N)
    f = rng.uniform(0.0, 2.0, nev)
    P = oracle.density_matrix(C, f)
    # int n(r) dr = sum_ij P_ij S_ij = sum_l f_l  (Eqs. 3 and 4 with <psi_l|psi_l> = 1)
    assert abs(np.sum(P * S) - f.sum()) <= 1e-10 * max(1.0, f.sum())
    # Hermitian, real non-negative diagonal
    assert np.abs(P - P.conj().T).max() <= 1e-12 * np.abs(P).max()
    assert np.all(np.diag(P).real >= 0) and np.abs(np.diag(P).imag).max() <= 1e-15 * np.abs(P).max()
    # 0/1 occupations: D = P^T = C C^H is the S-projector onto the occupied space, D S D = D
    P1 = oracle.density_matrix(C, np.ones(nev))
    D = P1.T
    assert np.abs(D @ S @ D - D).max() <= 1e-9 * max(1.0, np.abs(D).max())
    # library cross-check
    np.testing.assert_allclose(P, np.einsum("l,il,jl->ij", f, C.conj(), C), rtol=0, atol=1e-12 * np.abs(P).max())


def test_zero_states_gives_zero():
    P = oracle.density_matrix(np.zeros((5, 0)), np.zeros(0))
    assert P.shape == (5, 5) and np.all(P == 0)
