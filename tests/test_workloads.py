"""The seeded input recipe (no method arithmetic): what both sides rely on.

Step 3 on the GPU reads one triangle of H, the oracle reads the whole matrix, so the generator must
hand out H (and S) that are Hermitian BIT FOR BIT -- not merely to rounding.  A vectorised exp is not
guaranteed to return the same bits for the same argument at two places of a tensor, hence the explicit
mirroring in workloads.overlap / hamiltonian; these tests pin that contract.
"""
import numpy as np
import pytest
import torch

from paper_2502_02460_b200 import workloads as wl


@pytest.mark.parametrize("N,cplx", [(1, False), (5, False), (257, False), (700, False), (450, True), (2100, False)])
def test_pencil_is_exactly_hermitian(N, cplx):
    p = wl.small_pencil(N, seed=9, complex=cplx)
    assert wl.is_colmajor(p.H) and wl.is_colmajor(p.S)
    assert torch.equal(p.H, p.H.conj().t())
    assert torch.equal(p.S, p.S.conj().t())
    if cplx:
        assert torch.count_nonzero(p.H.diagonal().imag) == 0 and torch.count_nonzero(p.S.diagonal().imag) == 0
    # S: unit Gaussian overlap + 1e-3 on the diagonal, entries in (0, 1]
    assert torch.allclose(p.S.diagonal().real, torch.full((N,), 1.001, dtype=torch.float64), rtol=0, atol=1e-15)
    assert p.S.abs().max().item() <= 1.001 + 1e-15


def test_pencil_is_reproducible():
    a = wl.small_pencil(300, seed=4)
    b = wl.small_pencil(300, seed=4)
    c = wl.small_pencil(300, seed=5)
    assert torch.equal(a.H, b.H) and torch.equal(a.S, b.S)
    assert not torch.equal(a.H, c.H)


def test_mirror_upper_repairs_an_inconsistent_lower_triangle():
    g = torch.Generator().manual_seed(1)
    A = torch.randn((70, 70), dtype=torch.float64, generator=g)
    up = torch.triu(A).clone()
    wl.mirror_upper_(A, chunk=32)        # several blocks and a ragged one
    assert torch.equal(torch.triu(A), up)
    assert torch.equal(A, A.t())
    Z = torch.complex(torch.randn((33, 33), dtype=torch.float64, generator=g), torch.randn((33, 33), dtype=torch.float64, generator=g))
    upz = torch.triu(Z, 1).clone()
    wl.mirror_upper_(Z, chunk=16)
    assert torch.equal(torch.triu(Z, 1), upz)
    assert torch.equal(Z, Z.conj().t())
    assert torch.count_nonzero(Z.diagonal().imag) == 0


def test_spd_and_scale_of_the_recipe():
    p = wl.small_pencil(256, seed=2)
    ev = np.linalg.eigvalsh(p.S.numpy())
    assert ev.min() > 5e-4 and ev.max() < 40.0      # jitter keeps S positive definite, well conditioned
