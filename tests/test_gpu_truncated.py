"""(5) The truncated-basis route for an ill-conditioned overlap matrix on the GPU (gs_truncated_to_standard,
gs_standard_eigh, gs_backtransform_dense) against the oracle's step-by-step version (oracle.truncated_eigh).

Unique and compared element-wise: sigma (eigenvalues of S), the number of kept directions, eps of the reduced problem.
Valid but not unique (phases, rotations in clusters), hence checked by their defining identities: C^H S C = I,
X^H (H C - S C eps) = 0, and C has no component along the dropped eigenvectors of S.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _dev(a):
    return wl.to_colmajor(torch.from_numpy(np.ascontiguousarray(a)).cuda())


def _pencil_with_near_null_directions(n, cplx, seed):
    """BASELINE recipe at order n - 4, plus 4 basis functions that nearly duplicate existing ones (distance 1e-5):
    four eigenvalues of S drop to ~1e-10 while the rest stays at >= 1e-3."""
    rng = np.random.default_rng(seed)
    m = n - 4
    box = 6.0 * (m / 256.0) ** (1.0 / 3.0)
    r = rng.uniform(0, box, (m, 3))
    r = np.concatenate([r, r[:4] + 1e-5 * rng.standard_normal((4, 3))])
    d2 = ((r[:, None, :] - r[None, :, :]) ** 2).sum(-1)
    jitter = np.full(n, 1e-3)
    jitter[:4] = 0.0                                 # no diagonal jitter on the four duplicated pairs: each pair's
    jitter[m:] = 0.0                                 # 2 x 2 block [[1, 1 - 1.5e-10], [., 1]] keeps S near-singular
    S = np.exp(-0.5 * d2) + np.diag(jitter)
    g = rng.standard_normal((n, n))
    g = np.triu(g) + np.triu(g, 1).T
    H = -S * (1.0 + 0.1 * g) + np.diag(rng.uniform(-2, 0, n))
    if cplx:
        ph = np.exp(1j * 0.7 * (r[:, 0][:, None] - r[:, 0][None, :]))
        S, H = S * ph, H * ph
    S, H = 0.5 * (S + S.conj().T), 0.5 * (H + H.conj().T)
    return H, S


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("n", [40, 150, 300])
def test_truncated_route_against_oracle(n, cplx):
    from paper_2502_02460_b200 import gs
    H, S = _pencil_with_near_null_directions(n, cplx, seed=n)
    delta = 1e-5
    ref = oracle.truncated_eigh(H, S, delta)
    assert 0 < ref["kept"] < n                      # the input does have directions to drop
    nev = ref["kept"] // 2
    plan = gs.Plan(n, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
    S_in = np.array(S, copy=True)
    S_in[np.tril_indices(n, -1)] = np.nan           # only the upper triangle of S may be read
    X, Hr, sigma = plan.truncated_to_standard(_dev(H), _dev(S_in), delta)
    assert plan.last_info() == 0
    assert plan.truncated_rank() == ref["kept"]
    np.testing.assert_allclose(sigma.cpu().numpy(), ref["sigma"], rtol=0, atol=1e-12 * ref["sigma"].max())
    ndrop = n - ref["kept"]
    Xn = X.cpu().numpy()
    assert np.all(Xn[:, :ndrop] == 0)                # dropped directions: zero columns
    np.testing.assert_allclose(Xn[:, ndrop:].conj().T @ S @ Xn[:, ndrop:], np.eye(ref["kept"]), rtol=0, atol=1e-8)
    eps, Ct = plan.standard_eigh(Hr)
    C = wl.colmajor_empty(n, nev, dtype=X.dtype, device="cuda")
    plan.backtransform_dense(X, Ct, C)
    assert plan.last_info() == 0
    en, Cn = eps.cpu().numpy(), C.cpu().numpy()
    scale = np.abs(ref["eps"]).max()
    np.testing.assert_allclose(en, ref["eps"][:nev], rtol=0, atol=1e-8 * scale)     # 1/sqrt(sigma) <= 316 amplifies rounding
    np.testing.assert_allclose(Cn.conj().T @ S @ Cn, np.eye(nev), rtol=0, atol=1e-8)
    Xk = ref["X"]
    assert np.abs(Xk.conj().T @ (H @ Cn - S @ Cn * en[None, :])).max() <= 1e-7 * scale
    # no component along the dropped eigenvectors of S (taken from the ORACLE's Jacobi)
    _, D, _ = oracle.jacobi(S)
    assert np.abs(D[:, :ndrop].conj().T @ S @ Cn).max() <= 1e-8
    plan.close()


def test_delta_zero_agrees_with_the_cholesky_route_on_the_gpu():
    from paper_2502_02460_b200 import gs
    n, nev = 260, 100
    p = wl.small_pencil(n, seed=77)
    plan = gs.Plan(n, nev)
    X, Hr, sigma = plan.truncated_to_standard(wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda()), 0.0)
    assert plan.truncated_rank() == n
    eps_t, _ = plan.standard_eigh(Hr)
    plan2, U, V, Ht = gs.generalized_to_standard(wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda()), nev)
    eps_c, _ = plan2.standard_eigh(Ht)
    assert plan.last_info() == 0 and plan2.last_info() == 0
    assert (eps_t - eps_c).abs().max().item() <= 1e-9 * eps_c.abs().max().item()
    plan.close()
    plan2.close()
