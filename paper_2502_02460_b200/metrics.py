"""Acceptance metrics of BASELINE.json `north_star`, evaluated identically for the oracle's and the
CUDA path's results (plain torch FP64 ops, CPU or GPU; never inside a timed region).

  - relative Frobenius error on upper triangles   <= 1e-11   (U, U^-1, H~)
  - eigenvector residual  ||H C - S C eps||_F / (||H||_F * N * 2^-52)   <= 100
  - S-orthonormality      ||C^H S C - I||_max                            <= 1e-10
"""
from __future__ import annotations

import numpy as np
import torch

TOL_FROB = 1e-11
TOL_RESIDUAL = 100.0
TOL_SORTH = 1e-10


def _t(a, device=None) -> torch.Tensor:
    if isinstance(a, np.ndarray):
        a = torch.from_numpy(np.ascontiguousarray(a))
    if device is not None:
        a = a.to(device)
    return a


def rel_frob_upper(X, X_ref) -> float:
    """||triu(X) - triu(X_ref)||_F / ||triu(X_ref)||_F  (reading Q4: parity on upper triangles)."""
    X_ref = _t(X_ref)
    X = _t(X, X_ref.device)
    d = torch.triu(X - X_ref)
    den = torch.triu(X_ref).norm().item()
    return d.norm().item() / (den if den > 0 else 1.0)


def rel_frob(X, X_ref) -> float:
    X_ref = _t(X_ref)
    X = _t(X, X_ref.device)
    den = X_ref.norm().item()
    return (X - X_ref).norm().item() / (den if den > 0 else 1.0)


def strictly_lower_max(X) -> float:
    """max |X_ij| over i > j: the zeroing contract of U and U^-1."""
    X = _t(X)
    if X.shape[0] < 2:
        return 0.0
    return torch.tril(X, -1).abs().max().item()


def eig_residual(H, S, C, eps) -> float:
    """||H C - S C diag(eps)||_F / (||H||_F * N * 2^-52)."""
    H = _t(H)
    S, C, eps = _t(S, H.device), _t(C, H.device), _t(eps, H.device)
    N = H.shape[0]
    R = H @ C - (S @ C) * eps.to(C.dtype).unsqueeze(0)
    return R.norm().item() / (H.norm().item() * N * 2.0 ** -52)


def s_orthonormality(S, C) -> float:
    """||C^H S C - I||_max."""
    S = _t(S)
    C = _t(C, S.device)
    G = C.conj().t() @ (S @ C)
    G.diagonal().sub_(1.0)
    return G.abs().max().item() if G.numel() else 0.0
