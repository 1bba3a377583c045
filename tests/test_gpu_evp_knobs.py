"""The alternative forms of the standard eigensolver's kernels stay correct (NEXT-4): the plain-load
symmetric product with three launches per column (GS_EVP_SYMV=0: the form odd real N always takes), the TMA form
without the fused F step (GS_EVP_FUSE=0), strips of one and two blocks per work item (GS_EVP_CHUNK), one streaming CTA
per SM (GS_EVP_CTAS=1), no programmatic dependent launch (GS_EVP_PDL=0), the back-transformation without split k-ranges
(GS_EVP_BACK_SPLIT=0).  The knobs are read once per process, so each configuration runs in its own process; the checks
are those of tests/test_gpu_evp.py: eigenvalues against the oracle's Jacobi, the tridiagonal matrix against Sturm
bisection, residual and orthonormality of the eigenvectors."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SNIPPET = r"""
import numpy as np, torch
import oracle
from paper_2502_02460_b200 import gs, workloads as wl
bad = 0
for cplx, N, nev in ((False, 300, 100), (True, 200, 200), (False, 700, 64), (False, 257, 257)):
    p = wl.small_pencil(N, seed=21 + N, complex=cplx)
    plan, U, V, Ht = gs.generalized_to_standard(wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda()), nev)
    Hs = oracle.hermitian_from_upper(Ht.cpu().numpy())
    eps_o, _, _ = oracle.jacobi(Hs)
    A = Ht.clone()
    low = torch.tril(torch.ones(N, N, dtype=torch.bool, device="cuda"), -1)
    A[low] = float("nan")                                   # the strictly-lower part is never read
    d, e, tau = plan.evp_tridiagonalize(A)
    plan.last_info()
    t_eigs = oracle.tridiag_eigenvalues(d.cpu().numpy(), e.cpu().numpy())
    eps, Z = plan.evp_tridiag_solve(d, e)
    Ct = plan.evp_backtransform(A, Z)
    plan.last_info()
    scale = max(1.0, np.abs(eps_o).max())
    Cn, en = Ct.cpu().numpy(), eps.cpu().numpy()
    errs = {"tridiag": np.abs(t_eigs - eps_o).max() / scale, "eps": np.abs(en - eps_o[:nev]).max() / scale,
            "resid": np.linalg.norm(Hs @ Cn - Cn * en[None, :]) / (N * np.finfo(float).eps * np.linalg.norm(Hs)),
            "orth": np.abs(Cn.conj().T @ Cn - np.eye(nev)).max()}
    ok = errs["tridiag"] <= 1e-12 and errs["eps"] <= 1e-12 and errs["resid"] <= 10.0 and errs["orth"] <= 1e-12
    if not ok:
        bad += 1
        print("MISMATCH", cplx, N, nev, errs, flush=True)
    plan.close()
print("OK" if bad == 0 else "FAILED")
"""


@pytest.mark.parametrize("env", [
    {"GS_EVP_SYMV": "0"},
    {"GS_EVP_FUSE": "0"},
    {"GS_EVP_CHUNK": "1", "GS_EVP_CTAS": "1"},
    {"GS_EVP_CHUNK": "2", "GS_EVP_PDL": "0"},
    {"GS_EVP_BACK_SPLIT": "0"},
])
def test_eigensolver_configuration(env):
    e = dict(os.environ)
    e.update(env)
    e["PYTHONPATH"] = ROOT + os.pathsep + e.get("PYTHONPATH", "")
    r = subprocess.run([sys.executable, "-c", SNIPPET], env=e, cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and r.stdout.strip().endswith("OK"), r.stdout[-3000:] + r.stderr[-4000:]
