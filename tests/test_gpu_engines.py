"""The alternative engine configurations stay correct: the 128 x 128-tile real engine (GS_TILE64=0),
the 64 x 64-tile complex engine (GS_CTILE_HALF=0), no super-tile rasterisation, other POTRF panel
schedules, the recursive form of the panel's diagonal block (GS_POTRF_FLAT=0), the alternative diagonal-block kernels (GS_LEAF=0: rank-1 sweep over 256 threads; GS_LEAF_BLOCKED=1: 4-row panels).  The knobs are read at plan creation, so each configuration runs in its own process."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SNIPPET = r"""
import numpy as np, torch
import oracle
from paper_2502_02460_b200 import gs, metrics as M, workloads as wl
bad = 0
for cplx, N in ((False, 700), (True, 450), (False, 1500)):
    p = wl.small_pencil(N, seed=9, complex=cplx)
    H, S = p.H.numpy(), p.S.numpy()
    U_o = oracle.cholesky(S); V_o = oracle.invert_upper(U_o); Ht_o = oracle.to_standard(H, V_o)
    plan, U, V, Ht = gs.generalized_to_standard(wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda()), N // 2)
    Ct = wl.dense_rhs(N, N // 2, seed=1, complex=cplx)
    C = wl.colmajor_empty(N, N // 2, dtype=p.H.dtype, device="cuda")
    plan.backtransform(V, wl.to_colmajor(Ct.cuda()), C); plan.last_info()
    errs = {"U": M.rel_frob_upper(U.cpu(), U_o), "V": M.rel_frob_upper(V.cpu(), V_o), "Ht": M.rel_frob_upper(Ht.cpu(), Ht_o),
            "C": M.rel_frob(C.cpu(), oracle.backtransform(V.cpu().numpy(), Ct.numpy()))}
    if not max(errs.values()) <= M.TOL_FROB:
        bad += 1
        D = (torch.triu(Ht.cpu()) - torch.triu(torch.from_numpy(np.ascontiguousarray(Ht_o)))).abs()
        idx = (D > 1e-9).nonzero()
        print("MISMATCH", cplx, N, errs, "bad H~ entries", idx.shape[0],
              "rows", (idx[:, 0].min().item(), idx[:, 0].max().item()) if idx.numel() else None,
              "cols", (idx[:, 1].min().item(), idx[:, 1].max().item()) if idx.numel() else None, flush=True)
    plan.close()
print("OK" if bad == 0 else "FAILED")
"""


@pytest.mark.parametrize("env", [
    {"GS_TILE64": "0", "GS_CTILE_HALF": "0"},
    {"GS_TILE64": "1"},
    {"GS_SUPER_TILE": "0"},
    {"GS_POTRF_NB": "2", "GS_POTRF_TAIL": "6", "GS_POTRF_NB_TAIL": "2", "GS_POTRF_END": "3", "GS_POTRF_NB_END": "1"},
    {"GS_POTRF_NB": "16", "GS_POTRF_TAIL": "0", "GS_POTRF_END": "0"},
    {"GS_LEAF_BLOCKED": "1"},
    {"GS_LEAF": "0"},
    {"GS_POTRF_FLAT": "0"},
])
def test_engine_configuration(env):
    e = dict(os.environ)
    e.update(env)
    e["PYTHONPATH"] = ROOT + os.pathsep + e.get("PYTHONPATH", "")
    r = subprocess.run([sys.executable, "-c", SNIPPET], env=e, cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and r.stdout.strip().endswith("OK"), r.stdout[-3000:] + r.stderr[-4000:]
