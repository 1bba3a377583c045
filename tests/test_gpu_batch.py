"""NEXT-2: K independent pencils in flight on K streams give, pencil by pencil, exactly what a
single-pencil run gives (same kernels, same order per pencil), and match the oracle."""
import numpy as np
import pytest
import torch

import oracle
from paper_2502_02460_b200 import metrics as M
from paper_2502_02460_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cplx", [False, True])
def test_batch_matches_single_runs_and_oracle(cplx):
    from paper_2502_02460_b200 import gs
    from paper_2502_02460_b200.batch import Batch
    K, N, nev = 6, 384, 100
    pens = [wl.small_pencil(N, seed=50 + k, complex=cplx, device="cuda") for k in range(K)]
    b = Batch(K, N, nev, complex=cplx)
    U, V, Ht = b.alloc(), b.alloc(), b.alloc(zeros=True)
    b.reduce([p.H for p in pens], [p.S for p in pens], U, V, Ht)
    Ct = [wl.dense_rhs(N, nev, seed=k, complex=cplx, device="cuda") for k in range(K)]
    C = b.alloc(cols=nev)
    b.backtransform(V, Ct, C)
    assert b.last_info() == [0] * K
    torch.cuda.synchronize()
    for k in range(K):
        plan, U1, V1, Ht1 = gs.generalized_to_standard(pens[k].H, pens[k].S, nev)
        assert torch.equal(torch.triu(U[k]), torch.triu(U1))
        assert torch.equal(torch.triu(V[k]), torch.triu(V1))
        assert torch.equal(torch.triu(Ht[k]), torch.triu(Ht1))
        plan.close()
    # oracle parity on two of them
    for k in (0, K - 1):
        U_o = oracle.cholesky(pens[k].S.cpu().numpy())
        V_o = oracle.invert_upper(U_o)
        assert M.rel_frob_upper(Ht[k].cpu(), oracle.to_standard(pens[k].H.cpu().numpy(), V_o)) <= M.TOL_FROB
        assert M.rel_frob(C[k].cpu(), oracle.backtransform(V_o, Ct[k].cpu().numpy())) <= 1e-10
    b.close()
