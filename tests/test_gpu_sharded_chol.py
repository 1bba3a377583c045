"""gs_cholesky_sharded (include/gs.h): step 1 over the ranks of one NVSwitch
domain, panels dealt round-robin, the row panels all-gathered by the producing side, ordered by device-side flags.

One process, one GPU, R emulated ranks = R plans on R streams with R copies of S, one host thread per rank (as one
process per GPU would be); every rank's whole program is enqueued up front and the stream waits order them.  Nothing
spins in a kernel (stream memory operations), so the streams cannot starve each other; the run sits in a child process
with a timeout because a wait that is never signalled would block a stream for good.  Checked: every rank ends with the
complete factor, equal bit for bit on all ranks, against the oracle's unblocked Cholesky (O1) at the 1e-11 bar; zeros
below the diagonal; a second factorisation with advanced epochs on the same flags; nranks = 1."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SNIPPET = r"""
import sys, threading
import numpy as np, torch
import oracle
from paper_2502_02460_b200 import gs, metrics as M, workloads as wl
torch.cuda.set_device(0)
ok = True
for cplx, N, R in ((False, 1500, 2), (False, 1100, 3), (True, 700, 2), (False, 1300, 4), (False, 300, 3)):
    dt = gs.GS_COMPLEX128 if cplx else gs.GS_REAL64
    p = wl.small_pencil(N, seed=50 + N, complex=cplx)
    S0 = wl.to_colmajor(p.S.cuda())
    U_o = oracle.cholesky(p.S.numpy())
    plans = [gs.Plan(N, 0, dtype=dt) for _ in range(R)]
    streams = [torch.cuda.Stream() for _ in range(R)]
    S = [S0.clone() for _ in range(R)]
    low = torch.tril(torch.ones(N, N, dtype=torch.bool, device="cuda"), -1)
    flags = [torch.zeros(R, dtype=torch.int32, device="cuda") for _ in range(R)]
    nep = plans[0].cholesky_sharded_epochs()
    torch.cuda.synchronize()
    for rnd in range(2):
        for r in range(R):
            S[r].copy_(S0)
            S[r][low] = float("nan")                      # the strictly-lower triangle is never read
        torch.cuda.synchronize()
        def rank_program(r):
            torch.cuda.set_device(0)
            plans[r].cholesky_sharded(S[r], r, R, [x.data_ptr() for x in S], [pl.workspace.data_ptr() for pl in plans],
                                      [f.data_ptr() for f in flags], epoch0=rnd * nep, stream=streams[r])
        th = [threading.Thread(target=rank_program, args=(r,)) for r in reversed(range(R))]
        for t in th:
            t.start()
        for t in th:
            t.join()
        torch.cuda.synchronize()
        for r in range(R):
            assert plans[r].last_info() == 0
            e = M.rel_frob_upper(S[r].cpu(), U_o)
            z = bool((S[r][low] == 0).all())
            same = bool(torch.equal(S[r], S[0]))
            print("cplx", cplx, "N", N, "R", R, "round", rnd, "rank", r, "err", e, "zeros below", z, "equal to rank 0", same, flush=True)
            ok = ok and e <= M.TOL_FROB and z and same
    for pl in plans:
        pl.close()
# a pivot that is not positive on ONE rank's panel: nobody hangs (every rank signals whatever its status: its kernels are
# no-ops, its signals are not), the owner of the bad block reports the pivot, and the flags reach their final values
N, R = 900, 2
p = wl.small_pencil(N, seed=77)
Sbad = p.S.clone()
Sbad[400, 400] = -1.0                                  # block 3 = panel 1 (panels of GS_POTRF_NB blocks) or panel 3 (nb = 1)
S0 = wl.to_colmajor(Sbad.cuda())
plans = [gs.Plan(N, 0) for _ in range(R)]
streams = [torch.cuda.Stream() for _ in range(R)]
S = [S0.clone() for _ in range(R)]
flags = [torch.zeros(R, dtype=torch.int32, device="cuda") for _ in range(R)]
torch.cuda.synchronize()
def bad_program(r):
    torch.cuda.set_device(0)
    plans[r].cholesky_sharded(S[r], r, R, [x.data_ptr() for x in S], [pl.workspace.data_ptr() for pl in plans],
                              [f.data_ptr() for f in flags], epoch0=0, stream=streams[r])
th = [threading.Thread(target=bad_program, args=(r,)) for r in range(R)]
for t in th: t.start()
for t in th: t.join()
torch.cuda.synchronize()                               # returns: no stream is left waiting
infos = [pl.last_info(raise_on_failure=False) for pl in plans]
print("non-PD: infos", infos, "statuses", [getattr(pl, "last_status", None) for pl in plans], "flags", [f.tolist() for f in flags], flush=True)
ok = ok and 401 in [abs(int(i)) for i in infos]
for pl in plans:
    pl.close()
# nranks = 1: no peers, no flags
N = 900
p = wl.small_pencil(N, seed=7)
plan = gs.Plan(N, 0)
S1 = wl.to_colmajor(p.S.cuda())
plan.cholesky_sharded(S1, 0, 1)
assert plan.last_info() == 0
e1 = M.rel_frob_upper(S1.cpu(), oracle.cholesky(p.S.numpy()))
print("nranks 1 err", e1)
ok = ok and e1 <= M.TOL_FROB
print("OK" if ok else "FAILED")
"""


@pytest.mark.parametrize("nb", ["2", "1"])
def test_sharded_cholesky_emulated_ranks(nb):
    e = dict(os.environ)
    e["PYTHONPATH"] = ROOT + os.pathsep + e.get("PYTHONPATH", "")
    e["GS_POTRF_NB"] = nb                                  # panels of 2 (1) blocks: several panels per rank at test sizes
    r = subprocess.run([sys.executable, "-c", SNIPPET], env=e, cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip().endswith("OK"), r.stdout[-4000:] + r.stderr[-3000:]


def test_sharded_cholesky_argument_errors():
    import ctypes

    import torch
    from paper_2502_02460_b200 import gs, workloads as wl
    L = gs.lib()
    plan = gs.Plan(256, 0)
    S = wl.colmajor_zeros(256, 256, device="cuda")
    f = torch.zeros(2, dtype=torch.int32, device="cuda")
    two = lambda a, b: (ctypes.c_void_p * 2)(a, b)
    ws = plan.workspace.data_ptr()
    assert L.gs_cholesky_sharded(plan._h, S.data_ptr(), 0, 0, None, None, None, 0, None) == 1          # nranks < 1
    assert L.gs_cholesky_sharded(plan._h, S.data_ptr(), 2, 2, None, None, None, 0, None) == 1          # rank out of range
    assert L.gs_cholesky_sharded(plan._h, S.data_ptr(), 0, 9, None, None, None, 0, None) == 1          # more than 8 ranks
    assert L.gs_cholesky_sharded(plan._h, S.data_ptr(), 0, 2, None, None, None, 0, None) == 1          # peers missing
    assert L.gs_cholesky_sharded(plan._h, S.data_ptr(), 0, 2, two(S.data_ptr() + 16, S.data_ptr()), two(ws, ws),
                                 two(f.data_ptr(), f.data_ptr()), 0, None) == 1                       # own entry is not S_inout
    assert L.gs_cholesky_sharded(plan._h, None, 0, 1, None, None, None, 0, None) == 1
    n = ctypes.c_uint32(0)
    assert L.gs_cholesky_sharded_epochs(plan._h, ctypes.byref(n)) == 0 and n.value == 3               # one panel: entry + 2
    assert L.gs_cholesky_sharded_epochs(None, ctypes.byref(n)) == 1
    plan.close()
