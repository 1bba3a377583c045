"""Device-side ordering of the fused exchange (include/gs.h: gs_exchange_signal / gs_exchange_wait; sharded.py sync="device").

One process, one GPU, two emulated ranks = two plans on two streams that share the GPU's memory: rank r's column-range
kernels push their slabs into the other rank's buffers from their epilogues, signal the round's epoch into both flag arrays
behind those kernels, and rank r's consuming launch waits on its own flags.  Rank 1 is enqueued FIRST, although its step 3
needs the slabs rank 0 produces later: without the wait it would read the NaN the buffers are poisoned with.  Nothing
here spins in a kernel (stream memory operations), so the two streams cannot starve each other.  The whole exchange runs in
a child process with a timeout: a wait that is never signalled would block a stream for good.
"""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SNIPPET = r"""
import numpy as np, torch
import oracle
from paper_2502_02460_b200 import gs, metrics as M, sharded, workloads as wl
torch.cuda.set_device(0)
N, R = 1300, 2
p = wl.small_pencil(N, seed=31)
H, S = wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda())
H2 = wl.to_colmajor(3.0 * p.H.cuda())                  # round 2 reduces another H: stale slabs of round 1 would show
V_o = oracle.invert_upper(oracle.cholesky(p.S.numpy()))
Ht_o = 3.0 * oracle.to_standard(p.H.numpy(), V_o)
ranges = sharded.column_ranges(N, R, 128)
plans = [gs.Plan(N, 0) for _ in range(R)]
streams = [torch.cuda.Stream() for _ in range(R)]
nan = float("nan")
U = [wl.colmajor_empty(N, N, device="cuda") for _ in range(R)]
Vw = [wl.colmajor_empty(N, N, device="cuda") for _ in range(R)]
V = [wl.colmajor_zeros(N, N, device="cuda") for _ in range(R)]
G = [wl.colmajor_empty(N, N, device="cuda") for _ in range(R)]
Ht = [wl.colmajor_empty(N, N, device="cuda") for _ in range(R)]
flags = [torch.zeros(2 * R, dtype=torch.int32, device="cuda") for _ in range(R)]
for r in range(R):
    V[r].copy_(torch.triu(torch.full((N, N), nan, dtype=torch.float64, device="cuda")))     # upper: to be delivered; lower: zeros
    G[r].fill_(nan); Ht[r].fill_(nan)
    o = 1 - r
    plans[r].set_push_targets(gs.GS_PUSH_UINV, [V[0].data_ptr(), V[1].data_ptr()])
    plans[r].set_push_targets(gs.GS_PUSH_G, [G[o].data_ptr()])
    plans[r].set_push_targets(gs.GS_PUSH_HTILDE, [Ht[o].data_ptr()])
torch.cuda.synchronize()
for epoch in (1, 2):
    for r in (1, 0):                                  # the rank that DEPENDS on the other one goes first
        c0, c1 = ranges[r]
        st = streams[r]
        plan = plans[r]
        ready_out = [flags[s].data_ptr() + 4 * r for s in range(R)]
        ready_in = [flags[r].data_ptr() + 4 * s for s in range(R)]
        done_out = [flags[s].data_ptr() + 4 * (R + r) for s in range(R)]
        done_in = [flags[r].data_ptr() + 4 * (R + s) for s in range(R)]
        with torch.cuda.stream(st):
            if epoch > 1:
                plan.exchange_wait(done_in, epoch - 1, stream=st)      # the peers have finished reading round 1's slabs
            U[r].copy_(S)
            plan.cholesky_leading(U[r], c1, stream=st)
            plan.invert_triangular_cols(U[r], Vw[r], c0, c1 - c0, stream=st)
            plan.to_standard_g_cols(H if epoch == 1 else H2, Vw[r], G[r], c0, c1 - c0, stream=st)
            plan.exchange_signal(ready_out, epoch, stream=st)
            plan.exchange_wait(ready_in, epoch, stream=st)
            plan.to_standard_cols(V[r], G[r], Ht[r], c0, c1 - c0, stream=st)
            plan.exchange_signal(done_out, epoch, stream=st)
    # (no host synchronisation between the rounds: the done flags order them)
torch.cuda.synchronize()
ok = True
for r in range(R):
    assert plans[r].last_info() == 0
    eV, eH = M.rel_frob_upper(V[r].cpu(), V_o), M.rel_frob_upper(Ht[r].cpu(), Ht_o)
    print("rank", r, "V", eV, "Ht", eH, "flags", flags[r].tolist())
    ok = ok and eV <= 1e-11 and eH <= 1e-11 and flags[r].tolist() == [2] * (2 * R)
print("OK" if ok else "FAILED")
"""


def test_signal_and_wait_order_two_emulated_ranks_without_host_synchronisation():
    e = dict(os.environ)
    e["PYTHONPATH"] = ROOT + os.pathsep + e.get("PYTHONPATH", "")
    r = subprocess.run([sys.executable, "-c", SNIPPET], env=e, cwd=ROOT, capture_output=True, text=True, timeout=180)
    assert r.returncode == 0 and r.stdout.strip().endswith("OK"), r.stdout[-3000:] + r.stderr[-3000:]


def test_argument_errors():
    import torch
    from paper_2502_02460_b200 import gs
    plan = gs.Plan(64, 0)
    L = gs.lib()
    st = int(torch.cuda.current_stream().cuda_stream)
    f = torch.zeros(4, dtype=torch.int32, device="cuda")
    import ctypes
    arr = (ctypes.c_void_p * 1)(f.data_ptr() + 2)                 # not 4-byte aligned
    assert L.gs_exchange_signal(plan._h, 1, arr, 1, st) == 1
    assert L.gs_exchange_wait(plan._h, 1, None, 1, st) == 1
    assert L.gs_exchange_wait(plan._h, 65, arr, 1, st) == 1
    assert L.gs_exchange_signal(plan._h, 0, None, 1, st) == 0    # nothing to do
    plan.exchange_signal([f.data_ptr(), f.data_ptr() + 4], 7)
    plan.exchange_wait([f.data_ptr(), f.data_ptr() + 4], 7)      # already satisfied: must not block
    torch.cuda.synchronize()
    assert f.tolist() == [7, 7, 0, 0]
    plan.close()
