"""The fused exchange of the sharded path across PROCESSES (paper_2502_02460_b200/sharded.py, exchange="push";
include/gs.h: gs_plan_set_push_targets, gs_ipc_*): two ranks, one process each, both on cuda:0 -- the
box has one GPU, and CUDA IPC maps another process's allocation the same way whether it lives on
this GPU or on a peer across NVLink.  Each rank's column-range kernels store their tiles into the
other process's buffers from their epilogues; no kernel of one rank ever waits on the other (the
hosts meet at gloo barriers with the GPU idle).  Every rank must end up with all of U^-1, G,
triu(H~) and C, equal to the CPU oracle's, in two consecutive rounds (buffer re-use).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, nev, cplx, out):
    try:
        import torch.distributed as dist

        import oracle
        from paper_2502_02460_b200 import gs, metrics as M, sharded
        from paper_2502_02460_b200 import workloads as wl
        os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
        torch.cuda.set_device(0)
        dist.init_process_group("gloo", rank=rank, world_size=world)
        p = wl.small_pencil(N, seed=21, complex=cplx)
        H, S = wl.to_colmajor(p.H.cuda()), wl.to_colmajor(p.S.cuda())
        Ct = wl.dense_rhs(N, nev, seed=6, complex=cplx)
        Ctd = wl.to_colmajor(Ct.cuda())
        plan = gs.Plan(N, nev, dtype=gs.GS_COMPLEX128 if cplx else gs.GS_REAL64)
        drv = sharded.ShardedReduction(plan, rank, world, exchange="push")
        bufs = drv.alloc(H)
        U_o = oracle.cholesky(p.S.numpy())
        V_o = oracle.invert_upper(U_o)
        Ht_o = oracle.to_standard(p.H.numpy(), V_o)
        C_o = oracle.backtransform(V_o, Ct.numpy())
        errs = []
        for rnd in range(2):
            if rnd == 1:      # poison what the peers must deliver again
                bufs.Uinv.copy_(torch.tril(torch.zeros_like(bufs.Uinv), -1) + torch.triu(torch.full_like(bufs.Uinv, float("nan"))))
                bufs.G.fill_(float("nan"))
                bufs.Htilde.fill_(float("nan"))
                bufs.C.fill_(float("nan"))
                torch.cuda.synchronize()
            res = drv.reduce(H, S, out=bufs)
            Ht = drv.gather_htilde(res)
            C = drv.backtransform(res.Uinv, Ctd, out=res.C)
            errs.append({"V": M.rel_frob_upper(res.Uinv.cpu(), V_o), "V_lower": M.strictly_lower_max(res.Uinv.cpu()),
                         "Ht": M.rel_frob_upper(Ht.cpu(), Ht_o), "C": M.rel_frob(C.cpu(), C_o),
                         "G_finite": bool(torch.isfinite(torch.view_as_real(torch.triu(res.G)) if cplx else torch.triu(res.G)).all())})
        drv.close()
        plan.close()
        out.put((rank, errs, None))
        dist.barrier()
        dist.destroy_process_group()
    except Exception as e:  # noqa: BLE001 -- reported to the parent, which fails the test
        import traceback
        out.put((rank, None, traceback.format_exc()))
        raise


@pytest.mark.parametrize("N,cplx", [(1500, False), (900, True)])
def test_push_exchange_between_two_processes(N, cplx):
    world, nev = 2, N // 3
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, N, nev, cplx, out)) for r in range(world)]
    for p in procs:
        p.start()
    try:
        res = sorted((out.get(timeout=300) for _ in range(world)), key=lambda t: t[0])
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.terminate()
    for rank, errs, tb in res:
        assert tb is None, tb
        for e in errs:
            assert e["V"] <= 1e-11 and e["Ht"] <= 1e-11 and e["C"] <= 1e-11, (rank, errs)
            assert e["V_lower"] == 0.0 and e["G_finite"], (rank, errs)
