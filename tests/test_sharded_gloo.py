"""world_size-2 and -3 gloo tests (CPU) of the host logic of the sharded path (paper_2502_02460_b200/sharded.py;
SURVEY.md section 8(f) NEXT-3): column ranges, the order of the calls, the one
exchange of unequal column slabs, the gather of H~ and of C.

There is no GPU here, so the `plan` the driver calls is a TEST-ONLY stand-in defined in this file: it
does each column-range call with numpy from the rank's OWN buffers (poisoning with NaN everything the
call does not produce), so a slab that the exchange fails to deliver, or a call issued before the data
it needs has arrived, shows up as NaNs or as a mismatch with the oracle's whole-matrix result.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

import oracle
from paper_2502_02460_b200 import sharded
from paper_2502_02460_b200 import workloads as wl


class _NumpyColsPlan:
    """Same method names and buffer conventions as gs.Plan's column-range calls; CPU, test only."""

    def __init__(self, N, nev, block):
        self.N, self.nev, self.block = N, nev, block
        self.calls = []
        self.fail_info = 0

    def cholesky_leading(self, S, ncols, stream=None):
        full = S.numpy().copy()
        full[:ncols, :ncols] = oracle.cholesky(np.ascontiguousarray(full[:ncols, :ncols]))
        full[:, ncols:] = np.nan                      # nothing right of the leading block may be used
        S.copy_(torch.from_numpy(full))
        self.calls.append("cholesky")

    def invert_triangular_cols(self, U, Uinv, c0, w, stream=None):
        c1 = c0 + w
        Uinv.fill_(float("nan"))
        if w > 0:
            Ul = np.triu(U.numpy()[:c1, :c1])
            V = np.zeros((self.N, w), dtype=U.numpy().dtype)
            V[:c1] = np.triu(np.linalg.solve(Ul, np.eye(c1, dtype=Ul.dtype)))[:, c0:c1]
            Uinv[:, c0:c1] = torch.from_numpy(V)
        self.calls.append("invert_cols")

    def to_standard_g_cols(self, H, Uinv, G, c0, w, stream=None):
        Hn = H.numpy()
        T = np.triu(Hn, 1) + np.diag(np.diag(Hn)) / 2
        G.fill_(float("nan"))
        G[:, c0:c0 + w] = torch.from_numpy(T @ Uinv.numpy()[:, c0:c0 + w])
        self.calls.append("g_cols")

    def to_standard_cols(self, Uinv, G, Ht, c0, w, stream=None):
        c1 = c0 + w
        V, Gn = Uinv.numpy()[:, :c1], G.numpy()[:, :c1]        # nothing to the right of the range is read
        X = V.conj().T @ Gn[:, c0:c1] + Gn.conj().T @ V[:, c0:c1]
        Ht[:c1, c0:c1] = torch.from_numpy(np.triu(X, -c0))     # rows <= column (global indices)
        self.calls.append("syr2k_cols")

    def backtransform_cols(self, Uinv, Ct, C, k0, w, stream=None):
        C.fill_(float("nan"))
        C[:, k0:k0 + w] = torch.from_numpy(Uinv.numpy() @ Ct.numpy()[:, k0:k0 + w])
        self.calls.append("back_cols")

    def last_info(self, stream=None, raise_on_failure=True):
        return self.fail_info


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(target, world, extra_args, timeout=240, attempts=2):
    """Runs `target(rank, world, port, *extra_args, out)` in `world` spawned processes and returns their
    results sorted by rank.  A rendezvous that does not come up (port taken between _free_port() and the
    workers' bind, a slow import under load) is retried once on a fresh port; a real failure fails twice."""
    last = None
    for _ in range(attempts):
        ctx = mp.get_context("spawn")
        out = ctx.Queue()
        port = _free_port()
        procs = [ctx.Process(target=target, args=(r, world, port) + tuple(extra_args) + (out,)) for r in range(world)]
        for p in procs:
            p.start()
        try:
            res = sorted((out.get(timeout=timeout) for _ in range(world)), key=lambda t: t[0])
            for p in procs:
                p.join(timeout=60)
            if all(p.exitcode == 0 for p in procs):
                return res
            last = AssertionError(f"worker exit codes {[p.exitcode for p in procs]}")
        except Exception as e:  # noqa: BLE001 -- queue.Empty on a hung rendezvous
            last = e
        finally:
            for p in procs:
                if p.is_alive():
                    p.terminate()
    raise last


def _worker(rank, world, port, N, nev, block, cplx, out):
    import torch.distributed as dist
    os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = wl.small_pencil(N, seed=11, complex=cplx)                # identical on every rank
    H, S = wl.to_colmajor(p.H), wl.to_colmajor(p.S)
    plan = _NumpyColsPlan(N, nev, block)
    drv = sharded.ShardedReduction(plan, rank, world)
    res = drv.reduce(H, S)
    own = res.Htilde[:, res.cols[0]:res.cols[1]].clone()
    Ht = drv.gather_htilde(res)
    Ct = wl.to_colmajor(wl.dense_rhs(N, nev, seed=4, complex=cplx))
    C = drv.backtransform(res.Uinv, Ct)
    out.put((rank, res.cols, plan.calls, res.Uinv.numpy().copy(), np.triu(Ht.numpy()), C.numpy().copy(),
             np.triu(own.numpy(), -res.cols[0])))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,N,block,cplx", [(2, 300, 32, False), (3, 257, 16, True), (2, 40, 64, False), (3, 100, 64, False)])
def test_sharded_driver_over_gloo(world, N, block, cplx):
    nev = N // 3
    res = _spawn(_worker, world, (N, nev, block, cplx))
    pen = wl.small_pencil(N, seed=11, complex=cplx)
    U_o = oracle.cholesky(pen.S.numpy())
    V_o = oracle.invert_upper(U_o)
    Ht_o = np.triu(oracle.to_standard(pen.H.numpy(), V_o))
    C_o = oracle.backtransform(V_o, wl.dense_rhs(N, nev, seed=4, complex=cplx).numpy())
    ranges = sharded.column_ranges(N, world, block)
    for rank, cols, calls, V, Ht, C, own in res:
        assert tuple(cols) == ranges[rank]
        assert calls == (["cholesky", "invert_cols", "g_cols", "syr2k_cols", "back_cols"] if cols[1] > cols[0] else ["back_cols"])
        assert np.isfinite(V).all() and np.isfinite(Ht).all() and np.isfinite(C).all()
        assert np.linalg.norm(V - V_o) <= 1e-11 * np.linalg.norm(V_o)        # every rank ends with all of U^-1
        assert np.linalg.norm(Ht - Ht_o) <= 1e-11 * np.linalg.norm(Ht_o)     # ... and all of triu(H~)
        assert np.linalg.norm(C - C_o) <= 1e-11 * np.linalg.norm(C_o)
        c0, c1 = cols
        assert np.linalg.norm(own - Ht_o[:, c0:c1]) <= 1e-11 * max(np.linalg.norm(Ht_o[:, c0:c1]), 1e-300)


def test_column_ranges_cover_align_and_balance():
    for N, world, block in ((16384, 8, 128), (16384, 2, 128), (8192, 4, 64), (1000, 8, 128), (100, 3, 128), (32768, 8, 128)):
      for kappa in (0.0, sharded.CHOL_WEIGHT):
        r = sharded.column_ranges(N, world, block, kappa)
        assert len(r) == world and r[0][0] == 0 and r[-1][1] == N
        for (a0, a1), (b0, b1) in zip(r, r[1:]):
            assert a1 == b0 and a0 <= a1
        for c0, c1 in r:
            assert c0 % block == 0 or c0 == N
            assert c1 % block == 0 or c1 == N
    # equal sums of (leading Cholesky + share of steps 2-3): at the headline size no rank carries more than
    # 1.12 x the mean, with and without the Cholesky term
    for world in (2, 4, 8):
        for kappa in (0.0, sharded.CHOL_WEIGHT):
            r = sharded.column_ranges(16384, world, 128, kappa)
            cost = [sharded.range_cost(c0, c1, 16384, kappa) for c0, c1 in r]
            assert max(cost) <= 1.12 * sum(cost) / world, (world, kappa, cost)
    # the plain cube rule is the kappa = 0 case
    assert sharded.column_ranges(16384, 8, 128, 0.0)[0] == (0, 8192)
    # with the Cholesky term the last rank, which factors all of S, gets the narrowest range
    r = sharded.column_ranges(16384, 8, 128)
    assert r[-1][1] - r[-1][0] == min(c1 - c0 for c0, c1 in r)


def test_even_ranges():
    assert sharded.even_ranges(4096, 8, 2) == [(512 * k, 512 * (k + 1)) for k in range(8)]
    r = sharded.even_ranges(5, 3, 2)
    assert r[0][0] == 0 and r[-1][1] == 5 and all(a1 == b0 for (_, a1), (b0, _) in zip(r, r[1:]))
    assert all(k0 % 2 == 0 for k0, _ in r)
    assert sharded.even_ranges(0, 4) == [(0, 0)] * 4


def test_slab_is_a_contiguous_view():
    X = wl.colmajor_zeros(6, 5)
    v = sharded.slab(X, 1, 3)
    assert v.is_contiguous() and v.shape == (2, 6)
    v.fill_(7.0)
    assert float(X[:, 1:3].min()) == 7.0 and float(X[:, 0].abs().max()) == 0.0 and float(X[:, 3:].abs().max()) == 0.0
    with pytest.raises(ValueError):
        sharded.slab(torch.zeros(6, 5), 1, 3)


def _failing_worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_2502_02460_b200.gs import GsError
    os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    dist.init_process_group("gloo", rank=rank, world_size=world)
    N = 96
    p = wl.small_pencil(N, seed=2)
    plan = _NumpyColsPlan(N, 8, 16)
    plan.fail_info = 77 if rank == 1 else 0          # only rank 1's leading block hits the bad pivot
    drv = sharded.ShardedReduction(plan, rank, world)
    try:
        drv.reduce(wl.to_colmajor(p.H), wl.to_colmajor(p.S))
        out.put((rank, None))
    except GsError as e:
        out.put((rank, (e.status, e.info)))
    dist.barrier()                                   # nobody is left behind in the exchange
    dist.destroy_process_group()


def test_a_failing_rank_stops_every_rank():
    res = _spawn(_failing_worker, 2, ())
    assert res == [(0, (2, 77)), (1, (2, 77))]


def test_sharded_cholesky_option_needs_the_push_exchange_with_device_ordering():
    """chol='sharded' (gs_cholesky_sharded) stores into the peers' buffers: only with exchange='push', sync='device'."""
    from paper_2502_02460_b200 import sharded

    class P:
        N, nev, block = 1024, 0, 128
    for kw in ({"exchange": "collective"}, {"exchange": "push", "sync": "host"}):
        with pytest.raises(ValueError):
            sharded.ShardedReduction(P(), rank=0, world=2, chol="sharded", **kw)
    with pytest.raises(ValueError):
        sharded.ShardedReduction(P(), rank=0, world=2, chol="cyclic")
    with pytest.raises(ValueError):
        sharded.ShardedReduction(P(), rank=0, world=9, exchange="push", sync="device", chol="sharded")
    r = sharded.ShardedReduction(P(), rank=0, world=1, chol="sharded")      # one rank: nothing to shard
    assert not r.chol_sharded
