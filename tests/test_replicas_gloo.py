"""world_size-2 gloo test (CPU) of the multi-GPU host logic: replicas only, no data-path collective
(DESIGN.md section 9).  Covers per-rank seeds, the barrier, max-over-ranks timing and the whole-job
aggregate that bench.py prints."""
import os
import socket

import torch
import torch.multiprocessing as mp

from paper_2502_02460_b200 import replicas
from paper_2502_02460_b200 import workloads as wl


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update({"RANK": str(rank), "WORLD_SIZE": str(world), "LOCAL_RANK": str(rank),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    info = replicas.rank_info()
    replicas.init(info, "gloo")
    seed = replicas.replica_seed(wl.CONFIGS[0].seed, info.rank)
    # each rank builds its own (different) small pencil, as bench.py does on its own GPU
    p = wl.make_pencil(32, 3.0, seed)
    replicas.barrier(info)
    my_ms = 10.0 + 5.0 * info.rank                      # rank 1 is the slow replica
    step_ms = replicas.max_over_ranks(info, my_ms)
    value = replicas.aggregate_throughput(info, 1e12, step_ms)
    out.put((info.rank, seed, float(p.S[0, 1]), step_ms, value))
    replicas.barrier(info)
    replicas.finalize(info)


def test_two_replicas_over_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, seed0, s0, ms0, v0), (r1, seed1, s1, ms1, v1) = res
    assert (r0, r1) == (0, 1)
    assert seed0 != seed1 and s0 != s1                  # independent pencils
    assert ms0 == ms1 == 15.0                           # max over ranks, seen by every rank
    assert v0 == v1 == 2 * 1e12 / 15e-3 / 1e12          # all ranks' flops / slowest replica's time


def test_single_rank_needs_no_process_group():
    info = replicas.RankInfo(0, 1, 0)
    replicas.barrier(info)
    assert replicas.max_over_ranks(info, 3.5) == 3.5
    assert replicas.aggregate_throughput(info, 2e12, 1000.0) == 2.0
    assert replicas.replica_seed(7, 0) == 7 and replicas.replica_seed(7, 3) == 307
