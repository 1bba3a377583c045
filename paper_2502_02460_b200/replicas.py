"""Multi-GPU mode of the path: replicas only.

The factorisation does not shard into independent units, so N GPUs run N independent pencils --
the paper's "trivial parallelism (e.g., for separate k-points or spin channels)" (PAPER.md:114,
PAPER.md:92).  There is no data-path collective: torch.distributed is used only for the barrier and
for the max-over-ranks of the device time.  This module holds that host logic so that it can be
tested with the gloo backend on CPU (tests/test_replicas_gloo.py); bench.py uses it with NCCL.
"""
from __future__ import annotations

import os
from dataclasses import dataclass

import torch
import torch.distributed as dist


@dataclass(frozen=True)
class RankInfo:
    rank: int
    world: int
    local_rank: int


def rank_info() -> RankInfo:
    return RankInfo(int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
                    int(os.environ.get("LOCAL_RANK", "0")))


def replica_seed(base_seed: int, rank: int) -> int:
    """Every rank reduces its own pencil: same recipe, different seed."""
    return base_seed + 100 * rank


def init(info: RankInfo, backend: str, device=None) -> None:
    if info.world > 1 and not dist.is_initialized():
        kwargs = {}
        if backend == "nccl" and device is not None:
            kwargs["device_id"] = device
        dist.init_process_group(backend, rank=info.rank, world_size=info.world, **kwargs)


def barrier(info: RankInfo) -> None:
    if info.world > 1:
        dist.barrier()


def max_over_ranks(info: RankInfo, x: float, device="cpu") -> float:
    """The job's step time is the slowest replica's."""
    if info.world == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(info: RankInfo, flops_per_replica: float, step_ms_max: float) -> float:
    """Whole-job TFLOP/s: all ranks' nominal flops over the max-over-ranks step time (weak scaling)."""
    return info.world * flops_per_replica / (step_ms_max * 1e-3) / 1e12


def finalize(info: RankInfo) -> None:
    if info.world > 1 and dist.is_initialized():
        dist.destroy_process_group()
