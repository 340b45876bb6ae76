"""Host-side plumbing for ``bench.py --gpus N``: one process per GPU, no data-path collective.

Views and frames are independent (the paper itself runs one view per GPU chip
and sends the hologram to every chip), so the path shards by whole frames: rank r reconstructs its
own frames with its own plan.  The only cross-rank traffic is control: a barrier on both sides of
the timed region and a MAX over the per-rank device times.  ``torch.distributed`` carries both
(NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import os

from .workloads import shard_range  # re-exported: block partition of independent units

__all__ = ["RankInfo", "rank_info", "init", "barrier", "max_over_ranks", "sum_over_ranks",
           "finalize", "shard_range", "aggregate_throughput"]


class RankInfo:
    def __init__(self, rank=0, local_rank=0, world=1):
        self.rank, self.local_rank, self.world = int(rank), int(local_rank), int(world)

    @property
    def is_root(self):
        return self.rank == 0


def rank_info(env=None):
    """RANK / LOCAL_RANK / WORLD_SIZE as torchrun exports them; a bare run is rank 0 of 1."""
    env = os.environ if env is None else env
    return RankInfo(env.get("RANK", 0), env.get("LOCAL_RANK", 0), env.get("WORLD_SIZE", 1))


def init(info, backend):
    """Join the process group when world > 1 (rendezvous from MASTER_ADDR / MASTER_PORT)."""
    if info.world == 1:
        return False
    import torch.distributed as dist
    if not dist.is_initialized():
        dist.init_process_group(backend=backend, rank=info.rank, world_size=info.world)
    return True


def _dev(device):
    import torch
    return torch.device("cpu") if device is None else device


def barrier(info):
    if info.world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(info, value, device=None):
    """MAX of a per-rank float (the timed region's device time)."""
    if info.world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=_dev(device))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(info, value, device=None):
    """SUM of a per-rank float (units processed, kernel launches, bytes)."""
    if info.world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=_dev(device))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(info, units_this_rank, seconds_this_rank, device=None):
    """Whole-job throughput: units all ranks processed / the slowest rank's time.
    Returns ``(units_total, seconds_max, units_per_second)``."""
    units = sum_over_ranks(info, units_this_rank, device)
    sec = max_over_ranks(info, seconds_this_rank, device)
    return units, sec, (units / sec if sec > 0 else 0.0)


def finalize(info):
    if info.world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
