"""Multi-GPU plumbing for bench.py: one process per GPU, REPLICAS ONLY.

The paper's code is single-device (multi-device is future work) and the
north_star says one GPU, so `--gpus N` runs N independent replicas of the workload (independent
gauge configurations / right-hand sides, seed offset by rank) with NO data-path collective.
torch.distributed is used only for the barrier and for the max-over-ranks of the device time.
Everything here is host logic and is covered by a world_size-2 gloo test on CPU.
"""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str):
    """Initialise torch.distributed when WORLD_SIZE > 1.  Returns (rank, local_rank, world)."""
    rank, local_rank, world = env_world()
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value: float, world: int, device=None) -> float:
    """MAX all-reduce of a host scalar (device time in ms)."""
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_seed(base_seed: int, rank: int) -> int:
    """Each replica draws its own fields: seed = base + 1000 * rank."""
    return int(base_seed) + 1000 * int(rank)


def aggregate_ns_per_site(ms_total: float, steps: int, sites_per_step_per_rank: int, world: int) -> float:
    """Whole-job Dslash cost: time / (sites processed by ALL ranks).  Weak scaling: each rank
    processes `sites_per_step_per_rank` sites per step."""
    return ms_total * 1e6 / (float(steps) * sites_per_step_per_rank * world)


def finalize(world: int):
    if world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
