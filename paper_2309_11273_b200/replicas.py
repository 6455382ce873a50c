"""Host logic of the multi-GPU mode ("replicas only"): the path is not sharded, every rank
advances an independent replica of the workload, there is NO data-path collective.  The only exchange
is the timing reduction of the measurement protocol: device time is the MAX over ranks, the job's
throughput is the units all ranks processed divided by that time.  Works on any torch.distributed
backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def max_over_ranks(value: float, device="cpu") -> float:
    """max of a per-rank scalar over all ranks (identity without an initialised process group)"""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_throughput(units_per_rank: float, steps: int, ms_max: float, world: int) -> float:
    """units (node-steps, bond-updates) per second of the whole job: every rank does `units_per_rank`
    per step (weak scaling), all ranks are done after `ms_max` milliseconds"""
    return world * units_per_rank * steps / (ms_max * 1e-3)


def rank_info(env=None):
    """(rank, local_rank, world_size) from the torchrun environment"""
    import os
    env = os.environ if env is None else env
    return int(env.get("RANK", "0")), int(env.get("LOCAL_RANK", "0")), int(env.get("WORLD_SIZE", "1"))
