"""Replica bookkeeping for `bench.py --gpus N` ("replicas only").

north_star fixes the library to one GPU with no sharding and no collectives, so N GPUs run N
independent replicas of the planner.  The only thing the ranks exchange is the TIMING: the step
time of the job is the maximum over ranks, and the whole-job throughput is the units all ranks
processed divided by that time.  No data-path collective exists.  These helpers hold that logic so
that it is testable with the `gloo` backend on CPU (tests/test_replicas_gloo.py).
"""
import os


def env_rank_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_seed(base_seed: int, rank: int, step: int, call: int) -> int:
    """Seed of call `call` (0 rollout, 1 belief update) of planning step `step` on replica `rank`:
    distinct per (rank, step, call), equal to the single-GPU sequence for rank 0."""
    return int(base_seed) + 2 * int(step) + int(call) + (int(rank) << 32)


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of one scalar (a duration); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: float, world: int, ms_per_step_max: float) -> float:
    """Units per second of the whole job: every replica processes `units_per_rank` per step."""
    return world * units_per_rank / (ms_per_step_max * 1e-3)
