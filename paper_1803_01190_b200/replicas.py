"""Rank bookkeeping for `bench.py --gpus N`: N independent replicas of the single-GPU path ("replicas only",
DESIGN.md section 8).  Nothing here touches particle data: the path has no exchange step, so there is no data-path
collective -- only a barrier and a max-over-ranks of the measured time (torch.distributed; NCCL on GPUs, gloo in the
CPU tests)."""
import os


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_seed(base_seed, rank):
    """Each replica integrates its own system: same recipe, a distinct seed."""
    return int(base_seed) + 1000 * int(rank)


def max_over_ranks(x, device="cpu"):
    """max of a python float over all ranks (identity without an initialised process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def job_value(units_per_rank_per_step, steps, ms_max, world):
    """Whole-job throughput: units of all ranks / the slowest rank's time."""
    return float(world) * float(units_per_rank_per_step) * float(steps) / (float(ms_max) * 1e-3)
