"""Multi-GPU: replicas only.  The path does not shard -- a slab decomposition would need a halo
exchange per stencil pass and an all-reduce per dot product -- so N ranks run N independent simulations (different
seeds), with no collective on the data path.  This module holds the host logic bench.py uses for that: the per-rank
seed shift, the barrier, and the max-over-ranks timing reduction.  It works on any torch.distributed backend (nccl on
the GPUs; gloo in the CPU tests)."""
import os


def rank_world():
    """(rank, world_size, local_rank) from the torchrun environment (1 process: 0, 1, 0)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def seed_shift(rank):
    """Replica `rank` simulates its own instance of the workload: generators take seed + seed_shift(rank)."""
    return int(rank)


def barrier(dist=None):
    if dist is not None and dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def max_over_ranks(value, dist=None, device="cpu"):
    """The slowest replica defines the job's time: MAX all-reduce of a scalar (timing plumbing only)."""
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value_ms(ms_total_max, steps, world):
    """Whole-job metric for N replicas: time per (step of one replica) = max-over-ranks time / (steps * N):
    weak scaling -- per-GPU work is fixed, N replicas finish N steps' worth of work per step time."""
    return ms_total_max / (steps * world)
