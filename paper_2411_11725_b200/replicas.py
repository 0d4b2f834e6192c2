"""Host logic of the multi-GPU mode: replicas only.

The demag convolution couples every cell to every other, so the path does not shard at the
config sizes; `bench.py --gpus N` runs N independent meshes, one per rank, with no data-path
collective.  What is left for `torch.distributed` is the rendezvous, the barrier and the
max-over-ranks of the timing; those few lines live here so that they can be tested with the
gloo backend on CPU (tests/test_replicas_gloo.py).
"""
import os


def rank_info(env=None):
    """(rank, world_size, local_rank) from the torchrun environment (1 process: 0, 1, 0)."""
    env = os.environ if env is None else env
    return int(env.get("RANK", "0")), int(env.get("WORLD_SIZE", "1")), int(env.get("LOCAL_RANK", "0"))


def replica_seed(N, rank):
    """Seed of replica `rank` of the config-4 grid N^3: rank 0 is config 4's own seed 4 + N."""
    return 4 + int(N) + int(rank)


def max_over_ranks(seconds, device=None):
    """Slowest rank's time: every multi-GPU number is the max over ranks, never a wall clock."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(seconds)
    t = torch.tensor([float(seconds)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, evals_per_step, cells, steps, seconds):
    """Whole-job throughput in Mcells/s: every rank processed the same number of cells."""
    return world * evals_per_step * cells * steps / seconds / 1e6
