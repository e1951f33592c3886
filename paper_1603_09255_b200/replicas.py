"""N > 1: "replicas only".

A single panmictic population does not shard -- every father row may live on any GPU
 -- so each rank runs an independent replica of the workload with its own
seed and there is NO data-path collective.  This module holds the only cross-rank logic there is:
the per-rank seed and the reduction of the timing (max over ranks) and of the processed units
(sum over ranks).  It is backend-agnostic (`nccl` on the GPUs, `gloo` in the CPU tests).
"""
import os

SEED_STRIDE = 1000


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_config(cfg, rank):
    """The rank's replica: same parameters, seed shifted by SEED_STRIDE * rank (rank 0 = cfg)."""
    out = dict(cfg)
    out["seed"] = cfg["seed"] + SEED_STRIDE * rank
    return out


def patch_block(n_patches, rank, world):
    """Contiguous block [first, first + count) of a sweep's patches owned by `rank`: unlinked patches
    (m = 0) are independent replicates, so a sweep shards by patch with no data-path
    collective.  Blocks differ in size by at most one patch."""
    base, extra = divmod(int(n_patches), int(world))
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def sweep_shard(n_patches, rank, world, **kw):
    """The rank's share of an `n_patches` sweep (workloads.sweep_config), with the parameters the
    patches have in the whole sweep and a seed of its own."""
    from . import workloads
    first, count = patch_block(n_patches, rank, world)
    seed = kw.pop("seed", 6)
    return workloads.sweep_config(n_patches=count, first_patch=first, total_patches=n_patches,
                                  seed=seed + SEED_STRIDE * rank, **kw)


def reduce_over_ranks(dist, times, units, device="cpu"):
    """times -> element-wise MAX over ranks, units -> element-wise SUM over ranks.
    `dist` is torch.distributed (initialised) or None for a single process."""
    times = [float(t) for t in times]
    units = [float(u) for u in units]
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return times, units
    import torch
    t = torch.tensor(times, device=device, dtype=torch.float64)
    u = torch.tensor(units, device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()], [float(x) for x in u.tolist()]


def throughput(units_all_ranks, max_ms):
    """Whole-job units per second: units of all ranks over the slowest rank's time."""
    return units_all_ranks / (max_ms * 1e-3)
