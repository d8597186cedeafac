"""Multi-GPU: the path shards by ensemble.  Each slow-time ensemble is an
independent problem, so rank r of W filters the ensembles `ensemble_shard(n, r, W)` with its own
plan on its own GPU and there is no data-path collective (weak scaling).  The only communication
a driver needs is gathering the finished 2-D images, which `gather_images` does with
torch.distributed (NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def ensemble_shard(n_ensembles: int, rank: int, world_size: int) -> list[int]:
    """Round-robin assignment: consecutive (overlapping) ensembles land on different GPUs, so a
    streaming sequence keeps every GPU busy from the first packets on."""
    if world_size < 1 or not (0 <= rank < world_size) or n_ensembles < 0:
        raise ValueError((n_ensembles, rank, world_size))
    return list(range(rank, n_ensembles, world_size))


def gather_images(local: dict, n_ensembles: int, group=None) -> list:
    """local: {ensemble index: image tensor}.  Returns the images of all ensembles, in order, on
    every rank (all_gather_object: images are small 2-D float32 arrays)."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    parts = [None] * world
    dist.all_gather_object(parts, {int(k): v for k, v in local.items()}, group=group)
    merged = {}
    for part in parts:
        for k, v in part.items():
            if k in merged:
                raise RuntimeError(f"ensemble {k} filtered by two ranks")
            merged[k] = v
    missing = [e for e in range(n_ensembles) if e not in merged]
    if missing:
        raise RuntimeError(f"ensembles {missing} were not filtered by any rank")
    return [merged[e] for e in range(n_ensembles)]
