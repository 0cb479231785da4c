"""Replica sharding across GPUs.

Replicas are independent (the batch dimension), so the path shards with no data-path collective:
rank r of N runs `batch` replicas keyed as replica r*batch .. (r+1)*batch - 1 (the handle's `replica_offset`),
which keeps every replica's Philox stream independent of N.  Only timings (max over ranks) and the per-replica
observables (an all-gather of 2 * batch int64) cross ranks.  No arithmetic of the method lives here.
"""
import torch
import torch.distributed as dist


def replica_offset(rank, batch_per_rank):
    """First global replica index of a rank (weak scaling: every rank runs batch_per_rank replicas)."""
    if rank < 0 or batch_per_rank < 1:
        raise ValueError("rank must be >= 0 and batch_per_rank >= 1")
    return int(rank) * int(batch_per_rank)


def global_batch(world, batch_per_rank):
    return int(world) * int(batch_per_rank)


def _active():
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def max_over_ranks(value, device="cpu"):
    """Max of a python float over all ranks (the job is as slow as its slowest rank)."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if _active():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier():
    if _active():
        dist.barrier()


def gather_observables(E, M):
    """All-gather per-replica int64 tensors E, M of the local shard into [world * batch] tensors, rank-major
    (= global replica order, since rank r owns replicas r*batch ..)."""
    if not _active():
        return E.clone(), M.clone()
    world = dist.get_world_size()
    Es = [torch.empty_like(E) for _ in range(world)]
    Ms = [torch.empty_like(M) for _ in range(world)]
    dist.all_gather(Es, E)
    dist.all_gather(Ms, M)
    return torch.cat(Es), torch.cat(Ms)
