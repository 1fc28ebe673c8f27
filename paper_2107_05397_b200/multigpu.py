"""Multi-GPU plumbing of the shard mode (the problem is split into independent sets of stripes whose
results "have to be eventually merged").  One process per GPU calls unifrac_dm_shard with (rank, world); a rank's buffer
then holds the distances of the tile-pair blocks it owns and 0 everywhere else, so the merge is an element-wise sum over the
ranks: one all-reduce over NCCL / NVLink (gloo in the CPU tests).  No UniFrac arithmetic here."""
from __future__ import annotations


def merge_shards(out, group=None):
    """In-place merge of the ranks' shard buffers (torch tensor on the backend's device: CUDA for nccl, CPU for gloo).
    Every pair has exactly one owner and is 0 on the other ranks, so SUM reproduces the owner's value bit for bit."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return out
    dist.all_reduce(out, op=dist.ReduceOp.SUM, group=group)
    return out


def owner_of_pairs(pairs, world: int):
    """Owner rank of each (i, j) sample pair -- the library's host helper unifrac_shard_of_pair."""
    from . import binding
    return [binding.unifrac_shard_of_pair(int(a), int(b), world) for a, b in pairs]
