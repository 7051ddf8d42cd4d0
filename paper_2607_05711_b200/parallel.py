"""Multi-GPU plumbing.  The layer shards over tokens: every step of the hot
path is row-independent except the LoRA weight gradients, which sum over tokens.  One process
per GPU; each rank runs the whole path on its own rows and the only exchange is the ordinary
data-parallel all-reduce of (dA, dB) -- (K + N) * r fp32 values, latency-bound on NVLink."""
import torch
import torch.distributed as dist


def shard_rows(M, rank, world):
    """Contiguous row range [lo, hi) of rank `rank`; the ranges partition [0, M)."""
    base, extra = divmod(M, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def allreduce_lora_grads(dA, dBt, group=None):
    """Sum the adapter gradients over the data-parallel group, in place, as ONE flat bucket
    (sized for launch latency, not link count)."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return dA, dBt
    flat = torch.cat([dA.reshape(-1), dBt.reshape(-1)])
    dist.all_reduce(flat, op=dist.ReduceOp.SUM, group=group)
    dA.copy_(flat[:dA.numel()].view_as(dA))
    dBt.copy_(flat[dA.numel():].view_as(dBt))
    return dA, dBt


def allreduce_amax(amax, group=None):
    """Optional: a global tensor scale (bit-parity with the unsharded run) needs max over ranks."""
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(amax, op=dist.ReduceOp.MAX, group=group)
    return amax
