"""Replica bookkeeping for N > 1 GPUs (replicas only, no data-path collective).

Conversations are independent units bound to one decoder for life, so N GPUs
are N pools and N independent tail steps.  The only cross-rank traffic is measurement: a barrier
and two scalar reductions (max time, summed work).  Works on any torch.distributed backend
(nccl on GPUs; gloo in the CPU tests).
"""
import torch


def rank_seed(base_seed, rank):
    """Every replica serves its own conversations: same length recipe, different seed."""
    return int(base_seed) + 100 * int(rank)


def bind_conversations(need_blocks, pool_blocks, world):
    """The paper's placement rule across `world` decoders, host-only replay:
    each arriving conversation goes to the decoder with the lowest active occupancy that fits.
    Returns the decoder index per conversation (-1 = nobody fits)."""
    used = [0] * world
    out = []
    for need in need_blocks:
        best = -1
        for r in range(world):
            if pool_blocks - used[r] < need:
                continue
            if best < 0 or used[r] < used[best]:
                best = r
        if best >= 0:
            used[best] += int(need)
        out.append(best)
    return out


def aggregate(dist, local_ms, local_units, device="cpu"):
    """(max over ranks of the step time, sum over ranks of the units) -> whole-job rate inputs."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(local_ms), float(local_units)
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())
