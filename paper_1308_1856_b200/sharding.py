"""Multi-GPU plumbing: the path shards only over independent batch members.

One process per GPU; members are partitioned across ranks; there is NO collective on the data path.  The only
communication is the final gather of per-member result rows and the max-over-ranks of the device time, done with
torch.distributed (NCCL on GPUs, gloo in the CPU tests).  Holds no arithmetic of the method.
"""
import numpy as np


def member_slice(n_members_total, rank, world):
    """Contiguous near-equal partition of members [0, n_members_total): returns (first, count) of `rank`."""
    if world < 1 or not (0 <= rank < world) or n_members_total < 0:
        raise ValueError((n_members_total, rank, world))
    base, extra = divmod(n_members_total, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def _device():
    import torch
    dist = _dist()
    if dist is not None and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def max_over_ranks(x):
    """max of a python float over all ranks (device time of the slowest rank)."""
    import torch
    dist = _dist()
    if dist is None or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x):
    import torch
    dist = _dist()
    if dist is None or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_rows(local_rows, n_members_total):
    """local_rows: [b_local][w] float64 of this rank's members (partitioned by member_slice) -> [n_total][w] on
    every rank, in global member order."""
    import torch
    dist = _dist()
    local_rows = np.ascontiguousarray(local_rows, dtype=np.float64)
    if dist is None or dist.get_world_size() == 1:
        assert local_rows.shape[0] == n_members_total
        return local_rows
    world, rank = dist.get_world_size(), dist.get_rank()
    w = local_rows.shape[1]
    cap = max(member_slice(n_members_total, r, world)[1] for r in range(world))
    pad = np.zeros((cap, w))
    pad[: local_rows.shape[0]] = local_rows
    mine = torch.from_numpy(pad).to(_device())
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    out = np.zeros((n_members_total, w))
    for r in range(world):
        first, cnt = member_slice(n_members_total, r, world)
        out[first:first + cnt] = parts[r][:cnt].cpu().numpy()
    return out


def barrier():
    dist = _dist()
    if dist is not None and dist.get_world_size() > 1:
        dist.barrier()
