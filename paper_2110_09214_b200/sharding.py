"""Target sharding for multi-GPU runs: every rank holds all sources and evaluates a
contiguous slice of the charges.  Host-side logic only -- no arithmetic of the method."""
from __future__ import annotations


def shard_range(n: int, world: int, rank: int):
    """(first, count) of rank `rank`'s contiguous target slice; sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def all_gather_rows(local, n_total: int, out=None):
    """All-gather row slices made with shard_range: rank r contributes its [count_r, k] rows and every rank gets
    the [n_total, k] whole (same device / backend as `local`).  Equal slices go through one
    all_gather_into_tensor; ragged ones are padded to the largest slice first (collectives need equal sizes)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size()
    k = local.shape[1]
    if out is None:
        out = torch.empty((n_total, k), dtype=local.dtype, device=local.device)
    if world == 1:
        out.copy_(local)
        return out
    if n_total % world == 0:
        dist.all_gather_into_tensor(out, local.contiguous())
        return out
    maxc = -(-n_total // world)
    padded = torch.zeros((maxc, k), dtype=local.dtype, device=local.device)
    padded[:local.shape[0]] = local
    buf = torch.empty((world * maxc, k), dtype=local.dtype, device=local.device)
    dist.all_gather_into_tensor(buf, padded)
    for r in range(world):
        first, count = shard_range(n_total, world, r)
        out[first:first + count] = buf[r * maxc:r * maxc + count]
    return out


def all_gather_charges(local_slice, n_total: int, out=None):
    """The one exchange of a time step: every rank contributes its [count,4] slice of the charges and gets the
    full [n_total,4] array."""
    return all_gather_rows(local_slice, n_total, out=out)
