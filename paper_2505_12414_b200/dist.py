"""Host-side helpers for running the path on N GPUs, one process per GPU (``torch.distributed``).

The path shards without a data-path collective (Eq. 1: the events of a
likelihood are independent, and so are pseudo-experiments):

* toys (BASELINE.json configs[4]) are dealt to ranks in contiguous blocks; every rank uploads, evaluates
  and fits only its own toys; the per-toy results are gathered at the end (``gather_toy_rows``);
* the events of ONE dataset may be split into contiguous shards (multiples of 64 events, the kernels'
  item size); every rank evaluates its shard with ``mf_nll_grad`` and the K+1 partial sums are combined
  by ``combine_partials``: an all-gather followed by a compensated sum in RANK ORDER on every rank, so
  that all ranks hold bit-identical results and the result does not depend on the collective's
  reduction tree (an all-reduce's order may).  K+1 <= 17 doubles: latency bound on any fabric.

Nothing here computes anything: it is plumbing over ``torch.distributed`` (gloo on CPU in the tests, nccl on
GPUs); the rank-ordered compensated sum itself is the library's ``mf_combine_partials`` (host C).
"""
from __future__ import annotations

import numpy as np

ITEM = 64  # events per warp item of the kernels (mf_kernels.cuh kItem)


def shard_toys(n_toys: int, rank: int, world: int) -> tuple[int, int]:
    """(first toy, number of toys) of `rank`: contiguous blocks whose sizes differ by at most one."""
    if not (0 <= rank < world) or n_toys < 0:
        raise ValueError("bad rank / world / n_toys")
    base, extra = divmod(n_toys, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def shard_events(n_events: int, rank: int, world: int) -> tuple[int, int]:
    """(first event, number of events) of `rank`: contiguous shards of whole 64-event items, the last
    shard takes the ragged tail."""
    if not (0 <= rank < world) or n_events < 0:
        raise ValueError("bad rank / world / n_events")
    items = (n_events + ITEM - 1) // ITEM
    first_item, n_items = shard_toys(items, rank, world)
    first = min(first_item * ITEM, n_events)
    last = min((first_item + n_items) * ITEM, n_events)
    return first, last - first


def ordered_sum(rows: np.ndarray) -> np.ndarray:
    """Compensated sum of rows[0], rows[1], ... in that order: the library's mf_combine_partials (host C)."""
    from . import combine_partials as _c
    rows = np.asarray(rows, dtype=np.float64)
    return _c(rows.reshape(rows.shape[0], -1)).reshape(rows.shape[1:])


def combine_partials(local: np.ndarray, group=None) -> np.ndarray:
    """All ranks pass their K+1 partial sums (-ln L and gradient of their event shard); all ranks get the
    same, rank-ordered compensated total."""
    import torch
    import torch.distributed as dist
    local = np.ascontiguousarray(local, dtype=np.float64)
    world = dist.get_world_size(group)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    mine = torch.from_numpy(local).to(dev)
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine, group=group)
    return ordered_sum(np.stack([p.cpu().numpy() for p in parts]))


def gather_toy_rows(local_rows: np.ndarray, n_toys: int, group=None) -> np.ndarray:
    """local_rows: [my toys][C] results of this rank's block (shard_toys order).  Returns [n_toys][C] on
    every rank, in toy order."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    local_rows = np.ascontiguousarray(local_rows, dtype=np.float64)
    if local_rows.ndim == 1:
        local_rows = local_rows[:, None]
    first, count = shard_toys(n_toys, rank, world)
    if local_rows.shape[0] != count:
        raise ValueError(f"rank {rank} holds {local_rows.shape[0]} rows, its block has {count}")
    width = local_rows.shape[1]
    cap = (n_toys + world - 1) // world
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    pad = np.zeros((cap, width))
    pad[:count] = local_rows
    mine = torch.from_numpy(pad).to(dev)
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine, group=group)
    out = np.empty((n_toys, width))
    for r in range(world):
        f, c = shard_toys(n_toys, r, world)
        out[f:f + c] = parts[r].cpu().numpy()[:c]
    return out
