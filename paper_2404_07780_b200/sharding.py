"""Galaxy sharding across ranks.

Galaxies are independent units: the path shards by galaxy
with no collective inside the iteration loop.  The only communication is the final
gather of the fitted parameters and chi^2 (a few hundred KB).  Host-side logic only;
works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import Sequence

import numpy as np
import torch


def shard_galaxies(pixels_per_galaxy: Sequence[int], world: int) -> list[np.ndarray]:
    """Partition galaxy indices over `world` ranks, balanced by pixel count.

    Cost per galaxy per iteration is proportional to its pixel count (2 K^2 FMAs per
    pixel), so galaxies are dealt largest-first to the least loaded rank (LPT); ties
    and equal sizes fall back to round-robin order.  Every index appears exactly once;
    each rank's list is sorted so that a rank's batch keeps the input order.
    """
    px = np.asarray(pixels_per_galaxy, dtype=np.int64)
    if world < 1:
        raise ValueError("world must be >= 1")
    order = np.argsort(-px, kind="stable")
    load = np.zeros(world, dtype=np.int64)
    count = np.zeros(world, dtype=np.int64)
    owner = np.empty(len(px), dtype=np.int64)
    for g in order:
        r = int(np.lexsort((count, load))[0])      # least load, then fewest galaxies
        owner[g] = r
        load[r] += px[g]
        count[r] += 1
    return [np.flatnonzero(owner == r) for r in range(world)]


def gather_results(local_index: np.ndarray, params: torch.Tensor, chi2: torch.Tensor,
                   n_total: int, group=None):
    """All-gather the per-rank results into full `[n_total, P]` / `[n_total]` tensors
    in the original galaxy order.  Shards may have different lengths."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    P = params.shape[1]
    dev = params.device
    n_local = torch.tensor([len(local_index)], dtype=torch.int64, device=dev)
    counts = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(counts, n_local, group=group)
    n_max = int(max(c.item() for c in counts))
    pad = lambda t, shape: torch.cat([t, t.new_zeros((n_max - t.shape[0],) + shape)], 0)
    idx_t = pad(torch.as_tensor(local_index, dtype=torch.int64, device=dev), ())
    buf_i = [torch.empty_like(idx_t) for _ in range(world)]
    buf_p = [torch.empty((n_max, P), dtype=params.dtype, device=dev) for _ in range(world)]
    buf_c = [torch.empty(n_max, dtype=chi2.dtype, device=dev) for _ in range(world)]
    dist.all_gather(buf_i, idx_t, group=group)
    dist.all_gather(buf_p, pad(params, (P,)), group=group)
    dist.all_gather(buf_c, pad(chi2, ()), group=group)
    full_p = torch.empty((n_total, P), dtype=params.dtype, device=dev)
    full_c = torch.empty(n_total, dtype=chi2.dtype, device=dev)
    for r in range(world):
        n = int(counts[r].item())
        full_p[buf_i[r][:n]] = buf_p[r][:n]
        full_c[buf_i[r][:n]] = buf_c[r][:n]
    return full_p, full_c
