"""Host-side multi-GPU plumbing: structures are independent units, so a job shards by structure
with no data-path collective; the only exchange is an optional all-gather of the per-structure energies.
No arithmetic of the method lives here."""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np


def partition(cost: Sequence[float], world: int) -> List[Tuple[int, int]]:
    """Contiguous ranges [lo, hi) of structures, one per rank, balancing the summed cost (e.g. atoms + edges).

    Greedy prefix split at the ideal cumulative boundaries; every structure lands in exactly one range, ranges are
    ordered by rank, and empty ranges are allowed when there are fewer structures than ranks."""
    cost = np.asarray(cost, np.float64)
    n = cost.size
    if world < 1:
        raise ValueError("world must be >= 1")
    csum = np.concatenate([[0.0], np.cumsum(cost)])
    total = csum[-1]
    cuts = [0]
    for r in range(1, world):
        target = total * r / world
        k = int(np.searchsorted(csum, target, side="left"))
        if k > 0 and abs(csum[k - 1] - target) <= abs(csum[min(k, n)] - target):
            k -= 1
        cuts.append(min(max(k, cuts[-1]), n))
    cuts.append(n)
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


def gather_energies(local, counts: Sequence[int], group=None):
    """All-gather of variable-length per-structure energy vectors (torch tensors on the backend's device)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    m = int(max(counts)) if len(counts) else 0
    pad = torch.zeros(m, dtype=local.dtype, device=local.device)
    pad[: local.numel()] = local
    out = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(out, pad, group=group)
    return torch.cat([out[r][: counts[r]] for r in range(world)])
