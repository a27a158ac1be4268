"""Multi-GPU host logic: the path shards over realisations with no data-path collective.

`partition` gives each rank its contiguous slice of the batch; `merge_welford` combines per-rank
ensemble accumulators (count, mean, M2) with Chan's pairwise formula after one all_gather.  Works on
any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

from typing import Tuple

import torch
import torch.distributed as dist


def partition(B: int, world: int, rank: int) -> Tuple[int, int]:
    """(first realisation, count) of `rank`: sizes differ by at most one, earlier ranks get the extras."""
    if B < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad partition arguments")
    base, extra = divmod(B, world)
    count = base + (1 if rank < extra else 0)
    start = rank * base + min(rank, extra)
    return start, count


def chan_merge(n_a: int, mean_a: torch.Tensor, M2_a: torch.Tensor,
               n_b: int, mean_b: torch.Tensor, M2_b: torch.Tensor):
    """Merge two (count, mean, M2) accumulators (Chan et al.); either side may be empty."""
    if n_a == 0:
        return n_b, mean_b.clone(), M2_b.clone()
    if n_b == 0:
        return n_a, mean_a.clone(), M2_a.clone()
    n = n_a + n_b
    delta = mean_b - mean_a
    mean = mean_a + delta * (n_b / n)
    M2 = M2_a + M2_b + delta * delta * (n_a * n_b / n)
    return n, mean, M2


def merge_welford(count: int, mean: torch.Tensor, M2: torch.Tensor, group=None):
    """All ranks contribute their accumulator; every rank returns the merged (count, mean, M2)."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return count, mean, M2
    world = dist.get_world_size(group)
    cnt = torch.tensor([count], dtype=torch.int64, device=mean.device)
    counts = [torch.zeros_like(cnt) for _ in range(world)]
    means = [torch.zeros_like(mean) for _ in range(world)]
    M2s = [torch.zeros_like(M2) for _ in range(world)]
    dist.all_gather(counts, cnt, group=group)
    dist.all_gather(means, mean.contiguous(), group=group)
    dist.all_gather(M2s, M2.contiguous(), group=group)
    n, m, s = 0, torch.zeros_like(mean), torch.zeros_like(M2)
    for r in range(world):
        n, m, s = chan_merge(n, m, s, int(counts[r].item()), means[r], M2s[r])
    return n, m, s


def gather_stats(stats_bytes: torch.Tensor, group=None) -> torch.Tensor:
    """Concatenate per-rank ssp_stats records (uint8 tensors of equal length) in rank order."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return stats_bytes
    world = dist.get_world_size(group)
    out = [torch.zeros_like(stats_bytes) for _ in range(world)]
    dist.all_gather(out, stats_bytes.contiguous(), group=group)
    return torch.cat(out)
