"""Host-side sharding of the seed x hit scan over ranks (one process per GPU, torch.distributed).

The scan shards in two ways:

* by event -- independent events (BASELINE.json configs[2]) go to ranks round-robin, no
  communication at all (`shard_events`); this is what `bench.py --gpus N` does (weak scaling);
* by seed -- the seeds of every turn partition are cut into contiguous, chunk-aligned ranges
  (`shard_partitions`), each rank scans its ranges, and ONE exchange step picks the global
  winner per partition: `merge_best` = all_reduce(MIN) of the local best RSS, then all_reduce(MIN)
  of the seed index among the ranks that hold that RSS, which reproduces the single-process rule
  "lowest RSS, ties -> lowest global seed index" (reading R15) exactly.  Every rank then classifies
  the winning seeds itself (one seed per partition: comet_select_and_classify on P seeds), so no
  broadcast of masks is needed.

Only index arithmetic and collectives live here; the scan itself is libcomet.  Works with the
`gloo` backend on CPU tensors (tests) and `nccl` on CUDA tensors.
"""
from typing import List, Sequence, Tuple

import numpy as np
import torch
import torch.distributed as dist

CHUNK = 32
_I64_MAX = np.iinfo(np.int64).max


def shard_events(n_events: int, rank: int, world: int) -> List[int]:
    """Indices of the events rank `rank` of `world` processes (round-robin)."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    return list(range(rank, n_events, world))


def shard_partitions(part_off: Sequence[int], rank: int, world: int, align: int = CHUNK) -> List[Tuple[int, int]]:
    """Per partition, the global seed range [begin, end) this rank scans.

    Every partition is split into `world` contiguous pieces whose interior boundaries are multiples
    of `align` seeds from the partition start (track chunks stay whole); pieces differ by at most
    one aligned block, trailing ranks may get an empty range."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    out = []
    for p in range(len(part_off) - 1):
        lo, hi = int(part_off[p]), int(part_off[p + 1])
        blocks = -(-(hi - lo) // align)
        b0 = (blocks * rank) // world
        b1 = (blocks * (rank + 1)) // world
        out.append((min(hi, lo + b0 * align), min(hi, lo + b1 * align)))
    return out


def local_best(rss: torch.Tensor, ranges: Sequence[Tuple[int, int]], offset: int = 0):
    """(best_rss [P] float64, best_seed [P] int64) of this rank's ranges; `rss[i]` belongs to global
    seed `offset + i`.  Empty range -> (+inf, int64 max).  Ties -> lowest index (first minimum)."""
    P = len(ranges)
    v = torch.full((P,), float("inf"), dtype=torch.float64, device=rss.device)
    i = torch.full((P,), _I64_MAX, dtype=torch.int64, device=rss.device)
    for p, (b, e) in enumerate(ranges):
        if e > b:
            seg = rss[b - offset:e - offset]
            m = torch.min(seg)
            first = torch.nonzero(seg == m, as_tuple=False)[0, 0]
            v[p] = m
            i[p] = first + b
    return v, i


def merge_best(best_rss: torch.Tensor, best_seed: torch.Tensor, group=None):
    """The exchange step: global (best_rss, best_seed) per partition on every rank."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return best_rss.clone(), best_seed.clone()
    g = best_rss.clone()
    dist.all_reduce(g, op=dist.ReduceOp.MIN, group=group)
    cand = torch.where(best_rss == g, best_seed, torch.full_like(best_seed, _I64_MAX))
    dist.all_reduce(cand, op=dist.ReduceOp.MIN, group=group)
    return g, cand
