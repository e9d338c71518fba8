"""Host-side sharding of one pair list over ranks.

Pairs are independent (one read against one candidate region), so the path shards
with no data-path collective: rank r aligns the contiguous pair range ``pair_range(P, world, r)``
against the (replicated) packed sequences, and the per-rank results are concatenated in rank order
with ``cigar_off`` rebased by the number of CIGAR runs of the preceding ranks. The paper's own
multi-GPU use is the same thing with one process per GPU and no communication.

Nothing here computes an alignment: ``align_fn`` is the caller's (``Context.align_batch_host`` on a
GPU box; the tests pass the CPU oracle). ``torch.distributed`` (NCCL or gloo) is used only to gather
the results on rank 0.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import numpy as np

FIELDS = ("score", "ref_start", "ref_end", "read_start", "read_end", "passed", "n_match", "n_cols",
          "cigar_off", "cigar_len", "cigar_ops")


def pair_range(n_pairs: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous, balanced split: the first ``n_pairs % world`` ranks take one pair more."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad world/rank")
    base, extra = divmod(int(n_pairs), world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_batch(batch, world: int, rank: int):
    """This rank's share of ``batch``: same sequences, its contiguous slice of the pair list."""
    lo, hi = pair_range(batch.n_pairs, world, rank)
    return batch.subset(np.arange(lo, hi, dtype=np.int64))


def stitch(parts) -> dict:
    """Concatenate per-rank results (rank order) into one result in caller pair order."""
    out = {}
    for f in FIELDS:
        if f == "cigar_off":
            continue
        out[f] = np.concatenate([np.asarray(getattr(p, f) if not isinstance(p, dict) else p[f]) for p in parts])
    offs, base = [], 0
    for p in parts:
        get = (lambda k: p[k]) if isinstance(p, dict) else (lambda k: getattr(p, k))
        offs.append(np.asarray(get("cigar_off"), dtype=np.uint64) + np.uint64(base))
        base += int(np.asarray(get("cigar_ops")).shape[0])
    out["cigar_off"] = np.concatenate(offs) if offs else np.zeros(0, np.uint64)
    return out


def align_sharded(batch, align_fn: Callable, group=None) -> Optional[dict]:
    """Align this rank's shard with ``align_fn`` and gather everything on rank 0.

    Returns the stitched result (dict of numpy arrays, fields ``FIELDS``) on rank 0, None elsewhere.
    Works without an initialised process group (world size 1).
    """
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        world, rank = dist.get_world_size(group), dist.get_rank(group)
    else:
        world, rank = 1, 0
    res = align_fn(shard_batch(batch, world, rank))
    mine = {f: np.ascontiguousarray(getattr(res, f)) for f in FIELDS}
    if world == 1:
        return stitch([mine])
    gathered = [None] * world if rank == 0 else None
    dist.gather_object(mine, gathered, dst=0, group=group)
    return stitch(gathered) if rank == 0 else None
