"""Multi-GPU batches: shard by sequence, no data-path collective.

A single fold does not shard (every cell needs its whole row and column): N GPUs run N
replicas.  A batch of independent sequences shards naturally: the length-sorted list is dealt round-robin
to the ranks (equal counts, near-equal work: the cost of a fold grows like n^3), every rank folds its own
sequences with its own R table, and only the int32 scores travel -- one gather of `count` integers to
rank 0, plumbing outside the timed data path.  This module is host logic only (no kernels, no arithmetic
of the method); the world-size-2 gloo test in tests/test_shard_gloo.py covers it on CPU.
"""
from __future__ import annotations

import numpy as np


def shard_indices(lens, world: int, rank: int) -> np.ndarray:
    """Indices (into the caller's batch) of the sequences rank `rank` of `world` folds.

    Longest first, dealt round-robin; ties keep the original order, so the partition is deterministic."""
    lens = np.asarray(lens)
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad world/rank")
    order = np.argsort(-lens.astype(np.int64), kind="stable")
    return order[rank::world]


def fold_batch_sharded(fold_fn, seqs, lens, world: int, rank: int, dist=None):
    """Folds this rank's shard with `fold_fn(list_of_bytes, int32 lens) -> int32 scores` (on a GPU rank:
    a closure over Rna4r.fold_batch_host) and returns the scores of the WHOLE batch in the caller's order on
    rank 0 (None on the other ranks).  `dist` is torch.distributed (any backend) or None for world == 1."""
    idx = shard_indices(lens, world, rank)
    mine = np.asarray(fold_fn([seqs[i] for i in idx], np.asarray(lens, dtype=np.int32)[idx]), dtype=np.int32)
    if mine.shape != idx.shape:
        raise ValueError("fold_fn returned the wrong number of scores")
    if world == 1:
        out = np.empty(len(lens), dtype=np.int32)
        out[idx] = mine
        return out
    gathered = [None] * world if rank == 0 else None
    dist.gather_object((idx, mine), gathered, dst=0)
    if rank != 0:
        return None
    out = np.full(len(lens), np.iinfo(np.int32).min, dtype=np.int32)
    seen = np.zeros(len(lens), dtype=bool)
    for ridx, rsc in gathered:
        if seen[ridx].any():
            raise RuntimeError("a sequence was folded by two ranks")
        seen[ridx] = True
        out[ridx] = rsc
    if not seen.all():
        raise RuntimeError("a sequence was folded by no rank")
    return out
