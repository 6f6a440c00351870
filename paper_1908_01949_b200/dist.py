"""Host-side sharding helpers for more than one GPU.  The path shards by independent
problems: whole events across ranks (no collective), or -- one event on several GPUs -- contiguous slabs of the
slowest grid axis (theta), followed by ONE all_reduce(MAX) of the packed 64-bit (score, ~index) keys.
Plumbing only: no arithmetic of the method."""
from __future__ import annotations

import copy
from typing import Tuple

import numpy as np

INDEX_MASK = 0xFFFFFFFF


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [begin, end) of n items for `rank`; sizes differ by at most one; empty when n < world."""
    base, rem = divmod(n, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def shard_theta(grid, rank: int, world: int):
    """Sub-grid holding this rank's slab of the theta axis, and the offset that maps its linear seed indices
    back to the full grid's (theta is the slowest axis of the linear index).  Returns (None, 0) for an empty slab."""
    b, e = shard_range(int(grid.n[0]), rank, world)
    if e <= b:
        return None, 0
    sub = copy.deepcopy(grid)
    sub.lo = np.array(grid.lo, dtype=np.float64).copy()
    sub.n = np.array(grid.n, dtype=np.int32).copy()
    sub.lo[0] = grid.lo[0] + b * grid.step[0]
    sub.n[0] = e - b
    inner = int(np.prod(np.asarray(grid.n[1:], dtype=np.int64)))
    return sub, b * inner


def globalize_keys(keys: np.ndarray, index_offset: int) -> np.ndarray:
    """Packed keys (bits(S) << 32 | 0xFFFFFFFF - local index) -> the same with the full grid's index."""
    k = np.asarray(keys, dtype=np.uint64)
    idx = np.uint64(INDEX_MASK) - (k & np.uint64(INDEX_MASK)) + np.uint64(index_offset)
    return (k & ~np.uint64(INDEX_MASK)) | (np.uint64(INDEX_MASK) - idx)


def all_reduce_best_keys(keys_i64):
    """In-place all_reduce(MAX) of packed keys held in an int64 torch tensor (S >= 0, so the sign bit is clear
    and signed order equals unsigned order).  Works on any backend (nccl on GPUs, gloo in the CPU tests)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(keys_i64, op=dist.ReduceOp.MAX)
    return keys_i64


def unpack_key(key: int) -> Tuple[float, int]:
    s = np.array([key >> 32], dtype=np.uint32).view(np.float32)[0]
    return float(s), int(INDEX_MASK - (key & INDEX_MASK))
