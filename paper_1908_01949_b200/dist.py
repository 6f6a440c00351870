"""Host-side sharding for more than one GPU.  The path shards by independent problems
(seeds are independent): whole events across ranks (no collective at all), or -- one event on several
GPUs -- contiguous slabs of the slowest grid axis (theta).  A slab is scanned with node values that are BIT-IDENTICAL
to the full grid's (cdc_grid_spec.first carries the integer node offset, so node i of the slab is lo + (i0 + i) step),
each rank re-scores its own near-best seeds exactly (cdc_best_track, fp64), and the ranks' exact winners are merged:
the highest S = n_match - chi2 / lambda (a double, formed exactly as the single-GPU path and the oracle form it) wins,
ties go to the lowest global linear index (reading C10) -- so a sharded run returns the very seed, chi2 and labels of
the single-GPU path.  The exchange is a few bytes per event (latency only): one all_gather of (S, index, n_match, chi2)
and one all_reduce(MAX) of the owner's labels.  Plumbing only: no arithmetic of the method beyond that comparison."""
from __future__ import annotations

import copy
from typing import List, Optional, Sequence, Tuple

import numpy as np

INDEX_MASK = 0xFFFFFFFF
NO_LABEL = np.iinfo(np.int32).min


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [begin, end) of n items for `rank`; sizes differ by at most one; empty when n < world."""
    base, rem = divmod(n, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def shard_theta(grid, rank: int, world: int):
    """This rank's slab of the theta axis as a grid with the same lo / step and an integer node offset `first`, and the
    offset that maps its linear seed indices back to the full grid's (theta is the slowest axis of the linear index).
    Returns (None, 0) for an empty slab."""
    b, e = shard_range(int(grid.n[0]), rank, world)
    if e <= b:
        return None, 0
    sub = copy.deepcopy(grid)
    sub.lo = np.array(grid.lo, dtype=np.float64).copy()
    sub.n = np.array(grid.n, dtype=np.int32).copy()
    first = np.array(getattr(grid, "first", np.zeros(5)), dtype=np.int32).copy()
    first[0] += b
    sub.first = first
    sub.n[0] = e - b
    inner = int(np.prod(np.asarray(grid.n[1:], dtype=np.int64)))
    return sub, b * inner


def slab_node(sub, idx: Sequence[int]) -> np.ndarray:
    """Node values of a slab exactly as the library forms them: lo + (first + i) step."""
    first = np.asarray(getattr(sub, "first", np.zeros(5)), dtype=np.float64)
    return np.asarray(sub.lo, dtype=np.float64) + (first + np.asarray(idx, dtype=np.float64)) * np.asarray(sub.step, dtype=np.float64)


def exact_score(n_match, chi2, window_mm: float) -> np.ndarray:
    """S = n_match - chi2 / lambda in fp64 (reading C10), the quantity the exact arg max is taken over."""
    return np.asarray(n_match, dtype=np.float64) - np.asarray(chi2, dtype=np.float64) / (float(window_mm) ** 2)


def merge_slab_results(results: Sequence[Optional[dict]], offsets: Sequence[Sequence[int]], window_mm: float,
                       hit_offsets: np.ndarray) -> dict:
    """Merge per-rank results of a theta-sharded scan held in ONE process (the single-GPU test and the reference for the
    collective merge).  results[r] = output of SeedScanner.scan on rank r's slabs (or None: no slab at all);
    offsets[r][e] = index offset of event e's slab on rank r, or -1 where rank r has no slab of event e."""
    E = len(hit_offsets) - 1
    best_S = np.full(E, -1.0); best_idx = np.full(E, -1, dtype=np.int64); owner = np.full(E, -1, dtype=np.int64)
    for r, res in enumerate(results):
        if res is None:
            continue
        S = exact_score(res["best_n_match"], res["best_chi2"], window_mm)
        for e in range(E):
            if offsets[r][e] < 0 or res["best_seed"][e] < 0:
                continue
            gi = int(res["best_seed"][e]) + int(offsets[r][e])
            if S[e] > best_S[e] or (S[e] == best_S[e] and gi < best_idx[e]):
                best_S[e], best_idx[e], owner[e] = S[e], gi, r
    out = dict(best_seed=best_idx, best_S=best_S, owner=owner,
               best_n_match=np.zeros(E, dtype=np.uint32), best_chi2=np.zeros(E),
               labels=np.full(int(hit_offsets[-1]), -1, dtype=np.int32))
    for e in range(E):
        if owner[e] >= 0:
            res = results[owner[e]]
            out["best_n_match"][e] = res["best_n_match"][e]; out["best_chi2"][e] = res["best_chi2"][e]
            out["labels"][hit_offsets[e]:hit_offsets[e + 1]] = res["labels"][hit_offsets[e]:hit_offsets[e + 1]]
    return out


def merge_slab_results_collective(res: Optional[dict], offset_e: Sequence[int], window_mm: float, hit_offsets: np.ndarray,
                                  device=None, group=None) -> dict:
    """The same merge across ranks with torch.distributed (nccl on GPUs, gloo in the CPU tests): every rank passes its own
    result and gets the merged one.  Two small collectives: all_gather of (S, global index, n_match, chi2) per event and
    all_reduce(MAX) of the labels (the owner's labels, INT_MIN elsewhere)."""
    import torch
    import torch.distributed as dist
    E = len(hit_offsets) - 1
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    rec = np.zeros((E, 4), dtype=np.float64)
    rec[:, 0] = -1.0; rec[:, 1] = -1.0
    if res is not None:
        S = exact_score(res["best_n_match"], res["best_chi2"], window_mm)
        for e in range(E):
            if offset_e[e] >= 0 and res["best_seed"][e] >= 0:
                rec[e] = (S[e], float(int(res["best_seed"][e]) + int(offset_e[e])), float(res["best_n_match"][e]), 0.0)
        chi_bits = np.asarray(res["best_chi2"], dtype=np.float64).view(np.int64)
    else:
        chi_bits = np.zeros(E, dtype=np.int64)
    # indices < 2^31 and n_match are exact in a double; chi2 travels as its bit pattern in a second int64 tensor
    t = torch.from_numpy(rec).to(device) if device is not None else torch.from_numpy(rec)
    cb = torch.from_numpy(chi_bits.copy()).to(t.device)
    if world > 1:
        allrec = [torch.empty_like(t) for _ in range(world)]; allchi = [torch.empty_like(cb) for _ in range(world)]
        dist.all_gather(allrec, t, group=group); dist.all_gather(allchi, cb, group=group)
    else:
        allrec, allchi = [t], [cb]
    R = np.stack([x.cpu().numpy() for x in allrec]); CB = np.stack([x.cpu().numpy() for x in allchi])
    best_S = np.full(E, -1.0); best_idx = np.full(E, -1, dtype=np.int64); owner = np.full(E, -1, dtype=np.int64)
    for r in range(world):
        for e in range(E):
            S, gi = R[r, e, 0], int(R[r, e, 1])
            if gi < 0:
                continue
            if S > best_S[e] or (S == best_S[e] and gi < best_idx[e]):
                best_S[e], best_idx[e], owner[e] = S, gi, r
    lab = np.full(int(hit_offsets[-1]), NO_LABEL, dtype=np.int32)
    for e in range(E):
        if owner[e] == rank and res is not None:
            lab[hit_offsets[e]:hit_offsets[e + 1]] = res["labels"][hit_offsets[e]:hit_offsets[e + 1]]
    tl = torch.from_numpy(lab).to(t.device)
    if world > 1:
        dist.all_reduce(tl, op=dist.ReduceOp.MAX, group=group)
    lab = tl.cpu().numpy()
    lab[lab == NO_LABEL] = -1
    nm = np.zeros(E, dtype=np.uint32); chi2 = np.zeros(E)
    for e in range(E):
        if owner[e] >= 0:
            nm[e] = np.uint32(R[owner[e], e, 2]); chi2[e] = CB[owner[e], e:e + 1].view(np.float64)[0]
    return dict(best_seed=best_idx, best_S=best_S, owner=owner, best_n_match=nm, best_chi2=chi2, labels=lab)


def globalize_keys(keys: np.ndarray, index_offset: int) -> np.ndarray:
    """Packed fp32 keys (bits(S) << 32 | 0xFFFFFFFF - local index) -> the same with the full grid's index."""
    k = np.asarray(keys, dtype=np.uint64)
    idx = np.uint64(INDEX_MASK) - (k & np.uint64(INDEX_MASK)) + np.uint64(index_offset)
    return (k & ~np.uint64(INDEX_MASK)) | (np.uint64(INDEX_MASK) - idx)


def all_reduce_best_keys(keys_i64):
    """In-place all_reduce(MAX) of packed fp32 keys held in an int64 torch tensor (S >= 0, so the sign bit is clear
    and signed order equals unsigned order): the fused fp32 arg max across ranks (a diagnostic; the exact merge is
    merge_slab_results_collective).  Works on any backend (nccl on GPUs, gloo in the CPU tests)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(keys_i64, op=dist.ReduceOp.MAX)
    return keys_i64


def unpack_key(key: int) -> Tuple[float, int]:
    s = np.array([key >> 32], dtype=np.uint32).view(np.float32)[0]
    return float(s), int(INDEX_MASK - (key & INDEX_MASK))
