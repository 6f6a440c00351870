"""World-size-2 gloo tests (CPU) of the multi-GPU host logic: event / theta-slab sharding and the packed-key
all_reduce(MAX) that merges per-rank best seeds."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1908_01949_b200 import dist as D, synth


def _pack(S, idx):
    return (np.array(S, dtype=np.float32).view(np.uint32).astype(np.uint64) << np.uint64(32)) | \
        (np.uint64(0xFFFFFFFF) - np.asarray(idx, dtype=np.uint64))


def test_shard_range_partitions_exactly():
    for n in (0, 1, 2, 7, 16, 256):
        for world in (1, 2, 3, 8):
            parts = [D.shard_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
            sizes = [e - b for b, e in parts]
            assert max(sizes) - min(sizes) <= 1


def test_theta_slabs_cover_the_grid_in_index_order():
    grid, _ = synth.truth_anchored_grid(np.array([0.3, 10.0, 50.0, 60.0, 40.0]), [5, 3, 2, 4, 3])
    seen = []
    for r in range(3):
        sub, off = D.shard_theta(grid, r, 3)
        assert np.array_equal(sub.lo, grid.lo) and int(sub.first[0]) == off // int(np.prod(grid.n[1:]))
        for lin in range(sub.n_seeds):
            node = D.slab_node(sub, sub.unravel(lin))                   # lo + (first + i) step, as the library forms it
            assert np.array_equal(node, grid.node(grid.unravel(lin + off)))    # bit-identical to the full grid's node
            seen.append(lin + off)
    assert seen == list(range(grid.n_seeds))
    assert D.shard_theta(grid, 7, 8) == (None, 0)          # more ranks than theta nodes: empty slab


def test_globalize_and_unpack_keys():
    k = _pack([3.5, 0.0], [7, 0])
    g = D.globalize_keys(k, 1000)
    assert D.unpack_key(int(g[0])) == (3.5, 1007) and D.unpack_key(int(g[1])) == (0.0, 1000)
    # higher score wins; equal score -> lower index wins under MAX
    assert _pack([4.0], [9])[0] > _pack([3.5], [1])[0] and _pack([4.0], [2])[0] > _pack([4.0], [3])[0]


def _fake_rank_result(rank, world, E, hit_offsets, seed=5):
    """Per-rank 'exact winners' of a theta-sharded scan with many ties across ranks (same for every caller)."""
    rng = np.random.default_rng(seed + rank)
    nm = rng.integers(20, 24, size=E).astype(np.uint32)
    chi2 = rng.integers(0, 3, size=E).astype(np.float64) * 0.25
    seedidx = rng.integers(0, 50, size=E).astype(np.int64)
    labels = rng.integers(-1, 3, size=int(hit_offsets[-1])).astype(np.int32)
    offs = [rank * 1000 if (e + rank) % 4 != 3 else -1 for e in range(E)]          # some ranks own no slab of some events
    return dict(best_seed=seedidx, best_n_match=nm, best_chi2=chi2, labels=labels), offs


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(5)
    E, n_theta, inner = 4, 6, 40
    S = rng.integers(0, 30, size=(E, n_theta * inner)).astype(np.float32) * 0.25     # many ties
    b, e = D.shard_range(n_theta, rank, world)
    local = S[:, b * inner:e * inner]
    li = np.array([int(np.flatnonzero(row == row.max())[0]) for row in local])
    keys = D.globalize_keys(_pack(local[np.arange(E), li], li), b * inner)
    t = torch.from_numpy(keys.view(np.int64).copy())
    D.all_reduce_best_keys(t)
    q.put((rank, t.numpy().view(np.uint64).tolist()))
    # event sharding: ranks own disjoint event ranges, nothing to reduce
    q.put((rank, D.shard_range(E, rank, world)))
    # the exact merge of a theta-sharded scan (fp64 S, lowest global index, owner's labels) as a collective
    hit_offsets = np.array([0, 3, 7, 7, 12, 20, 21])
    res, offs = _fake_rank_result(rank, world, 6, hit_offsets)
    m = D.merge_slab_results_collective(res, offs, 1.0, hit_offsets)
    q.put((rank, {k: m[k].tolist() for k in ("best_seed", "best_n_match", "best_chi2", "labels", "owner")}))
    dist.destroy_process_group()


def test_two_rank_key_reduction_equals_single_process_argmax():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in procs]
    got = [q.get(timeout=120) for _ in range(6)]
    [p.join(timeout=60) for p in procs]
    assert all(p.exitcode == 0 for p in procs)
    rng = np.random.default_rng(5)
    S = rng.integers(0, 30, size=(4, 240)).astype(np.float32) * 0.25
    want = [(float(row.max()), int(np.flatnonzero(row == row.max())[0])) for row in S]
    keys = [g[1] for g in got if isinstance(g[1], list)]
    assert len(keys) == 2 and keys[0] == keys[1]
    assert [D.unpack_key(k) for k in keys[0]] == want
    ranges = sorted(g[1] for g in got if isinstance(g[1], tuple))
    assert ranges == [(0, 2), (2, 4)]
    # collective merge == the single-process merge of the same per-rank results, on both ranks
    hit_offsets = np.array([0, 3, 7, 7, 12, 20, 21])
    per_rank = [_fake_rank_result(r, 2, 6, hit_offsets) for r in range(2)]
    ref = D.merge_slab_results([p[0] for p in per_rank], [p[1] for p in per_rank], 1.0, hit_offsets)
    merged = [g[1] for g in got if isinstance(g[1], dict)]
    assert len(merged) == 2
    for m in merged:
        for k in ("best_seed", "best_n_match", "best_chi2", "labels", "owner"):
            assert m[k] == ref[k].tolist(), k
    assert (ref["owner"] >= 0).all() and len(set(ref["owner"].tolist())) == 2          # both ranks win somewhere
