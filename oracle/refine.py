"""Coarse-to-fine refinement of the seed scan -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see cdc_oracle.c header).

PAPER.md:69: "After calculating E for all seeds, we took the several candidate seeds with the lowest E, and make
other seed sets around them with finer granularity.  Afterwards, the same scanning process was repeated ten times
to get enough resolution for the seed selection."  The paper gives neither the number of candidates nor the shrink
factor; reading C17:

  * every seed lives on the integer lattice of the FINEST pitch: value[a] = lo0[a] + q[a] * s_T[a], s_T = s_0 / 2^T,
    so a node of the initial grid G0 has q = i * 2^T;
  * iteration 0 scans G0; iteration t = 1..T scans, around each parent, the 3^5 nodes q_parent + {-d, 0, +d}^5 with
    d = 2^(T - t) (pitch halves every iteration; the parent is the centre node, so the best S never decreases);
  * after each iteration the parents are the K scanned seeds with the highest S = n_match - chi2 / lambda, ordered by
    (S descending, rank of the sub-grid they were scanned in, linear index in it); a seed whose lattice point q was
    already taken is skipped (overlapping sub-grids scan some points twice);
  * the result is the first parent of the last iteration.

Plain and slow: each sub-grid is handed to the exhaustive oracle scan as an ordinary 3^5 grid (lo, step, n), the
selection is a Python sort.
"""
from __future__ import annotations

import types

import numpy as np

from . import Bound, scan, scan_parallel

N_SUB = 3


def _subgrid(lo0, s_fine, q_parent, d):
    lo = lo0 + (np.asarray(q_parent, dtype=np.int64) - d).astype(np.float64) * s_fine
    return types.SimpleNamespace(lo=lo, step=float(d) * s_fine, n=np.full(5, N_SUB, dtype=np.int32))


def _unravel(idx, n):
    out = []
    for a in reversed(range(5)):
        out.append(idx % int(n[a])); idx //= int(n[a])
    return tuple(reversed(out))


def _select(cands, K):
    """cands: list of (S, rank, idx, q-tuple, n_match, chi2).  -> first K distinct lattice points in the order
    (S desc, rank asc, idx asc)."""
    cands = sorted(cands, key=lambda c: (-c[0], c[1], c[2]))
    taken, seen = [], set()
    for c in cands:
        if c[3] in seen:
            continue
        seen.add(c[3]); taken.append(c)
        if len(taken) == K:
            break
    return taken


def refine(geom, field, params: dict, wire_id, drift, grid0, K: int = 8, T: int = 10, n_proc=None):
    """Returns dict(seed (5,), S, n_match, chi2, q (5,), trace = per-iteration list of parents (q, S))."""
    lam = float(params["window"]) ** 2
    lo0 = np.asarray(grid0.lo, dtype=np.float64)
    s_fine = np.asarray(grid0.step, dtype=np.float64) / float(2 ** T)
    n0 = np.asarray(grid0.n, dtype=np.int64)
    # iteration 0: the initial grid
    out = scan_parallel(geom, field, params, wire_id, drift, grid0, n_proc=n_proc)
    S = out["n_match"].astype(np.float64) - out["chi2"] / lam
    order = np.lexsort((np.arange(S.size), -S))[:K]               # (S desc, index asc); G0 nodes are distinct
    parents = [(float(S[i]), 0, int(i), tuple(int(c) * 2 ** T for c in _unravel(int(i), n0)),
                int(out["n_match"][i]), float(out["chi2"][i])) for i in order]
    trace = [[(p[3], p[0]) for p in parents]]
    bound = Bound(geom, field, params)
    for t in range(1, T + 1):
        d = 2 ** (T - t)
        cands = []
        for rank, par in enumerate(parents):
            g = _subgrid(lo0, s_fine, par[3], d)
            o = scan(bound, wire_id, drift, g, details=False)
            Ss = o["n_match"].astype(np.float64) - o["chi2"] / lam
            for idx in range(N_SUB ** 5):
                off = _unravel(idx, g.n)
                q = tuple(int(par[3][a]) + (off[a] - 1) * d for a in range(5))
                cands.append((float(Ss[idx]), rank, idx, q, int(o["n_match"][idx]), float(o["chi2"][idx])))
        parents = _select(cands, K)
        trace.append([(p[3], p[0]) for p in parents])
    best = parents[0]
    q = np.array(best[3], dtype=np.int64)
    # the value the winning sub-grid handed to the scan: lo + i * step of that 3^5 grid (one rounding per axis)
    if T > 0:
        seed = None
        d = 1
        for rank, par in enumerate(trace[T - 1]):
            g = _subgrid(lo0, s_fine, par[0], d)
            off = (q - (np.asarray(par[0], dtype=np.int64) - d)) // d
            if np.all((off >= 0) & (off < N_SUB)) and rank == best[1]:
                seed = g.lo + off.astype(np.float64) * g.step
        assert seed is not None
    else:
        seed = lo0 + np.array(_unravel(best[2], n0), dtype=np.float64) * np.asarray(grid0.step, dtype=np.float64)
    return dict(seed=seed, S=best[0], n_match=best[4], chi2=best[5], q=q, trace=trace)
