"""Convenience layer over binding.py for tests, bench.py and smoke(): allocates the caller-owned device
buffers with PyTorch and returns numpy views of the results.  Marshalling only -- no arithmetic of the method.
"""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np

from . import binding as B


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1908_01949_b200 needs a CUDA device: there is no CPU fallback")
    return torch


class SeedScanner:
    """Geometry + field on the device; runs the hot path on batches of events."""

    def __init__(self, geom, field, use_wire_table: bool = True):
        self.geometry = B.Geometry(geom, field, use_wire_table=use_wire_table)
        self.charge = -1

    def upload(self, hit_offsets, wire_id, drift_mm) -> B.Events:
        return B.Events(self.geometry, hit_offsets, wire_id, drift_mm)

    def hough(self, events: B.Events, zref: Sequence[float], hp: Optional[B.HoughParams] = None,
              want_accum: bool = False, charge: int = -1) -> dict:
        torch = _torch()
        hp = hp or B.hough_params()
        dims = B.cdc_hough_dims(hp)
        E = events.n_events
        d_zref = torch.tensor(np.asarray(zref, dtype=np.float32), device="cuda")
        d_ranges = torch.zeros((E, 3, 2), dtype=torch.float64, device="cuda")
        d_peak = torch.zeros((E, 4), dtype=torch.int32, device="cuda")
        d_acc = torch.zeros((E,) + dims, dtype=torch.int32, device="cuda") if want_accum else None
        B.cdc_hough_seed_ranges(self.geometry, events, hp, charge, d_zref, d_ranges, d_peak, d_acc)
        torch.cuda.synchronize()
        return dict(ranges=d_ranges.cpu().numpy(), peak=d_peak.cpu().numpy(), dims=dims,
                    accum=None if d_acc is None else d_acc.cpu().numpy().astype(np.uint32))

    def scan(self, events: B.Events, grids: Sequence, params: B.ScanParams, per_seed: bool = True,
             debug: bool = False, best: bool = True) -> dict:
        """cdc_seed_scan (+ cdc_best_track).  Returns numpy arrays; per-seed outputs are concatenated over events."""
        torch = _torch()
        E = events.n_events
        specs = B.grid_specs(grids)
        n_seeds = [int(np.prod(np.asarray(g.n, dtype=np.int64))) for g in grids]
        total = int(sum(n_seeds))
        d_key = torch.zeros(E, dtype=torch.int64, device="cuda")
        d_nm = torch.zeros(total, dtype=torch.int32, device="cuda") if per_seed else None
        d_c2 = torch.zeros(total, dtype=torch.float32, device="cuda") if per_seed else None
        d_dbg = torch.zeros(total * B.SEED_DEBUG_DTYPE.itemsize, dtype=torch.uint8, device="cuda") if debug else None
        B.cdc_seed_scan(self.geometry, events, specs, params, d_key, d_nm, d_c2, d_dbg)
        out = dict(n_seeds=n_seeds)
        if best:
            d_seed = torch.zeros(E, dtype=torch.int64, device="cuda")
            d_bnm = torch.zeros(E, dtype=torch.int32, device="cuda")
            d_bc2 = torch.zeros(E, dtype=torch.float64, device="cuda")
            d_lab = torch.zeros(max(events.n_hits, 1), dtype=torch.int32, device="cuda")
            B.cdc_best_track(self.geometry, events, specs, params, d_key, d_seed, d_bnm, d_bc2, d_lab)
            torch.cuda.synchronize()
            out.update(best_seed=d_seed.cpu().numpy(), best_n_match=d_bnm.cpu().numpy().astype(np.uint32),
                       best_chi2=d_bc2.cpu().numpy(), labels=d_lab.cpu().numpy()[:events.n_hits])
        torch.cuda.synchronize()
        key = d_key.cpu().numpy().view(np.uint64)
        out["best_key"] = key
        out["S32_max"] = (key >> np.uint64(32)).astype(np.uint32).view(np.float32)
        out["S32_argmax"] = (np.uint64(0xFFFFFFFF) - (key & np.uint64(0xFFFFFFFF))).astype(np.int64)
        out["stats"] = B.cdc_scan_get_stats(events)
        if per_seed:
            out["n_match"] = d_nm.cpu().numpy().astype(np.uint32)
            out["chi2"] = d_c2.cpu().numpy()
        if debug:
            out["debug"] = d_dbg.cpu().numpy().view(B.SEED_DEBUG_DTYPE)
        return out

    def scan_adaptive(self, events: B.Events, grids: Sequence, params: B.ScanParams, tol_mm: float, h_max_mm: float) -> dict:
        """cdc_seed_scan_adaptive with every per-seed output; numpy arrays concatenated over events."""
        torch = _torch()
        E = events.n_events
        n_seeds = [int(np.prod(np.asarray(g.n, dtype=np.int64))) for g in grids]
        total = int(sum(n_seeds))
        d_key = torch.zeros(E, dtype=torch.int64, device="cuda")
        d_nm = torch.zeros(total, dtype=torch.int32, device="cuda"); d_c2 = torch.zeros(total, dtype=torch.float32, device="cuda")
        d_dbg = torch.zeros(total * B.SEED_DEBUG_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
        d_lev = torch.zeros((total, 8), dtype=torch.int32, device="cuda")
        B.cdc_seed_scan_adaptive(self.geometry, events, B.grid_specs(grids), params, tol_mm, h_max_mm, d_key, d_nm, d_c2,
                                 d_dbg, d_lev)
        torch.cuda.synchronize()
        key = d_key.cpu().numpy().view(np.uint64)
        lev = d_lev.cpu().numpy()
        return dict(n_seeds=n_seeds, n_match=d_nm.cpu().numpy().astype(np.uint32), chi2=d_c2.cpu().numpy(),
                    debug=d_dbg.cpu().numpy().view(B.SEED_DEBUG_DTYPE), n_level=lev[:, :7], seq_hash=lev[:, 7].view(np.uint32),
                    best_key=key, S32_max=(key >> np.uint64(32)).astype(np.uint32).view(np.float32),
                    S32_argmax=(np.uint64(0xFFFFFFFF) - (key & np.uint64(0xFFFFFFFF))).astype(np.int64),
                    stats=B.cdc_scan_get_stats(events))

    def slabs(self, grids: Sequence, rank: int, world: int):
        """This rank's theta slab of every grid (dist.shard_theta) and the index offsets back to the full grids; an
        event whose theta axis has fewer nodes than ranks gets a one-node placeholder here and offset -1 (ignored)."""
        import copy
        from . import dist as D
        subs, offs = [], []
        for g in grids:
            sub, off = D.shard_theta(g, rank, world)
            if sub is None:
                sub = copy.deepcopy(g)
                sub.n = np.ones(5, dtype=np.int32); sub.first = np.zeros(5, dtype=np.int32)
                off = -1
            subs.append(sub); offs.append(off)
        return subs, offs

    def scan_sharded(self, events: B.Events, grids: Sequence, params: B.ScanParams, rank: int, world: int,
                     hit_offsets, collective: bool = True) -> dict:
        """One event batch whose seed grids are split over `world` GPUs along theta: this rank
        scans its slabs (node values bit-identical to the full grids'), re-scores its near-best seeds exactly, and the
        ranks' exact winners are merged (highest fp64 S, then lowest global index).  collective=True merges over
        torch.distributed and returns the merged result on every rank; collective=False returns this rank's own
        (result, offsets) for dist.merge_slab_results."""
        from . import dist as D
        subs, offs = self.slabs(grids, rank, world)
        res = self.scan(events, subs, params, per_seed=False, debug=False)
        if not collective:
            return dict(result=res, offsets=offs)
        torch = _torch()
        return D.merge_slab_results_collective(res, offs, float(params.window_mm), np.asarray(hit_offsets),
                                               device=torch.device("cuda", torch.cuda.current_device()))

    def find_tracks_host(self, hit_offsets, wire_id, drift_mm, grids: Sequence, params: B.ScanParams,
                         hp: Optional[B.HoughParams] = None, zref=None, hough_sets_axes: bool = True) -> dict:
        return B.cdc_find_tracks_host(self.geometry, hit_offsets, wire_id, drift_mm, B.grid_specs(grids), params,
                                      hp, zref, hough_sets_axes)

    def refine(self, events: B.Events, grids: Sequence, params: B.ScanParams, n_parents: int = 8,
               n_iterations: int = 10, **kw) -> dict:
        """Coarse-to-fine refinement around the best seeds of `grids` (cdc_refine_tracks)."""
        return B.cdc_refine_tracks(self.geometry, events, B.grid_specs(grids), params, n_parents=n_parents,
                                   n_iterations=n_iterations, **kw)

    def peel(self, events: B.Events, grids0: Sequence, params: B.ScanParams, n: Sequence[int],
             half_width: Sequence[float], **kw) -> dict:
        """Turn-partition peeling from partition 0's grids (cdc_peel_turns)."""
        return B.cdc_peel_turns(self.geometry, events, B.grid_specs(grids0), params, n, half_width, **kw)

    def close(self):
        self.geometry.close()
