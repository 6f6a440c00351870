"""ctypes front end of oracle/cdc_oracle.c.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
never imports paper_1908_01949_b200 (geometry/field/event objects are taken by
attribute, i.e. anything shaped like the records of the seeded input generator).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

_lib = None


class OrcGeom(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("r_mm", C.c_void_p), ("n_wires", C.c_void_p),
                ("phi0", C.c_void_p), ("stereo", C.c_void_p), ("offset", C.c_void_p),
                ("n_wires_total", C.c_int32), ("wire", C.c_void_p),
                ("z_half", C.c_double), ("R0", C.c_double), ("r_out", C.c_double)]


class OrcField(C.Structure):
    _fields_ = [("kind", C.c_int32), ("bz", C.c_double), ("nr", C.c_int32), ("nz", C.c_int32),
                ("r0", C.c_double), ("z0", C.c_double), ("dr", C.c_double), ("dz", C.c_double),
                ("tab", C.c_void_p)]


class OrcParams(C.Structure):
    _fields_ = [("h", C.c_double), ("max_steps", C.c_int32), ("window", C.c_double),
                ("eloss", C.c_double), ("charge", C.c_int32)]


class OrcHits(C.Structure):
    _fields_ = [("n_hits", C.c_int32), ("wire_id", C.c_void_p), ("drift", C.c_void_p)]


class OrcApproach(C.Structure):
    _fields_ = [("interval", C.c_int32), ("hit", C.c_int32), ("wire", C.c_int32), ("turn", C.c_int32),
                ("matched", C.c_int32), ("D", C.c_double), ("resid", C.c_double), ("zw", C.c_double)]


class OrcResult(C.Structure):
    _fields_ = [("n_match", C.c_int32), ("n_steps", C.c_int32), ("turns", C.c_int32), ("m_gas", C.c_int32),
                ("chi2", C.c_double), ("r", C.c_double * 3), ("T", C.c_double * 3), ("p", C.c_double),
                ("n_rec", C.c_int32)]


class OrcHoughParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("bin_xy", "bin_R", "tol", "R_lo", "R_hi", "half_xy", "origin",
                                          "half_theta", "half_pt")]


APPROACH_DTYPE = np.dtype([("interval", "i4"), ("hit", "i4"), ("wire", "i4"), ("turn", "i4"),
                           ("matched", "i4"), ("pad", "i4"), ("D", "f8"), ("resid", "f8"), ("zw", "f8")])
assert APPROACH_DTYPE.itemsize == C.sizeof(OrcApproach)

HOUGH_DEFAULT = dict(bin_xy=4.0, bin_R=4.0, tol=6.0, R_lo=240.0, R_hi=364.0, half_xy=460.0, origin=100.0,
                     half_theta=0.03, half_pt=7.5)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_argmax.restype = C.c_int64
    return _lib


def timed_with_fast_build(fn):
    """Run fn() with the speed build of the same source loaded (bench.py's second CPU number), then restore the
    parity build.  Timing only."""
    global _lib
    lib()
    keep = _lib
    fast = C.CDLL(_build.build_fast())
    fast.orc_argmax.restype = C.c_int64
    try:
        _lib = fast
        return fn()
    finally:
        _lib = keep


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Bound:
    """Keeps the numpy buffers alive behind the C structs."""

    def __init__(self, geom, field, params: dict):
        self.keep = []
        k = self.keep
        def arr(a, dt):
            a = np.ascontiguousarray(a, dtype=dt); k.append(a); return a
        self.n_wires_total = int(geom.offset[-1])
        self.g = OrcGeom(int(len(geom.r_mm)), _p(arr(geom.r_mm, np.float64)), _p(arr(geom.n_wires, np.int32)),
                         _p(arr(geom.phi0_rad, np.float64)), _p(arr(geom.stereo_rad, np.float64)),
                         _p(arr(geom.offset, np.int32)), self.n_wires_total, _p(arr(geom.wire, np.float32)),
                         float(geom.z_half_mm), float(geom.R0_mm), float(geom.r_out_mm))
        tab = arr(field.table, np.float32) if field.kind == 1 else None
        self.f = OrcField(int(field.kind), float(field.bz_T), int(field.nr), int(field.nz), float(field.r0_mm),
                          float(field.z0_mm), float(field.dr_mm), float(field.dz_mm), _p(tab))
        self.P = OrcParams(float(params["h"]), int(params["max_steps"]), float(params["window"]),
                           float(params.get("eloss", 0.0)), int(params.get("charge", -1)))
        self.window = float(params["window"])

    def hits(self, wire_id, drift):
        w = np.ascontiguousarray(wire_id, dtype=np.int32)
        d = np.ascontiguousarray(drift, dtype=np.float32)
        self.keep += [w, d]
        how = -np.ones(self.n_wires_total, dtype=np.int32)
        how[w] = np.arange(w.size, dtype=np.int32)
        return OrcHits(int(w.size), _p(w), _p(d)), how


def field_at(bound: Bound, xyz: Sequence[float]) -> np.ndarray:
    B = np.zeros(3)
    lib().orc_field_at(C.byref(bound.f), C.c_double(xyz[0]), C.c_double(xyz[1]), C.c_double(xyz[2]), _p(B))
    return B


def rkn_step(bound: Bound, a: float, h: float, r, T):
    r = np.ascontiguousarray(r, dtype=np.float64); T = np.ascontiguousarray(T, dtype=np.float64)
    rn = np.zeros(3); Tn = np.zeros(3)
    lib().orc_rkn_step(C.byref(bound.f), C.c_double(a), C.c_double(h), _p(r), _p(T), _p(rn), _p(Tn))
    return rn, Tn


def rkn_step_err(bound: Bound, a: float, h: float, r, T):
    """One RKN step and the local error estimate h^2 max|k1 - k2 - k3 + k4| of PAPER.md ref. [5] (reading C19)."""
    r = np.ascontiguousarray(r, dtype=np.float64); T = np.ascontiguousarray(T, dtype=np.float64)
    rn = np.zeros(3); Tn = np.zeros(3); err = C.c_double()
    lib().orc_rkn_step_err(C.byref(bound.f), C.c_double(a), C.c_double(h), _p(r), _p(T), _p(rn), _p(Tn), C.byref(err))
    return rn, Tn, float(err.value)


def eval_seed(bound: Bound, wire_id, drift, seed, mode: int = 1, records: bool = False,
              rec_slack: float = 0.0, trajectory: bool = False):
    """Evaluate one seed.  Returns dict(n_match, chi2, n_steps, turns, m_gas, r, T, p[, rec][, traj])."""
    H, how = bound.hits(wire_id, drift)
    seed = np.ascontiguousarray(seed, dtype=np.float64)
    res = OrcResult()
    cap = (64 * max(int(H.n_hits), 1) + 4096) if records else 0
    rec = np.zeros(cap, dtype=APPROACH_DTYPE) if records else None
    traj = np.zeros((bound.P.max_steps + 1, 6)) if trajectory else None
    lib().orc_eval_seed(C.byref(bound.g), C.byref(bound.f), C.byref(H), _p(how), _p(seed), C.byref(bound.P),
                        C.c_int32(mode), C.byref(res), _p(rec), C.c_int32(cap), C.c_double(rec_slack), _p(traj))
    out = dict(n_match=res.n_match, chi2=res.chi2, n_steps=res.n_steps, turns=res.turns, m_gas=res.m_gas,
               r=np.array(res.r[:]), T=np.array(res.T[:]), p=res.p)
    if records:
        assert res.n_rec < cap, "approach record buffer overflow"
        out["rec"] = rec[:res.n_rec]
    if trajectory:
        out["traj"] = traj[:res.n_steps + 1]
    return out


def scan(bound: Bound, wire_id, drift, grid, begin: int = 0, end: Optional[int] = None,
         index_list: Optional[np.ndarray] = None, mode: int = 1, details: bool = True):
    """Exhaustive evaluation of seeds [begin, end) of `grid` (or of index_list[begin:end])."""
    H, _ = bound.hits(wire_id, drift)
    lo = np.ascontiguousarray(grid.lo, dtype=np.float64)
    st = np.ascontiguousarray(grid.step, dtype=np.float64)
    nn = np.ascontiguousarray(grid.n, dtype=np.int32)
    il = None if index_list is None else np.ascontiguousarray(index_list, dtype=np.int64)
    if end is None:
        end = int(il.size) if il is not None else int(np.prod(nn.astype(np.int64)))
    n = end - begin
    nm = np.zeros(n, dtype=np.int32); c2 = np.zeros(n)
    ns = np.zeros(n, dtype=np.int32) if details else None
    tu = np.zeros(n, dtype=np.int32) if details else None
    fr = np.zeros((n, 3)) if details else None
    mg = np.zeros(n, dtype=np.int32) if details else None
    lib().orc_scan(C.byref(bound.g), C.byref(bound.f), C.byref(H), _p(lo), _p(st), _p(nn), _p(il),
                   C.c_int64(begin), C.c_int64(end), C.byref(bound.P), C.c_int32(mode),
                   _p(nm), _p(c2), _p(ns), _p(tu), _p(fr), _p(mg))
    return dict(n_match=nm, chi2=c2, n_steps=ns, turns=tu, final_r=fr, m_gas=mg)


def _scan_worker(args):
    geom, field, params, wire_id, drift, grid, b, e, il, mode = args
    return scan(Bound(geom, field, params), wire_id, drift, grid, b, e, il, mode)


def scan_parallel(geom, field, params: dict, wire_id, drift, grid, index_list=None, mode: int = 1,
                  n_proc: Optional[int] = None):
    """The same exhaustive scan split over host cores by seed range; every process is still the
    single-threaded oracle (used only to keep the test suite's wall time down)."""
    import multiprocessing as mp
    total = int(index_list.size) if index_list is not None else grid.n_seeds
    n_proc = n_proc or min(os.cpu_count() or 1, 8)
    n_chunks = max(1, min(total, n_proc * 4))
    edges = np.linspace(0, total, n_chunks + 1).astype(np.int64)
    jobs = [(geom, field, params, wire_id, drift, grid, int(edges[i]), int(edges[i + 1]), index_list, mode)
            for i in range(n_chunks) if edges[i + 1] > edges[i]]
    if n_proc == 1 or len(jobs) == 1:
        parts = [_scan_worker(j) for j in jobs]
    else:
        with mp.get_context("fork").Pool(n_proc) as pool:
            parts = pool.map(_scan_worker, jobs)
    return {k: np.concatenate([p[k] for p in parts]) for k in parts[0]}


def argmax(n_match: np.ndarray, chi2: np.ndarray, window: float):
    nm = np.ascontiguousarray(n_match, dtype=np.int32); c2 = np.ascontiguousarray(chi2, dtype=np.float64)
    S = C.c_double()
    i = lib().orc_argmax(C.c_int64(nm.size), _p(nm), _p(c2), C.c_double(window), C.byref(S))
    return int(i), float(S.value)


def labels(bound: Bound, wire_id, drift, seed, mode: int = 1):
    H, _ = bound.hits(wire_id, drift)
    seed = np.ascontiguousarray(seed, dtype=np.float64)
    lab = np.zeros(max(int(H.n_hits), 1), dtype=np.int32)
    res = OrcResult()
    lib().orc_labels(C.byref(bound.g), C.byref(bound.f), C.byref(H), _p(seed), C.byref(bound.P), C.c_int32(mode),
                     _p(lab), C.byref(res))
    return lab[:H.n_hits], dict(n_match=res.n_match, chi2=res.chi2, n_steps=res.n_steps, turns=res.turns)


def seed_of_index(grid, idx: int) -> np.ndarray:
    lo = np.ascontiguousarray(grid.lo, dtype=np.float64); st = np.ascontiguousarray(grid.step, dtype=np.float64)
    nn = np.ascontiguousarray(grid.n, dtype=np.int32); s = np.zeros(5)
    lib().orc_seed_of_index(_p(lo), _p(st), _p(nn), C.c_int64(idx), _p(s))
    return s


def hough(bound: Bound, wire_id, drift, zref: float, hp: Optional[dict] = None, want_accum: bool = True,
          bz: float = 1.0, charge: int = -1):
    H, _ = bound.hits(wire_id, drift)
    d = dict(HOUGH_DEFAULT); d.update(hp or {})
    HP = OrcHoughParams(*[float(d[k]) for k, _ in OrcHoughParams._fields_])
    dims = np.zeros(3, dtype=np.int32)
    lib().orc_hough_dims(C.byref(HP), _p(dims))
    acc = np.zeros(tuple(int(x) for x in dims), dtype=np.uint32) if want_accum else None
    peak = np.zeros(4, dtype=np.int32); ranges = np.zeros(6)
    lib().orc_hough(C.byref(bound.g), C.byref(H), C.c_double(zref), C.byref(HP), C.c_double(bz), C.c_int32(charge),
                    _p(acc), _p(peak), _p(ranges))
    return dict(accum=acc, peak=peak, ranges=ranges.reshape(3, 2), dims=dims)


def bin_event(bound: Bound, wire_id, drift) -> np.ndarray:
    H, _ = bound.hits(wire_id, drift)
    out = np.zeros(bound.n_wires_total, dtype=np.float32)
    lib().orc_bin_event(C.byref(bound.g), C.byref(H), _p(out))
    return out


class OrcAdaptiveInfo(C.Structure):
    _fields_ = [("units", C.c_int32), ("n_level", C.c_int32 * 8), ("margin_tol", C.c_double), ("margin_up", C.c_double),
                ("seq_hash", C.c_uint32), ("kmargin_tol", C.c_double), ("kmargin_up", C.c_double),
                ("r0_margin", C.c_double), ("exit_margin", C.c_double)]


def eval_seed_adaptive(bound: Bound, wire_id, drift, seed, tol: float, h_max: float, records: bool = False,
                       rec_slack: float = 0.0):
    """One seed with the adaptive step of reading C19 applied to the scan (orc_eval_seed_adaptive).  Returns the fields
    of eval_seed plus units (path in units of h), n_level (accepted steps per level) and the decision margins."""
    H, _ = bound.hits(wire_id, drift)
    seed = np.ascontiguousarray(seed, dtype=np.float64)
    res = OrcResult(); info = OrcAdaptiveInfo()
    cap = (64 * max(int(H.n_hits), 1) + 4096) if records else 0
    rec = np.zeros(cap, dtype=APPROACH_DTYPE) if records else None
    lib().orc_eval_seed_adaptive(C.byref(bound.g), C.byref(bound.f), C.byref(H), _p(seed), C.byref(bound.P),
                                 C.c_double(tol), C.c_double(h_max), C.byref(res), C.byref(info), _p(rec), C.c_int32(cap),
                                 C.c_double(rec_slack))
    out = dict(n_match=res.n_match, chi2=res.chi2, n_steps=res.n_steps, turns=res.turns, m_gas=res.m_gas,
               r=np.array(res.r[:]), T=np.array(res.T[:]), p=res.p, units=info.units, n_level=np.array(info.n_level[:]),
               margin_tol=info.margin_tol, margin_up=info.margin_up, seq_hash=int(info.seq_hash),
               kmargin_tol=info.kmargin_tol, kmargin_up=info.kmargin_up, r0_margin=info.r0_margin,
               exit_margin=info.exit_margin)
    if records:
        out["rec"] = rec[:res.n_rec]
    return out


def scan_adaptive(bound: Bound, wire_id, drift, grid, tol: float, h_max: float, index_list=None, begin: int = 0,
                  end: Optional[int] = None):
    H, _ = bound.hits(wire_id, drift)
    lo = np.ascontiguousarray(grid.lo, dtype=np.float64); st = np.ascontiguousarray(grid.step, dtype=np.float64)
    nn = np.ascontiguousarray(grid.n, dtype=np.int32)
    il = None if index_list is None else np.ascontiguousarray(index_list, dtype=np.int64)
    if end is None:
        end = int(il.size) if il is not None else int(np.prod(nn.astype(np.int64)))
    n = end - begin
    nm = np.zeros(n, dtype=np.int32); c2 = np.zeros(n); ns = np.zeros(n, dtype=np.int32); un = np.zeros(n, dtype=np.int32)
    mg = np.zeros(n, dtype=np.int32); fr = np.zeros((n, 3)); nl = np.zeros((n, 8), dtype=np.int32); mar = np.zeros((n, 6))
    sh = np.zeros(n, dtype=np.uint32)
    lib().orc_scan_adaptive(C.byref(bound.g), C.byref(bound.f), C.byref(H), _p(lo), _p(st), _p(nn), _p(il),
                            C.c_int64(begin), C.c_int64(end), C.byref(bound.P), C.c_double(tol), C.c_double(h_max),
                            _p(nm), _p(c2), _p(ns), _p(un), _p(mg), _p(fr), _p(nl), _p(mar), _p(sh))
    return dict(n_match=nm, chi2=c2, n_steps=ns, units=un, m_gas=mg, final_r=fr, n_level=nl, margins=mar, seq_hash=sh)


def _scan_adaptive_worker(args):
    geom, field, params, wire_id, drift, grid, tol, h_max, il, b, e = args
    return scan_adaptive(Bound(geom, field, params), wire_id, drift, grid, tol, h_max, il, b, e)


def scan_adaptive_parallel(geom, field, params: dict, wire_id, drift, grid, tol: float, h_max: float, index_list=None,
                           n_proc: Optional[int] = None):
    import multiprocessing as mp
    total = int(index_list.size) if index_list is not None else grid.n_seeds
    n_proc = n_proc or min(os.cpu_count() or 1, 8)
    edges = np.linspace(0, total, max(1, min(total, n_proc * 4)) + 1).astype(np.int64)
    jobs = [(geom, field, params, wire_id, drift, grid, tol, h_max, index_list, int(edges[i]), int(edges[i + 1]))
            for i in range(len(edges) - 1) if edges[i + 1] > edges[i]]
    if n_proc == 1 or len(jobs) == 1:
        parts = [_scan_adaptive_worker(j) for j in jobs]
    else:
        with mp.get_context("fork").Pool(n_proc) as pool:
            parts = pool.map(_scan_adaptive_worker, jobs)
    return {k: np.concatenate([p[k] for p in parts]) for k in parts[0]}
