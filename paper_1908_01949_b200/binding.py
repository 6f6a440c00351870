"""Thin ctypes binding of include/cdc_seedscan.h: same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of libcdc_seedscan.so; PyTorch supplies device memory
and streams.  There is no CPU fallback: loading fails loudly when the library is missing, and every
compute call raises CdcError on a non-zero status.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcdc_seedscan.so")

EXPORTS = ["cdc_last_error", "cdc_geometry_create", "cdc_geometry_destroy", "cdc_geometry_wire_table",
           "cdc_event_upload", "cdc_events_destroy", "cdc_events_tables", "cdc_hough_dims",
           "cdc_hough_seed_ranges", "cdc_hough_seed_ranges_noalloc", "cdc_seed_scan", "cdc_scan_get_stats", "cdc_best_track",
           "cdc_find_tracks_host", "cdc_refine_tracks", "cdc_peel_turns", "cdc_classification_quality", "cdc_common_hits", "cdc_seed_scan_paper_mapping", "cdc_seed_scan_paper_mapping_v2", "cdc_seed_scan_adaptive", "cdc_fp32_peak_probe", "cdc_fp32_issue_probe", "cdc_kernel_launch_count"]


class CdcError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"cdc status {status}: {message}")
        self.status = status


class GeometryDesc(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("r_mm", C.c_void_p), ("n_wires", C.c_void_p), ("phi0_rad", C.c_void_p),
                ("stereo_rad", C.c_void_p), ("h_wire", C.c_void_p), ("z_half_mm", C.c_double),
                ("R0_mm", C.c_double), ("r_out_mm", C.c_double)]


class FieldDesc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("bz_T", C.c_double), ("nr", C.c_int32), ("nz", C.c_int32),
                ("r0_mm", C.c_double), ("z0_mm", C.c_double), ("dr_mm", C.c_double), ("dz_mm", C.c_double),
                ("h_br_bz", C.c_void_p)]


class GridSpec(C.Structure):
    _fields_ = [("lo", C.c_double * 5), ("step", C.c_double * 5), ("n", C.c_int32 * 5), ("first", C.c_int32 * 5)]


class ScanParams(C.Structure):
    _fields_ = [("h_mm", C.c_double), ("max_steps", C.c_int32), ("window_mm", C.c_double),
                ("eloss_MeV_per_mm", C.c_double), ("charge", C.c_int32), ("rescore_margin", C.c_double),
                ("kernel_variant", C.c_int32)]


class HoughParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("bin_xy_mm", "bin_R_mm", "tol_mm", "R_lo_mm", "R_hi_mm", "half_xy_mm",
                                          "origin_mm", "half_theta_rad", "half_pt_MeV")]


class RefineParams(C.Structure):
    _fields_ = [("n_parents", C.c_int32), ("n_iterations", C.c_int32)]


class PeelParams(C.Structure):
    _fields_ = [("max_partitions", C.c_int32), ("min_hits", C.c_int32), ("min_classified", C.c_int32),
                ("extrap_max_steps", C.c_int32), ("n", C.c_int32 * 5), ("pad_", C.c_int32), ("half_width", C.c_double * 5),
                ("extrap_tol_mm", C.c_double), ("extrap_h_max_mm", C.c_double)]


class ScanStats(C.Structure):
    _fields_ = [(k, C.c_uint64) for k in ("n_seeds", "n_steps", "n_gas_steps", "n_approach_tests", "n_pool",
                                          "pool_cap", "n_lookups", "n_g1", "n_approaches")] + [("kernel_ms", C.c_double)]


SEED_DEBUG_DTYPE = np.dtype([("n_steps", "i4"), ("turns", "i4"), ("m_gas", "i4"), ("pad", "i4"),
                             ("x", "f8"), ("y", "f8"), ("z", "f8")])
HOUGH_DEFAULT = dict(bin_xy_mm=4.0, bin_R_mm=4.0, tol_mm=6.0, R_lo_mm=240.0, R_hi_mm=364.0, half_xy_mm=460.0,
                     origin_mm=100.0, half_theta_rad=0.03, half_pt_MeV=7.5)

_lib = None


def lib():
    """The loaded C-ABI library.  Builds it in-tree if the sources are newer (needs nvcc); never falls back."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            from . import build as _build
            _build.build()
        L = C.CDLL(LIB_PATH)
        L.cdc_last_error.restype = C.c_char_p
        for name in EXPORTS[1:]:
            getattr(L, name).restype = C.c_int32
        L.cdc_kernel_launch_count.restype = C.c_uint64
        _lib = L
    return _lib


def _check(status: int):
    if status != 0:
        raise CdcError(status, lib().cdc_last_error().decode())


def _hp(a: Optional[np.ndarray]):
    return None if a is None else C.c_void_p(a.ctypes.data)


def _dp(t):
    """Device pointer of a torch tensor (or None)."""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _stream(stream) -> C.c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(int(stream.cuda_stream))


def scan_params(h_mm: float, max_steps: int, window_mm: float = 1.0, eloss_MeV_per_mm: float = 0.0,
                charge: int = -1, rescore_margin: float = 0.0, kernel_variant: int = 0) -> ScanParams:
    return ScanParams(float(h_mm), int(max_steps), float(window_mm), float(eloss_MeV_per_mm), int(charge),
                      float(rescore_margin), int(kernel_variant))


def hough_params(**kw) -> HoughParams:
    d = dict(HOUGH_DEFAULT); d.update(kw)
    return HoughParams(*[float(d[k]) for k, _ in HoughParams._fields_])


def grid_specs(grids: Sequence) -> C.Array:
    """Objects with .lo, .step, .n (5 each) and optionally .first (node offset per axis) -> array of cdc_grid_spec."""
    arr = (GridSpec * len(grids))()
    for i, g in enumerate(grids):
        first = getattr(g, "first", None)
        for a in range(5):
            arr[i].lo[a] = float(g.lo[a]); arr[i].step[a] = float(g.step[a]); arr[i].n[a] = int(g.n[a])
            arr[i].first[a] = 0 if first is None else int(first[a])
    return arr


class Geometry:
    """cdc_geometry handle (A0).  `geom` / `field` are records shaped like synth.Geometry / synth.Field."""

    def __init__(self, geom, field, use_wire_table: bool = True):
        self._keep = []
        def arr(a, dt):
            a = np.ascontiguousarray(a, dtype=dt); self._keep.append(a); return a
        wire = arr(geom.wire, np.float32) if (use_wire_table and getattr(geom, "wire", None) is not None) else None
        gd = GeometryDesc(int(len(geom.r_mm)), _hp(arr(geom.r_mm, np.float64)), _hp(arr(geom.n_wires, np.int32)),
                          _hp(arr(geom.phi0_rad, np.float64)), _hp(arr(geom.stereo_rad, np.float64)), _hp(wire),
                          float(geom.z_half_mm), float(geom.R0_mm), float(geom.r_out_mm))
        tab = arr(field.table, np.float32) if int(field.kind) == 1 else None
        fd = FieldDesc(int(field.kind), float(field.bz_T), int(field.nr), int(field.nz), float(field.r0_mm),
                       float(field.z0_mm), float(field.dr_mm), float(field.dz_mm), _hp(tab))
        self.handle = C.c_void_p()
        _check(lib().cdc_geometry_create(C.byref(gd), C.byref(fd), C.byref(self.handle)))
        self.n_wires_total = int(np.sum(np.asarray(geom.n_wires)))

    def wire_table(self) -> np.ndarray:
        out = np.zeros((self.n_wires_total, 5), dtype=np.float32)
        n = C.c_int32()
        _check(lib().cdc_geometry_wire_table(self.handle, _hp(out), C.byref(n)))
        assert n.value == self.n_wires_total
        return out

    def close(self):
        if self.handle:
            lib().cdc_geometry_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Events:
    """cdc_events handle (A1).  wire_id / drift are numpy arrays (host) or torch CUDA tensors (device)."""

    def __init__(self, geometry: Geometry, hit_offsets, wire_id, drift_mm, stream=None):
        self.geometry = geometry
        self.offsets = np.ascontiguousarray(hit_offsets, dtype=np.int32)
        self.n_events = int(self.offsets.size - 1)
        self.n_hits = int(self.offsets[-1])
        on_device = hasattr(wire_id, "is_cuda")
        if on_device:
            import torch
            assert wire_id.dtype == torch.int32 and drift_mm.dtype == torch.float32
            pw, pd = _dp(wire_id), _dp(drift_mm)
        else:
            w = np.ascontiguousarray(wire_id, dtype=np.int32); d = np.ascontiguousarray(drift_mm, dtype=np.float32)
            pw, pd = _hp(w), _hp(d)
        self.handle = C.c_void_p()
        _check(lib().cdc_event_upload(geometry.handle, C.c_int32(self.n_events), _hp(self.offsets), pw, pd,
                                      C.c_int32(1 if on_device else 0), _stream(stream), C.byref(self.handle)))

    def tables(self):
        W = self.geometry.n_wires_total
        drift = np.zeros((self.n_events, W), dtype=np.float32)
        bits = np.zeros((self.n_events, (W + 31) // 32), dtype=np.uint32)
        _check(lib().cdc_events_tables(self.handle, _hp(drift), _hp(bits)))
        return drift, bits

    def close(self):
        if self.handle:
            lib().cdc_events_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def cdc_hough_dims(hp: HoughParams):
    dims = (C.c_int32 * 3)()
    _check(lib().cdc_hough_dims(C.byref(hp), dims))
    return tuple(int(x) for x in dims)


def cdc_hough_seed_ranges(geometry: Geometry, events: Events, hp: HoughParams, charge: int, d_zref, d_ranges,
                          d_peak, d_accum=None, stream=None):
    _check(lib().cdc_hough_seed_ranges(geometry.handle, events.handle, C.byref(hp), C.c_int32(charge), _dp(d_zref),
                                       _dp(d_ranges), _dp(d_peak), _dp(d_accum), _stream(stream)))


HOUGH_NOALLOC_MAX_EVENTS = 4096


def cdc_hough_seed_ranges_noalloc(geometry: Geometry, n_events: int, d_hit_offsets, d_wire_id, hp: HoughParams, charge: int,
                                  d_zref, d_ranges, d_peak, d_accum=None, stream=None):
    """The Hough vote with its scratch in a static device array: no allocation, no Events handle (include/cdc_seedscan.h)."""
    _check(lib().cdc_hough_seed_ranges_noalloc(geometry.handle, C.c_int32(n_events), _dp(d_hit_offsets), _dp(d_wire_id),
                                               C.byref(hp), C.c_int32(charge), _dp(d_zref), _dp(d_ranges), _dp(d_peak),
                                               _dp(d_accum), _stream(stream)))


def cdc_seed_scan(geometry: Geometry, events: Events, grids: C.Array, params: ScanParams, d_best_key,
                  d_n_match=None, d_chi2=None, d_debug=None, stream=None):
    _check(lib().cdc_seed_scan(geometry.handle, events.handle, grids, C.byref(params), _dp(d_n_match), _dp(d_chi2),
                               _dp(d_debug), _dp(d_best_key), _stream(stream)))


def cdc_scan_get_stats(events: Events, stream=None) -> dict:
    st = ScanStats()
    _check(lib().cdc_scan_get_stats(events.handle, C.byref(st), _stream(stream)))
    return {k: (float if k == "kernel_ms" else int)(getattr(st, k)) for k, _ in ScanStats._fields_}


def cdc_best_track(geometry: Geometry, events: Events, grids: C.Array, params: ScanParams, d_best_key, d_best_seed,
                   d_best_n_match, d_best_chi2, d_labels, stream=None):
    _check(lib().cdc_best_track(geometry.handle, events.handle, grids, C.byref(params), _dp(d_best_key),
                                _dp(d_best_seed), _dp(d_best_n_match), _dp(d_best_chi2), _dp(d_labels),
                                _stream(stream)))


def cdc_seed_scan_adaptive(geometry: Geometry, events: Events, grids: C.Array, params: ScanParams, tol_mm: float,
                           h_max_mm: float, d_best_key, d_n_match=None, d_chi2=None, d_debug=None, d_levels=None,
                           stream=None) -> None:
    """the scan with the adaptive RKN step (device outputs, caller-owned torch tensors)."""
    _check(lib().cdc_seed_scan_adaptive(geometry.handle, events.handle, grids, C.byref(params), C.c_double(tol_mm),
                                        C.c_double(h_max_mm), _dp(d_n_match), _dp(d_chi2), _dp(d_debug), _dp(d_levels),
                                        _dp(d_best_key), _stream(stream)))


def cdc_find_tracks_host(geometry: Geometry, hit_offsets, wire_id, drift_mm, grids: C.Array, params: ScanParams,
                         hp: Optional[HoughParams] = None, zref=None, hough_sets_axes: bool = True, stream=None) -> dict:
    """End-to-end call with host (numpy) buffers in and out.  With hp the Hough vote runs; its ranges replace the
    (theta, px, py) axes of the grids unless hough_sets_axes is False."""
    off = np.ascontiguousarray(hit_offsets, dtype=np.int32)
    w = np.ascontiguousarray(wire_id, dtype=np.int32); d = np.ascontiguousarray(drift_mm, dtype=np.float32)
    E = int(off.size - 1)
    seed = np.zeros(E, dtype=np.int64); nm = np.zeros(E, dtype=np.uint32); chi2 = np.zeros(E)
    key = np.zeros(E, dtype=np.uint64); lab = np.zeros(max(int(off[-1]), 1), dtype=np.int32)
    ranges = np.zeros((E, 3, 2)) if hp is not None else None
    zr = None if zref is None else np.ascontiguousarray(zref, dtype=np.float32)
    _check(lib().cdc_find_tracks_host(geometry.handle, C.c_int32(E), _hp(off), _hp(w), _hp(d), grids, C.byref(params),
                                      None if hp is None else C.byref(hp), _hp(zr), C.c_int32(1 if hough_sets_axes else 0),
                                      _hp(seed), _hp(nm), _hp(chi2),
                                      _hp(key), _hp(lab), _hp(ranges), _stream(stream)))
    return dict(best_seed=seed, best_n_match=nm, best_chi2=chi2, best_key=key, labels=lab[:int(off[-1])],
                ranges=ranges)


def cdc_refine_tracks(geometry: Geometry, events: Events, grids: C.Array, params: ScanParams, n_parents: int = 8,
                      n_iterations: int = 10, want_labels: bool = True, want_trace: bool = True, stream=None) -> dict:
    """Coarse-to-fine refinement.  Host (numpy) outputs."""
    E, K, T = events.n_events, int(n_parents), int(n_iterations)
    seed = np.zeros((E, 5)); S = np.zeros(E); nm = np.zeros(E, dtype=np.uint32); chi2 = np.zeros(E)
    q = np.zeros((E, 5), dtype=np.int64)
    lab = np.zeros(max(events.n_hits, 1), dtype=np.int32) if want_labels else None
    tS = np.zeros((E, T + 1, K)) if want_trace else None
    tq = np.zeros((E, T + 1, K, 5), dtype=np.int64) if want_trace else None
    rp = RefineParams(K, T)
    _check(lib().cdc_refine_tracks(geometry.handle, events.handle, grids, C.byref(params), C.byref(rp), _hp(seed), _hp(S),
                                   _hp(nm), _hp(chi2), _hp(q), _hp(lab), _hp(tS), _hp(tq), _stream(stream)))
    return dict(seed=seed, S=S, n_match=nm, chi2=chi2, q=q, labels=None if lab is None else lab[:events.n_hits],
                trace_S=tS, trace_q=tq)


def cdc_peel_turns(geometry: Geometry, events: Events, grids0: C.Array, params: ScanParams, n: Sequence[int],
                   half_width: Sequence[float], max_partitions: int = 4, min_hits: int = 10, min_classified: int = 5,
                   extrap_max_steps: int = 3000, extrap_tol: float = 0.0, extrap_h_max: float = 0.0, stream=None) -> dict:
    """Turn-partition peeling.  Host (numpy) outputs; `partition` is read back from the device."""
    import torch
    E, P = events.n_events, int(max_partitions)
    pp = PeelParams(P, int(min_hits), int(min_classified), int(extrap_max_steps), (C.c_int32 * 5)(*[int(v) for v in n]), 0,
                    (C.c_double * 5)(*[float(v) for v in half_width]), float(extrap_tol), float(extrap_h_max))
    n_part = np.zeros(E, dtype=np.int32); status = np.zeros(E, dtype=np.int32)
    seeds = np.zeros((E, P, 5)); nm = np.zeros((E, P), dtype=np.uint32); chi2 = np.zeros((E, P)); centres = np.zeros((E, P, 5))
    d_part = torch.empty(max(events.n_hits, 1), dtype=torch.int32, device="cuda")
    _check(lib().cdc_peel_turns(geometry.handle, events.handle, grids0, C.byref(params), C.byref(pp), _hp(n_part),
                                _hp(status), _hp(seeds), _hp(nm), _hp(chi2), _hp(centres), _dp(d_part), _stream(stream)))
    torch.cuda.synchronize()
    return dict(n_partitions=n_part, status=status, seeds=seeds, n_match=nm, chi2=chi2, centres=centres,
                partition=d_part[:events.n_hits].cpu().numpy(), d_partition=d_part)


def cdc_classification_quality(events: Events, n_turns: int, d_labels, d_truth, stream=None) -> dict:
    """Eq. (2), (3) of the paper per event and turn partition; returns numpy arrays."""
    import torch
    E, n = events.n_events, int(n_turns)
    conf = torch.zeros((E, n, n), dtype=torch.int32, device="cuda"); ct = torch.zeros((E, n), dtype=torch.int32, device="cuda")
    ni = torch.zeros((E, n), dtype=torch.int32, device="cuda")
    eff = torch.zeros((E, n), dtype=torch.float64, device="cuda"); pur = torch.zeros((E, n), dtype=torch.float64, device="cuda")
    _check(lib().cdc_classification_quality(events.handle, C.c_int32(n), _dp(d_labels), _dp(d_truth), _dp(conf), _dp(ct),
                                            _dp(ni), _dp(eff), _dp(pur), _stream(stream)))
    torch.cuda.synchronize()
    return dict(confusion=conf.cpu().numpy(), c_true=ct.cpu().numpy(), noise_into=ni.cpu().numpy(),
                efficiency=eff.cpu().numpy(), purity=pur.cpu().numpy())


def cdc_common_hits(events: Events, d_labels_a, d_labels_b, turn_a: int = -1, turn_b: int = -1, stream=None) -> np.ndarray:
    import torch
    out = torch.zeros(events.n_events, dtype=torch.int32, device="cuda")
    _check(lib().cdc_common_hits(events.handle, _dp(d_labels_a), _dp(d_labels_b), C.c_int32(turn_a), C.c_int32(turn_b),
                                 _dp(out), _stream(stream)))
    torch.cuda.synchronize()
    return out.cpu().numpy()


def cdc_seed_scan_paper_mapping(geometry: Geometry, events: Events, event: int, grid, params: ScanParams, d_seed_index,
                                d_n_match, d_chi2, stream=None):
    """The paper's block-per-seed / thread-per-fired-wire mapping (comparison point only)."""
    _check(lib().cdc_seed_scan_paper_mapping(geometry.handle, events.handle, C.c_int32(event), grid_specs([grid]),
                                             C.byref(params), _dp(d_seed_index), C.c_int32(int(d_seed_index.numel())),
                                             _dp(d_n_match), _dp(d_chi2), _stream(stream)))


def cdc_seed_scan_paper_mapping_v2(geometry: Geometry, events: Events, event: int, grid, params: ScanParams, d_seed_index,
                                   d_n_match, d_chi2, timed: bool = False, stream=None):
    """The paper's two-kernel mapping (record all steps, then DCA per wire; comparison point only).
    timed=True returns the device times (ms) of the two kernels."""
    ms = np.zeros(2) if timed else None
    _check(lib().cdc_seed_scan_paper_mapping_v2(geometry.handle, events.handle, C.c_int32(event), grid_specs([grid]),
                                                C.byref(params), _dp(d_seed_index), C.c_int32(int(d_seed_index.numel())),
                                                _dp(d_n_match), _dp(d_chi2), _hp(ms), _stream(stream)))
    return ms


def cdc_kernel_launch_count() -> int:
    return int(lib().cdc_kernel_launch_count())


def cdc_fp32_issue_probe(mode: int, iters: int = 4096, stream=None):
    ms = C.c_double(); wi = C.c_double(); fl = C.c_double()
    _check(lib().cdc_fp32_issue_probe(C.c_int32(mode), C.c_int32(iters), C.byref(ms), C.byref(wi), C.byref(fl), _stream(stream)))
    return float(ms.value), float(wi.value), float(fl.value)


def cdc_fp32_peak_probe(iters: int = 4096, stream=None):
    f = C.c_double(); ms = C.c_double()
    _check(lib().cdc_fp32_peak_probe(C.c_int32(iters), C.byref(f), C.byref(ms), _stream(stream)))
    return float(f.value), float(ms.value)
