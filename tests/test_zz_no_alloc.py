"""cdc_hough_seed_ranges_noalloc (csrc/hough_noalloc.cu): the Hough vote with its scratch -- one packed peak key per
event -- in a static device array, for callers that cannot allocate (CUDA graph capture, serving loops).  Same kernels
as cdc_hough_seed_ranges, so accumulator, peak and ranges must be IDENTICAL to the existing path's (which
test_gpu_parity.py checks against the oracle), on two calls in a row that share the scratch: the second call has fewer
events and other hits, so a key left over from the first call would show.  Collected last (zz): the suite runs with
pytest -x."""
import numpy as np
import pytest

from paper_1908_01949_b200 import api, binding as B, synth

import parity_util as U

pytestmark = pytest.mark.gpu


def _existing_path(sc, events, zref):
    off, w, d = synth.pack_hits(events)
    return sc.hough(sc.upload(off, w, d), zref, want_accum=True)


def _noalloc(sc, events, zref, torch):
    off, w, _ = synth.pack_hits(events)
    E = len(events)
    hp = B.hough_params()
    dims = B.cdc_hough_dims(hp)
    d_off = torch.tensor(np.asarray(off, dtype=np.int32), device="cuda")
    d_w = torch.tensor(np.asarray(w, dtype=np.int32), device="cuda")
    d_zref = torch.tensor(np.asarray(zref, dtype=np.float32), device="cuda")
    # outputs pre-filled with garbage: every element must be written
    d_ranges = torch.full((E, 3, 2), -7.0, dtype=torch.float64, device="cuda")
    d_peak = torch.full((E, 4), -7, dtype=torch.int32, device="cuda")
    d_acc = torch.full((E,) + tuple(dims), -7, dtype=torch.int32, device="cuda")
    B.cdc_hough_seed_ranges_noalloc(sc.geometry, E, d_off, d_w, hp, -1, d_zref, d_ranges, d_peak, d_acc)
    torch.cuda.synchronize()
    return dict(ranges=d_ranges.cpu().numpy(), peak=d_peak.cpu().numpy(), accum=d_acc.cpu().numpy().astype(np.uint32))


def test_hough_noalloc_equals_the_existing_path_on_two_calls_in_a_row():
    import torch
    cfg, geom, field, events, _ = U.make_workload(3, n_events=6)
    sc = api.SeedScanner(geom, field)
    B.cdc_hough_seed_ranges_noalloc(sc.geometry, 0, None, None, B.hough_params(), -1, None, None, None)     # set-up call
    first, second = events, events[4:1:-1]                    # 6 events, then 3 of them in another order
    for evs in (first, second):
        zref = [float(ev.seed[1]) for ev in evs]
        ref = _existing_path(sc, evs, zref)
        got = _noalloc(sc, evs, zref, torch)
        assert int(ref["peak"][:, 3].min()) >= 10            # a real peak in every event
        assert np.array_equal(got["accum"], ref["accum"])
        assert np.array_equal(got["peak"], ref["peak"])
        assert np.array_equal(got["ranges"], ref["ranges"])
    # the same call again: nothing of the previous one is left in the scratch
    again = _noalloc(sc, second, [float(ev.seed[1]) for ev in second], torch)
    assert np.array_equal(again["peak"], got["peak"]) and np.array_equal(again["ranges"], got["ranges"])
    sc.close()


def test_hough_noalloc_rejects_more_events_than_the_static_scratch_holds():
    import torch
    cfg, geom, field, events, _ = U.make_workload(0, n_events=1)
    sc = api.SeedScanner(geom, field)
    E = B.HOUGH_NOALLOC_MAX_EVENTS + 1
    d_off = torch.zeros(E + 1, dtype=torch.int32, device="cuda")
    d_w = torch.zeros(1, dtype=torch.int32, device="cuda")
    d_zref = torch.zeros(E, dtype=torch.float32, device="cuda")
    d_ranges = torch.zeros((E, 3, 2), dtype=torch.float64, device="cuda")
    d_peak = torch.zeros((E, 4), dtype=torch.int32, device="cuda")
    with pytest.raises(B.CdcError) as err:
        B.cdc_hough_seed_ranges_noalloc(sc.geometry, E, d_off, d_w, B.hough_params(), -1, d_zref, d_ranges, d_peak)
    assert err.value.status == -2 and "4096" in str(err.value)          # CDC_ERR_RANGE
    # the limit itself is accepted (events without hits: peak votes 0)
    B.cdc_hough_seed_ranges_noalloc(sc.geometry, E - 1, d_off, d_w, B.hough_params(), -1, d_zref, d_ranges, d_peak)
    torch.cuda.synchronize()
    assert int(d_peak[:E - 1, 3].max()) == 0
    sc.close()
