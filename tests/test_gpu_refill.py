"""The lane-refill variant of the scan kernel (params.kernel_variant = 2, csrc/scan_refill.cu: a thread runs two seeds in
a row -- seed l of one 32-seed chunk, then seed 31 - l of the next -- and a per-step vote ends the warp) against the
production kernel (csrc/scan.cu).  The per-seed arithmetic is the same code (scan_one.cuh) in the same order; only the
first hold of a second seed's lookup cadence is shorter, which changes which wires are HELD, never which approaches
are owned.  So per-seed n_match, step / turn / in-gas counts, final positions (bitwise), the exact best seed, its chi2
and the labels must be IDENTICAL; the fp32 chi2 of a seed is the same set of terms, added in the order of the slot list
where one interval owns two approaches (a few ulp of the sum).  Parity of the production kernel with the fp64 oracle is
test_gpu_parity.py / test_gpu_edges.py / test_gpu_sizes.py."""
import dataclasses

import numpy as np
import pytest

from paper_1908_01949_b200 import api, binding as B, synth

import parity_util as U

pytestmark = pytest.mark.gpu


def _both(sc, events, grids, cfg, debug):
    off, w, d = synth.pack_hits(events)
    out = []
    for variant in (2, 0):
        E = sc.upload(off, w, d)
        out.append(sc.scan(E, grids, U.gpu_params(cfg, kernel_variant=variant), per_seed=True, debug=debug))
    return out


def _assert_identical(a, b, debug):
    assert np.array_equal(a["n_match"], b["n_match"])
    # the same terms; two approaches owned by the same interval are added in slot order, which follows the lookups
    assert np.all(np.abs(a["chi2"].astype(np.float64) - b["chi2"]) <= 2e-5 * np.maximum(b["n_match"], 1))
    for k in ("best_seed", "best_n_match", "best_chi2", "labels"):
        assert np.array_equal(a[k], b[k]), k
    assert a["stats"]["n_steps"] == b["stats"]["n_steps"]       # (sign changes of held wires that end outside the window are
                                                                 # counted per held wire and may differ: the held sets do)
    if debug:
        for k in ("n_steps", "turns", "m_gas", "x", "y", "z"):
            assert np.array_equal(a["debug"][k], b["debug"][k]), k


@pytest.mark.parametrize("cfg_id,n_events,grid_n", [(0, 2, 8), (1, 2, (6, 9, 5, 5, 5)), (2, 1, (5, 7, 5, 5, 4)),
                                                    (3, 3, (5, 16, 5, 5, 5)), (3, 2, (4, 1, 6, 5, 5)), (1, 1, (1, 3, 1, 1, 1))])
@pytest.mark.parametrize("debug", [False, True])
def test_refill_kernel_equals_one_seed_kernel(cfg_id, n_events, grid_n, debug):
    """Seed counts that are and are not multiples of 64 (a last chunk without a partner, a grid smaller than one chunk),
    z0 node counts that do and do not fill half a warp, both fields, energy loss; with and without the debug record."""
    cfg, geom, field, events, grids = U.make_workload(cfg_id, n_events=n_events, grid_n=grid_n)
    sc = api.SeedScanner(geom, field)
    a, b = _both(sc, events, grids, cfg, debug)
    _assert_identical(a, b, debug)
    if grids[0].n_seeds > 64:
        assert int(a["n_match"].max()) >= 10


def test_refill_kernel_events_of_different_size():
    """Grids of different sizes in one launch: blocks beyond an event's last chunk pair leave at once."""
    cfg, geom, field, events, _ = U.make_workload(1, n_events=3)
    grids = [synth.truth_anchored_grid(ev.seed, n)[0] for ev, n in zip(events, ((4, 16, 4, 4, 4), (3, 5, 3, 3, 3), (6, 8, 5, 4, 3)))]
    sc = api.SeedScanner(geom, field)
    a, b = _both(sc, events, grids, cfg, True)
    _assert_identical(a, b, True)


def test_refill_kernel_step_cap_and_slow_seeds():
    """max_steps = 1 and 2, and seeds at or below 1 MeV/c (one step, reading C7): a lane can take its second seed at once."""
    cfg, geom, field, events, _ = U.make_workload(1, n_events=1)
    ev = events[0]
    grid = synth.Grid(lo=np.array([0.1, -100.0, -0.6, -0.6, -0.3]), step=np.array([0.4, 50.0, 0.4, 0.4, 0.3]),
                      n=np.array([3, 5, 4, 4, 3], dtype=np.int32))
    sc = api.SeedScanner(geom, field)
    for ms in (1, 2, 300):
        a, b = _both(sc, [ev], [grid], dataclasses.replace(cfg, max_steps=ms), True)
        _assert_identical(a, b, True)
