"""the scan with the adaptive RKN step (cdc_seed_scan_adaptive, csrc/scan_adaptive.cu) against the
oracle's adaptive-step evaluation (oracle/cdc_oracle.c orc_eval_seed_adaptive), same seeded inputs, through the C ABI.

Parity protocol of this variant.  The step-size decisions are taken in fp32 by the kernel and in
fp64 by the oracle, and a different decision changes every later vertex, so:
  (a) a seed whose oracle-side error estimate comes within DECISION_EPS (relative) of tol, or of tol / 32, at any
      decision -- or within DECISION_K_EPS H^2 of it: the fp32 rounding noise of the estimate, a few ulp of the stage
      derivatives, which is the larger of the two at tol <= 1e-6 -- is an explicit EXCEPTION CLASS: listed and counted,
      not compared further (parity_util.compare_scan_adaptive); so is a seed whose in-gas units differ while one of
      the oracle's vertices lies within 1e-3 mm of R0 (the in-gas flag of that vertex is a threshold decision), or
      whose step counts differ while one lies within 1e-3 mm of |z| = z_half or r_out (the exit tests);
  (b) every other seed must take the IDENTICAL sequence of step lengths (equal hash of the level sequence, equal number
      of steps, path units and steps per level), and then
  (c) final positions agree within 1e-3 mm, in-gas units are equal, and n_match is identical except the usual listed
      threshold classes of the fixed-step protocol (checked on the oracle's adaptive records: an approach within
      1e-3 mm of the window edge or of a wire end), chi2 within the fp32 bound."""
import numpy as np
import pytest

import oracle
from paper_1908_01949_b200 import api, binding as B, synth

import parity_util as U

pytestmark = pytest.mark.gpu

@pytest.mark.parametrize("cfg_id,grid_n,tol,h_max", [(1, 6, 1e-5, 8.0), (3, 6, 1e-5, 8.0), (3, 5, 1e-4, 8.0), (3, 5, 3e-7, 4.0),
                                                     (2, 5, 1e-5, 8.0)])
def test_adaptive_scan_against_the_adaptive_oracle(cfg_id, grid_n, tol, h_max):
    cfg, geom, field, events, grids = U.make_workload(cfg_id, n_events=2, grid_n=grid_n)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    gpu = sc.scan_adaptive(E, grids, U.gpu_params(cfg), tol, h_max)
    n_exc = n_edge = n_cmp = 0
    o = 0
    for e, (ev, grid) in enumerate(zip(events, grids)):
        ns = grid.n_seeds
        exc, cmp_, edge = U.compare_scan_adaptive(cfg, geom, field, ev, grid, gpu, o, e, tol, h_max)
        n_exc += exc; n_cmp += cmp_; n_edge += edge
        o += ns
    assert n_exc <= 0.05 * (n_exc + n_cmp) and n_edge <= max(2, int(2e-3 * n_cmp))
    assert int(gpu["n_level"][:, 1:].sum()) > 0 or tol < 1e-6            # longer steps were actually taken
    print(f"adaptive cfg{cfg_id} tol {tol} h_max {h_max}: {n_cmp} seeds with the identical step sequence, {n_exc} decision-"
          f"threshold exceptions, {n_edge} window / wire-end exceptions; levels {gpu['n_level'].sum(axis=0).tolist()}")


def test_adaptive_scan_with_tiny_tolerance_equals_the_fixed_step_scan():
    """tol -> 0: every step at level 0; per-seed n_match, step counts and positions of the adaptive kernel equal the
    fixed-step production kernel's (positions to fp32 rounding: the two kernels order the arithmetic differently)."""
    cfg, geom, field, events, grids = U.make_workload(3, n_events=2, grid_n=5)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    ad = sc.scan_adaptive(sc.upload(off, w, d), grids, U.gpu_params(cfg), 1e-13, 8.0)
    fx = sc.scan(sc.upload(off, w, d), grids, U.gpu_params(cfg), per_seed=True, debug=True)
    assert int(ad["n_level"][:, 1:].sum()) == 0
    assert np.array_equal(ad["debug"]["n_steps"], fx["debug"]["n_steps"])
    assert (ad["n_match"] != fx["n_match"]).mean() < 2e-3
    for k in ("x", "y", "z"):
        assert np.abs(ad["debug"][k] - fx["debug"][k]).max() < 2e-4


def test_adaptive_scan_rejects_bad_arguments():
    cfg, geom, field, events, grids = U.make_workload(1, n_events=1, grid_n=2)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    for tol, h_max in ((0.0, 8.0), (-1.0, 8.0), (1e-5, 1.0), (1e-5, 16.0)):
        with pytest.raises(B.CdcError):
            sc.scan_adaptive(E, grids, U.gpu_params(cfg), tol, h_max)
