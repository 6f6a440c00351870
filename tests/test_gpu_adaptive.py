"""the scan with the adaptive RKN step (cdc_seed_scan_adaptive, csrc/scan_adaptive.cu) against the
oracle's adaptive-step evaluation (oracle/cdc_oracle.c orc_eval_seed_adaptive), same seeded inputs, through the C ABI.

Parity protocol of this variant.  The step-size decisions are taken in fp32 by the kernel and in
fp64 by the oracle, and a different decision changes every later vertex, so:
  (a) a seed whose oracle-side error estimate comes within DECISION_EPS (relative) of tol, or of tol / 32, at any
      decision is an explicit EXCEPTION CLASS: listed and counted, not compared further;
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

DECISION_EPS = 0.03


def _explain_adaptive(bound, ev, seed, cfg, geom, tol, h_max):
    r = oracle.eval_seed_adaptive(bound, ev.wire_id, ev.drift_mm, seed, tol, h_max, records=True, rec_slack=0.1)
    rec = r["rec"]
    return bool((np.abs(np.abs(rec["resid"]) - cfg.window_mm) < U.EDGE_TOL_MM).any() or
                (np.abs(np.abs(rec["zw"]) - geom.z_half_mm) < U.EDGE_TOL_MM).any())


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
        orc = oracle.scan_adaptive_parallel(geom, field, U.oracle_params(cfg), ev.wire_id, ev.drift_mm, grid, tol, h_max)
        dbg = gpu["debug"][o:o + ns]
        exc = (orc["margins"][:, 0] < DECISION_EPS) | (orc["margins"][:, 1] < DECISION_EPS)           # (a)
        ok = ~exc
        n_exc += int(exc.sum()); n_cmp += int(ok.sum())
        # (b) identical step-length sequence
        assert np.array_equal(gpu["seq_hash"][o:o + ns][ok], orc["seq_hash"][ok])
        assert np.array_equal(dbg["n_steps"][ok], orc["n_steps"][ok]) and np.array_equal(dbg["pad"][ok], orc["units"][ok])
        assert np.array_equal(gpu["n_level"][o:o + ns][ok], orc["n_level"][ok][:, :7])
        # (c) positions, in-gas units, match counts
        pos = np.stack([dbg["x"], dbg["y"], dbg["z"]], axis=1)
        assert np.linalg.norm(pos - orc["final_r"], axis=1)[ok].max() < U.POS_TOL_MM
        assert np.array_equal(dbg["m_gas"][ok], orc["m_gas"][ok])
        nm_g = gpu["n_match"][o:o + ns]; c2_g = gpu["chi2"][o:o + ns]
        bad = np.flatnonzero(ok & (nm_g != orc["n_match"]))
        bound = oracle.Bound(geom, field, U.oracle_params(cfg))
        for i in bad:
            assert _explain_adaptive(bound, ev, grid.node(grid.unravel(int(i))), cfg, geom, tol, h_max), \
                f"seed {i}: n_match {nm_g[i]} vs {orc['n_match'][i]} without a threshold case"
        n_edge += bad.size
        good = ok.copy(); good[bad] = False
        assert np.all(np.abs(c2_g[good] - orc["chi2"][good]) <= 1e-3 * np.maximum(orc["n_match"][good], 1))
        # the fused fp32 arg max is the arg max of the per-seed fp32 scores
        S32 = nm_g.astype(np.float32) - c2_g / np.float32(cfg.window_mm ** 2)
        assert abs(float(gpu["S32_max"][e]) - float(np.maximum(S32, 0).max())) < 1e-5
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
