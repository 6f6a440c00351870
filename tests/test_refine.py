"""Coarse-to-fine refinement (reading C17): pins of the plain CPU statement
(oracle/refine.py) on CPU, and GPU parity against it (-m gpu)."""
import numpy as np
import pytest

import oracle
from oracle import refine as R
from paper_1908_01949_b200 import synth


def _setup(noise=0.0, sigma=0.0, cfg_id=0):
    cfg = synth.CONFIGS[cfg_id]
    geom = synth.make_geometry()
    field = synth.make_uniform_field()
    ev = synth.generate_events(cfg, geom, field, 1, sigma_drift=sigma, noise=noise)[0]
    params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm)
    return cfg, geom, field, ev, params


def test_refinement_equals_explicit_enumeration_of_the_lattice():
    """T = 2, K = 2 on a 3^5 grid: evaluate every lattice point the definition can visit one by one and replay the
    selection rule by hand."""
    cfg, geom, field, ev, params = _setup()
    shift = np.array([0.2, -0.3, 0.25, 0.15, -0.2]) * synth.HALF_WIDTH
    g0, _ = synth.truth_anchored_grid(ev.seed + shift, 3)
    K, T = 2, 2
    r = R.refine(geom, field, params, ev.wire_id, ev.drift_mm, g0, K=K, T=T, n_proc=2)
    b = oracle.Bound(geom, field, params)
    s_fine = g0.step / 2 ** T
    cache = {}
    def S_of(q):
        q = tuple(int(x) for x in q)
        if q not in cache:
            e = oracle.eval_seed(b, ev.wire_id, ev.drift_mm, g0.lo + np.array(q, dtype=np.float64) * s_fine)
            cache[q] = e["n_match"] - e["chi2"] / cfg.window_mm ** 2
        return cache[q]
    import itertools
    scanned = [tuple(4 * i for i in idx) for idx in itertools.product(range(3), repeat=5)]
    for t in range(0, T + 1):
        vals = sorted(((S_of(q), q) for q in set(scanned)), key=lambda x: -x[0])
        top = vals[:K]
        got = r["trace"][t]
        assert [q for q, _ in got] == [q for _, q in top]                       # the same lattice points, in order
        assert np.allclose([s for _, s in got], [s for s, _ in top], rtol=0, atol=1e-9)
        assert top[0][0] - top[1][0] > 1e-6                                      # no near-tie decided the order
        if t < T:
            d = 2 ** (T - t - 1)
            scanned = [tuple(p[a] + o[a] * d for a in range(5)) for _, p in top
                       for o in itertools.product((-1, 0, 1), repeat=5)]
    assert tuple(r["q"]) == r["trace"][T][0][0]
    assert np.allclose(r["seed"], g0.lo + r["q"] * s_fine, rtol=0, atol=1e-9)


def test_refinement_never_loses_score_and_keeps_distinct_parents():
    cfg, geom, field, ev, params = _setup(noise=0.05, sigma=0.2)
    g0, _ = synth.truth_anchored_grid(ev.seed + np.array([0.3, 0.4, -0.35, 0.25, 0.45]) * synth.HALF_WIDTH / 2, 5)
    r = R.refine(geom, field, params, ev.wire_id, ev.drift_mm, g0, K=4, T=5)
    best = [tr[0][1] for tr in r["trace"]]
    # the parent is the centre node of its sub-grid (re-evaluated from lo + 1 * step: the same point up to an ulp)
    assert all(b1 >= b0 - 1e-9 for b0, b1 in zip(best, best[1:]))
    assert best[-1] > best[0]
    for tr in r["trace"]:
        assert len({q for q, _ in tr}) == len(tr)                               # duplicates skipped
        assert all(s0 >= s1 for (_, s0), (_, s1) in zip(tr, tr[1:]))


def test_truth_node_stays_first_parent_on_a_smear_free_event():
    """G0 contains the truth: S(truth) = number of hits is the global maximum, so refinement must return it."""
    cfg, geom, field, ev, params = _setup()
    g0, anchor = synth.truth_anchored_grid(ev.seed, 4)
    r = R.refine(geom, field, params, ev.wire_id, ev.drift_mm, g0, K=3, T=4)
    assert tuple(r["q"]) == tuple(int(a) * 2 ** 4 for a in anchor)
    assert r["n_match"] == ev.wire_id.size and r["S"] > ev.wire_id.size - 1e-3
    assert np.allclose(r["seed"], ev.seed, rtol=0, atol=1e-9)
    assert all(tr[0][0] == tuple(r["q"]) for tr in r["trace"])


@pytest.mark.gpu
@pytest.mark.parametrize("cfg_id,n0,K,T", [(0, 5, 4, 6), (1, 4, 8, 10), (2, 3, 3, 4), (3, 4, 2, 5)])
def test_gpu_refinement_equals_oracle(cfg_id, n0, K, T):
    """uniform field, noise, energy loss (cfg2) and tabulated field (cfg3)"""
    from paper_1908_01949_b200 import api, binding as B
    cfg = synth.CONFIGS[cfg_id]
    geom = synth.make_geometry()
    field = synth.make_uniform_field() if cfg.field_kind == 0 else synth.make_table_field()
    events = synth.generate_events(cfg, geom, field, 2)
    shift = np.array([0.3, 0.4, -0.35, 0.25, 0.45]) * synth.HALF_WIDTH / 2
    grids = [synth.truth_anchored_grid(ev.seed + shift, n0)[0] for ev in events]
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    P = B.scan_params(cfg.h_mm, cfg.max_steps, cfg.window_mm, cfg.eloss_MeV_per_mm)
    out = B.cdc_refine_tracks(sc.geometry, E, B.grid_specs(grids), P, n_parents=K, n_iterations=T)
    params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm, eloss=cfg.eloss_MeV_per_mm)
    for e, (ev, g0) in enumerate(zip(events, grids)):
        r = R.refine(geom, field, params, ev.wire_id, ev.drift_mm, g0, K=K, T=T)
        for t in range(T + 1):
            assert [tuple(q) for q in out["trace_q"][e, t].tolist()] == [q for q, _ in r["trace"][t]], (e, t)
            assert out["trace_S"][e, t].tolist() == [s for _, s in r["trace"][t]]           # bit-equal doubles
        assert out["q"][e].tolist() == r["q"].tolist()
        assert out["seed"][e].tolist() == r["seed"].tolist()
        assert out["S"][e] == r["S"] and out["n_match"][e] == r["n_match"] and out["chi2"][e] == r["chi2"]
        lab, _ = oracle.labels(oracle.Bound(geom, field, params), ev.wire_id, ev.drift_mm, r["seed"])
        assert np.array_equal(out["labels"][off[e]:off[e + 1]], lab)
        assert out["S"][e] >= out["trace_S"][e, 0, 0] - 1e-9
