"""GPU tests of the boundary's remaining calls and of the degenerate cases: A1 tables, error reporting,
empty / ragged / single-seed inputs, the wire-table builder, device-resident hits, the end-to-end host call."""
import numpy as np
import pytest

import oracle
from paper_1908_01949_b200 import api, binding as B, synth

import parity_util as U

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def setup():
    import torch
    assert torch.cuda.is_available()
    cfg, geom, field, events, grids = U.make_workload(1, n_events=3, grid_n=4)
    return cfg, geom, field, events, grids, api.SeedScanner(geom, field)


def test_event_tables_equal_oracle_binning(setup):
    cfg, geom, field, events, grids, sc = setup
    off, w, d = synth.pack_hits(events)
    rng = np.random.default_rng(1)
    perm = np.concatenate([off[e] + rng.permutation(off[e + 1] - off[e]) for e in range(len(events))])
    E = sc.upload(off, w[perm], d[perm])                       # hits need not be sorted
    tab, bits = E.tables()
    bound = oracle.Bound(geom, field, U.oracle_params(cfg))
    for e, ev in enumerate(events):
        assert np.array_equal(tab[e], oracle.bin_event(bound, ev.wire_id, ev.drift_mm))
        want = np.zeros(bits.shape[1] * 32, dtype=bool); want[ev.wire_id] = True
        got = ((bits[e][:, None] >> np.arange(32, dtype=np.uint32)[None, :]) & 1).astype(bool).ravel()
        assert np.array_equal(got, want)


def test_upload_errors_are_reported(setup):
    cfg, geom, field, events, grids, sc = setup
    off = np.array([0, 3], dtype=np.int32)
    with pytest.raises(B.CdcError) as ei:
        sc.upload(off, np.array([1, 2, geom.n_wires_total], dtype=np.int32), np.ones(3, dtype=np.float32))
    assert ei.value.status == -2
    with pytest.raises(B.CdcError) as ei:
        sc.upload(off, np.array([1, 2, 2], dtype=np.int32), np.ones(3, dtype=np.float32))
    assert ei.value.status == -1 and "duplicate" in str(ei.value)
    for bad in (-0.5, np.nan, np.inf):
        with pytest.raises(B.CdcError) as ei:
            sc.upload(off, np.array([1, 2, 3], dtype=np.int32), np.array([1.0, bad, 1.0], dtype=np.float32))
        assert ei.value.status == -1
    E = sc.upload(off, np.array([1, 2, 3], dtype=np.int32), np.ones(3, dtype=np.float32))
    g = synth.truth_anchored_grid(events[0].seed, 2)[0]
    import torch
    key = torch.zeros(1, dtype=torch.int64, device="cuda")
    with pytest.raises(B.CdcError):
        B.cdc_seed_scan(sc.geometry, E, B.grid_specs([g]), B.scan_params(0.0, 100), key)       # h <= 0
    g.n[0] = 0
    with pytest.raises(B.CdcError):
        B.cdc_seed_scan(sc.geometry, E, B.grid_specs([g]), B.scan_params(2.0, 100), key)       # n < 1
    with pytest.raises(B.CdcError) as ei:                                                        # call order
        B.cdc_best_track(sc.geometry, E, B.grid_specs([g]), B.scan_params(2.0, 100), key, key, key, key, key)
    assert ei.value.status == -5


def test_energy_loss_beyond_the_curvature_bounds_is_rejected(setup):
    cfg, geom, field, events, grids, sc = setup
    off, w, d = synth.pack_hits(events[:1])
    E = sc.upload(off, w, d)
    import torch
    key = torch.zeros(1, dtype=torch.int64, device="cuda")
    B.cdc_seed_scan(sc.geometry, E, B.grid_specs(grids[:1]), B.scan_params(2.0, 50, 1.0, 2.5e-3), key)     # accepted
    with pytest.raises(B.CdcError) as ei:
        B.cdc_seed_scan(sc.geometry, E, B.grid_specs(grids[:1]), B.scan_params(2.0, 50, 1.0, 0.01), key)
    assert ei.value.status == -2


def test_field_table_too_small_is_rejected(setup):
    cfg, geom, *_ = setup
    small = synth.make_table_field(r_max=800.0)
    with pytest.raises(B.CdcError) as ei:
        api.SeedScanner(geom, small)
    assert ei.value.status == -2


def test_empty_event_and_ragged_grid(setup):
    cfg, geom, field, events, grids, sc = setup
    ev = events[0]
    # event 0 has no hits at all; event 1 is a real one with a ragged 5 x 3 x 7 x 2 x 3 grid (630 seeds: 4 full
    # blocks of 128 and a tail of 118)
    g_empty = synth.truth_anchored_grid(ev.seed, [2, 3, 1, 2, 2])[0]
    g_rag = synth.truth_anchored_grid(ev.seed, [5, 3, 7, 2, 3])[0]
    off = np.array([0, 0, ev.wire_id.size], dtype=np.int32)
    E = sc.upload(off, ev.wire_id, ev.drift_mm)
    gpu = sc.scan(E, [g_empty, g_rag], U.gpu_params(cfg), per_seed=True, debug=True)
    n0 = g_empty.n_seeds
    assert gpu["n_seeds"] == [n0, 630]
    assert not gpu["n_match"][:n0].any() and not gpu["chi2"][:n0].any()
    assert gpu["best_seed"][0] == 0 and gpu["best_n_match"][0] == 0 and gpu["best_chi2"][0] == 0.0   # ties -> index 0
    assert (gpu["debug"]["n_steps"][:n0] > 0).all()
    orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), ev.wire_id, ev.drift_mm, g_rag)
    U.compare_scan(cfg, geom, field, ev, g_rag, gpu, orc, np.arange(630), offset=n0)
    U.check_best(cfg, geom, field, ev, g_rag, gpu, e=1, orc_full=orc)
    assert gpu["labels"].size == ev.wire_id.size


def test_event_without_hits_on_a_grid_larger_than_the_candidate_pool(setup):
    """Every seed of an event without hits scores S = 0: the tie goes to index 0 and the 65 536-entry candidate pool
    must not overflow (only index 0 stands in for the seeds without a match)."""
    cfg, geom, field, events, grids, sc = setup
    ev = events[0]
    g_big = synth.truth_anchored_grid(ev.seed, 12)[0]                    # 248 832 seeds
    off = np.array([0, 0, ev.wire_id.size], dtype=np.int32)
    E = sc.upload(off, ev.wire_id, ev.drift_mm)
    gpu = sc.scan(E, [g_big, g_big], B.scan_params(cfg.h_mm, 60, cfg.window_mm), per_seed=False)
    assert gpu["stats"]["n_pool"] <= gpu["stats"]["pool_cap"]
    assert gpu["best_seed"][0] == 0 and gpu["best_n_match"][0] == 0 and gpu["best_chi2"][0] == 0.0
    assert gpu["best_seed"][1] >= 0


def test_single_seed_and_step_cap(setup):
    cfg, geom, field, events, grids, sc = setup
    ev = events[1]
    g1 = synth.truth_anchored_grid(ev.seed, 1)[0]
    off, w, d = synth.pack_hits([ev])
    E = sc.upload(off, w, d)
    for cap in (1, 37, cfg.max_steps):
        gpu = sc.scan(E, [g1], B.scan_params(cfg.h_mm, cap, cfg.window_mm), per_seed=True, debug=True)
        bound = oracle.Bound(geom, field, dict(h=cfg.h_mm, max_steps=cap, window=cfg.window_mm))
        r = oracle.eval_seed(bound, ev.wire_id, ev.drift_mm, ev.seed)
        assert gpu["debug"]["n_steps"][0] == r["n_steps"] == min(cap, r["n_steps"])
        assert gpu["n_match"][0] == r["n_match"] and gpu["best_seed"][0] == 0
        assert gpu["best_chi2"][0] == r["chi2"]
        assert np.linalg.norm([gpu["debug"][k][0] - r["r"][i] for i, k in enumerate("xyz")]) < U.POS_TOL_MM


def test_degenerate_seeds_terminate(setup):
    """Inward-pointing, stiff and very soft seeds are propagated like any other (reading C4) and end by the same rule."""
    cfg, geom, field, events, grids, sc = setup
    ev = events[0]
    off, w, d = synth.pack_hits([ev])
    E = sc.upload(off, w, d)
    bound = oracle.Bound(geom, field, U.oracle_params(cfg))
    for seed in ([0.3, 0.0, -80.0, -30.0, 20.0], [0.0, 0.0, 400.0, 0.0, 1.0], [1.0, 700.0, 0.3, 0.2, 0.5],
                 [2.0, -749.9, 10.0, 10.0, -50.0]):
        g = synth.Grid(lo=np.array(seed, dtype=np.float64), step=np.zeros(5), n=np.ones(5, dtype=np.int32))
        gpu = sc.scan(E, [g], U.gpu_params(cfg), per_seed=True, debug=True)
        r = oracle.eval_seed(bound, ev.wire_id, ev.drift_mm, np.array(seed))
        assert gpu["debug"]["n_steps"][0] == r["n_steps"], seed
        assert gpu["n_match"][0] == r["n_match"]


def test_wire_table_builder_matches_generator(setup):
    cfg, geom, field, *_ = setup
    sc2 = api.SeedScanner(geom, field, use_wire_table=False)
    built = sc2.geometry.wire_table()
    ulp = np.spacing(np.abs(geom.wire).astype(np.float32))
    assert np.all(np.abs(built - geom.wire) <= ulp)          # same fp64 formula, rounded once: <= 1 ulp (libm vs numpy)
    assert (built == geom.wire).mean() > 0.999
    assert np.array_equal(api.SeedScanner(geom, field).geometry.wire_table(), geom.wire)


def test_device_resident_hits_and_host_call_agree(setup):
    import torch
    cfg, geom, field, events, grids, sc = setup
    off, w, d = synth.pack_hits(events)
    E_host = sc.upload(off, w, d)
    E_dev = sc.upload(off, torch.tensor(w, device="cuda"), torch.tensor(d, device="cuda"))
    P = U.gpu_params(cfg)
    a = sc.scan(E_host, grids, P, per_seed=True)
    b = sc.scan(E_dev, grids, P, per_seed=True)
    c = sc.find_tracks_host(off, w, d, grids, P)
    for k in ("best_seed", "best_n_match", "best_chi2", "labels", "best_key"):
        assert np.array_equal(a[k], b[k]) and np.array_equal(a[k], c[k]), k
    assert np.array_equal(a["n_match"], b["n_match"]) and np.array_equal(a["chi2"], b["chi2"])   # deterministic
    for e, (ev, grid) in enumerate(zip(events, grids)):
        orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), ev.wire_id, ev.drift_mm, grid)
        U.check_best(cfg, geom, field, ev, grid, a, e=e, hit_slice=slice(off[e], off[e + 1]), orc_full=orc)


def test_host_call_with_hough_ranges(setup):
    cfg2, geom, field, events, _ = U.make_workload(2, grid_n=6)
    sc = api.SeedScanner(geom, field)
    ev = events[0]
    off, w, d = synth.pack_hits(events)
    g0 = synth.truth_anchored_grid(ev.seed, 6)[0]
    P = U.gpu_params(cfg2)
    out = sc.find_tracks_host(off, w, d, [g0], P, hp=B.hough_params(), zref=[float(ev.seed[1])])
    E = sc.upload(off, w, d)
    h = sc.hough(E, [float(ev.seed[1])])
    assert np.array_equal(out["ranges"], h["ranges"])
    lo = g0.lo.copy(); hi = g0.lo + g0.step * (g0.n - 1)
    lo[[0, 2, 3]] = h["ranges"][0][:, 0]; hi[[0, 2, 3]] = h["ranges"][0][:, 1]
    grid = synth.ranges_grid(lo, hi, 6)
    staged = sc.scan(E, [grid], P, per_seed=True)
    for k in ("best_seed", "best_n_match", "best_chi2", "labels"):
        assert np.array_equal(out[k], staged[k]), k
    U.check_best(cfg2, geom, field, ev, grid, staged)
    # the vote without the replacement of the axes (bench.py's end-to-end arm on truth-anchored grids): same ranges
    # reported, the grid scanned as given
    keep = sc.find_tracks_host(off, w, d, [g0], P, hp=B.hough_params(), zref=[float(ev.seed[1])], hough_sets_axes=False)
    plain = sc.scan(E, [g0], P, per_seed=False)
    assert np.array_equal(keep["ranges"], h["ranges"])
    for k in ("best_seed", "best_n_match", "best_chi2", "labels", "best_key"):
        assert np.array_equal(keep[k], plain[k]), k


def test_fp32_peak_probe_is_near_nominal():
    f, ms = B.cdc_fp32_peak_probe(2048)
    assert 40e12 < f < 80e12 and ms > 0


@pytest.mark.parametrize("cfg_id", [1, 3])
def test_paper_thread_mapping_gives_the_same_scores(cfg_id):
    """The re-created v1 mapping of the paper (one block per seed, one thread per fired wire) is a comparison point:
    same arithmetic, same scoring rule, so its per-seed n_match equals the product kernel's (and the oracle's)."""
    import torch
    cfg, geom, field, events, grids = U.make_workload(cfg_id, n_events=2, grid_n=6)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    P = U.gpu_params(cfg)
    ref = sc.scan(E, grids, P, per_seed=True, best=False)
    sel = synth.stratified_seed_sample(grids[1].n_seeds, 300, key=9)
    d_sel = torch.tensor(sel, dtype=torch.int64, device="cuda")
    d_nm = torch.zeros(sel.size, dtype=torch.int32, device="cuda"); d_c2 = torch.zeros(sel.size, dtype=torch.float32, device="cuda")
    B.cdc_seed_scan_paper_mapping(sc.geometry, E, 1, grids[1], P, d_sel, d_nm, d_c2)
    torch.cuda.synchronize()
    nm = d_nm.cpu().numpy(); c2 = d_c2.cpu().numpy()
    o = grids[0].n_seeds
    same = nm == ref["n_match"][o + sel]
    assert same.mean() > 0.99                                   # uniform field: stage form vs closed form, edge cases only
    assert np.all(np.abs(c2[same] - ref["chi2"][o + sel][same]) <= 1e-3 * np.maximum(nm[same], 1))
    orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), events[1].wire_id, events[1].drift_mm, grids[1], index_list=sel)
    bound = oracle.Bound(geom, field, U.oracle_params(cfg))
    for i in np.nonzero(nm != orc["n_match"])[0]:
        assert U.explain_mismatch(bound, events[1], grids[1].node(grids[1].unravel(int(sel[i]))), cfg, geom)
    assert (nm != orc["n_match"]).sum() <= 2
    # the two-kernel mapping (record every step, then DCA per wire from the record): same arithmetic,
    # so bit-equal to the one-kernel mapping
    d_nm2 = torch.zeros_like(d_nm); d_c22 = torch.zeros_like(d_c2)
    ms = B.cdc_seed_scan_paper_mapping_v2(sc.geometry, E, 1, grids[1], P, d_sel, d_nm2, d_c22, timed=True)
    torch.cuda.synchronize()
    assert np.array_equal(d_nm2.cpu().numpy(), nm) and ms[0] > 0 and ms[1] > 0
    assert np.allclose(d_c22.cpu().numpy(), c2, rtol=1e-5, atol=1e-6)       # block-level float atomics: order differs
    with pytest.raises(B.CdcError):                                         # 32 B x seeds x steps beyond 16 GiB
        B.cdc_seed_scan_paper_mapping_v2(sc.geometry, E, 1, grids[1], B.scan_params(cfg.h_mm, 2_000_000, cfg.window_mm),
                                         d_sel, d_nm2, d_c22)


def test_tightly_curling_seeds_use_the_short_lookup_cadence(setup):
    """Seeds with a small track radius (here below 20 mm) cannot use the look-ahead lookup centre; they fall
    back to a lookup around their own position.  Every wire of the two innermost layers is fired, so any wire the
    candidate set missed would show up as a missing match."""
    cfg, geom, field, events, grids, sc = setup
    w = np.arange(0, int(geom.offset[2]), dtype=np.int32)
    d = np.full(w.size, 4.0, dtype=np.float32)
    off = np.array([0, w.size], dtype=np.int32)
    E = sc.upload(off, w, d)
    # p between 3.5 and 6.5 MeV/c (radius 10-20 mm), pointing outward at R0 + a bit, mostly transverse
    g = synth.Grid(lo=np.array([0.2, -50.0, 3.0, 1.0, 0.2]), step=np.array([0.9, 40.0, 0.6, 0.5, 0.15]),
                   n=np.array([3, 3, 4, 4, 3], dtype=np.int32))
    geom2 = synth.make_geometry(R0=522.0)                     # start close to the first layer so the curl reaches it
    sc2 = api.SeedScanner(geom2, field)
    E2 = sc2.upload(off, w, d)
    P = B.scan_params(cfg.h_mm, 600, cfg.window_mm)
    gpu = sc2.scan(E2, [g], P, per_seed=True, debug=True, best=False)
    params = dict(h=cfg.h_mm, max_steps=600, window=cfg.window_mm)
    orc = oracle.scan_parallel(geom2, field, params, w, d, g)
    assert orc["n_match"].max() >= 3                          # the curls do reach fired wires
    bound = oracle.Bound(geom2, field, params)
    bad = np.nonzero((gpu["n_match"] != orc["n_match"]) | (gpu["debug"]["n_steps"] != orc["n_steps"]))[0]
    for i in bad:
        ev = synth.Event(wire_id=w, drift_mm=d, truth_turn=np.zeros_like(w), seed=np.zeros(5), n_turns=1, n_signal=0)
        same = gpu["debug"]["n_steps"][i] == orc["n_steps"][i] and gpu["debug"]["m_gas"][i] == orc["m_gas"][i]
        assert U.explain_mismatch(bound, ev, g.node(g.unravel(int(i))), cfg, geom2,
                                  dn=int(gpu["n_match"][i]) - int(orc["n_match"][i]),
                                  dchi2=float(gpu["chi2"][i]) - float(orc["chi2"][i]), same_track=bool(same))
    assert bad.size <= 3


@pytest.mark.parametrize("field_kind", [0, 1])
def test_moderately_curling_seeds_dense_hits_every_seed(setup, field_kind):
    """Seeds with a track radius of 30-150 mm (9-45 MeV/c) use the look-ahead lookup and the slot-pruning bounds with a
    large curvature term; every wire of the four innermost layers carries a hit with a random drift distance, so a wire
    that was wrongly kept out of the live slots would show up as a missing match."""
    cfg, geom, _, events, grids, sc = setup
    field = synth.make_uniform_field() if field_kind == 0 else synth.make_table_field()
    rng = np.random.default_rng(17)
    w = np.arange(0, int(geom.offset[4]), dtype=np.int32)
    d = rng.uniform(0.0, 8.0, size=w.size).astype(np.float32)
    off = np.array([0, w.size], dtype=np.int32)
    geom2 = synth.make_geometry(R0=522.0)
    sc2 = api.SeedScanner(geom2, field)
    E2 = sc2.upload(off, w, d)
    g = synth.Grid(lo=np.array([0.1, -300.0, 6.0, 2.0, -6.0]), step=np.array([0.7, 150.0, 6.0, 5.0, 4.0]),
                   n=np.array([4, 5, 6, 6, 4], dtype=np.int32))
    P = B.scan_params(cfg.h_mm, 800, 2.0)
    gpu = sc2.scan(E2, [g], P, per_seed=True, debug=True, best=False)
    params = dict(h=cfg.h_mm, max_steps=800, window=2.0)
    orc = oracle.scan_parallel(geom2, field, params, w, d, g)
    assert orc["n_match"].max() >= 6 and (orc["n_match"] > 0).mean() > 0.3
    bound = oracle.Bound(geom2, field, params)
    cfg2 = __import__("dataclasses").replace(cfg, window_mm=2.0)
    bad = np.nonzero((gpu["n_match"] != orc["n_match"]) | (gpu["debug"]["n_steps"] != orc["n_steps"]))[0]
    for i in bad:
        ev = synth.Event(wire_id=w, drift_mm=d, truth_turn=np.zeros_like(w), seed=np.zeros(5), n_turns=1, n_signal=0)
        same = gpu["debug"]["n_steps"][i] == orc["n_steps"][i] and gpu["debug"]["m_gas"][i] == orc["m_gas"][i]
        assert U.explain_mismatch(bound, ev, g.node(g.unravel(int(i))), cfg2, geom2,
                                  dn=int(gpu["n_match"][i]) - int(orc["n_match"][i]),
                                  dchi2=float(gpu["chi2"][i]) - float(orc["chi2"][i]), same_track=bool(same)), int(i)
    print(f"field {field_kind}: {bad.size} listed threshold cases of {g.n_seeds} seeds: {bad.tolist()}")
    assert bad.size <= int(1e-2 * g.n_seeds)                  # ~40 approaches per seed here, each with two window edges
    sc2.close()


@pytest.mark.parametrize("field_kind,h,window,steps", [(0, 4.0, 7.0, 750), (1, 0.5, 0.5, 3000), (1, 3.0, 5.0, 1000)])
def test_every_wire_fired_at_the_corners_of_step_and_window(field_kind, h, window, steps):
    """All 4512 wires carry a hit with a random drift distance; the largest window the 2 x 2 lookup admits at h = 4 mm
    (lookup every step), a small step with a narrow window (lookup every 16 steps), and one in between.  Every seed
    against the oracle; differences must be window-edge cases (chi2 difference = dn * lambda) or track thresholds."""
    import dataclasses
    geom = synth.make_geometry()
    field = synth.make_uniform_field() if field_kind == 0 else synth.make_table_field()
    rng = np.random.default_rng(23)
    w = np.arange(0, int(geom.offset[-1]), dtype=np.int32)
    d = rng.uniform(0.0, 8.0, size=w.size).astype(np.float32)
    cfg = dataclasses.replace(synth.CONFIGS[1], h_mm=h, window_mm=window, max_steps=steps, field_kind=field_kind)
    base = synth.generate_events(synth.CONFIGS[1 if field_kind == 0 else 3], geom, field, 1, first_event=7)[0]
    ev = synth.Event(wire_id=w, drift_mm=d, truth_turn=-np.ones_like(w), seed=base.seed, n_turns=1, n_signal=0)
    grid = synth.truth_anchored_grid(base.seed, 5)[0]
    sc = api.SeedScanner(geom, field)
    E = sc.upload(np.array([0, w.size], dtype=np.int32), w, d)
    gpu = sc.scan(E, [grid], U.gpu_params(cfg), per_seed=True, debug=True)
    orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), w, d, grid)
    assert orc["n_match"].mean() > 5
    dbg = gpu["debug"]
    same = (dbg["n_steps"] == orc["n_steps"]) & (dbg["m_gas"] == orc["m_gas"])
    bad = np.nonzero((gpu["n_match"] != orc["n_match"]) | ~same)[0]
    bound = oracle.Bound(geom, field, U.oracle_params(cfg))
    for i in bad:
        assert U.explain_mismatch(bound, ev, grid.node(grid.unravel(int(i))), cfg, geom,
                                  dn=int(gpu["n_match"][i]) - int(orc["n_match"][i]),
                                  dchi2=float(gpu["chi2"][i]) - float(orc["chi2"][i]), same_track=bool(same[i])), int(i)
    assert bad.size <= int(5e-3 * grid.n_seeds)
    U.check_best(cfg, geom, field, ev, grid, gpu, orc_full=orc)
    sc.close()


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_candidate_pool_overflow_is_recovered_by_a_second_pass(setup, variant):
    """More near-ties than the candidate pool holds: a plateau grid -- step = 0 on four
    axes, 16^5 = 1,048,576 nodes of which only 16 are distinct, each 65,536 times -- fills the 65,536-entry pool in
    launch order, against the running maximum.  cdc_best_track must collect the near-ties of the FINAL maximum again
    (second pass of the scan into a pool sized for them) and return the exact best seed: the LOWEST linear index among
    the copies of the best node (reading C10), its n_match / chi2 bit-equal to the oracle's, and the labels."""
    cfg, geom, field, events, grids, sc = setup
    ev = events[0]
    full, _ = synth.truth_anchored_grid(ev.seed, 16)
    lo = ev.seed.copy(); lo[4] = full.lo[4]
    step = np.zeros(5); step[4] = full.step[4]
    grid = synth.Grid(lo=lo, step=step, n=np.full(5, 16, dtype=np.int32))
    off, w, d = synth.pack_hits([ev])
    E = sc.upload(off, w, d)
    gpu = sc.scan(E, [grid], U.gpu_params(cfg, kernel_variant=variant), per_seed=False, debug=False)
    st = gpu["stats"]
    assert st["pool_cap"] == 65536 and st["n_pool"] >= 65536          # the second pass's count: every copy of the best node
    line = synth.Grid(lo=lo, step=step, n=np.array([1, 1, 1, 1, 16], dtype=np.int32))
    bound = oracle.Bound(geom, field, U.oracle_params(cfg))
    o = oracle.scan(bound, ev.wire_id, ev.drift_mm, line)
    k, _ = oracle.argmax(o["n_match"], o["chi2"], cfg.window_mm)
    assert int(gpu["best_seed"][0]) == k                               # theta, z, px, py indices 0: linear index = i_pz
    assert int(gpu["best_n_match"][0]) == int(o["n_match"][k]) and float(gpu["best_chi2"][0]) == float(o["chi2"][k])
    lab, _ = oracle.labels(bound, ev.wire_id, ev.drift_mm, line.node((0, 0, 0, 0, k)))
    assert np.array_equal(gpu["labels"], lab)
    # an ordinary scan on the same handle afterwards is unaffected
    g2 = grids[0]
    again = sc.scan(E, [g2], U.gpu_params(cfg, kernel_variant=variant), per_seed=False, debug=False)
    E2 = sc.upload(off, w, d)
    fresh = sc.scan(E2, [g2], U.gpu_params(cfg, kernel_variant=variant), per_seed=False, debug=False)
    for key in ("best_seed", "best_n_match", "best_chi2", "labels", "best_key"):
        assert np.array_equal(again[key], fresh[key]), key


@pytest.mark.parametrize("world", [2, 3])
def test_theta_sharded_scan_equals_the_unsharded_scan(setup, world):
    """One event batch split over `world` GPUs along theta, the ranks run one after the
    other on this one device: the merged best seed, chi2 (as doubles), n_match and labels must equal the unsharded call's,
    bit for bit, and the slab node values must be bit-identical to the full grid's (the node offset travels in
    cdc_grid_spec.first)."""
    from paper_1908_01949_b200 import dist as D
    cfg, geom, field, events, _, sc = setup
    grids = [synth.truth_anchored_grid(ev.seed, (7, 6, 5, 5, 5))[0] for ev in events]     # 7 theta nodes: uneven slabs
    grids[2] = synth.truth_anchored_grid(events[2].seed, (2, 6, 5, 5, 5))[0]              # fewer theta nodes than 3 ranks
    off, w, d = synth.pack_hits(events)
    P = U.gpu_params(cfg)
    whole = sc.scan(sc.upload(off, w, d), grids, P, per_seed=False)
    results, offsets = [], []
    for rank in range(world):
        subs, offs = sc.slabs(grids, rank, world)
        for g, sub, o in zip(grids, subs, offs):
            if o >= 0:
                for i in range(int(sub.n[0])):
                    lin = sub.linear((i, 0, 0, 0, 0))
                    assert D.slab_node(sub, sub.unravel(lin))[0] == g.node(g.unravel(lin + o))[0]      # bit-identical
        r = sc.scan_sharded(sc.upload(off, w, d), grids, P, rank, world, off, collective=False)
        results.append(r["result"]); offsets.append(r["offsets"])
    assert offsets[world - 1][2] == (-1 if world == 3 else offsets[world - 1][2])
    merged = D.merge_slab_results(results, offsets, cfg.window_mm, off)
    for k in ("best_seed", "best_n_match", "best_chi2", "labels"):
        assert np.array_equal(merged[k], whole[k]), k
    assert np.array_equal(merged["best_S"], D.exact_score(whole["best_n_match"], whole["best_chi2"], cfg.window_mm))
    # the collective form of the merge in a single process (world size 1 degenerates to the rank's own result)
    one = sc.scan_sharded(sc.upload(off, w, d), grids, P, 0, 1, off, collective=True)
    for k in ("best_seed", "best_n_match", "best_chi2", "labels"):
        assert np.array_equal(one[k], whole[k]), k


def test_field_reuse_decision_boundary_positions(setup):
    """Tabulated field: the kernel carries B at a step's start vertex over from the previous step's 4th-stage point only
    where the two provably differ by less than half an ulp32 of B_max (reading C22; about 25 MeV/c for this
    table at 2 mm steps).  Seeds from 12 to 60 MeV/c -- both sides of that decision -- end within 1e-3 mm of the oracle,
    which evaluates B at every vertex, with identical step counts."""
    cfg, geom, _, events, grids, sc = setup
    field = synth.make_table_field()
    cfg3 = synth.CONFIGS[3]
    ev = synth.generate_events(cfg3, geom, field, 1)[0]
    u = ev.seed[2:5] / np.linalg.norm(ev.seed[2:5])
    # |p| of the nodes: the three momentum axes scale the truth direction by 0.12 .. 0.57 independently
    lo = np.concatenate([ev.seed[:2], 0.12 * 104.97 * u]); step = np.concatenate([[0.0, 0.0], 0.09 * 104.97 * u])
    g = synth.Grid(lo=lo, step=step, n=np.array([1, 1, 6, 6, 6], dtype=np.int32))
    p = np.array([np.linalg.norm(g.node(g.unravel(i))[2:5]) for i in range(g.n_seeds)])
    assert p.min() < 20.0 and p.max() > 50.0 and ((p > 20) & (p < 30)).any()
    sc3 = api.SeedScanner(geom, field)
    E3 = sc3.upload(*synth.pack_hits([ev]))
    P = B.scan_params(cfg3.h_mm, 900, cfg3.window_mm)
    gpu = sc3.scan(E3, [g], P, per_seed=True, debug=True, best=False)
    orc = oracle.scan_parallel(geom, field, dict(h=cfg3.h_mm, max_steps=900, window=cfg3.window_mm), ev.wire_id, ev.drift_mm, g)
    same = gpu["debug"]["n_steps"] == orc["n_steps"]
    assert (~same).sum() <= 2
    pos = np.stack([gpu["debug"][k] for k in "xyz"], axis=1)
    err = np.linalg.norm(pos - orc["final_r"], axis=1)
    print(f"|p| {p.min():.1f} .. {p.max():.1f} MeV/c, steps {orc['n_steps'].min()} .. {orc['n_steps'].max()}, max position error "
          f"{err[same].max():.2e} mm (below 25 MeV/c: {err[same & (p < 25)].max():.2e}, above: {err[same & (p >= 25)].max():.2e})")
    assert err[same].max() < U.POS_TOL_MM
    sc3.close()


def test_field_reuse_on_and_off_give_the_same_tracks(setup):
    """A / B of the one decision of reading C22 (params.kernel_variant = 3 evaluates B at every start vertex): per seed the
    same step counts, final positions within 2e-5 mm of one another (both within 1e-3 mm of the oracle, test above and
    test_gpu_parity.py), n_match equal up to a handful of window-edge cases, and the same exact best seed, chi2 and labels."""
    cfg3, geom, field, events, grids = U.make_workload(3, n_events=3, grid_n=9)
    sc3 = api.SeedScanner(geom, field)
    out = []
    for variant in (0, 3):
        E3 = sc3.upload(*synth.pack_hits(events))
        out.append(sc3.scan(E3, grids, U.gpu_params(cfg3, kernel_variant=variant), per_seed=True, debug=True))
    a, b = out
    assert np.array_equal(a["debug"]["n_steps"], b["debug"]["n_steps"])
    d = np.sqrt(sum((a["debug"][k] - b["debug"][k]) ** 2 for k in "xyz"))
    n_diff = int((a["n_match"] != b["n_match"]).sum())
    print(f"reuse on / off: {a['n_match'].size} seeds, max position difference {d.max():.2e} mm, n_match differs on {n_diff}")
    assert d.max() < 2e-5
    assert n_diff <= max(2, int(2e-4 * a["n_match"].size))
    for k in ("best_seed", "best_n_match", "best_chi2", "labels"):
        assert np.array_equal(a[k], b[k]), k
    sc3.close()
