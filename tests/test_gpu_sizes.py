"""Parity at the sizes BASELINE.json's configs[2..4] state: configs[3] with its 256 events,
configs[4] at 32^5 seeds per event and at a batch of 1024 events, and -- gated, because the oracle needs ~8 minutes on
16 cores -- the oracle's arg max over EVERY seed of one configs[2] event.  The GPU side runs in the launch
configuration bench.py times (production kernel, no per-seed outputs) and, where per-seed comparisons need them, again
with the per-seed outputs; the two must agree bit for bit.  Tolerances: parity_util.py (BASELINE.json north_star)."""
import os

import numpy as np
import pytest

import oracle
from paper_1908_01949_b200 import api, binding as B, synth

import parity_util as U

pytestmark = pytest.mark.gpu

BEST_KEYS = ("best_seed", "best_n_match", "best_chi2", "labels", "best_key")


def _oracle_best_from_near_set(cfg, geom, field, ev, grid, S32, slack=1.0):
    """The oracle's arg max over every seed whose fp32 score is within `slack` of the fp32 maximum (the fp32 score is
    good to ~1e-2, reading C11), with its n_match, chi2 and labels."""
    bound = oracle.Bound(geom, field, U.oracle_params(cfg))
    near = np.nonzero(S32 >= S32.max() - slack)[0].astype(np.int64)
    o = oracle.scan(bound, ev.wire_id, ev.drift_mm, grid, index_list=near, details=False)
    k, _ = oracle.argmax(o["n_match"], o["chi2"], cfg.window_mm)
    b = int(near[k])
    lab, _ = oracle.labels(bound, ev.wire_id, ev.drift_mm, grid.node(grid.unravel(b)))
    return b, int(o["n_match"][k]), float(o["chi2"][k]), lab, near.size


def _near_job(job):
    cfg, geom, field, ev, grid, S32 = job
    return _oracle_best_from_near_set(cfg, geom, field, ev, grid, S32)


# ------------------------------------------------------------------ configs[3]: 256 events x 16^5
def test_cfg3_full_batch_of_256_events():
    """configs[3] as stated: 256 events x 16^5 seeds in the tabulated field.  (i) the whole batch in bench.py's launch
    configuration and again with per-seed outputs: identical best seeds, labels and fused arg-max keys; the candidate pool
    did not overflow; (ii) for ALL 256 events the best seed, its n_match / chi2 (bit-equal doubles) and the labels equal
    the oracle's arg max over every seed within 1.0 of the fp32 maximum; (iii) positions, step counts, n_match, chi2 on
    32 of the events: one on every seed, 250 stratified seeds on each of the others."""
    import multiprocessing as mp
    cfg = synth.CONFIGS[3]
    geom = synth.make_geometry(); field = synth.make_table_field()
    events = synth.generate_events_parallel(3, 256)
    assert len(events) == cfg.n_events == 256
    grids = [synth.truth_anchored_grid(ev.seed, cfg.grid_n)[0] for ev in events]
    assert all(g.n_seeds == 16 ** 5 for g in grids)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    P = U.gpu_params(cfg)
    E = sc.upload(off, w, d)
    bare = sc.scan(E, grids, P, per_seed=False, debug=False)               # what bench.py times
    assert bare["stats"]["n_pool"] <= bare["stats"]["pool_cap"] and bare["stats"]["n_seeds"] == 256 * 16 ** 5
    full = sc.scan(E, grids, P, per_seed=True, debug=False)
    for k in BEST_KEYS:
        assert np.array_equal(bare[k], full[k]), k
    assert (bare["best_seed"] >= 0).all()
    # (ii) every event against the oracle
    ns = 16 ** 5
    jobs = []
    for e, (ev, grid) in enumerate(zip(events, grids)):
        S32 = full["n_match"][e * ns:(e + 1) * ns].astype(np.float64) - full["chi2"][e * ns:(e + 1) * ns] / cfg.window_mm ** 2
        jobs.append((cfg, geom, field, ev, grid, S32))
    with mp.get_context("fork").Pool(os.cpu_count() or 1) as pool:
        res = pool.map(_near_job, jobs)
    near_total = 0
    for e, (b, nm, c2, lab, n_near) in enumerate(res):
        assert int(bare["best_seed"][e]) == b, f"event {e}: best seed {bare['best_seed'][e]} vs oracle {b}"
        assert int(bare["best_n_match"][e]) == nm and float(bare["best_chi2"][e]) == c2, f"event {e}"
        assert np.array_equal(bare["labels"][off[e]:off[e + 1]], lab), f"event {e}: labels"
        near_total += n_near
    # (iii) per-seed parity on 32 events (debug records: positions, step and in-gas counts)
    sub = list(range(0, 256, 8))
    ev_s = [events[i] for i in sub]; gr_s = [grids[i] for i in sub]
    off_s, w_s, d_s = synth.pack_hits(ev_s)
    Es = sc.upload(off_s, w_s, d_s)
    dbg = sc.scan(Es, gr_s, P, per_seed=True, debug=True)
    listed = 0
    for j, (i, ev, grid) in enumerate(zip(sub, ev_s, gr_s)):
        assert np.array_equal(dbg["n_match"][j * ns:(j + 1) * ns], full["n_match"][i * ns:(i + 1) * ns])       # batch-independent
        if j == 1:
            sel = np.arange(ns)
            orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), ev.wire_id, ev.drift_mm, grid, n_proc=os.cpu_count())
        else:
            sel = synth.stratified_seed_sample(ns, 250, key=300 + i)
            orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), ev.wire_id, ev.drift_mm, grid, index_list=sel)
        listed += len(U.compare_scan(cfg, geom, field, ev, grid, dbg, orc, sel, offset=j * ns))
    print(f"cfg3 x 256: best seed / n_match / chi2 / labels bit-exact on 256 of 256 events (oracle on {near_total} near-maximum "
          f"seeds); {listed} listed threshold exceptions of {ns + 31 * 250} compared seeds; pool {bare['stats']['n_pool']} of "
          f"{bare['stats']['pool_cap']}")


# ------------------------------------------------------------------ configs[4]: 32^5 seeds, one event
def test_cfg4_grid_32_to_the_5th():
    """33,554,432 seeds of one event (grid.x = 262,144 blocks): 4096 stratified seeds + the truth node's neighbourhood
    against the oracle, the best seed against the oracle's arg max over every seed within 1.0 of the fp32 maximum."""
    cfg, geom, field, events, grids = U.make_workload(4, n_events=1, grid_n=32)
    ev, grid = events[0], grids[0]
    assert grid.n_seeds == 32 ** 5
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    gpu = sc.scan(E, grids, U.gpu_params(cfg), per_seed=True, debug=True)
    bare = sc.scan(E, grids, U.gpu_params(cfg), per_seed=False, debug=False)
    for k in BEST_KEYS:
        assert np.array_equal(bare[k], gpu[k]), k
    sel = synth.stratified_seed_sample(grid.n_seeds, 4096, key=41)
    anchor = np.array([16] * 5)
    nb = [grid.linear(tuple(anchor + np.array(dlt))) for dlt in np.ndindex(3, 3, 3, 3, 3)]     # truth node .. +2 on every axis
    sel = np.unique(np.concatenate([sel, np.array(nb, dtype=np.int64)]))
    orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), ev.wire_id, ev.drift_mm, grid, index_list=sel)
    listed = U.compare_scan(cfg, geom, field, ev, grid, gpu, orc, sel)
    U.check_best(cfg, geom, field, ev, grid, gpu)
    print(f"cfg4 32^5: {len(listed)} listed threshold exceptions of {sel.size}; pool {gpu['stats']['n_pool']}")


# ------------------------------------------------------------------ configs[4]: batch of 1024 events
def test_cfg4_batch_of_1024_events():
    """1024 x 16^5 = 1.07e9 seeds in one call (grid.y = 1024): 128 generated events, each eight times in the batch (every
    copy is uploaded, binned and scanned on its own).  All copies of an event must give the same answer; for 16 events
    best seed, n_match, chi2 and labels are checked against the oracle (arg max over the near-maximum seeds of a separate
    per-seed scan) and 200 stratified seeds each against the oracle's per-seed results."""
    cfg = synth.CONFIGS[4]
    geom = synth.make_geometry(); field = synth.make_table_field()
    base = synth.generate_events_parallel(4, 128)
    events = [base[i % 128] for i in range(1024)]
    grids = [synth.truth_anchored_grid(ev.seed, 16)[0] for ev in events]
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    P = U.gpu_params(cfg)
    E = sc.upload(off, w, d)
    big = sc.scan(E, grids, P, per_seed=False, debug=False)
    assert big["stats"]["n_seeds"] == 1024 * 16 ** 5 and (big["best_seed"] >= 0).all()
    for k in ("best_seed", "best_n_match", "best_chi2", "best_key"):
        v = big[k].reshape(8, 128)
        assert (v == v[0]).all(), k
    ns = 16 ** 5
    sub = list(range(0, 128, 8))
    ev_s = [base[i] for i in sub]; gr_s = [grids[i] for i in sub]
    off_s, w_s, d_s = synth.pack_hits(ev_s)
    small = sc.scan(sc.upload(off_s, w_s, d_s), gr_s, P, per_seed=True, debug=True)
    listed = 0
    for j, (i, ev, grid) in enumerate(zip(sub, ev_s, gr_s)):
        for k in ("best_seed", "best_n_match", "best_chi2", "best_key"):
            assert small[k][j] == big[k][i], (k, i)
        assert np.array_equal(small["labels"][off_s[j]:off_s[j + 1]], big["labels"][off[i]:off[i + 1]])
        U.check_best(cfg, geom, field, ev, grid, small, e=j, hit_slice=slice(off_s[j], off_s[j + 1]))
        sel = synth.stratified_seed_sample(ns, 200, key=500 + i)
        orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), ev.wire_id, ev.drift_mm, grid, index_list=sel)
        listed += len(U.compare_scan(cfg, geom, field, ev, grid, small, orc, sel, offset=j * ns))
    print(f"cfg4 batch 1024: {listed} listed threshold exceptions of {16 * 200}; pool {big['stats']['n_pool']} of {big['stats']['pool_cap']}")


# ------------------------------------------------------------------ configs[2]: the oracle's arg max over the WHOLE grid
@pytest.mark.skipif(os.environ.get("CDC_SLOW_PARITY") != "1",
                    reason="~8 min of oracle on 16 cores (3.6e10 RKN steps): set CDC_SLOW_PARITY=1; the result of the "
                           "round's run is committed under profiles/")
def test_cfg2_full_grid_oracle_argmax():
    """One configs[2] event (24^5 = 7,962,624 seeds, Hough-derived axes, energy loss): the oracle evaluates EVERY seed
    (split over the host cores by seed range; every process is the single-threaded oracle) and its arg max must be the
    GPU's best seed -- no GPU score enters the oracle's candidate set (VERDICT r1 missing #4)."""
    cfg, geom, field, events, _ = U.make_workload(2)
    ev = events[0]
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    h = sc.hough(E, [float(ev.seed[1])])
    g0, _ = synth.truth_anchored_grid(ev.seed, cfg.grid_n)
    lo = g0.lo.copy(); hi = g0.lo + g0.step * (g0.n - 1)
    lo[[0, 2, 3]] = h["ranges"][0][:, 0]; hi[[0, 2, 3]] = h["ranges"][0][:, 1]
    grid = synth.ranges_grid(lo, hi, cfg.grid_n)
    gpu = sc.scan(E, [grid], U.gpu_params(cfg), per_seed=True, debug=True)
    orc = oracle.scan_parallel(geom, field, U.oracle_params(cfg), ev.wire_id, ev.drift_mm, grid, n_proc=os.cpu_count())
    listed = U.compare_scan(cfg, geom, field, ev, grid, gpu, orc, np.arange(grid.n_seeds))
    b = U.check_best(cfg, geom, field, ev, grid, gpu, orc_full=orc)
    S = orc["n_match"] - orc["chi2"] / cfg.window_mm ** 2
    top2 = np.sort(S)[-2:]
    print(f"cfg2 full grid: oracle arg max over {grid.n_seeds} seeds = GPU best seed {b}; S gap of the two best seeds "
          f"{top2[1] - top2[0]:.4f}; {len(listed)} listed threshold exceptions of {grid.n_seeds}")
