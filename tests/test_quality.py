"""Classification efficiency / purity (Eq. (2), (3)) and N_c: pins of the plain CPU
statement (oracle/quality.py) and GPU parity (-m gpu)."""
import numpy as np
import pytest

from oracle import quality as Q
from paper_1908_01949_b200 import synth


def test_eq2_eq3_on_a_hand_counted_example():
    #        hit:   0  1  2  3  4  5  6  7  8  9 10 11
    truth = [0, 0, 0, 0, 1, 1, 1, 1, 1, -1, -1, 0]
    label = [0, 0, 1, -1, 1, 1, 0, 1, -1, 1, -1, 0]
    r = Q.classification_quality(label, truth, 2)
    # turn 0: 5 true hits, 3 classified 0, 1 classified 1, 1 unclassified; turn 1: 5 true, 3 -> 1, 1 -> 0, 1 unclassified
    assert r["confusion"].tolist() == [[3, 1], [1, 3]]
    assert r["c_true"].tolist() == [5, 5] and r["noise_into"].tolist() == [0, 1]
    assert r["efficiency"].tolist() == [3 / 5, 3 / 5]                   # Eq. (2): C_{n'->n'} / C_n'
    assert r["purity"].tolist() == [3 / 4, 3 / 4]                       # Eq. (3): C_{n'->n'} / sum_i C_{i->n'} (noise not in the sum)
    other = [0, -1, 1, 1, -1, 0, 0, 0, 0, 0, 0, -1]
    assert Q.common_hits(label, other) == 6                              # hits 0, 2, 5, 6, 7, 9
    assert Q.common_hits(label, other, 1, 0) == 3 and Q.common_hits(label, other, 0, 0) == 2   # 5, 7, 9 / 0, 6


def test_perfect_and_empty_classification():
    truth = np.array([0, 0, 1, 1, 1, -1])
    r = Q.classification_quality(truth, truth, 3)
    assert r["efficiency"].tolist() == [1.0, 1.0, -1.0] and r["purity"].tolist() == [1.0, 1.0, -1.0]
    r = Q.classification_quality(-np.ones(6, dtype=int), truth, 2)
    assert r["efficiency"].tolist() == [0.0, 0.0] and r["purity"].tolist() == [-1.0, -1.0]
    assert Q.common_hits(truth, -np.ones(6, dtype=int)) == 0 and Q.common_hits(truth, truth) == 5


@pytest.mark.gpu
def test_gpu_quality_and_common_hits_equal_oracle():
    import torch
    from paper_1908_01949_b200 import api, binding as B
    cfg = synth.CONFIGS[3]
    geom = synth.make_geometry(); field = synth.make_table_field()
    events = synth.generate_events(cfg, geom, field, 6)
    grids = [synth.truth_anchored_grid(ev.seed, 6)[0] for ev in events]
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    out = sc.scan(E, grids, B.scan_params(cfg.h_mm, cfg.max_steps, cfg.window_mm), per_seed=False)
    truth = np.concatenate([ev.truth_turn for ev in events]).astype(np.int32)
    d_lab = torch.tensor(out["labels"], device="cuda"); d_tr = torch.tensor(truth, device="cuda")
    q = B.cdc_classification_quality(E, 3, d_lab, d_tr)
    rng = np.random.default_rng(3)
    other = np.where(rng.random(truth.size) < 0.5, out["labels"], -1).astype(np.int32)
    nc = B.cdc_common_hits(E, d_lab, torch.tensor(other, device="cuda"))
    nc10 = B.cdc_common_hits(E, d_lab, torch.tensor(other, device="cuda"), 1, 0)
    eff_sig = []
    for e in range(len(events)):
        sl = slice(off[e], off[e + 1])
        r = Q.classification_quality(out["labels"][sl], truth[sl], 3)
        for k in ("confusion", "c_true", "noise_into"):
            assert np.array_equal(q[k][e], r[k]), k
        assert q["efficiency"][e].tolist() == r["efficiency"].tolist()          # one IEEE division each
        assert q["purity"][e].tolist() == r["purity"].tolist()
        assert nc[e] == Q.common_hits(out["labels"][sl], other[sl])
        assert nc10[e] == Q.common_hits(out["labels"][sl], other[sl], 1, 0)
        eff_sig.append(r["efficiency"][0])
    # the truth is a node of every grid: the first partition is found with high efficiency and purity
    assert np.mean(eff_sig) > 0.8


@pytest.mark.gpu
def test_bidirectional_scan_and_common_hits():
    """the scan run independently from the entrance and from the exit of the turn partition; the backward
    scan is the same kernel with the opposite charge from the exit-side seed (momentum reversed).  Labels of both scans
    bit-exact against the oracle and N_c equal."""
    import dataclasses
    import torch
    import oracle
    from paper_1908_01949_b200 import api, binding as B
    cfg = dataclasses.replace(synth.CONFIGS[0], noise_occupancy=0.05)
    geom = synth.make_geometry(); field = synth.make_uniform_field()
    events = [ev for ev in synth.generate_events(cfg, geom, field, 12) if ev.seed_exit is not None][:3]
    assert len(events) == 3
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    gf = [synth.truth_anchored_grid(ev.seed, 6)[0] for ev in events]
    gb = [synth.truth_anchored_grid(ev.seed_exit, 6)[0] for ev in events]
    fwd = sc.scan(E, gf, B.scan_params(cfg.h_mm, cfg.max_steps, cfg.window_mm, charge=-1), per_seed=False)
    bwd = sc.scan(E, gb, B.scan_params(cfg.h_mm, cfg.max_steps, cfg.window_mm, charge=+1), per_seed=False)
    nc = B.cdc_common_hits(E, torch.tensor(fwd["labels"], device="cuda"), torch.tensor(bwd["labels"], device="cuda"), 0, 0)
    for e, ev in enumerate(events):
        sl = slice(off[e], off[e + 1])
        labs = []
        for grid, q, got in ((gf[e], -1, fwd), (gb[e], +1, bwd)):
            params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm, charge=q)
            o = oracle.scan_parallel(geom, field, params, ev.wire_id, ev.drift_mm, grid)
            best, _ = oracle.argmax(o["n_match"], o["chi2"], cfg.window_mm)
            assert int(got["best_seed"][e]) == best and float(got["best_chi2"][e]) == float(o["chi2"][best])
            lab, _ = oracle.labels(oracle.Bound(geom, field, params), ev.wire_id, ev.drift_mm, grid.node(grid.unravel(best)))
            assert np.array_equal(got["labels"][sl], lab)
            labs.append(lab)
        assert nc[e] == Q.common_hits(labs[0], labs[1], 0, 0)
        assert nc[e] >= 0.6 * ev.n_signal                     # both directions find most of the partition
    assert max(nc) >= 20                                      # the paper's quality cut N_c >= 20 is reachable
