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
    assert Q.common_hits(label, [0, -1, 1, 1, -1, 0, 0, 0, 0, 0, 0, -1]) == 6      # hits 0, 2, 5, 6, 7, 9


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
    eff_sig = []
    for e in range(len(events)):
        sl = slice(off[e], off[e + 1])
        r = Q.classification_quality(out["labels"][sl], truth[sl], 3)
        for k in ("confusion", "c_true", "noise_into"):
            assert np.array_equal(q[k][e], r[k]), k
        assert q["efficiency"][e].tolist() == r["efficiency"].tolist()          # one IEEE division each
        assert q["purity"][e].tolist() == r["purity"].tolist()
        assert nc[e] == Q.common_hits(out["labels"][sl], other[sl])
        eff_sig.append(r["efficiency"][0])
    # the truth is a node of every grid: the first partition is found with high efficiency and purity
    assert np.mean(eff_sig) > 0.8
