"""The two-seeds-per-thread variant of the scan kernel (params.kernel_variant = 1, csrc/scan_pair.cu: two z0-neighbour
seeds per thread, every quantity a packed fp32 pair, ONE wire lookup for both) against the production kernel (one
seed per thread, csrc/scan.cu).  Every half of a packed instruction rounds like the scalar one and the operation order
of the propagation and of every g, D and residual is the same, so per-seed n_match and step / turn / in-gas counts must
be IDENTICAL, and so must the exact (fp64) best seed, its n_match / chi2 and the labels; final positions are
bit-identical in the uniform field and within 1e-4 mm in the tabulated one; the fp32 chi2 of a seed is the same set of
terms, added in the order of the shared lookup's slot list (a few ulp of the sum).  Parity of the production kernel with
the fp64 oracle is test_gpu_parity.py / test_gpu_edges.py / test_gpu_sizes.py."""
import dataclasses

import numpy as np
import pytest

from paper_1908_01949_b200 import api, binding as B, synth

import parity_util as U

pytestmark = pytest.mark.gpu


def _both(sc, events, grids, cfg, debug):
    off, w, d = synth.pack_hits(events)
    out = []
    for variant in (1, 0):
        E = sc.upload(off, w, d)
        out.append(sc.scan(E, grids, U.gpu_params(cfg, kernel_variant=variant), per_seed=True, debug=debug))
    return out


def _assert_identical(a, b, debug):
    assert np.array_equal(a["n_match"], b["n_match"])
    assert np.all(np.abs(a["chi2"].astype(np.float64) - b["chi2"]) <= 2e-5 * np.maximum(b["n_match"], 1))
    for k in ("best_seed", "best_n_match", "best_chi2", "labels"):
        assert np.array_equal(a[k], b[k]), k
    assert a["stats"]["n_steps"] == b["stats"]["n_steps"]
    if debug:
        for k in ("n_steps", "turns", "m_gas"):
            assert np.array_equal(a["debug"][k], b["debug"][k]), k
        for k in ("x", "y", "z"):
            assert np.all(np.abs(a["debug"][k] - b["debug"][k]) <= 1e-4), k


@pytest.mark.parametrize("cfg_id,n_events,grid_n", [(0, 2, 8), (1, 2, (6, 9, 5, 5, 5)), (2, 1, (5, 7, 5, 5, 4)),
                                                    (3, 3, (5, 9, 5, 5, 5)), (3, 2, (4, 1, 6, 5, 5))])
@pytest.mark.parametrize("debug", [False, True])
def test_pair_kernel_equals_one_seed_kernel(cfg_id, n_events, grid_n, debug):
    """Even and odd z0 node counts (an odd count leaves the last node without a partner), a single z0 node, both
    fields, energy loss; with and without the debug record (the variant without in-gas bookkeeping)."""
    cfg, geom, field, events, grids = U.make_workload(cfg_id, n_events=n_events, grid_n=grid_n)
    sc = api.SeedScanner(geom, field)
    a, b = _both(sc, events, grids, cfg, debug)
    _assert_identical(a, b, debug)
    assert int(a["n_match"].max()) >= 10


@pytest.mark.parametrize("fieldname", ["uniform", "table"])
def test_pair_kernel_dense_hits_spill_slots(fieldname):
    """Every wire of the inner layers fired and soft, curling seeds: the union of the two seeds' candidate sets exceeds
    the four register slots and spills to shared memory."""
    geom = synth.make_geometry()
    field = synth.make_uniform_field() if fieldname == "uniform" else synth.make_table_field()
    cfg = dataclasses.replace(synth.CONFIGS[1 if fieldname == "uniform" else 3], max_steps=1200)
    w = np.arange(0, int(geom.offset[6]), dtype=np.int32)                  # six inner layers, every wire
    rng = np.random.default_rng(5)
    d = rng.uniform(0.0, 8.0, w.size).astype(np.float32)
    ev = dataclasses.replace(synth.generate_events(cfg, geom, field, 1)[0], wire_id=w, drift_mm=d,
                             truth_turn=np.zeros(w.size, np.int32))
    grid = synth.Grid(lo=np.array([0.2, -350.0, -40.0, -40.0, -12.0]), step=np.array([0.3, 100.0, 16.0, 16.0, 6.0]),
                      n=np.array([4, 8, 6, 6, 5], dtype=np.int32))
    sc = api.SeedScanner(geom, field)
    a, b = _both(sc, [ev], [grid], cfg, True)
    _assert_identical(a, b, True)
    assert int(a["n_match"].max()) >= 5
