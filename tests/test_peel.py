"""Turn-partition peeling (reading C18): pins of the plain CPU statement
(oracle/peel.py) and GPU parity of cdc_peel_turns (-m gpu)."""
import math

import numpy as np
import pytest

import oracle
from oracle import peel as OP
from oracle import quality as Q
from paper_1908_01949_b200 import synth

HALF_WIDTH = [0.01, 26.0, 2.5, 2.5, 1.7]        # PAPER.md:51 (0.01 rad, 2.5 MeV) and :83 (2.6 cm, 1.7 MeV)


def _two_turn_event(**kw):
    cfg = synth.CONFIGS[1]
    geom = synth.make_geometry(); field = synth.make_uniform_field()
    ev = synth.generate_events(cfg, geom, field, 1, **kw)[0]
    return cfg, geom, field, ev


def test_next_entrance_is_one_helix_period_later_in_a_uniform_field():
    # closed form: without energy loss the (x, y) projection in a uniform field is a closed circle, so the next
    # outward crossing of rho = R0 is the seed's own (x, y) and direction, one period later:
    # z advances by 2 pi p_z / (kappa |q| B).  The chord / lerp of the crossing are exact to the sagitta
    # h^2 / (8 R) ~ 1.5e-3 mm and to theta^2 / 8 ~ 5e-6 in direction.
    cfg, geom, field, ev = _two_turn_event()
    params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm)
    th, z0, px, py, pz = ev.seed
    nx = OP.next_entrance(geom, field, params, ev.seed, 3000)
    assert nx is not None
    x0, y0 = geom.R0_mm * math.cos(th), geom.R0_mm * math.sin(th)
    dz = 2.0 * math.pi * pz / (0.299792458 * 1.0)
    assert abs(nx[0] - x0) < 3e-3 and abs(nx[1] - y0) < 3e-3
    assert abs(math.hypot(nx[0], nx[1]) - geom.R0_mm) < 1e-9            # on the cylinder
    assert abs(nx[2] - (z0 + dz)) < 3e-3
    p = math.sqrt(px * px + py * py + pz * pz)
    assert abs(nx[3] - px) < 1e-5 * p and abs(nx[4] - py) < 1e-5 * p and abs(nx[5] - pz) < 1e-5 * p
    assert abs(math.sqrt(nx[3] ** 2 + nx[4] ** 2 + nx[5] ** 2) - p) < 1e-9 * p


def test_next_entrance_lies_on_the_chord_of_the_c_oracles_trajectory_and_loses_the_gas_energy():
    # the Python loop of next_entrance against the C oracle's own vertices (orc_eval_seed trajectory): the crossing
    # interval is the first (rho_n < R0 <= rho_{n+1}) after the start, the point lies on that chord at rho = R0, and
    # with energy loss |p| = p0 - eloss * h * (vertices with rho >= R0 before it, the start counted in)  (C6)
    cfg = synth.CONFIGS[2]
    geom = synth.make_geometry(); field = synth.make_uniform_field()
    ev = synth.generate_events(cfg, geom, field, 1)[0]
    params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm, eloss=cfg.eloss_MeV_per_mm)
    bound = oracle.Bound(geom, field, params)
    traj = oracle.eval_seed(bound, ev.wire_id, ev.drift_mm, ev.seed, trajectory=True)["traj"]
    rho2 = traj[:, 0] ** 2 + traj[:, 1] ** 2
    inside = rho2 >= geom.R0_mm ** 2
    inside[0] = True                                                       # reading C7: the seed is in the gas
    n = int(np.nonzero(~inside[:-1] & inside[1:])[0][0])
    nx = OP.next_entrance(geom, field, params, ev.seed, 3000)
    a, b = traj[n, :3], traj[n + 1, :3]
    pos = np.array(nx[:3])
    tau = np.dot(pos - a, b - a) / np.dot(b - a, b - a)
    assert 0.0 <= tau <= 1.0
    assert np.abs(a + tau * (b - a) - pos).max() < 1e-9
    assert abs(math.hypot(nx[0], nx[1]) - geom.R0_mm) < 1e-9
    p0 = math.sqrt(sum(float(v) ** 2 for v in ev.seed[2:]))
    m_gas = int(inside[:n + 1].sum())
    pn = math.sqrt(nx[3] ** 2 + nx[4] ** 2 + nx[5] ** 2)
    assert abs(pn - (p0 - cfg.eloss_MeV_per_mm * cfg.h_mm * m_gas)) < 1e-9
    u = np.array(nx[3:]) / pn                                              # direction between T_n and T_{n+1}
    assert np.dot(u, traj[n, 3:]) > 1 - 1e-4 and np.dot(u, traj[n + 1, 3:]) > 1 - 1e-4


def test_error_estimate_of_the_adaptive_step_equals_its_uniform_field_closed_form():
    # reading C19 / PAPER.md ref. [5]: err = h^2 max_i |k1 - k2 - k3 + k4|_i.  In a uniform field k = c J U with
    # c = a B_z and J (Ux, Uy) = (Uy, -Ux); expanding the four stages gives
    #   k1 - k2 - k3 + k4 = -(c^3 h^2 / 4) J T + (c^4 h^3 / 4) T_xy        (z component 0)
    # and the step itself must be the plain step bit for bit
    geom = synth.make_geometry(); field = synth.make_uniform_field(0.9)
    bound = oracle.Bound(geom, field, dict(h=2.0, max_steps=10, window=1.0))
    rng = np.random.default_rng(5)
    for _ in range(20):
        T = rng.normal(size=3); T /= np.linalg.norm(T)
        r = rng.uniform(-600, 600, size=3)
        a = -0.299792458 / rng.uniform(20.0, 110.0); h = float(rng.choice([1.0, 2.0, 4.0, 16.0]))
        rn, Tn, err = oracle.rkn_step_err(bound, a, h, r, T)
        rn0, Tn0 = oracle.rkn_step(bound, a, h, r, T)
        assert np.array_equal(rn, rn0) and np.array_equal(Tn, Tn0)
        c = a * 0.9
        e = -(c ** 3 * h ** 2 / 4.0) * np.array([T[1], -T[0]]) + (c ** 4 * h ** 3 / 4.0) * T[:2]
        assert abs(err - h * h * np.abs(e).max()) <= 1e-6 * err + 1e-22


def test_adaptive_extrapolation_takes_fewer_longer_steps_to_the_same_entrance():
    cfg, geom, field, ev = _two_turn_event()
    params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm)
    fixed = np.array(OP.next_entrance(geom, field, params, ev.seed, 3000))
    tr = []
    tiny = np.array(OP.next_entrance_adaptive(geom, field, params, ev.seed, 3000, 1e-12, 32.0, trace=tr))
    assert set(tr) == {cfg.h_mm} and np.array_equal(tiny, fixed)        # never below h: the fixed-step form itself
    tr = []
    ad = np.array(OP.next_entrance_adaptive(geom, field, params, ev.seed, 3000, 1e-3, 32.0, trace=tr))
    assert set(tr) <= {2.0, 4.0, 8.0, 16.0, 32.0} and max(tr) >= 8.0 and len(tr) < 300
    assert np.abs(ad[:3] - fixed[:3]).max() < 1e-4 and np.abs(ad[3:] - fixed[3:]).max() < 1e-5
    assert abs(math.hypot(ad[0], ad[1]) - geom.R0_mm) < 1e-9
    capped = []
    OP.next_entrance_adaptive(geom, field, params, ev.seed, 3000, 1.0, 4.0, trace=capped)
    assert max(capped) == 4.0                                            # h_max
    # tabulated field: the estimate follows the field's variation, same entrance
    cfg2 = synth.CONFIGS[2]
    tf = synth.make_table_field()
    ev2 = synth.generate_events(cfg2, geom, tf, 1)[0]
    p2 = dict(h=cfg2.h_mm, max_steps=cfg2.max_steps, window=cfg2.window_mm)
    f2 = np.array(OP.next_entrance(geom, tf, p2, ev2.seed, 3000))
    a2 = np.array(OP.next_entrance(geom, tf, p2, ev2.seed, 3000, 1e-4, 16.0))
    assert np.abs(a2[:3] - f2[:3]).max() < 1e-3 and np.abs(a2[3:] - f2[3:]).max() < 1e-4
    # with energy loss the momentum is constant over a step (C6), so the step length enters at first order:
    # the loss over one 16 mm step is 3.2e-3 MeV/c, 3e-5 of p, which bends ~1 m of path by ~0.02 mm; |p| itself
    # differs by less than one step's loss
    p2["eloss"] = cfg2.eloss_MeV_per_mm
    f2 = np.array(OP.next_entrance(geom, tf, p2, ev2.seed, 3000))
    a2 = np.array(OP.next_entrance(geom, tf, p2, ev2.seed, 3000, 1e-4, 16.0))
    assert np.abs(a2[:3] - f2[:3]).max() < 0.05
    assert abs(np.linalg.norm(a2[3:]) - np.linalg.norm(f2[3:])) <= 16.0 * cfg2.eloss_MeV_per_mm


def test_centred_grid_nodes():
    g = OP.centred_grid([1.0, 2.0, 3.0, 4.0, 5.0], [0.5, 1.0, 0.0, 2.0, 4.0], [3, 5, 1, 2, 9])
    nodes = [[g.lo[a] + i * g.step[a] for i in range(int(g.n[a]))] for a in range(5)]
    assert nodes[0] == [0.5, 1.0, 1.5] and nodes[1] == [1.0, 1.5, 2.0, 2.5, 3.0]
    assert nodes[2] == [3.0] and nodes[3] == [2.0, 6.0] and nodes[4][0] == 1.0 and nodes[4][4] == 5.0 and nodes[4][8] == 9.0
    assert g.n_seeds == 3 * 5 * 2 * 9


def test_peeling_a_smear_free_noise_free_event_returns_the_truth_partitions():
    # every signal hit of a two-turn event ends in the partition of its truth turn, nothing is left, the loop stops
    # because fewer than min_hits hits remain: efficiency = purity = 1 for both partitions (Eq. 2, 3)
    cfg, geom, field, ev = _two_turn_event(sigma_drift=0.0, noise=0.0)
    params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm)
    grid0, _ = synth.truth_anchored_grid(ev.seed, 3)
    r = OP.peel(geom, field, params, ev.wire_id, ev.drift_mm, grid0, [3] * 5, HALF_WIDTH, max_partitions=4,
                min_hits=10, min_classified=5, n_proc=4)
    assert r["status"] == 1 and r["seeds"].shape == (2, 5)
    q = Q.classification_quality(r["partition"], ev.truth_turn, 2)
    assert q["efficiency"].tolist() == [1.0, 1.0] and q["purity"].tolist() == [1.0, 1.0]
    assert np.array_equal(r["partition"], ev.truth_turn)
    assert np.abs(r["seeds"][0] - ev.seed).max() == 0.0                    # the truth is a node of the first grid
    # the second partition's seed is one helix period after the first (uniform field, no loss)
    dz = 2.0 * math.pi * ev.seed[4] / 0.299792458
    assert abs(r["seeds"][1][1] - (ev.seed[1] + dz)) <= 26.0
    assert r["n_match"].sum() >= int((ev.truth_turn >= 0).sum())


def test_peeling_stops_for_each_listed_reason():
    cfg, geom, field, ev = _two_turn_event()
    params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm)
    grid0, _ = synth.truth_anchored_grid(ev.seed, 3)
    kw = dict(n_proc=4)
    r = OP.peel(geom, field, params, ev.wire_id, ev.drift_mm, grid0, [1] * 5, HALF_WIDTH, max_partitions=1, **kw)
    assert r["status"] == 3 and r["seeds"].shape[0] == 1 and set(np.unique(r["partition"])) <= {-1, 0}
    r = OP.peel(geom, field, params, ev.wire_id, ev.drift_mm, grid0, [1] * 5, HALF_WIDTH, min_hits=10 ** 6, **kw)
    assert r["status"] == 1 and r["seeds"].shape[0] == 0 and (r["partition"] == -1).all()
    r = OP.peel(geom, field, params, ev.wire_id, ev.drift_mm, grid0, [1] * 5, HALF_WIDTH, min_classified=10 ** 6, **kw)
    assert r["status"] == 2 and r["seeds"].shape[0] == 0 and (r["partition"] == -1).all()
    # a track that leaves through the end plate before it comes back: |z| > 750 mm (C7)
    far = np.array(ev.seed); far[1] = 700.0 * np.sign(ev.seed[4]); far = far.astype(np.float32).astype(np.float64)
    gfar, _ = synth.truth_anchored_grid(far, 1)
    r = OP.peel(geom, field, params, ev.wire_id, ev.drift_mm, gfar, [1] * 5, HALF_WIDTH, min_classified=0, **kw)
    assert r["status"] == 4 and r["seeds"].shape[0] == 1
    # classified hits are disjoint between partitions and never noise-free-of-charge: every label is a recorded partition
    r = OP.peel(geom, field, params, ev.wire_id, ev.drift_mm, grid0, [3] * 5, HALF_WIDTH, max_partitions=3, **kw)
    assert r["partition"].max() < r["seeds"].shape[0]


def _gpu_vs_oracle(cfg_id, n_events, n0, n, max_steps, P=3, extrap_tol=0.0, extrap_h_max=0.0, **gen_kw):
    from paper_1908_01949_b200 import api, binding as B
    cfg = synth.CONFIGS[cfg_id]
    geom = synth.make_geometry()
    field = synth.make_uniform_field() if cfg.field_kind == 0 else synth.make_table_field()
    events = synth.generate_events(cfg, geom, field, n_events, **gen_kw)
    grids = [synth.truth_anchored_grid(ev.seed, n0)[0] for ev in events]
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = sc.upload(off, w, d)
    bits_before = E.tables()[1].copy()
    params = dict(h=cfg.h_mm, max_steps=max_steps, window=cfg.window_mm, eloss=cfg.eloss_MeV_per_mm)
    Pg = B.scan_params(cfg.h_mm, max_steps, cfg.window_mm, cfg.eloss_MeV_per_mm)
    out = B.cdc_peel_turns(sc.geometry, E, B.grid_specs(grids), Pg, n, HALF_WIDTH, max_partitions=P, min_hits=10,
                           min_classified=5, extrap_max_steps=3000, extrap_tol=extrap_tol, extrap_h_max=extrap_h_max)
    assert np.array_equal(E.tables()[1], bits_before)                       # the events are handed back unchanged
    res = []
    for e, (ev, g0) in enumerate(zip(events, grids)):
        r = OP.peel(geom, field, params, ev.wire_id, ev.drift_mm, g0, n, HALF_WIDTH, max_partitions=P, min_hits=10,
                    min_classified=5, extrap_max_steps=3000, extrap_tol=extrap_tol, extrap_h_max=extrap_h_max)
        k = r["seeds"].shape[0]
        assert out["status"][e] == r["status"] and out["n_partitions"][e] == k, (e, out["status"][e], r["status"])
        assert np.array_equal(out["partition"][off[e]:off[e + 1]], r["partition"]), e       # bit-exact labels
        assert np.array_equal(out["seeds"][e, :k], r["seeds"]), e                           # seeds as doubles
        assert np.array_equal(out["n_match"][e, :k].astype(np.int64), r["n_match"]), e
        assert np.array_equal(out["chi2"][e, :k], r["chi2"]), e
        assert np.array_equal(out["centres"][e, 1:1 + r["centres"].shape[0]], r["centres"]), e   # extrapolation, fp64
        assert not out["seeds"][e, k:].any()
        res.append((ev, r))
    sc.close()
    return res


@pytest.mark.gpu
def test_gpu_peeling_equals_oracle_two_turn_events_uniform_field():
    res = _gpu_vs_oracle(1, 3, 6, [5, 5, 5, 5, 5], 1500)
    # the method works on these events: both partitions found, most of their hits in the right one
    for ev, r in res:
        assert r["seeds"].shape[0] >= 2
        q = Q.classification_quality(r["partition"], ev.truth_turn, 2)
        assert q["efficiency"].min() > 0.5 and q["purity"].min() > 0.6


@pytest.mark.gpu
def test_gpu_peeling_equals_oracle_with_energy_loss_three_turns():
    _gpu_vs_oracle(2, 1, 6, [5, 5, 5, 5, 5], 1500, P=4)


@pytest.mark.gpu
def test_gpu_peeling_equals_oracle_table_field_mixed_turn_counts():
    _gpu_vs_oracle(3, 4, 5, [4, 4, 4, 4, 4], 1500)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg_id,n_events,P", [(1, 2, 3), (2, 1, 4), (3, 4, 3)])
def test_gpu_peeling_with_adaptive_extrapolation_equals_oracle(cfg_id, n_events, P):
    # reading C19: step lengths up to 16 mm between the partitions; every step-size decision is taken in fp64 on both
    # sides, so the extrapolated centres (hence everything after them) are still bit-equal
    res = _gpu_vs_oracle(cfg_id, n_events, 6, [5, 5, 5, 5, 5], 1500, P=P, extrap_tol=1e-4, extrap_h_max=16.0)
    assert any(r["centres"].shape[0] >= 1 for _, r in res)


@pytest.mark.gpu
def test_gpu_peeling_rejects_bad_arguments():
    from paper_1908_01949_b200 import api, binding as B
    cfg, geom, field, ev = _two_turn_event()
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits([ev])
    E = sc.upload(off, w, d)
    g = B.grid_specs([synth.truth_anchored_grid(ev.seed, 2)[0]])
    Pg = B.scan_params(cfg.h_mm, 500, cfg.window_mm)
    for kw in (dict(max_partitions=0), dict(max_partitions=9), dict(min_hits=-1), dict(extrap_max_steps=0),
               dict(extrap_tol=-1.0), dict(extrap_tol=1e-4, extrap_h_max=1.0), dict(extrap_tol=float("nan"))):
        with pytest.raises(B.CdcError):
            B.cdc_peel_turns(sc.geometry, E, g, Pg, [2] * 5, HALF_WIDTH, **kw)
    with pytest.raises(B.CdcError):
        B.cdc_peel_turns(sc.geometry, E, g, Pg, [0, 2, 2, 2, 2], HALF_WIDTH)
    with pytest.raises(B.CdcError):
        B.cdc_peel_turns(sc.geometry, E, g, Pg, [2] * 5, [0.01, -1.0, 1, 1, 1])
    out = B.cdc_peel_turns(sc.geometry, E, g, Pg, [2] * 5, HALF_WIDTH, min_hits=10 ** 6)      # nothing to do
    assert out["status"].tolist() == [1] and out["n_partitions"].tolist() == [0] and (out["partition"] == -1).all()
    sc.close()
