"""Pins of the oracle's adaptive-step scan propagator (oracle/cdc_oracle.c orc_eval_seed_adaptive; reading C19 applied
to the scan; "the RKN method was used for the track parameter propagation [5]").  None of
them re-derives the controller from itself: the fixed-step oracle (pinned elsewhere), the closed form of the error
estimate in a uniform field, the analytic helix and integer bookkeeping identities.  CPU only."""
import math

import numpy as np
import pytest

import oracle
from paper_1908_01949_b200 import synth

KAPPA = 0.299792458


def _bound(geom, field, cfg, **kw):
    p = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm, eloss=cfg.eloss_MeV_per_mm)
    p.update(kw)
    return oracle.Bound(geom, field, p)


@pytest.mark.parametrize("cfg_id,fieldname", [(1, "uniform"), (3, "table"), (2, "uniform")])
def test_tiny_tolerance_is_the_fixed_step_scan(geom, uniform_field, table_field, cfg_id, fieldname):
    """tol -> 0 keeps every step at level 0: the results must be those of the fixed-step evaluation (exhaustive mode),
    bit for bit -- n_match, chi2, step / turn / in-gas counts, final state and every approach record."""
    field = uniform_field if fieldname == "uniform" else table_field
    cfg = synth.CONFIGS[cfg_id]
    ev = synth.generate_events(cfg, geom, field, 1)[0]
    b = _bound(geom, field, cfg)
    rng = np.random.default_rng(cfg_id)
    for trial in range(3):
        seed = ev.seed + (0.0 if trial == 0 else 1.0) * rng.uniform(-1, 1, 5) * synth.HALF_WIDTH
        fx = oracle.eval_seed(b, ev.wire_id, ev.drift_mm, seed, mode=0, records=True, rec_slack=0.5)
        ad = oracle.eval_seed_adaptive(b, ev.wire_id, ev.drift_mm, seed, 1e-13, 16.0, records=True, rec_slack=0.5)
        assert ad["n_level"][0] == ad["n_steps"] == ad["units"] == fx["n_steps"] and ad["n_level"][1:].sum() == 0
        assert ad["n_match"] == fx["n_match"] and ad["chi2"] == fx["chi2"] and ad["turns"] == fx["turns"]
        assert ad["m_gas"] == fx["m_gas"] and ad["p"] == fx["p"]
        assert np.array_equal(ad["r"], fx["r"]) and np.array_equal(ad["T"], fx["T"])
        assert np.array_equal(ad["rec"], fx["rec"])


def test_level_sequence_follows_the_closed_form_of_the_estimate(geom, uniform_field):
    """Uniform field: k1 - k2 - k3 + k4 = -(c^3 H^2 / 4) J T + (c^4 H^3 / 4) T with c = a B_z (pinned for orc_rkn_step_err
    in test_peel.py), so err(H) = H^2 |c|^3 (H^2 / 4) |T_perp| sqrt(1 + (c H)^2) is known for every level H = h 2^j.  The
    controller must climb one level per accepted step while err <= tol / 32 and settle on the highest level whose
    estimate it has seen <= tol / 32 one level below -- computed here from the closed form alone."""
    cfg = synth.CONFIGS[1]
    b = _bound(geom, uniform_field, cfg, max_steps=2000)
    pt, p = 100.0, 104.97
    pz = math.sqrt(p * p - pt * pt)
    seed = np.array([0.4, -700.0, pt * math.cos(1.0), pt * math.sin(1.0), pz])
    c = KAPPA / p
    tperp = pt / p

    def est(H):
        return H ** 2 * c ** 3 * H ** 2 / 4.0 * tperp * math.sqrt(1.0 + (c * H) ** 2)

    hit_w = np.array([5], dtype=np.int32); drift = np.array([1.0], dtype=np.float32)
    for tol, h_max in ((1e-5, 16.0), (1e-4, 16.0), (3e-3, 16.0), (3e-3, 4.0), (1.0, 8.0)):
        J = int(math.floor(math.log2(h_max / cfg.h_mm) + 1e-9))
        j, seq = 0, []
        for _ in range(12):                         # replay the controller on the closed-form estimate
            while est(cfg.h_mm * 2 ** j) > tol and j > 0:
                j -= 1
            seq.append(j)
            if j < J and est(cfg.h_mm * 2 ** j) <= tol / 32.0:
                j += 1
        steady = seq[-1]
        ad = oracle.eval_seed_adaptive(b, hit_w, drift, seed, tol, h_max)
        want_climb = [seq.count(k) for k in range(steady)]              # steps spent on each level while climbing
        # (+ at most one step per lower level at the very end, where the path cap drops the level until the step fits)
        assert all(0 <= int(ad["n_level"][k]) - want_climb[k] <= 1 for k in range(steady)), (tol, h_max, ad["n_level"], seq)
        assert ad["n_level"][steady] > 50 and ad["n_level"][steady + 1:].sum() == 0
        assert ad["units"] == int((ad["n_level"] * 2 ** np.arange(8)).sum())


def test_adaptive_track_stays_on_the_helix(geom, uniform_field):
    """The adaptive track in a uniform field against the analytic helix at its own path length: the global error is at
    most a few times (number of steps) x tol / 16 (the estimate is ~ 16 x the true local error of the 4th-order step)
    and, separately, within the fixed-step bound scaled by 16^level."""
    cfg = synth.CONFIGS[1]
    b = _bound(geom, uniform_field, cfg, max_steps=3000)
    p = np.array([60.0, -55.0, 65.6]); p *= 104.97 / np.linalg.norm(p)
    seed = np.array([0.3, -120.0, p[0], p[1], p[2]])
    a = -KAPPA / 104.97
    r0 = np.array([500.0 * math.cos(0.3), 500.0 * math.sin(0.3), -120.0]); T0 = p / 104.97
    hit_w = np.array([5], dtype=np.int32); drift = np.array([1.0], dtype=np.float32)
    for tol in (1e-6, 1e-5, 1e-4):
        ad = oracle.eval_seed_adaptive(b, hit_w, drift, seed, tol, 16.0)
        s = cfg.h_mm * ad["units"]
        cs, sn = math.cos(a * s), math.sin(a * s)
        re = np.array([r0[0] + (T0[0] * sn + T0[1] * (1 - cs)) / a, r0[1] + (T0[1] * sn - T0[0] * (1 - cs)) / a, r0[2] + T0[2] * s])
        err = float(np.linalg.norm(ad["r"] - re))
        assert err < ad["n_steps"] * tol / 4.0, (tol, err)
        assert ad["n_steps"] < ad["units"] or tol < 2e-6           # it does take longer steps


def test_path_cap_in_gas_units_and_momentum(geom, uniform_field):
    """max_steps caps the PATH (units of h): a track that stays in the chamber ends on exactly max_steps units, dropping
    levels at the end; the in-gas count sums the units of the steps that start at rho >= R0 and p = p0 - eps h m."""
    cfg = synth.CONFIGS[2]
    ev = synth.generate_events(cfg, geom, uniform_field, 1)[0]
    for cap in (37, 1000, 1003):
        b = _bound(geom, uniform_field, cfg, max_steps=cap)
        ad = oracle.eval_seed_adaptive(b, ev.wire_id, ev.drift_mm, ev.seed, 1e-4, 16.0)
        assert ad["units"] == cap == int((ad["n_level"] * 2 ** np.arange(8)).sum())
        p0 = math.sqrt(float((ev.seed[2:] ** 2).sum()))
        assert ad["p"] == p0 - (cfg.eloss_MeV_per_mm * cfg.h_mm) * ad["m_gas"] and 0 < ad["m_gas"] <= cap


def test_adaptive_scan_finds_the_same_hits(geom, table_field):
    """With tol = 1e-5 mm (4 mm steps in this field) a configs[3] truth seed matches the same hits as the fixed 2 mm
    step: the chord's sagitta h^2 / 8R grows to 6e-3 mm, far inside the 1 mm window; chi2 moves by < 0.1."""
    cfg = synth.CONFIGS[3]
    evs = synth.generate_events(cfg, geom, table_field, 4)
    b = _bound(geom, table_field, cfg)
    for ev in evs:
        fx = oracle.eval_seed(b, ev.wire_id, ev.drift_mm, ev.seed, mode=0)
        ad = oracle.eval_seed_adaptive(b, ev.wire_id, ev.drift_mm, ev.seed, 1e-5, 8.0)
        assert ad["n_steps"] < 0.6 * fx["n_steps"] and abs(ad["units"] - fx["n_steps"]) <= 2
        assert abs(ad["n_match"] - fx["n_match"]) <= 1 and abs(ad["chi2"] - fx["chi2"]) < 0.1
        assert np.linalg.norm(ad["r"] - fx["r"]) < 2.0 * cfg.h_mm + 1e-3      # ends within one long step of it


def test_diagnostic_margins_against_independent_values(geom, uniform_field, table_field):
    """The decision and boundary margins the adaptive evaluation returns are what the parity protocol's exception classes
    rest on (tests/parity_util.compare_scan_adaptive), so they are pinned against values formed without them:
    (i) uniform field, tol -> 0 (every trial at level 0; the estimate at a vertex is h^2 times the maximum component of the
        closed form -(c^3 h^2 / 4) J T + (c^4 h^3 / 4) T of the test above): margin_tol = min |est - tol| / tol, margin_up =
        min |est - tol/32| / (tol/32), and the same two distances over h^2;
    (ii) tabulated field: the track is re-traced here vertex by vertex with the one-step routine (pinned elsewhere) and
        r0_margin = min_n>=1 | rho_n - R0 |, exit_margin = min_n>=1 min(| |z_n| - z_half |, | rho_n - r_out |)."""
    cfg = synth.CONFIGS[1]
    b = _bound(geom, uniform_field, cfg, max_steps=400)
    pt, p = 90.0, 104.97
    seed = np.array([0.4, -100.0, pt * math.cos(1.0), pt * math.sin(1.0), math.sqrt(p * p - pt * pt)])
    h, tol = cfg.h_mm, 1e-13
    w = np.array([5], dtype=np.int32); d = np.array([1.0], dtype=np.float32)
    r = oracle.eval_seed_adaptive(b, w, d, seed, tol, 16.0)
    assert r["n_level"][0] == r["n_steps"] > 100
    # the estimate at every vertex from the closed form (maximum norm, as the controller takes it), T_n from the one-step routine
    c = -KAPPA / p                                   # a B_z, electron
    pos = np.array([geom.R0_mm * math.cos(seed[0]), geom.R0_mm * math.sin(seed[0]), seed[1]]); T = seed[2:5] / p
    est = []
    for n in range(r["n_steps"]):
        vx = -(c ** 3 * h ** 2 / 4.0) * T[1] + (c ** 4 * h ** 3 / 4.0) * T[0]
        vy = (c ** 3 * h ** 2 / 4.0) * T[0] + (c ** 4 * h ** 3 / 4.0) * T[1]
        est.append(h ** 2 * max(abs(vx), abs(vy)))
        pos, T = oracle.rkn_step(b, c, h, pos, T)
    est = np.array(est)
    assert r["margin_tol"] == pytest.approx(np.min(np.abs(est - tol)) / tol, rel=1e-5)
    assert r["margin_up"] == pytest.approx(np.min(np.abs(est - tol / 32)) / (tol / 32), rel=1e-5)
    assert r["kmargin_tol"] == pytest.approx(np.min(np.abs(est - tol)) / h ** 2, rel=1e-5)
    assert r["kmargin_up"] == pytest.approx(np.min(np.abs(est - tol / 32)) / h ** 2, rel=1e-5)
    # (ii)
    cfg3 = synth.CONFIGS[3]
    ev = synth.generate_events(cfg3, geom, table_field, 1)[0]
    b3 = _bound(geom, table_field, cfg3)
    r3 = oracle.eval_seed_adaptive(b3, ev.wire_id, ev.drift_mm, ev.seed, 1e-13, 16.0)
    th, z0, px, py, pz = ev.seed
    p0 = math.sqrt(px * px + py * py + pz * pz)
    pos = np.array([geom.R0_mm * math.cos(th), geom.R0_mm * math.sin(th), z0]); T = np.array([px, py, pz]) / p0
    a = -KAPPA / p0
    r0m = exm = float("inf")
    for n in range(r3["n_steps"]):
        pos, T = oracle.rkn_step(b3, a, cfg3.h_mm, pos, T)
        rho = math.sqrt(pos[0] * pos[0] + pos[1] * pos[1])
        r0m = min(r0m, abs(rho - geom.R0_mm))
        exm = min(exm, abs(abs(pos[2]) - geom.z_half_mm), abs(rho - geom.r_out_mm))
    assert np.array_equal(pos, r3["r"])                                  # the same track
    assert r3["r0_margin"] == pytest.approx(r0m, rel=1e-12, abs=1e-12)
    assert r3["exit_margin"] == pytest.approx(exm, rel=1e-12, abs=1e-12)
    assert 0.0 < r3["exit_margin"] < cfg3.h_mm and r3["r0_margin"] < cfg3.h_mm     # a vertex near the exit / near R0 exists
