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
