"""Turn-partition peeling (full event reconstruction loop) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:83 (section 2.3): "For the neighboring previous turn partition, the track finding and fitting process are
same with that of the last turn partition except the preparation of the longitudinal seed (z0, pz0).  The
longitudinal seeds at the entrance and the exit were predicted by backwardly extrapolating the track that was already
fitted. [...] The whole event reconstruction process stops when the number of remaining unclassified hits becomes
less than ten."  PAPER.md:69: "The hits whose square of DCA is less than the cutoff value were classified as the hits
of the turn partition being investigated."

The Kalman fit is out of scope (GENFIT); reading C18 is the fit-free variant of
SURVEY.md 8(f) #3: the track that is extrapolated to the neighbouring partition is the BEST SEED itself.

  for k = 0, 1, ... (partition k; the neighbour is reached by extrapolating in the scan's own direction: a scan
  with the opposite charge from exit-side seeds, PAPER.md:71 / DESIGN.md section 13, makes this the paper's backward
  extrapolation):
    1. stop (status 1) if fewer than `min_hits` unclassified hits remain (checked before every scan: at the
       start and right after every classification)
    2. exhaustive scan of the partition's seed grid over the unclassified hits, best seed = arg max S   (A3-A8)
    3. the partition's hits = unclassified hits that the best seed's track matches in its FIRST passage
       through the gas (turn label 0 of reading C12)
    4. stop (status 2) if there are fewer than `min_classified` of them (the partition is discarded)
    5. record the partition, mark its hits classified; check 1. again; stop (status 3) if k + 1 == max_partitions
    6. extrapolate the best seed with the same RKN steps (C5-C7) to the next outward crossing of rho = R0 (the
       entrance of the neighbouring partition); stop (status 4) if the track ends first
    7. the neighbour's grid: n nodes per axis centred on the extrapolated (theta, z, px, py, pz), half-widths given

The crossing point of step 6, between the vertices r_n (rho < R0) and r_{n+1} (rho >= R0), d = r_{n+1} - r_n:
    A = dx dx + dy dy,  B = x dx + y dy,  C = x x + y y - R0 R0,  tau = (-B + sqrt(B B - A C)) / A,
    position r_n + tau d,  direction U / |U| with U = T_n + tau (T_{n+1} - T_n),  momentum p_n (no loss below R0),
every expression evaluated left to right in fp64; theta = atan2(y, x) of the position (libm).

Adaptive extrapolation (extrap_tol > 0; reading C19): PAPER.md:55 takes its propagator from ref. [5] (Lund et al.,
PAPER.md:151), whose Runge-Kutta-Nystroem step carries the local error estimate err = h^2 max_i |k1_i - k2_i - k3_i +
k4_i|.  Between two partitions nothing is scored, so step 6 may take longer steps where that estimate allows it:
    the step length starts at h and is always h 2^j, h <= h 2^j <= h_max;
    a trial step with err > tol is repeated with half the length (never below h);
    a trial step that crosses rho = R0 outward with a length above h is repeated with half the length (the crossing
    point is always taken on a chord of length h, as in the fixed-step form);
    after an accepted step with err <= tol / 32 the length doubles if that stays <= h_max (err grows ~16-fold);
    momentum: p = p0 - eloss * (path of the accepted steps that started at rho >= R0), the sum being exact in fp64.
Only accepted steps count against max_steps.  extrap_tol = 0 is the fixed-step form above.
Plain Python loops around the C oracle's single RKN step, exhaustive scan, arg max and labels.
"""
from __future__ import annotations

import math
import types

import numpy as np

from . import Bound, argmax, labels, rkn_step, rkn_step_err, scan_parallel, seed_of_index

KAPPA = 0.299792458          # reading C1 (same constant as cdc_oracle.c)

STATUS = {1: "fewer than min_hits unclassified hits", 2: "partition with fewer than min_classified hits",
          3: "max_partitions reached", 4: "track ended before the next entrance"}


def _crossing(r, T, rn, Tn, p, R0):
    d = [rn[i] - r[i] for i in range(3)]
    A = d[0] * d[0] + d[1] * d[1]
    B = r[0] * d[0] + r[1] * d[1]
    Cc = r[0] * r[0] + r[1] * r[1] - R0 * R0
    tau = (-B + math.sqrt(B * B - A * Cc)) / A
    pos = [r[i] + tau * d[i] for i in range(3)]
    U = [T[i] + tau * (Tn[i] - T[i]) for i in range(3)]
    nU = math.sqrt(U[0] * U[0] + U[1] * U[1] + U[2] * U[2])
    return pos + [p * (U[i] / nU) for i in range(3)]


def next_entrance_adaptive(geom, field, params: dict, seed, max_steps: int, tol: float, h_max: float, trace=None):
    """Step 6 with the step-doubling controller on the error estimate of ref. [5] (module docstring).
    trace (optional list): receives the length of every accepted step."""
    bound = Bound(geom, field, params)
    h0 = float(params["h"]); eloss = float(params.get("eloss", 0.0))
    kq = KAPPA * float(int(params.get("charge", -1)))
    R0 = float(geom.R0_mm); z_half = float(geom.z_half_mm); r_out = float(geom.r_out_mm)
    th, z0, px, py, pz = (float(v) for v in seed)
    r = [R0 * math.cos(th), R0 * math.sin(th), z0]                                   # C4
    p0 = math.sqrt(px * px + py * py + pz * pz)
    T = [px / p0, py / p0, pz / p0]
    p = p0
    n = 0; s_gas = 0.0; hc = h0
    c_n = True
    while n < max_steps:
        a = kq / p
        rn, Tn, err = rkn_step_err(bound, a, hc, r, T)
        rn = [float(v) for v in rn]; Tn = [float(v) for v in Tn]
        if err > tol and hc > h0:
            hc = hc / 2.0
            continue
        c_next = rn[0] * rn[0] + rn[1] * rn[1] >= R0 * R0
        if (not c_n) and c_next and hc > h0:
            hc = hc / 2.0
            continue
        s_next = s_gas + hc if c_n else s_gas                                        # C6
        p_next = p0 - eloss * s_next
        if (not c_n) and c_next:                                                     # C7: a new turn starts here
            return _crossing(r, T, rn, Tn, p_next, R0)
        if trace is not None:
            trace.append(hc)
        r, T = rn, Tn
        n += 1
        p = p_next; s_gas = s_next
        c_n = c_next
        if abs(r[2]) > z_half: break
        if r[0] * r[0] + r[1] * r[1] > r_out * r_out: break
        if not (p > 1.0): break
        if not all(math.isfinite(v) for v in r + T): break
        if err <= tol / 32.0 and hc * 2.0 <= h_max:
            hc = hc * 2.0
    return None


def next_entrance(geom, field, params: dict, seed, max_steps: int, tol: float = 0.0, h_max: float = 0.0):
    """Step 6.  Returns (x, y, z, px, py, pz) at the next outward crossing of rho = R0, or None."""
    if tol > 0.0:
        return next_entrance_adaptive(geom, field, params, seed, max_steps, tol, h_max)
    bound = Bound(geom, field, params)
    h = float(params["h"]); eloss_h = float(params.get("eloss", 0.0)) * h
    kq = KAPPA * float(int(params.get("charge", -1)))
    R0 = float(geom.R0_mm); z_half = float(geom.z_half_mm); r_out = float(geom.r_out_mm)
    th, z0, px, py, pz = (float(v) for v in seed)
    r = [R0 * math.cos(th), R0 * math.sin(th), z0]                                   # C4
    p0 = math.sqrt(px * px + py * py + pz * pz)
    T = [px / p0, py / p0, pz / p0]
    p = p0
    n = 0; m = 0
    c_n = True
    while n < max_steps:
        a = kq / p
        rn, Tn = rkn_step(bound, a, h, r, T)
        rn = [float(v) for v in rn]; Tn = [float(v) for v in Tn]
        if c_n:
            m += 1                                                                   # C6
        p_next = p0 - eloss_h * float(m)
        c_next = rn[0] * rn[0] + rn[1] * rn[1] >= R0 * R0
        if (not c_n) and c_next:                                                     # C7: a new turn starts here
            return _crossing(r, T, rn, Tn, p_next, R0)
        r, T = rn, Tn
        n += 1
        p = p_next
        c_n = c_next
        if abs(r[2]) > z_half: break
        if r[0] * r[0] + r[1] * r[1] > r_out * r_out: break
        if not (p > 1.0): break
        if not all(math.isfinite(v) for v in r + T): break
    return None


def centred_grid(centre, half_width, n):
    """Step 7: node i of axis a = lo[a] + i step[a], lo = c - hw, step = 2 hw / (n - 1); one node: the centre."""
    lo, step = [], []
    for a in range(5):
        if int(n[a]) > 1:
            lo.append(float(centre[a]) - float(half_width[a]))
            step.append(2.0 * float(half_width[a]) / float(int(n[a]) - 1))
        else:
            lo.append(float(centre[a])); step.append(0.0)
    nn = np.asarray(n, dtype=np.int32)
    return types.SimpleNamespace(lo=np.array(lo), step=np.array(step), n=nn, n_seeds=int(np.prod(nn.astype(np.int64))))


def peel(geom, field, params: dict, wire_id, drift, grid0, n, half_width, max_partitions: int = 4,
         min_hits: int = 10, min_classified: int = 5, extrap_max_steps: int = 3000, extrap_tol: float = 0.0,
         extrap_h_max: float = 0.0, n_proc=None):
    """Returns dict(partition (H,) int32: index of the partition a hit was classified into or -1, seeds (P, 5),
    n_match (P,), chi2 (P,), S (P,), status, centres: the extrapolated grid centres (P - 1 or P, 5))."""
    wire_id = np.asarray(wire_id, dtype=np.int32); drift = np.asarray(drift, dtype=np.float32)
    H = int(wire_id.size)
    part = -np.ones(H, dtype=np.int32)
    remaining = np.ones(H, dtype=bool)
    bound = Bound(geom, field, params)
    grid = grid0
    seeds, nms, c2s, Ss, centres = [], [], [], [], []
    status = 3
    if H < min_hits:
        status = 1; max_partitions = 0
    for k in range(max_partitions):
        idx = np.nonzero(remaining)[0]
        w, d = wire_id[idx], drift[idx]
        out = scan_parallel(geom, field, params, w, d, grid, n_proc=n_proc)
        best, S = argmax(out["n_match"], out["chi2"], float(params["window"]))
        seed = seed_of_index(grid, best)
        lab, _ = labels(bound, w, d, seed)
        cls = idx[np.asarray(lab) == 0]
        if cls.size < min_classified:
            status = 2; break
        seeds.append(seed); nms.append(int(out["n_match"][best])); c2s.append(float(out["chi2"][best])); Ss.append(S)
        part[cls] = k
        remaining[cls] = False
        if int(remaining.sum()) < min_hits:
            status = 1; break
        if k + 1 == max_partitions:
            status = 3; break
        nx = next_entrance(geom, field, params, seed, extrap_max_steps, extrap_tol, extrap_h_max)
        if nx is None:
            status = 4; break
        centre = [math.atan2(nx[1], nx[0]), nx[2], nx[3], nx[4], nx[5]]
        centres.append(centre)
        grid = centred_grid(centre, half_width, n)
    return dict(partition=part, seeds=np.array(seeds).reshape(-1, 5), n_match=np.array(nms, dtype=np.int64),
                chi2=np.array(c2s), S=np.array(Ss), status=status, centres=np.array(centres).reshape(-1, 5))
