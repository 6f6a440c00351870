"""Seeded synthetic inputs for the CDC seed scan: detector description, field
tables, Monte-Carlo-style events and seed grids.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA
path.  It holds none of the method's arithmetic: no Nystroem stepping, no
sign-change approach rule, no Eq. (1) score, no Hough vote.  Tracks are made by
an independent "truth" simulation (classical RK4 on the first-order Lorentz
system at a 1 mm sampling step, closest approach by Newton iteration on the
local osculating parabola), the way a detector Monte Carlo stands upstream of
a reconstruction program.

Recipe and citations:
  * geometry  - BASELINE.json configs[0]: 18 sense layers, r_i = 530 + 16.5 i mm,
                n_i = round(2 pi r_i / 16.8), wires |z| <= 750 mm, stereo
                +-70 mrad alternating ("eighteen layers with
                stereo configuration").
  * field     - 1 T solenoid; configs[3]: Bz = 1 - 0.05 (z/1 m)^2,
                Br from div B = 0, tabulated on a 10 mm (r, z) grid.
  * events    - |p| = 104.97 MeV/c electrons, start on a 100 mm
                disk, z in [-400, 400] mm; hits = DOCA + N(0, 0.2 mm) kept if
                < 8 mm; uniform noise occupancy.
  * seed grid - 5 axes (theta, z, px, py, pz) at R0 = 500 mm.

Units: mm, MeV/c, tesla, radians.  All draws come from numpy Philox streams
keyed by (base seed + 1000 * config + event index, purpose).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

KAPPA = 0.299792458          # curvature [1/mm] = KAPPA * q * B[T] / p[MeV/c]
P_SIGNAL = 104.97            # MeV/c
BASE_SEED = 19080194900
N_AXES = 5                   # theta, z, px, py, pz


# --------------------------------------------------------------------------
# detector description
# --------------------------------------------------------------------------
@dataclasses.dataclass
class Geometry:
    """Per-layer description plus the canonical fp32 per-wire table.

    wire[w] = (w0x, w0y, ux, uy, uz): the wire is the line w0 + t*u, w0 at z=0,
    u a unit vector (to fp32 rounding), restricted to |z| <= z_half.
    """
    r_mm: np.ndarray          # (L,) f64  waist radius (radius at z = 0)
    n_wires: np.ndarray       # (L,) i32
    phi0_rad: np.ndarray      # (L,) f64  azimuth of wire 0 at z = 0
    stereo_rad: np.ndarray    # (L,) f64  signed stereo angle
    wire: np.ndarray          # (W, 5) f32
    offset: np.ndarray        # (L+1,) i32 prefix sum of n_wires
    z_half_mm: float = 750.0
    R0_mm: float = 500.0
    r_out_mm: float = 827.0

    @property
    def n_layers(self) -> int:
        return int(self.r_mm.shape[0])

    @property
    def n_wires_total(self) -> int:
        return int(self.offset[-1])


def make_geometry(n_layers: int = 18, r_first: float = 530.0, dr: float = 16.5,
                  cell: float = 16.8, stereo: float = 0.070,
                  phi0: Optional[Sequence[float]] = None,
                  z_half: float = 750.0, R0: float = 500.0,
                  r_out: Optional[float] = None) -> Geometry:
    j = np.arange(n_layers)
    r = r_first + dr * j.astype(np.float64)
    n = np.rint(2.0 * math.pi * r / cell).astype(np.int32)
    eps = np.where(j % 2 == 0, stereo, -stereo).astype(np.float64)
    ph0 = np.zeros(n_layers) if phi0 is None else np.asarray(phi0, dtype=np.float64)
    off = np.zeros(n_layers + 1, dtype=np.int32)
    off[1:] = np.cumsum(n)
    wire = np.empty((int(off[-1]), 5), dtype=np.float64)
    for jj in range(n_layers):
        k = np.arange(int(n[jj]), dtype=np.float64)
        phi = ph0[jj] + 2.0 * math.pi * k / float(n[jj])
        s, c = np.sin(phi), np.cos(phi)
        sl = slice(int(off[jj]), int(off[jj + 1]))
        wire[sl, 0] = r[jj] * c
        wire[sl, 1] = r[jj] * s
        wire[sl, 2] = -math.sin(eps[jj]) * s
        wire[sl, 3] = math.sin(eps[jj]) * c
        wire[sl, 4] = math.cos(eps[jj])
    if r_out is None:
        r_out = float(r[-1] + dr)
    return Geometry(r_mm=r, n_wires=n, phi0_rad=ph0, stereo_rad=eps,
                    wire=wire.astype(np.float32), offset=off,
                    z_half_mm=z_half, R0_mm=R0, r_out_mm=r_out)


# --------------------------------------------------------------------------
# magnetic field
# --------------------------------------------------------------------------
@dataclasses.dataclass
class Field:
    """kind 0: uniform (0, 0, bz_T).  kind 1: (r, z) table, layout [iz][ir][2]
    = (B_r, B_z) fp32, nodes r = r0 + ir*dr, z = z0 + iz*dz, bilinear."""
    kind: int
    bz_T: float = 1.0
    nr: int = 0
    nz: int = 0
    r0_mm: float = 0.0
    z0_mm: float = 0.0
    dr_mm: float = 10.0
    dz_mm: float = 10.0
    table: Optional[np.ndarray] = None      # (nz, nr, 2) f32
    # closed form the table was sampled from (used by the truth simulation)
    quad_coeff: float = 0.0                 # Bz = bz_T * (1 - quad_coeff * (z/1000)^2)


def make_uniform_field(bz: float = 1.0) -> Field:
    return Field(kind=0, bz_T=bz)


def make_table_field(bz: float = 1.0, quad: float = 0.05, r_max: float = 900.0,
                     z_max: float = 1000.0, pitch: float = 10.0) -> Field:
    """configs[3]: Bz = bz (1 - quad (z/1 m)^2); div B = 0 gives
    B_r = bz * quad * (z/1 m) * (r/1 m)."""
    nr = int(round(r_max / pitch)) + 1
    nz = int(round(2.0 * z_max / pitch)) + 1
    rr = pitch * np.arange(nr, dtype=np.float64)
    zz = -z_max + pitch * np.arange(nz, dtype=np.float64)
    tab = np.empty((nz, nr, 2), dtype=np.float64)
    tab[:, :, 0] = bz * quad * (zz[:, None] / 1000.0) * (rr[None, :] / 1000.0)
    tab[:, :, 1] = (bz * (1.0 - quad * (zz / 1000.0) ** 2))[:, None]
    return Field(kind=1, bz_T=bz, nr=nr, nz=nz, r0_mm=0.0, z0_mm=-z_max,
                 dr_mm=pitch, dz_mm=pitch, table=tab.astype(np.float32),
                 quad_coeff=quad)


def _truth_field(field: Field, pos: np.ndarray) -> np.ndarray:
    """Closed-form field at pos (N,3) for the truth simulation (not the
    bilinear table: the Monte Carlo uses the 'real' field)."""
    B = np.zeros_like(pos)
    if field.kind == 0 or field.quad_coeff == 0.0:
        B[:, 2] = field.bz_T
        return B
    c = field.bz_T * field.quad_coeff * 1e-6
    B[:, 0] = c * pos[:, 2] * pos[:, 0]
    B[:, 1] = c * pos[:, 2] * pos[:, 1]
    B[:, 2] = field.bz_T - c * pos[:, 2] ** 2
    return B


# --------------------------------------------------------------------------
# truth simulation (Monte-Carlo stand-in)
# --------------------------------------------------------------------------
def _deriv(field, charge, eloss, R0sq, pos, T, p):
    B = _truth_field(field, pos)
    a = (KAPPA * charge) / p
    dT = a[:, None] * np.cross(T, B)
    gas = (pos[:, 0] ** 2 + pos[:, 1] ** 2) >= R0sq
    dp = np.where(gas, -eloss, 0.0)
    return T, dT, dp


def simulate_tracks(geom: Geometry, field: Field, pos0: np.ndarray, mom0: np.ndarray,
                    path_mm: float, charge: int = -1, eloss: float = 0.0,
                    ds: float = 1.0) -> Dict[str, np.ndarray]:
    """Classical RK4 on (r, T, p) with arc length as the variable, sampled every
    `ds` mm for `path_mm`.  Returns sampled pos (S,N,3), tan (S,N,3), p (S,N)
    and alive (S,N).  A track dies when |z| > z_half, rho > r_out or p <= 1."""
    N = pos0.shape[0]
    S = int(math.ceil(path_mm / ds)) + 1
    pos = np.empty((S, N, 3)); tan = np.empty((S, N, 3)); pp = np.empty((S, N))
    alive = np.zeros((S, N), dtype=bool)
    r = pos0.astype(np.float64).copy()
    p = np.linalg.norm(mom0, axis=1)
    T = mom0 / p[:, None]
    R0sq = geom.R0_mm ** 2
    live = np.ones(N, dtype=bool)
    for i in range(S):
        live = live & (np.abs(r[:, 2]) <= geom.z_half_mm) & \
            ((r[:, 0] ** 2 + r[:, 1] ** 2) <= geom.r_out_mm ** 2) & (p > 1.0)
        pos[i] = r; tan[i] = T; pp[i] = p; alive[i] = live
        if not live.any():
            alive[i + 1:] = False
            pos[i + 1:] = r; tan[i + 1:] = T; pp[i + 1:] = p
            break
        k1r, k1t, k1p = _deriv(field, charge, eloss, R0sq, r, T, p)
        k2r, k2t, k2p = _deriv(field, charge, eloss, R0sq, r + 0.5 * ds * k1r,
                               T + 0.5 * ds * k1t, p + 0.5 * ds * k1p)
        k3r, k3t, k3p = _deriv(field, charge, eloss, R0sq, r + 0.5 * ds * k2r,
                               T + 0.5 * ds * k2t, p + 0.5 * ds * k2p)
        k4r, k4t, k4p = _deriv(field, charge, eloss, R0sq, r + ds * k3r,
                               T + ds * k3t, p + ds * k3p)
        r = r + (ds / 6.0) * (k1r + 2 * k2r + 2 * k3r + k4r)
        T = T + (ds / 6.0) * (k1t + 2 * k2t + 2 * k3t + k4t)
        T = T / np.linalg.norm(T, axis=1)[:, None]
        p = p + (ds / 6.0) * (k1p + 2 * k2p + 2 * k3p + k4p)
    return {"pos": pos, "tan": tan, "p": pp, "alive": alive, "ds": ds}


def _perp(geom_wire: np.ndarray, w: np.ndarray, r: np.ndarray) -> np.ndarray:
    """Offset of points r (M,3) from the lines of wires w (M,), perpendicular part."""
    ww = geom_wire[w].astype(np.float64)
    d = r.copy()
    d[:, 0] -= ww[:, 0]; d[:, 1] -= ww[:, 1]
    u = ww[:, 2:5]
    t = np.einsum("ij,ij->i", d, u)
    return d - t[:, None] * u, u, t


def find_crossings(geom: Geometry, field: Field, sim: Dict[str, np.ndarray],
                   charge: int = -1, d_max: float = 9.0) -> List[np.ndarray]:
    """For every simulated track, every local minimum of the distance to a sense
    wire with DOCA < d_max while in the gas volume (rho >= R0).

    Returns, per track, a structured array sorted by path length with fields
    s (mm from the start), wire, doca, zw, turn."""
    pos, tan, pp, alive, ds = sim["pos"], sim["tan"], sim["p"], sim["alive"], sim["ds"]
    S, N, _ = pos.shape
    rho2 = pos[:, :, 0] ** 2 + pos[:, :, 1] ** 2
    gas = rho2 >= geom.R0_mm ** 2
    # turn index: number of outward crossings of R0 so far, minus one
    outward = np.zeros((S, N), dtype=np.int32)
    outward[1:] = (~gas[:-1]) & gas[1:]
    turn = np.cumsum(outward, axis=0) - 1
    ok = alive[:-1] & alive[1:] & gas[:-1]
    si, ti = np.nonzero(ok)
    x, y, z = pos[si, ti, 0], pos[si, ti, 1], pos[si, ti, 2]
    phi = np.arctan2(y, x)
    rec = []
    for j in range(geom.n_layers):
        te = math.tan(geom.stereo_rad[j])
        uj = np.sqrt(np.maximum(rho2[si, ti] - (z * te) ** 2, 0.0))
        m = np.abs(uj - geom.r_mm[j]) < d_max + 2.0 * ds + 1.0
        if not m.any():
            continue
        s_m, t_m = si[m], ti[m]
        nj = int(geom.n_wires[j])
        kf = (phi[m] - geom.phi0_rad[j] - np.arctan(z[m] * te / geom.r_mm[j])) * nj / (2 * math.pi)
        k0 = np.floor(kf).astype(np.int64)
        for dk in (0, 1):
            w = geom.offset[j] + np.mod(k0 + dk, nj)
            d0, u, _ = _perp(geom.wire, w, pos[s_m, t_m])
            d1, _, _ = _perp(geom.wire, w, pos[s_m + 1, t_m])
            g0 = np.einsum("ij,ij->i", d0, tan[s_m, t_m])
            g1 = np.einsum("ij,ij->i", d1, tan[s_m + 1, t_m])
            c = (g0 <= 0.0) & (g1 > 0.0)
            if not c.any():
                continue
            sc, tc, wc = s_m[c], t_m[c], w[c]
            r0 = pos[sc, tc]; T0 = tan[sc, tc]
            a = (KAPPA * charge) / pp[sc, tc]
            K = a[:, None] * np.cross(T0, _truth_field(field, r0))
            s = ds * g0[c] / (g0[c] - g1[c])
            for _ in range(4):          # Newton on f(s) = delta(s) . r'(s)
                rs = r0 + T0 * s[:, None] + 0.5 * K * (s ** 2)[:, None]
                vs = T0 + K * s[:, None]
                dl, uu, _ = _perp(geom.wire, wc, rs)
                vperp = vs - np.einsum("ij,ij->i", vs, uu)[:, None] * uu
                f = np.einsum("ij,ij->i", dl, vs)
                fp = np.einsum("ij,ij->i", vperp, vperp) + np.einsum("ij,ij->i", dl, K)
                s = s - f / fp
            rs = r0 + T0 * s[:, None] + 0.5 * K * (s ** 2)[:, None]
            dl, uu, tpar = _perp(geom.wire, wc, rs)
            doca = np.linalg.norm(dl, axis=1)
            zw = tpar * uu[:, 2]
            keep = (doca < d_max) & (np.abs(zw) <= geom.z_half_mm)
            rec.append(np.stack([tc[keep].astype(np.float64), (sc[keep] * ds + s[keep]),
                                 wc[keep].astype(np.float64), doca[keep], zw[keep],
                                 turn[sc[keep], tc[keep]].astype(np.float64)], axis=1))
    dt = np.dtype([("s", "f8"), ("wire", "i4"), ("doca", "f8"), ("zw", "f8"), ("turn", "i4")])
    out: List[np.ndarray] = []
    allrec = np.concatenate(rec, axis=0) if rec else np.zeros((0, 6))
    for t in range(N):
        a = allrec[allrec[:, 0] == t]
        a = a[np.argsort(a[:, 1], kind="stable")]
        o = np.empty(a.shape[0], dtype=dt)
        o["s"], o["wire"], o["doca"], o["zw"], o["turn"] = a[:, 1], a[:, 2].astype(np.int32), a[:, 3], a[:, 4], a[:, 5].astype(np.int32)
        out.append(o)
    return out


def truth_seed(geom: Geometry, field: Field, sim: Dict[str, np.ndarray], t: int,
               charge: int = -1, inward: bool = False) -> Optional[Tuple[np.ndarray, float]]:
    """State at the first outward crossing of rho = R0 of track t (the CDC entrance):
    (theta, z, px, py, pz) and the path length at which it happens.  inward=True: the first inward crossing
    after it (the CDC exit of the first turn partition), momentum as the particle has it there."""
    pos, tan, pp, alive, ds = sim["pos"][:, t], sim["tan"][:, t], sim["p"][:, t], sim["alive"][:, t], sim["ds"]
    rho2 = pos[:, 0] ** 2 + pos[:, 1] ** 2
    R0sq = geom.R0_mm ** 2
    idx = np.nonzero((rho2[:-1] < R0sq) & (rho2[1:] >= R0sq) & alive[1:])[0]
    if idx.size == 0:
        return None
    if inward:
        idx = np.nonzero((rho2[:-1] >= R0sq) & (rho2[1:] < R0sq) & alive[1:] & (np.arange(rho2.size - 1) > int(idx[0])))[0]
        if idx.size == 0:
            return None
    i = int(idx[0])
    r0, T0 = pos[i:i + 1], tan[i:i + 1]
    K = ((KAPPA * charge) / pp[i]) * np.cross(T0, _truth_field(field, r0))
    s = ds * (R0sq - rho2[i]) / (rho2[i + 1] - rho2[i])
    for _ in range(6):
        rs = r0 + T0 * s + 0.5 * K * s * s
        vs = T0 + K * s
        f = rs[0, 0] ** 2 + rs[0, 1] ** 2 - R0sq
        fp = 2.0 * (rs[0, 0] * vs[0, 0] + rs[0, 1] * vs[0, 1])
        s = s - f / fp
    rs = (r0 + T0 * s + 0.5 * K * s * s)[0]
    vs = (T0 + K * s)[0]
    vs = vs / np.linalg.norm(vs)
    p = pp[i] + (pp[i + 1] - pp[i]) * (s / ds)
    seed = np.array([math.atan2(rs[1], rs[0]), rs[2], p * vs[0], p * vs[1], p * vs[2]])
    return seed.astype(np.float32).astype(np.float64), i * ds + s


# --------------------------------------------------------------------------
# events
# --------------------------------------------------------------------------
@dataclasses.dataclass
class EventConfig:
    """One of BASELINE.json's configs made concrete."""
    cfg_id: int
    turns: Tuple[int, ...]                  # allowed turn counts
    turn_prob: Tuple[float, ...]            # probabilities of `turns`
    pt_range: Dict[int, Tuple[float, float]]
    noise_occupancy: float
    field_kind: int
    eloss_MeV_per_mm: float
    h_mm: float
    max_steps: int
    grid_n: int
    sigma_drift_mm: float = 0.2
    window_mm: float = 1.0
    drift_max_mm: float = 8.0
    n_events: int = 1
    hough_axes: bool = False                # (theta, px, py) ranges from the Hough vote

    @property
    def path_mm(self) -> float:
        return self.h_mm * self.max_steps


# Replacement p_t ranges for the multi-turn configs: BASELINE.json's ranges cannot
# reach the first sense layer (SURVEY.md 8(d) "config defect"; DESIGN.md readings).
PT_1, PT_2, PT_3 = (75.0, 95.0), (97.0, 103.0), (101.5, 104.5)

CONFIGS: Dict[int, EventConfig] = {
    0: EventConfig(0, (1,), (1.0,), {1: PT_1}, 0.0, 0, 0.0, 2.0, 1500, 8),
    1: EventConfig(1, (2,), (1.0,), {2: PT_2}, 0.10, 0, 0.0, 2.0, 3000, 16),
    2: EventConfig(2, (3,), (1.0,), {3: PT_3}, 0.15, 0, 2.0e-4, 2.0, 4500, 24, hough_axes=True),
    3: EventConfig(3, (1, 2, 3), (2.0 / 3.0, 1.0 / 6.0, 1.0 / 6.0), {1: PT_1, 2: PT_2, 3: PT_3},
                   0.20, 1, 0.0, 2.0, 4500, 16, n_events=256),
    4: EventConfig(4, (1, 2, 3), (2.0 / 3.0, 1.0 / 6.0, 1.0 / 6.0), {1: PT_1, 2: PT_2, 3: PT_3},
                   0.20, 1, 0.0, 2.0, 4500, 16, n_events=16),
}


@dataclasses.dataclass
class Event:
    wire_id: np.ndarray       # (H,) i32, ascending
    drift_mm: np.ndarray      # (H,) f32
    truth_turn: np.ndarray    # (H,) i32, -1 for noise
    seed: np.ndarray          # (5,) f64, fp32-representable truth seed at R0
    n_turns: int
    n_signal: int
    seed_exit: Optional[np.ndarray] = None   # (5,) f64: exit of the first turn partition with the momentum REVERSED
                                             # (a backward scan starts here with the opposite charge), or None


def _stream(seed: int, purpose: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[np.uint64(seed), np.uint64(purpose)]))


def _box_muller(u1: np.ndarray, u2: np.ndarray) -> np.ndarray:
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)


def generate_events(cfg: EventConfig, geom: Geometry, field: Field, n_events: Optional[int] = None,
                    first_event: int = 0, base_seed: int = BASE_SEED, charge: int = -1,
                    sigma_drift: Optional[float] = None, noise: Optional[float] = None,
                    tries_per_round: int = 12, chunk: int = 384) -> List[Event]:
    """Rejection-sample events: accept a candidate iff exactly its requested
    number of turn partitions have >= 10 wire crossings with DOCA < 8 mm
    (PAPER.md:83 stops below ten hits)."""
    n_events = cfg.n_events if n_events is None else n_events
    sigma = cfg.sigma_drift_mm if sigma_drift is None else sigma_drift
    occ = cfg.noise_occupancy if noise is None else noise
    seeds = [base_seed + 1000 * cfg.cfg_id + first_event + e for e in range(n_events)]
    cand = [_stream(s, 0) for s in seeds]
    want = []
    for e in range(n_events):
        u = cand[e].random()
        acc, k = 0.0, cfg.turns[-1]
        for t, pr in zip(cfg.turns, cfg.turn_prob):
            acc += pr
            if u < acc:
                k = t
                break
        want.append(k)
    done: List[Optional[Event]] = [None] * n_events
    pending = list(range(n_events))
    rounds = 0
    while pending:
        rounds += 1
        if rounds > 40:
            raise RuntimeError("event generation did not converge")
        U = np.stack([cand[e].random((tries_per_round, 6)) for e in pending])    # (P, tries, 6)
        P = len(pending)
        rr = 100.0 * np.sqrt(U[:, :, 0]); ph = 2 * math.pi * U[:, :, 1]
        z0 = -400.0 + 800.0 * U[:, :, 2]; az = 2 * math.pi * U[:, :, 3]
        lo = np.array([cfg.pt_range[want[e]][0] for e in pending])[:, None]
        hi = np.array([cfg.pt_range[want[e]][1] for e in pending])[:, None]
        pt = lo + (hi - lo) * U[:, :, 4]
        pz = np.where(U[:, :, 5] < 0.5, -1.0, 1.0) * np.sqrt(np.maximum(P_SIGNAL ** 2 - pt ** 2, 0.0))
        pos0 = np.stack([rr * np.cos(ph), rr * np.sin(ph), z0], axis=-1).reshape(-1, 3)
        mom0 = np.stack([pt * np.cos(az), pt * np.sin(az), pz], axis=-1).reshape(-1, 3)
        accepted: Dict[int, Tuple] = {}
        for c0 in range(0, pos0.shape[0], chunk):
            sl = slice(c0, min(c0 + chunk, pos0.shape[0]))
            sim = simulate_tracks(geom, field, pos0[sl], mom0[sl], 900.0 + cfg.path_mm,
                                  charge=charge, eloss=cfg.eloss_MeV_per_mm)
            cross = find_crossings(geom, field, sim, charge=charge)
            for loc in range(sl.stop - sl.start):
                glob = c0 + loc
                pe = glob // tries_per_round
                if pe in accepted:
                    continue
                ts = truth_seed(geom, field, sim, loc, charge=charge)
                if ts is None:
                    continue
                seed, s_seed = ts
                tx = truth_seed(geom, field, sim, loc, charge=charge, inward=True)
                cr = cross[loc]
                cr = cr[(cr["s"] <= s_seed + cfg.path_mm) & (cr["doca"] < cfg.drift_max_mm)]
                _, first = np.unique(cr["wire"], return_index=True)     # one hit per wire, first wins
                tfirst = cr["turn"][first]
                counts = np.bincount(tfirst[tfirst >= 0], minlength=1)
                if int((counts >= 10).sum()) != want[pending[pe]] or \
                        int((counts >= 10).sum()) != int((counts > 0).sum()):
                    continue
                accepted[pe] = (seed, cr, None if tx is None else tx[0])
        still = []
        for pe, e in enumerate(pending):
            if pe not in accepted:
                still.append(e)
                continue
            seed, cr, seed_x = accepted[pe]
            sm = _stream(seeds[e], 1)
            g = _box_muller(sm.random(cr.shape[0]), sm.random(cr.shape[0]))
            drift = np.abs(cr["doca"] + sigma * g)
            keep = drift < cfg.drift_max_mm
            wires, first = np.unique(cr["wire"][keep], return_index=True)   # first in path order wins
            sig_w = cr["wire"][keep][first]
            sig_d = drift[keep][first]
            sig_t = cr["turn"][keep][first]
            nz = _stream(seeds[e], 2)
            fire = nz.random(geom.n_wires_total) < occ
            nd = cfg.drift_max_mm * nz.random(geom.n_wires_total)
            fire[sig_w] = False
            nw = np.nonzero(fire)[0].astype(np.int32)
            w = np.concatenate([sig_w.astype(np.int32), nw])
            d = np.concatenate([sig_d, nd[nw]])
            t = np.concatenate([sig_t.astype(np.int32), -np.ones(nw.size, dtype=np.int32)])
            o = np.argsort(w, kind="stable")
            done[e] = Event(wire_id=w[o].astype(np.int32), drift_mm=d[o].astype(np.float32),
                            truth_turn=t[o].astype(np.int32), seed=seed, n_turns=want[e],
                            n_signal=int(sig_w.size),
                            seed_exit=None if seed_x is None else seed_x * np.array([1.0, 1.0, -1.0, -1.0, -1.0]))
        pending = still
    return done  # type: ignore[return-value]


def _generate_chunk(job):
    cfg_id, first, n, kw = job
    cfg = CONFIGS[cfg_id]
    geom = make_geometry()
    field = make_uniform_field() if cfg.field_kind == 0 else make_table_field()
    return generate_events(cfg, geom, field, n, first_event=first, **kw)


def generate_events_parallel(cfg_id: int, n_events: int, first_event: int = 0, chunk: int = 8, **kw) -> List["Event"]:
    """generate_events() for the default geometry / field of config cfg_id with the event ranges spread over the host
    cores (an event depends on its index only, so the result is the same list)."""
    import multiprocessing as mp
    import os
    jobs = [(cfg_id, first_event + i, min(chunk, n_events - i), kw) for i in range(0, n_events, chunk)]
    if len(jobs) <= 1:
        return _generate_chunk(jobs[0]) if jobs else []
    with mp.get_context("fork").Pool(min(len(jobs), os.cpu_count() or 1)) as pool:
        parts = pool.map(_generate_chunk, jobs)
    return [e for p in parts for e in p]


# --------------------------------------------------------------------------
# seed grids
# --------------------------------------------------------------------------
HALF_WIDTH = np.array([0.05, 37.5, 5.2485, 5.2485, 5.2485])   # "+-5 %" made concrete


@dataclasses.dataclass
class Grid:
    """Axis a has n[a] nodes lo[a] + i * step[a]; axes theta, z, px, py, pz;
    linear seed index = ((((i_theta*n_z + i_z)*n_px + i_px)*n_py + i_py)*n_pz + i_pz)."""
    lo: np.ndarray      # (5,) f64
    step: np.ndarray    # (5,) f64
    n: np.ndarray       # (5,) i32

    @property
    def n_seeds(self) -> int:
        return int(np.prod(self.n.astype(np.int64)))

    def node(self, idx: Sequence[int]) -> np.ndarray:
        return self.lo + np.asarray(idx, dtype=np.float64) * self.step

    def linear(self, idx: Sequence[int]) -> int:
        lin = 0
        for a in range(N_AXES):
            lin = lin * int(self.n[a]) + int(idx[a])
        return lin

    def unravel(self, lin: int) -> Tuple[int, ...]:
        out = []
        for a in reversed(range(N_AXES)):
            out.append(lin % int(self.n[a]))
            lin //= int(self.n[a])
        return tuple(reversed(out))


def truth_anchored_grid(seed: np.ndarray, n, half_width: np.ndarray = HALF_WIDTH) -> Tuple[Grid, Tuple[int, ...]]:
    """Truth is the node i* = floor(n/2) of every axis."""
    n = np.broadcast_to(np.asarray(n, dtype=np.int32), (N_AXES,)).copy()
    step = np.where(n > 1, 2.0 * half_width / np.maximum(n - 1, 1), 0.0)
    anchor = n // 2
    lo = seed - anchor * step
    return Grid(lo=lo.astype(np.float64), step=step.astype(np.float64), n=n), tuple(int(a) for a in anchor)


def ranges_grid(lo: np.ndarray, hi: np.ndarray, n) -> Grid:
    """Grid spanning [lo, hi] on every axis (used with the Hough ranges)."""
    n = np.broadcast_to(np.asarray(n, dtype=np.int32), (N_AXES,)).copy()
    step = np.where(n > 1, (hi - lo) / np.maximum(n - 1, 1), 0.0)
    return Grid(lo=np.asarray(lo, dtype=np.float64), step=step, n=n)


def pack_hits(events: Sequence[Event]) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Concatenate events: (hit_offsets i32 (E+1,), wire_id i32, drift f32)."""
    off = np.zeros(len(events) + 1, dtype=np.int32)
    off[1:] = np.cumsum([e.wire_id.size for e in events])
    return off, np.concatenate([e.wire_id for e in events]).astype(np.int32), \
        np.concatenate([e.drift_mm for e in events]).astype(np.float32)


def stratified_seed_sample(n_seeds: int, n_sample: int, key: int) -> np.ndarray:
    """Sorted, distinct linear seed indices, one per equal stratum (for sampled parity)."""
    n_sample = min(n_sample, n_seeds)
    rng = _stream(key, 3)
    edges = (np.arange(n_sample + 1, dtype=np.float64) * (n_seeds / n_sample)).astype(np.int64)
    width = np.maximum(edges[1:] - edges[:-1], 1)
    return np.minimum(edges[:-1] + (rng.random(n_sample) * width).astype(np.int64), n_seeds - 1)
