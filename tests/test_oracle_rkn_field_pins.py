"""Pins of the oracle's RKN step where the field DEPENDS ON POSITION.

In a uniform field orc_field_at ignores its argument, so the stage positions of the Nystroem scheme
(r_m = r + (h/2) T + (h^2/8) k1, r_e = r + h T + (h^2/2) k3; reading C5, sec. 2.2 ref. [5]) are dead
code there and the uniform-field pins of test_oracle_pins.py cannot see them.  Each test below fails for the mutation
    cdc_oracle.c  `(h * h / 8.0) * k1[i]` -> `(h * h / 4.0) * k1[i]`   and/or   `(h * h / 2.0) * k3[i]` -> `(h * h) * k3[i]`
(tests/test_oracle_mutations.py builds those mutants and checks that the pins turn red).  The energy-loss pin at the
end fails when a = kappa q / p is formed from p_{n+1} instead of p_n (reading C6).  CPU only.
"""
import math

import numpy as np

import oracle
from paper_1908_01949_b200 import synth

KAPPA = 0.299792458
P = 104.97


def _bound(geom, field, h=2.0, max_steps=10, eloss=0.0):
    return oracle.Bound(geom, field, dict(h=h, max_steps=max_steps, window=1.0, eloss=eloss, charge=-1))


def linear_field(c=2.0 ** -14, b0=1.0, pitch=10.0, r_max=900.0, z_max=1000.0):
    """B_z = b0 + c z, B_r = -c r / 2 (div B = 0), sampled on the cfg3 node lattice.  Every node value is a small
    multiple of 2^-15: exact in fp32, and bilinear interpolation reproduces a field that is linear in r and in z
    exactly -- so the tabulated field is smooth (no kinks at cell borders) and has a closed form."""
    nr = int(round(r_max / pitch)) + 1
    nz = int(round(2.0 * z_max / pitch)) + 1
    rr = pitch * np.arange(nr)
    zz = -z_max + pitch * np.arange(nz)
    tab = np.empty((nz, nr, 2))
    tab[:, :, 0] = (-c * rr / 2.0)[None, :]
    tab[:, :, 1] = (b0 + c * zz)[:, None]
    assert np.array_equal(tab.astype(np.float32).astype(np.float64), tab)
    return synth.Field(kind=1, bz_T=b0, nr=nr, nz=nz, r0_mm=0.0, z0_mm=-z_max, dr_mm=pitch, dz_mm=pitch,
                       table=tab.astype(np.float32))


def _three_turn_start():
    """An in-chamber three-turn track: p_t = 103 MeV/c, z from -600 mm upward (the one VERDICT r1 names)."""
    pt = 103.0
    pz = math.sqrt(P * P - pt * pt)
    r0 = np.array([500.0 * math.cos(0.3), 500.0 * math.sin(0.3), -600.0])
    T0 = np.array([pt * math.cos(0.9) / P, pt * math.sin(0.9) / P, pz / P])
    return r0, T0, -KAPPA / P


def _propagate(b, a, h, r, T, n):
    for _ in range(n):
        r, T = oracle.rkn_step(b, a, h, r, T)
    return r, T


def test_rkn_is_fourth_order_in_a_position_dependent_field(geom):
    """Self-convergence over three turns (6.6 m) in the smooth tabulated field B_z = 1 + c z: the error against
    h = 0.125 mm falls 16-fold per halving of h.  Wrong stage positions (the mutation above) leave a consistent but
    2nd-order scheme: ratio 4."""
    b = _bound(geom, linear_field())
    r0, T0, a = _three_turn_start()
    L = 6600.0
    ref, _ = _propagate(b, a, 0.125, r0, T0, int(L / 0.125))
    assert abs(ref[2]) < 990.0 and math.hypot(ref[0], ref[1]) < 890.0      # stayed inside the table
    err = {}
    for h in (8.0, 4.0, 2.0, 1.0):
        r, _ = _propagate(b, a, h, r0, T0, int(L / h))
        err[h] = float(np.linalg.norm(r - ref))
    for h in (8.0, 4.0, 2.0):
        assert 12.0 < err[h] / err[h / 2.0] < 20.0, err
    assert err[2.0] < 1e-7                                                  # same size as in the uniform field


def test_rkn_agrees_with_an_independent_integrator_in_the_cfg3_table(geom, table_field):
    """scipy's DOP853 (adaptive 8th-order Dormand-Prince on the FIRST-order system r' = T, T' = a T x B) with
    scipy's RegularGridInterpolator for the bilinear table shares neither the scheme nor the field code with the
    oracle.  After three turns in the BASELINE configs[3] field the oracle at h = 2 mm is within 1e-6 mm (its own
    truncation error; the north_star bound in the uniform field); with the stage-position mutation it is 1.7e-3 mm off."""
    from scipy.integrate import solve_ivp
    from scipy.interpolate import RegularGridInterpolator

    f = table_field
    rr = f.r0_mm + f.dr_mm * np.arange(f.nr)
    zz = f.z0_mm + f.dz_mm * np.arange(f.nz)
    iBr = RegularGridInterpolator((zz, rr), f.table[:, :, 0].astype(np.float64), method="linear")
    iBz = RegularGridInterpolator((zz, rr), f.table[:, :, 1].astype(np.float64), method="linear")
    r0, T0, a = _three_turn_start()

    def rhs(s, y):
        rho = math.hypot(y[0], y[1])
        Br = np.asarray(iBr((y[2], rho))).item()
        Bz = np.asarray(iBz((y[2], rho))).item()
        B = np.array([Br * y[0] / rho, Br * y[1] / rho, Bz])
        k = a * np.cross(y[3:], B)
        return [y[3], y[4], y[5], k[0], k[1], k[2]]

    L = 6600.0
    sol = solve_ivp(rhs, (0.0, L), np.concatenate([r0, T0]), method="DOP853", rtol=1e-13, atol=1e-13, max_step=5.0)
    assert sol.success
    b = _bound(geom, f)
    r, T = _propagate(b, a, 2.0, r0, T0, int(L / 2.0))
    assert abs(r[2]) < 750.0                                               # in the chamber to the end
    assert np.linalg.norm(r - sol.y[:3, -1]) < 1e-6
    assert np.linalg.norm(T - sol.y[3:, -1]) < 1e-8


def test_rkn_agrees_with_the_generator_truth_simulation(geom, table_field):
    """synth.simulate_tracks: classical RK4 on the first-order system in the CLOSED-FORM field at ds = 0.25 mm,
    written for the input generator, nothing shared with the oracle.  The table differs from the closed form by the
    interpolation error dB <= 1.25e-6 T of B_z (test_field_table_closed_forms), which bends a track of path L by at
    most |a| dB L^2 / 2; over 1 m that is 1.8e-3 mm.  The oracle at h = 20 mm must be inside that bound (measured
    1.0e-3 mm, of which its own truncation error is 7e-5 mm); with either stage-position mutation the scheme is
    2nd-order and 3.6e-3 mm off."""
    r0, T0, a = _three_turn_start()
    L, h = 1000.0, 20.0
    sim = synth.simulate_tracks(geom, table_field, r0[None, :], (P * T0)[None, :], L, ds=0.25)
    assert sim["alive"][-1, 0]
    b = _bound(geom, table_field)
    r, _ = _propagate(b, a, h, r0, T0, int(L / h))
    bound = abs(a) * 1.25e-6 * L * L / 2.0
    d = float(np.linalg.norm(r - sim["pos"][-1, 0]))
    assert d < bound + 1e-5, (d, bound)
    assert bound < 2e-3


def test_rkn_one_step_taylor_expansion_in_a_linear_field(geom):
    """One step against the Taylor series of the exact solution, derivatives written out by hand for the field
    B = (-c x / 2, -c y / 2, b0 + c z) with constant Jacobian J:  r'' = a T x B,  r''' = a (r'' x B + T x J T),
    r'''' = a (r''' x B + 2 r'' x J T + T x J r'').  A 4th-order Nystroem step reproduces r through h^4 and T through
    h^4 (r' through the h^4 r^(5)/24 term), so the defect is O(h^5) and falls 32-fold per halving.  The mutated
    stage positions put an error a T x J (h^2/8) k1 into k2, k3 and spoil the h^4 term of r: ratio 16."""
    c, b0 = 2.0 ** -10, 1.0
    b = _bound(geom, linear_field(c=c, b0=b0, z_max=400.0))
    a = -KAPPA / 30.0                                                      # a stiff curl makes the terms large
    r = np.array([310.0, -120.0, 55.0])
    T = np.array([0.48, 0.6, 0.64])
    J = np.diag([-c / 2.0, -c / 2.0, c])
    B = np.array([-c * r[0] / 2.0, -c * r[1] / 2.0, b0 + c * r[2]])
    assert np.allclose(oracle.field_at(b, r), B, rtol=0, atol=1e-15)
    d2 = a * np.cross(T, B)
    d3 = a * (np.cross(d2, B) + np.cross(T, J @ T))
    d4 = a * (np.cross(d3, B) + 2.0 * np.cross(d2, J @ T) + np.cross(T, J @ d2))

    def defect(h):
        rn, Tn = oracle.rkn_step(b, a, h, r, T)
        rt = r + h * T + h ** 2 / 2.0 * d2 + h ** 3 / 6.0 * d3 + h ** 4 / 24.0 * d4
        Tt = T + h * d2 + h ** 2 / 2.0 * d3 + h ** 3 / 6.0 * d4
        return float(np.linalg.norm(rn - rt)), float(np.linalg.norm(Tn - Tt))

    e8, t8 = defect(8.0)
    e4, t4 = defect(4.0)
    e2, t2 = defect(2.0)
    assert e2 > 1e-11                                                      # well above fp64 rounding at |r| ~ 300
    assert 26.0 < e8 / e4 < 38.0 and 26.0 < e4 / e2 < 38.0, (e8, e4, e2)   # position defect O(h^5)
    assert 13.0 < t8 / t4 < 19.0 and 13.0 < t4 / t2 < 19.0, (t8, t4, t2)   # direction defect O(h^4) beyond the h^3 term


def test_energy_loss_curvature_uses_p_n(geom, uniform_field):
    """Reading C6: a_n = kappa q / p_n with p_n = p0 - (eps h) m_n, m_n = in-gas steps BEFORE step n.  In a uniform
    field each step is then an exact helix arc of curvature a_n B (to the scheme's 1e-9 mm), so the vertex after N
    in-gas steps has a closed form: the composition of N arcs.  Forming a from p_{n+1} shifts every arc's angle by
    a h (eps h / p): 4e-3 mm after 400 steps."""
    eps, h, N = 2.0e-4, 2.0, 400
    pt = 85.0
    pz = math.sqrt(P * P - pt * pt)
    seed = np.array([0.7, -300.0, pt * math.cos(1.2), pt * math.sin(1.2), pz])     # 584 steps outside R0
    b = oracle.Bound(geom, uniform_field, dict(h=h, max_steps=N, window=1.0, eloss=eps, charge=-1))
    res = oracle.eval_seed(b, np.array([5], np.int32), np.array([1.0], np.float32), seed, trajectory=True)
    traj = res["traj"]
    assert res["n_steps"] == N
    assert np.all(traj[1:, 0] ** 2 + traj[1:, 1] ** 2 > 500.0 ** 2)       # in the gas all the way: m_n = n
    r = np.array([500.0 * math.cos(0.7), 500.0 * math.sin(0.7), -300.0])
    T = seed[2:] / P
    p0 = float(np.linalg.norm(seed[2:]))
    for n in range(N):
        a = -KAPPA / (p0 - (eps * h) * n)
        cs, sn = math.cos(a * h), math.sin(a * h)
        r = np.array([r[0] + (T[0] * sn + T[1] * (1.0 - cs)) / a, r[1] + (T[1] * sn - T[0] * (1.0 - cs)) / a,
                      r[2] + T[2] * h])
        T = np.array([T[0] * cs + T[1] * sn, T[1] * cs - T[0] * sn, T[2]])
    assert np.linalg.norm(traj[N, :3] - r) < 1e-6
    assert res["p"] == p0 - (eps * h) * N
