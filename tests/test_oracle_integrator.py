"""Pins for the oracle's KDK integrator (-m "not gpu"): Kepler closed forms, dt^2 scaling,
conservation laws, the Omega_p -> 0 limit, an independent rotating-frame integration, and the
bar symmetries of PAPER.md:77-90 Table 1."""
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

from paper_2607_00117_b200 import inputs

KEPLER = {"G": 1.0, "omega_p": 0.0, "phase0": 0.0, "components": [(inputs.PLUMMER, 0, [1.0, 0.0])]}
POT1 = inputs.CONFIGS[1]["potential"]


def kepler_ic(a=1.0, e=0.5):
    return np.array([[a * (1 - e), 0, 0, 0, math.sqrt((1 + e) / (a * (1 - e))), 0]])


def test_kepler_period_ellipse_and_second_order(smo):
    """Point mass G=M=1, a=1, e=0.5: period 2 pi sqrt(a^3/GM) = 2 pi; r = a(1-e^2)/(1+e cos f)."""
    ic = kepler_ic()
    errs = []
    for n in (2000, 4000, 8000):
        dt = 2 * math.pi / n
        tr = smo.integrate_trajectories(KEPLER, ic, dt, n, 1)[:, 0]
        errs.append(np.linalg.norm(tr[-1, :3] - ic[0, :3]))  # closed after exactly one period
        x, y = tr[:, 0], tr[:, 1]
        r = np.hypot(x, y)
        f = np.arctan2(y, x)
        ell = np.max(np.abs(r - 0.75 / (1 + 0.5 * np.cos(f))))
        E = 0.5 * (tr[:, 3:] ** 2).sum(1) - 1 / r
        L = x * tr[:, 4] - y * tr[:, 3]
        assert np.max(np.abs(L - L[0])) < 5e-14          # angular momentum: rounding only
        assert np.max(np.abs(E + 0.5)) < 40 * dt * dt     # E = -GM/2a, bounded O(dt^2) error
        assert ell < 30 * dt * dt
        assert np.all(np.abs(tr[:, 2]) == 0)
    assert errs[0] < 1e-3
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.05)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.05)


def test_circular_orbit_axisymmetric(smo):
    """Start on the circular orbit of MN+NFW (v_c^2 = R dPhi/dR, Eq.8, Eq.10): radius stays O(dt^2), L_z to rounding."""
    pot = {"G": POT1["G"], "omega_p": 0.0, "phase0": 0.0, "components": [POT1["components"][0], POT1["components"][2]]}
    R = 8.0
    G = pot["G"]
    vc2 = G * 5e10 * R ** 2 / (R ** 2 + 3.3 ** 2) ** 1.5 + G * 4 * math.pi * 1e7 * 15 ** 3 * (math.log1p(R / 15) - (R / 15) / (1 + R / 15)) / R
    ic = np.array([[R, 0, 0, 0, math.sqrt(vc2), 0]])
    dev = []
    for dt in (2e-3, 1e-3):
        tr = smo.integrate_trajectories(pot, ic, dt, int(0.5 / dt), 1)[:, 0]
        r = np.hypot(tr[:, 0], tr[:, 1])
        dev.append(np.max(np.abs(r - R)))
        Lz = tr[:, 0] * tr[:, 4] - tr[:, 1] * tr[:, 3]
        assert np.max(np.abs(Lz / Lz[0] - 1)) < 1e-14
    assert dev[1] < 3e-4 * R
    assert dev[0] / dev[1] == pytest.approx(4.0, rel=0.1)


def test_config0_energy_and_angular_momentum(smo):
    cfg = inputs.CONFIGS[0]
    ics = inputs.plummer_ics(200, cfg["seed"])
    tr = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], cfg["n_steps"], 10)
    E = lambda s: 0.5 * (s[..., 3:] ** 2).sum(-1) - 1 / np.sqrt(1 + (s[..., :3] ** 2).sum(-1))
    E0 = E(ics)
    dE = np.max(np.abs(E(tr) - E0) / np.abs(E0), axis=0)
    assert np.median(dE) < 5e-5 and dE.max() < 2e-3
    L0 = np.cross(ics[:, :3], ics[:, 3:])
    L = np.cross(tr[..., :3], tr[..., 3:])
    assert np.max(np.abs(L - L0)) < 5e-14 * max(1.0, np.abs(L0).max())


def test_jacobi_drift_and_second_order(smo, oracle_force):
    """Rotating bar: E_J = v^2/2 + Phi - Omega_p L_z (inertial v).  Gate: >=99% of orbits
    <= 1e-2, median <= 2e-4 (paper's own integrator: 1e-4..1e-2); halving dt divides the drift by ~4."""
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=48)
    drifts = []
    for dt, n in ((1e-3, 1500), (5e-4, 3000)):
        tr = smo.integrate_trajectories(cfg["potential"], ics, dt, n, n // 30)
        ej0 = smo.jacobi(cfg["potential"], ics, 0.0)
        d = np.zeros(len(ics))
        for k in range(tr.shape[0]):
            t = (k + 1) * (n // 30) * dt
            d = np.maximum(d, np.abs(smo.jacobi(cfg["potential"], tr[k], t) - ej0) / np.abs(ej0))
        drifts.append(d)
    assert np.median(drifts[0]) < 2e-4
    assert np.mean(drifts[0] <= 1e-2) >= 0.97
    ratio = np.median(drifts[0] / drifts[1])
    assert 3.2 < ratio < 4.8


def test_omega_zero_equals_static_path(smo):
    comp = POT1["components"]
    rot = {"G": POT1["G"], "omega_p": 0.0, "phase0": 0.0, "components": comp}
    sta = {"G": POT1["G"], "omega_p": 0.0, "phase0": 0.0, "components": [(k, 0, p) for k, _, p in comp]}
    ic = np.array([[3.0, 1.0, 0.2, -50.0, 180.0, 10.0], [0.5, -0.2, 0.05, 100.0, 40.0, -30.0]])
    a = smo.integrate_trajectories(rot, ic, 1e-3, 200, 20)
    b = smo.integrate_trajectories(sta, ic, 1e-3, 200, 20)
    assert np.array_equal(a, b)


def test_inertial_kdk_converges_to_rotating_frame_solution(smo):
    """Independent check of the frame handling (north_star: inertial frame, bar angle Omega_p t; PAPER.md:88
    integrates in the co-rotating frame): solve the rotating-frame equations
    x'' = F_bar-frame(x) - 2 Omega x v - Omega x (Omega x x) with DOP853 and map back."""
    Om = POT1["omega_p"]
    frozen = {"G": POT1["G"], "omega_p": 0.0, "phase0": 0.0, "components": POT1["components"]}

    def rhs(_t, s):
        F = smo.eval_force(frozen, [s[:3]], 0.0, want_phi=False)[0]
        x, y, _z, vx, vy, vz = s
        return [vx, vy, vz, F[0] + 2 * Om * vy + Om * Om * x, F[1] - 2 * Om * vx + Om * Om * y, F[2]]

    ic = np.array([2.5, 0.8, 0.15, -60.0, 190.0, 15.0])  # inertial; frames coincide at t=0
    s0 = ic.copy()
    s0[3] += Om * ic[1]   # v_rot = v - Omega x r
    s0[4] -= Om * ic[0]
    T = 0.08
    sol = solve_ivp(rhs, (0, T), s0, method="DOP853", rtol=1e-12, atol=1e-12)
    xr, vr = sol.y[:3, -1], sol.y[3:, -1]
    c, s = math.cos(Om * T), math.sin(Om * T)
    x_in = np.array([c * xr[0] - s * xr[1], s * xr[0] + c * xr[1], xr[2]])
    vr_in = vr + np.array([-Om * xr[1], Om * xr[0], 0.0])
    v_in = np.array([c * vr_in[0] - s * vr_in[1], s * vr_in[0] + c * vr_in[1], vr_in[2]])
    errs = []
    for n in (160, 320, 640):
        tr = smo.integrate_trajectories(POT1, ic[None], T / n, n, n)[0, 0]
        errs.append(np.linalg.norm(tr[:3] - x_in) + np.linalg.norm(tr[3:] - v_in) * 1e-2)
    assert errs[2] < 1e-3  # and Richardson: the O(dt^2) error extrapolates to the DOP853 solution
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.15)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.15)


def test_bar_symmetries_table1(smo):
    """PAPER.md:77-90 Table 1: (x,y,-z,vx,vy,-vz), (-x,-y,z,-vx,-vy,vz), (-x,-y,-z,-vx,-vy,-vz) map orbits to orbits."""
    ic = np.array([[2.0, 1.0, 0.3, -40.0, 170.0, 25.0]])
    base = smo.integrate_trajectories(POT1, ic, 1e-3, 300, 30)
    for sg in ([1, 1, -1, 1, 1, -1], [-1, -1, 1, -1, -1, 1], [-1, -1, -1, -1, -1, -1]):
        sg = np.array(sg, float)
        mir = smo.integrate_trajectories(POT1, ic * sg, 1e-3, 300, 30)
        assert np.array_equal(mir, base * sg)


def test_state_precision_floor(smo, oracle_force):
    """double vs long-double orbit state over 1000 config-1 steps: the chaos floor against which the
    GPU-vs-oracle 1e-10 gate is read."""
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=24)
    a = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], 1000, 100, state_prec=0)
    b = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], 1000, 100, state_prec=1)
    rel = np.max(np.linalg.norm(a[..., :3] - b[..., :3], axis=-1) / np.maximum(np.linalg.norm(b[..., :3], axis=-1), 1e-3), axis=0)
    assert np.median(rel) < 1e-11 and rel.max() < 1e-8


def test_double_force_instantiation_is_the_same_code_in_another_type(smo, oracle_force):
    """oracle/sm_oracle_forces.inc is compiled twice: __float128 (the parity oracle) and plain double (state_prec = 2, used only to
    TIME a CPU baseline without software quad arithmetic).  Same expressions, so the double run follows the quad run to the
    conditioning of the Ferrers recurrences in double (up to ~1e-9 relative for far lambda): trajectories within 1e-7
    over 300 steps of the barred potential, and every row still sums to n_rec."""
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=48)
    a = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], 300, 5, state_prec=0)
    b = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], 300, 5, state_prec=2)
    assert np.max(np.abs(a - b) / np.maximum(np.abs(a), 1e-3)) < 1e-7
    o = smo.build_library(cfg["potential"], ics, cfg["dt"], 300, 5, cfg["projections"], cfg["grids"], state_prec=2)
    assert np.array_equal(o["dens"].sum(1) + o["nout"][-1], np.full(48, 60))
    # the static Plummer sphere has no cancellation: the two agree to rounding
    c0 = inputs.CONFIGS[0]
    ic0 = inputs.plummer_ics(32, 5)
    a0 = smo.integrate_trajectories(c0["potential"], ic0, c0["dt"], 200, 1, state_prec=0)
    b0 = smo.integrate_trajectories(c0["potential"], ic0, c0["dt"], 200, 1, state_prec=2)
    assert np.max(np.abs(a0 - b0)) < 1e-12
