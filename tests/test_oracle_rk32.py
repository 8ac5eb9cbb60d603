"""Pins of the oracle's adaptive Bogacki-Shampine RK3(2) integrator in the bar's rotating frame (the paper's own
integrator; step control: DESIGN.md reading R23) against what the mathematics
and the paper fix: the analytic Kepler orbit, third-order convergence, the tolerance scaling of an embedded pair of order
3(2), equivalence of the rotating and the inertial frame in an axisymmetric potential, the separately pinned kick-drift-kick
oracle in the barred potential, the paper's printed range of the Jacobi-energy error, and the bookkeeping of the weights."""
import numpy as np
import pytest

from paper_2607_00117_b200 import inputs

KEPLER = {"G": 1.0, "omega_p": 0.0, "phase0": 0.0, "components": [(inputs.PLUMMER, 0, [1.0, 0.0])]}
ECC = 0.5
IC_KEPLER = np.array([[1.0 - ECC, 0.0, 0.0, 0.0, np.sqrt((1 + ECC) / (1 - ECC)), 0.0]])   # pericentre of a = 1, e = 0.5


def kepler_xy(t):
    """Position on the a = 1, e = 0.5 ellipse (G = M = 1) a time t after pericentre: Kepler's equation by Newton."""
    E = np.array(t, dtype=float)
    for _ in range(60):
        E = E - (E - ECC * np.sin(E) - t) / (1 - ECC * np.cos(E))
    return np.cos(E) - ECC, np.sqrt(1 - ECC ** 2) * np.sin(E)


def test_adaptive_kepler_orbit_matches_the_analytic_solution(smo):
    s, w, t_end = smo.integrate_rk32(KEPLER, IC_KEPLER, 6000, rtol=1e-9, atol_x=1e-12, atol_v=1e-12, h0=1e-3)
    t = np.cumsum(w[:, 0])
    assert t_end[0] == pytest.approx(t[-1], rel=1e-14) and t_end[0] > 2 * np.pi      # more than one period
    x, y = kepler_xy(t)
    assert np.max(np.hypot(s[:, 0, 0] - x, s[:, 0, 1] - y)) < 2e-6
    # energy and angular momentum of the samples
    E = 0.5 * (s[:, 0, 3:] ** 2).sum(1) - 1.0 / np.linalg.norm(s[:, 0, :3], axis=1)
    assert np.max(np.abs(E + 0.5)) < 1e-6
    assert np.max(np.abs(s[:, 0, 0] * s[:, 0, 4] - s[:, 0, 1] * s[:, 0, 3] - np.sqrt(1 - ECC ** 2))) < 1e-6
    # the controller takes its smallest steps at pericentre and its largest at apocentre
    acc = w[:, 0] > 0
    r = np.linalg.norm(s[:, 0, :3], axis=1)
    assert np.median(w[acc & (r < 0.6), 0]) < 0.35 * np.median(w[acc & (r > 1.4), 0])


def test_fixed_step_mode_is_third_order(smo):
    errs = []
    for n in (200, 400, 800):
        s, w, t_end = smo.integrate_rk32(KEPLER, IC_KEPLER, n, rtol=0.0, h0=1.0 / n)
        assert np.all(w == 1.0 / n) and t_end[0] == pytest.approx(1.0, rel=1e-12)
        x, y = kepler_xy(1.0)
        errs.append(np.hypot(s[-1, 0, 0] - x, s[-1, 0, 1] - y))
    assert 7.0 < errs[0] / errs[1] < 9.0 and 7.0 < errs[1] / errs[2] < 9.0


def test_tolerance_scaling_of_the_embedded_pair(smo):
    """The error estimate of a 3(2) pair is O(h^3), so the accepted step size scales as tol^(1/3): a tolerance 1000 times
    tighter needs 10 times as many steps for the same time span (a wrong estimator order or controller exponent breaks this)."""
    n_acc = []
    for rtol in (1e-5, 1e-8):
        s, w, t_end = smo.integrate_rk32(KEPLER, IC_KEPLER, 40000, rtol=rtol, atol_x=rtol * 1e-3, atol_v=rtol * 1e-3, h0=1e-4)
        t = np.cumsum(w[:, 0])
        n_acc.append(np.sum((w[:, 0] > 0) & (t <= 2 * np.pi)))
        assert t[-1] > 2 * np.pi
    assert 8.0 < n_acc[1] / n_acc[0] < 12.5


def test_rejected_attempts_have_zero_weight_and_leave_the_state(smo):
    s, w, t_end = smo.integrate_rk32(KEPLER, IC_KEPLER, 300, rtol=1e-6, atol_x=1e-9, atol_v=1e-9, h0=0.5)   # far too large a first step
    assert w[0, 0] == 0.0 and np.array_equal(s[0, 0], IC_KEPLER[0])
    rej = w[:, 0] == 0.0
    assert 1 <= rej.sum() < 60
    k = np.flatnonzero(rej)
    k = k[k > 0]
    assert np.array_equal(s[k, 0], s[k - 1, 0])
    assert t_end[0] == pytest.approx(w[:, 0].sum(), rel=1e-14)
    assert np.all(w[~rej, 0] > 0)
    # growth is capped at 5x and shrinkage at 0.2x per attempt
    acc = w[~rej, 0]
    assert np.all(acc[1:] / acc[:-1] < 5.0 + 1e-9)


@pytest.mark.parametrize("phase0", [0.0, 0.7])
def test_rotating_frame_equals_inertial_frame_in_an_axisymmetric_potential(smo, phase0):
    """With only axisymmetric components the rotating frame is fictitious: the samples of the Omega_p = 40 run, turned back by
    Omega_p t + phase0, must be the samples of the Omega_p = 0 run.  A wrong sign or factor in the Coriolis or centrifugal
    term, or in the velocity transformation, gives an O(1) difference that does not shrink with h; what remains is the
    O(h^3) truncation error of the two runs."""
    comps = [c for c in inputs.CONFIGS[1]["potential"]["components"] if c[0] != inputs.FERRERS2]
    ics = np.array([[3.0, 1.0, 0.2, -20.0, 180.0, 15.0], [0.5, -0.3, 0.1, 60.0, 90.0, -30.0], [9.0, 0.0, -1.0, 10.0, 150.0, 40.0]])
    diffs = []
    vd = []
    for h in (5e-4, 2.5e-4):
        n = int(round(0.3 / h))
        a, wa, _ = smo.integrate_rk32({"G": inputs.G_GALACTIC, "omega_p": 0.0, "phase0": 0.0, "components": comps}, ics, n, rtol=0.0, h0=h)
        b, wb, _ = smo.integrate_rk32({"G": inputs.G_GALACTIC, "omega_p": 40.0, "phase0": phase0, "components": comps}, ics, n, rtol=0.0, h0=h)
        th = 40.0 * np.cumsum(wb, axis=0) + phase0
        c, s_ = np.cos(th), np.sin(th)
        back = b.copy()
        for o in (0, 3):
            back[..., o] = c * b[..., o] - s_ * b[..., o + 1]
            back[..., o + 1] = s_ * b[..., o] + c * b[..., o + 1]
        diffs.append(np.max(np.linalg.norm(back[..., :3] - a[..., :3], axis=-1) / np.linalg.norm(a[..., :3], axis=-1)))
        vd.append(np.max(np.abs(back[..., 3:] - a[..., 3:])))
    # the two runs differ by their own O(h^3) truncation errors only: small, and 8 times smaller at half the step
    assert diffs[1] < 1e-4 and 7.0 < diffs[0] / diffs[1] < 9.0
    assert vd[1] < 1e-2 and 7.0 < vd[0] / vd[1] < 9.0


def test_converges_to_the_kick_drift_kick_oracle_in_the_barred_potential(smo, oracle_force):
    """The bar must sit at the same angle in both integrators: KDK in the inertial frame (pinned in test_oracle_integrator.py)
    against fixed-step RK3 in the rotating frame, config-1 orbits up to t = 0.1, samples compared on bar axes at the same times.
    The difference is the two truncation errors (dominated by RK3's h^3 on the tightest central orbits): it must be small and
    shrink about 8-fold when both steps are halved; a bar at a different angle or a wrong frame term would not converge."""
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=24)
    worst, typical = [], []
    for h in (5e-4, 2.5e-4):
        n = int(round(0.1 / h))
        kdk = smo.integrate_trajectories(cfg["potential"], ics, h / 10, 10 * n, 10)        # inertial, every h
        rk, w, t_end = smo.integrate_rk32(cfg["potential"], ics, n, rtol=0.0, h0=h)
        assert t_end == pytest.approx(np.full(24, 0.1), rel=1e-12)
        th = 40.0 * h * np.arange(1, n + 1)[:, None]
        c, s_ = np.cos(th), np.sin(th)
        xb = c * kdk[..., 0] + s_ * kdk[..., 1]
        yb = -s_ * kdk[..., 0] + c * kdk[..., 1]
        ub = c * kdk[..., 3] + s_ * kdk[..., 4]
        wb = -s_ * kdk[..., 3] + c * kdk[..., 4]
        d = np.sqrt((rk[..., 0] - xb) ** 2 + (rk[..., 1] - yb) ** 2 + (rk[..., 2] - kdk[..., 2]) ** 2) / np.linalg.norm(kdk[..., :3], axis=-1)
        dv = np.sqrt((rk[..., 3] - ub) ** 2 + (rk[..., 4] - wb) ** 2 + (rk[..., 5] - kdk[..., 5]) ** 2) / np.linalg.norm(kdk[..., 3:], axis=-1)
        worst.append(max(d.max(), dv.max()))
        typical.append(np.median(d.max(0)))
    assert worst[1] < 3e-3 and typical[1] < 3e-6
    assert 5.0 < worst[0] / worst[1] < 11.0 and 4.0 < typical[0] / typical[1] < 11.0


def test_jacobi_energy_error_in_the_papers_range(smo, oracle_force):
    """at rtol = 1e-4 'the Jacobi energy of the integrated orbits is typically conserved with a relative error of
    1e-4 - 1e-2' and fewer than 0.1% of the orbits drift by more than 1e-1."""
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=48)
    s, w, t_end = smo.integrate_rk32(cfg["potential"], ics, 5000, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3)
    ej0 = smo.jacobi(cfg["potential"], ics, 0.0)
    drift = np.zeros(48)
    for k in range(99, 5000, 100):
        ej = smo.jacobi(cfg["potential"], s[k], 0.0)     # E_J is invariant under the rotation to bar axes (theta = 0 at t = 0)
        drift = np.maximum(drift, np.abs(ej - ej0) / np.abs(ej0))
    print("RK3(2) rtol 1e-4: Jacobi drift median %.1e max %.1e; t_end median %.2f; rejected %.1f%%"
          % (np.median(drift), drift.max(), np.median(t_end), 100 * np.mean(w == 0)))
    assert 1e-6 < np.median(drift) < 1e-2 and drift.max() < 1e-1
    assert np.all(t_end > 0) and np.mean(w == 0) < 0.3


def test_weighted_rows_sum_to_one_and_match_the_counted_rows_for_equal_steps(smo, oracle_force):
    """weights dt/t_total.  Every row plus the weight outside its grid sums to 1.  With fixed steps all weights are
    equal, so n_steps x the weighted rows must be integer counts -- and the v_los marginal of the LOSVD row must be the orbit's
    surface-density image, i.e. the histogram of the projected positions alone, re-binned here with numpy."""
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=12)
    g = cfg["grids"]
    for rtol in (1e-4, 0.0):
        o = smo.build_library_rk32(cfg["potential"], ics, 600, cfg["projections"], g, rtol=rtol)
        assert o["losvd"][0].sum(1) + o["wout"][0] == pytest.approx(np.ones(12), rel=1e-12)
        assert o["dens"].sum(1) + o["wout"][1] == pytest.approx(np.ones(12), rel=1e-12)
    counts = o["losvd"][0] * 600
    assert np.max(np.abs(counts - np.rint(counts))) < 1e-9
    samples, dtw, _ = smo.integrate_rk32(cfg["potential"], ics, 600, rtol=0.0)
    al, be, ga = cfg["projections"][0]
    for i in range(12):
        xyz = np.array([smo.project((al, be, ga), s[:3], s[3:]) for s in samples[:, i]])
        img, _, _ = np.histogram2d(xyz[:, 1], xyz[:, 0], bins=[g["ny"], g["nx"]], range=[[g["y0"], g["y1"]], [g["x0"], g["x1"]]])
        inside = (xyz[:, 2] >= g["v0"]) & (xyz[:, 2] < g["v1"])
        img_v, _, _ = np.histogram2d(xyz[inside, 1], xyz[inside, 0], bins=[g["ny"], g["nx"]], range=[[g["y0"], g["y1"]], [g["x0"], g["x1"]]])
        marg = counts[i].reshape(g["ny"], g["nx"], g["nv"]).sum(2)
        assert np.array_equal(np.rint(marg), img_v) and np.all(img_v <= img)


def test_a_non_finite_error_estimate_shrinks_the_step_and_the_orbit_recovers(smo):
    """Reading R23: an attempt whose error estimate is NaN (a stage that overflowed) is rejected and the step is multiplied by 0.2
    -- so an absurd first step h0 = 1e300 (y + h k overflows to inf, inf - inf = NaN in the estimate) comes down by a factor 5 per
    attempt until attempts are accepted again.  With the growth factor 5 applied to a NaN estimate, the orbit never took a step."""
    n = 700   # 1e300 * 0.2^n reaches O(1) after ~430 attempts
    s, w, t_end = smo.integrate_rk32(KEPLER, IC_KEPLER, n, rtol=1e-6, atol_x=1e-9, atol_v=1e-9, h0=1e300)
    assert np.all(w[:300, 0] == 0)                        # the overflowing attempts are all rejected, the state stays in place
    assert np.all(s[:300, 0, :3] == [1.0 - ECC, 0.0, 0.0])
    assert t_end[0] > 0.1 and np.isfinite(s).all()        # ... and the orbit then moves along the ellipse
    x, y = kepler_xy(np.cumsum(w[:, 0]))
    assert np.max(np.hypot(s[:, 0, 0] - x, s[:, 0, 1] - y)) < 1e-3
