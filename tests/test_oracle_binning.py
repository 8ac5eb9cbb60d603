"""Pins for the oracle's projection and binning (-m "not gpu")."""
import math

import numpy as np
import pytest

from paper_2607_00117_b200 import inputs


def rot_z(t):
    c, s = math.cos(t), math.sin(t)
    return np.array([[c, -s, 0], [s, c, 0], [0, 0, 1.0]])


def rot_x(t):
    c, s = math.cos(t), math.sin(t)
    return np.array([[1.0, 0, 0], [0, c, -s], [0, s, c]])


def euler(alpha, beta, gamma):
    """PAPER.md:98 Eq.1: R = Rz(gamma) Rx(beta) Rz(alpha), active right-handed."""
    return rot_z(gamma) @ rot_x(beta) @ rot_z(alpha)


def test_projection_matches_matrix_product_and_is_a_rotation(smo):
    rng = np.random.default_rng(3)
    for _ in range(5):
        ang = tuple(rng.uniform(-math.pi, math.pi, 3))
        R = euler(*ang)
        rows = np.array([[smo.project(ang, e, e)[i] for e in np.eye(3)] for i in range(3)])
        # rows: X-row, Y-row (from positions) and the z'-row (from velocities)
        assert rows == pytest.approx(R, abs=1e-15)
        assert rows @ rows.T == pytest.approx(np.eye(3), abs=1e-15)
        assert np.linalg.det(rows) == pytest.approx(1.0, abs=1e-15)
    # beta = 0: (X,Y) = Rz(alpha+gamma)(x,y), v_los = v_z
    x, v = np.array([1.0, 2.0, 3.0]), np.array([4.0, 5.0, 6.0])
    out = smo.project((0.3, 0.0, 0.4), x, v)
    assert out[:2] == pytest.approx((rot_z(0.7) @ x)[:2], abs=1e-15)
    assert out[2] == 6.0
    # beta = 90 deg, alpha = gamma = 0: edge-on, line of sight along -y: v_los = +v_y? (Rx(90): z' = y)
    out = smo.project((0.0, math.pi / 2, 0.0), x, v)
    assert out == pytest.approx([1.0, -3.0, 5.0], abs=1e-15)


@pytest.fixture(scope="module")
def lib0(smo):
    cfg = inputs.CONFIGS[0]
    ics = inputs.plummer_ics(120, cfg["seed"])
    out = smo.build_library(cfg["potential"], ics, cfg["dt"], cfg["n_steps"], cfg["stride"], cfg["projections"],
                            cfg["grids"], want_diag=True)
    return cfg, ics, out


def test_row_sums_plus_nout_equal_nrec(lib0):
    cfg, ics, out = lib0
    n_rec = cfg["n_steps"] // cfg["stride"]
    assert np.array_equal(out["losvd"][0].sum(1) + out["nout"][0], np.full(len(ics), n_rec))
    assert np.array_equal(out["dens"].sum(1) + out["nout"][1], np.full(len(ics), n_rec))
    assert out["nout"].sum() > 0            # some samples do leave the grid (reading R6)
    assert out["diag"][:, 0].max() < 2e-3   # static potential: E_J = E, conserved O(dt^2)


def _rebin(cfg, pot_omega, traj, stride):
    """Brute-force re-binning of a dumped trajectory with numpy.histogramdd."""
    g = cfg["grids"]
    n_rec, n = traj.shape[:2]
    t = (np.arange(n_rec) + 1) * stride * cfg["dt"]
    th = pot_omega * t
    c, s = np.cos(th)[:, None], np.sin(th)[:, None]
    xb = np.stack([c * traj[..., 0] + s * traj[..., 1], -s * traj[..., 0] + c * traj[..., 1], traj[..., 2]], -1)
    vb = np.stack([c * traj[..., 3] + s * traj[..., 4], -s * traj[..., 3] + c * traj[..., 4], traj[..., 5]], -1)
    losvd, dens = [], []
    for i in range(n):
        d, _ = np.histogramdd(xb[:, i, ::-1], bins=(g["dz"], g["dy"], g["dx"]),
                              range=((g["bz0"], g["bz1"]), (g["by0"], g["by1"]), (g["bx0"], g["bx1"])))
        dens.append(d.ravel())
        rows = []
        for ang in cfg["projections"]:
            R = euler(*ang)
            xp = xb[:, i] @ R.T
            vp = vb[:, i] @ R.T
            h, _ = np.histogramdd(np.stack([xp[:, 1], xp[:, 0], vp[:, 2]], 1), bins=(g["ny"], g["nx"], g["nv"]),
                                  range=((g["y0"], g["y1"]), (g["x0"], g["x1"]), (g["v0"], g["v1"])))
            rows.append(h.ravel())
        losvd.append(rows)
    return np.array(losvd).transpose(1, 0, 2), np.array(dens)


def test_bruteforce_rebinning_config0(smo, lib0):
    cfg, ics, out = lib0
    traj = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], cfg["n_steps"], cfg["stride"])
    losvd, dens = _rebin(cfg, 0.0, traj, cfg["stride"])
    clean = out["near_edge"].sum(0) == 0
    assert clean.sum() > 100
    assert np.array_equal(out["losvd"][:, clean], losvd[:, clean])
    assert np.array_equal(out["dens"][clean], dens[clean])


def test_bruteforce_rebinning_barred_three_projections(smo, oracle_force):
    """Config-4-like geometry (3 inclinations) on the rotating potential, short run."""
    cfg = dict(inputs.CONFIGS[4])
    cfg["grids"] = inputs.CONFIGS[1]["grids"]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=16)
    n_steps, stride = 400, 4
    out = smo.build_library(cfg["potential"], ics, cfg["dt"], n_steps, stride, cfg["projections"], cfg["grids"], want_diag=True)
    traj = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], n_steps, stride)
    losvd, dens = _rebin(cfg, cfg["potential"]["omega_p"], traj, stride)
    clean = out["near_edge"].sum(0) == 0
    assert clean.sum() >= 12
    assert np.array_equal(out["losvd"][:, clean], losvd[:, clean])
    assert np.array_equal(out["dens"][clean], dens[clean])
    n_rec = n_steps // stride
    for p in range(3):
        assert np.array_equal(out["losvd"][p].sum(1) + out["nout"][p], np.full(16, n_rec))
    # v-marginal of the LOSVD block is the orbit's surface-density image
    g = cfg["grids"]
    img = out["losvd"][1].reshape(16, g["ny"], g["nx"], g["nv"]).sum(-1)
    R = euler(*cfg["projections"][1])
    th = cfg["potential"]["omega_p"] * (np.arange(n_rec) + 1) * stride * cfg["dt"]
    for i in np.flatnonzero(clean)[:4]:
        c, s = np.cos(th), np.sin(th)
        xb = np.stack([c * traj[:, i, 0] + s * traj[:, i, 1], -s * traj[:, i, 0] + c * traj[:, i, 1], traj[:, i, 2]], 1)
        vb = np.stack([c * traj[:, i, 3] + s * traj[:, i, 4], -s * traj[:, i, 3] + c * traj[:, i, 4], traj[:, i, 5]], 1)
        xp, vp = xb @ R.T, vb @ R.T
        ok = (vp[:, 2] >= g["v0"]) & (vp[:, 2] < g["v1"])
        h, _, _ = np.histogram2d(xp[ok, 1], xp[ok, 0], bins=(g["ny"], g["nx"]), range=((g["y0"], g["y1"]), (g["x0"], g["x1"])))
        assert np.array_equal(img[i], h)


def test_stride_not_dividing_nsteps_and_invalid_args(smo):
    cfg = inputs.CONFIGS[0]
    ics = inputs.plummer_ics(4, 1)
    out = smo.build_library(cfg["potential"], ics, 0.01, 103, 10, cfg["projections"], cfg["grids"])
    assert np.array_equal(out["dens"].sum(1) + out["nout"][1], np.full(4, 10))
    with pytest.raises(ValueError):
        smo.build_library(cfg["potential"], ics, -0.01, 100, 10, cfg["projections"], cfg["grids"])
    with pytest.raises(ValueError):
        smo.build_library(cfg["potential"], ics, 0.01, 100, 0, cfg["projections"], cfg["grids"])
    bad = {"G": 1.0, "omega_p": 0.0, "components": [(inputs.FERRERS2, 1, [1.0, 1.0, 2.0, 0.5])]}
    with pytest.raises(ValueError):
        smo.eval_force(bad, [[1, 2, 3]])
