"""GPU parity (-m gpu) of the paper's own integrator -- adaptive Bogacki-Shampine RK3(2) in the bar's rotating frame with
delta-t sample weights (reading R23) -- through the C ABI
(sm_integrate_rk32, sm_build_library_rk32) against the CPU oracle (pinned in tests/test_oracle_rk32.py).  The accept / reject
decision of a step attempt is a floating-point comparison taken in fp64 by both sides; where rounding flips one, the two step
sequences part ways for good, so the trajectory gate is read, as everywhere in this repo, against the oracle's own sensitivity
to a rounding-level perturbation."""
import numpy as np
import pytest

from paper_2607_00117_b200 import binding, inputs

from gpu_util import traj_rel_err

pytestmark = pytest.mark.gpu

CFG = inputs.CONFIGS[1]
TOL = dict(rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3)


@pytest.fixture(scope="module")
def cuda():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    return torch


def _gate(g, gw, gt, o, ow, ot, sens, name):
    err = traj_rel_err(g, o, 1.0)
    same = np.all((gw > 0) == (ow > 0), axis=0)
    print("%s: %d orbits; identical accept/reject sequence %.3f; err median %.2e max %.2e, frac<=1e-10 %.3f; oracle's own: median %.2e frac %.3f"
          % (name, len(err), same.mean(), np.median(err), err.max(), np.mean(err <= 1e-10), np.median(sens), np.mean(sens <= 1e-10)))
    certified = sens <= 1e-12
    assert certified.mean() >= 0.5
    assert np.all(err[certified] <= 1e-10) and np.all(same[certified])
    assert np.mean(err <= 1e-10) >= np.mean(sens <= 1e-10) - 0.03
    ok = err <= 1e-10
    assert np.max(np.abs(gw[:, ok] - ow[:, ok])) <= 1e-9 * np.max(ow)
    assert gt[ok] == pytest.approx(ot[ok], rel=1e-9)


@pytest.mark.parametrize("which", ["ferrers", "needle"])
def test_adaptive_trajectories_and_weights(cuda, smo, oracle_force, which):
    spec = CFG["potential"] if which == "ferrers" else inputs.paper_bar_potential()
    pot = binding.sm_make_potential(spec)
    ics = inputs.make_ics(CFG, oracle_force, n_orb=288, potential=spec)
    g, gw, gt = (t.cpu().numpy() for t in binding.sm_integrate_rk32(pot, ics, 1000, **TOL))
    o, ow, ot = smo.integrate_rk32(spec, ics, 1000, **TOL)
    tw, _, _ = smo.integrate_rk32(spec, ics * (1 + 1e-15), 1000, **TOL)
    _gate(g, gw, gt, o, ow, ot, traj_rel_err(tw, o, 1.0), "RK3(2) adaptive, " + which)
    assert 0.0 < np.mean(gw == 0) < 0.4          # some attempts are rejected, most are not


def test_fixed_step_trajectories(cuda, smo, oracle_force):
    """rtol <= 0: no decisions, plain third-order Runge-Kutta; also the static Plummer sphere (Omega_p = 0)."""
    pot = binding.sm_make_potential(CFG["potential"])
    ics = inputs.make_ics(CFG, oracle_force, n_orb=200)
    g, gw, gt = (t.cpu().numpy() for t in binding.sm_integrate_rk32(pot, ics, 1000, rtol=0.0, h0=1e-3))
    o, ow, ot = smo.integrate_rk32(CFG["potential"], ics, 1000, rtol=0.0, h0=1e-3)
    tw, _, _ = smo.integrate_rk32(CFG["potential"], ics * (1 + 1e-15), 1000, rtol=0.0, h0=1e-3)
    assert np.all(gw == 1e-3) and gt == pytest.approx(np.full(200, 1.0), rel=1e-12)
    _gate(g, gw, gt, o, ow, ot, traj_rel_err(tw, o, 1.0), "RK3 fixed steps")
    c0 = inputs.CONFIGS[0]
    p0 = binding.sm_make_potential(c0["potential"])
    ic0 = inputs.plummer_ics(300, 1)
    g0 = binding.sm_integrate_rk32(p0, ic0, 500, rtol=1e-6, atol_x=1e-8, atol_v=1e-8, h0=0.01)
    o0 = smo.integrate_rk32(c0["potential"], ic0, 500, rtol=1e-6, atol_x=1e-8, atol_v=1e-8, h0=0.01)
    assert traj_rel_err(g0[0].cpu().numpy(), o0[0], 1.0).max() < 1e-10
    assert g0[2].cpu().numpy() == pytest.approx(o0[2], rel=1e-10)


def test_non_finite_error_estimate_shrinks_the_step_as_in_the_oracle(cuda, smo):
    """Reading R23: a NaN error estimate (first step 1e300: the stages overflow) rejects the attempt and multiplies the step by 0.2;
    the orbits recover after ~430 attempts.  Same accept / reject sequence as the oracle, same integrated time."""
    c0 = inputs.CONFIGS[0]
    p0 = binding.sm_make_potential(c0["potential"])
    ic0 = inputs.plummer_ics(64, 2)
    tol = dict(rtol=1e-6, atol_x=1e-9, atol_v=1e-9, h0=1e300)
    g, gw, gt = (t.cpu().numpy() for t in binding.sm_integrate_rk32(p0, ic0, 700, **tol))
    o, ow, ot = smo.integrate_rk32(c0["potential"], ic0, 700, **tol)
    assert np.all(ow[:300] == 0) and np.all(ot > 0.05)
    assert np.array_equal(gw > 0, ow > 0)
    assert gt == pytest.approx(ot, rel=1e-9) and np.isfinite(g).all()
    assert traj_rel_err(g, o, 1.0).max() < 1e-9


def test_weighted_library_against_the_oracle(cuda, smo, oracle_force):
    """Rows = fp32 sums of dt/t_total.  Per row: L1 distance to the oracle's fp64 row at most the weight of the samples within
    1e-9 bin widths of an edge (either code is right) plus fp32 summation error; every row plus its outside weight sums to 1."""
    spec = inputs.paper_bar_potential()
    pot = binding.sm_make_potential(spec)
    cfg = inputs.CONFIGS[4]                      # three projections
    ics = inputs.make_ics(CFG, oracle_force, n_orb=70, potential=spec)    # ragged: not a multiple of the block size
    g = binding.sm_build_library_rk32(pot, ics, 800, cfg["projections"], cfg["grids"], **TOL)
    o = smo.build_library_rk32(spec, ics, 800, cfg["projections"], cfg["grids"], **TOL)
    t_ok = np.abs(g["t_end"].cpu().numpy() / o["t_end"] - 1) < 1e-9
    assert t_ok.mean() >= 0.95
    for p in range(3):
        gl = g["losvd"][p].cpu().numpy().astype(np.float64)
        l1 = np.abs(gl - o["losvd"][p]).sum(1)
        assert np.all(l1[t_ok] <= 2 * o["edge_w"][p][t_ok] + 2e-5), (p, l1.max())
        assert gl.sum(1) + g["wout"][p].cpu().numpy() == pytest.approx(np.ones(70), abs=2e-5)
        assert g["wout"][p].cpu().numpy()[t_ok] == pytest.approx(o["wout"][p][t_ok], abs=2e-5)
    gd = g["dens"].cpu().numpy().astype(np.float64)
    assert np.all(np.abs(gd - o["dens"]).sum(1)[t_ok] <= 2 * o["edge_w"][3][t_ok] + 2e-5)
    assert gd.sum(1) + g["wout"][3].cpu().numpy() == pytest.approx(np.ones(70), abs=2e-5)


def test_hash_rows_equal_global_atomic_rows(cuda, oracle_force):
    """The two weighted row builds (default: fixed-point shared-memory hash, non-zero cells into rows zeroed beside the integrator;
    debug flag 512: the first version, fp32 atomics on the global row) add the same terms in a different arithmetic: cells agree to
    fp32 summation error, the outside weights likewise, zero cells are exactly zero in both.  The default is reproducible bit for
    bit from call to call (order-independent sums), also through the segmented work queue (flag 8) and the orbit-chunk loop (1024)."""
    pot = binding.sm_make_potential(CFG["potential"])
    cfg = inputs.CONFIGS[4]
    ics = inputs.make_ics(CFG, oracle_force, n_orb=150)
    a = binding.sm_build_library_rk32(pot, ics, 700, cfg["projections"], cfg["grids"], **TOL)
    outs = {}
    for flags in (0, 512, 8, 1024):
        prev = binding.sm_set_debug_flags(flags)
        try:
            outs[flags] = binding.sm_build_library_rk32(pot, ics, 700, cfg["projections"], cfg["grids"], **TOL)
        finally:
            binding.sm_set_debug_flags(prev)
    b = outs[512]
    for k in ("losvd", "dens", "wout"):
        assert (a[k] - b[k]).abs().max().item() <= 2e-6, k
        assert ((a[k] == 0) == (b[k] == 0)).all().item(), k
        for flags in (0, 8, 1024):
            assert (a[k] == outs[flags][k]).all().item(), (k, flags)
    assert (a["t_end"] == b["t_end"]).all().item() and (a["t_end"] == outs[8]["t_end"]).all().item()


def _row_l1_ok(g, o, edge, total, what):
    l1 = np.abs(np.asarray(g, dtype=np.float64) - o).reshape(o.shape[0], -1).sum(1)
    assert np.all(l1 <= 2 * edge + 2e-5 * total), (what, l1.max(), edge.max())


def test_paper_observables_on_the_adaptive_integrator_match_oracle(cuda, smo, oracle_force):
    """SURVEY 8(f) NEXT-4 composed with NEXT-1/2: bundles, fourfold copies, aperture regrouping,
    cylindrical cells and Gauss-Hermite sums with weights dt / t_total, against oracle/smo.py build_observable_library_rk32 (pinned
    in tests/test_oracle_rk32_obs.py).  Per row: L1 distance <= 2 x (weight of the samples within 1e-9 bin widths of an edge)
    + 2e-5 x the row's total weight (fp32 cells; 2^-32 fixed-point sums); rows + outside weight = n_bundle x copies; the Jacobi
    diagnostic equal to the oracle's to 1e-6 relative; integration times to 1e-9."""
    from test_oracle_bundles import aperture_map, cyl_grids
    cfg = inputs.CONFIGS[4]
    pot = binding.sm_make_potential(CFG["potential"])
    ics = inputs.make_ics(CFG, oracle_force, n_orb=96)
    g_c, g_y = cfg["grids"], cyl_grids(cfg["grids"])
    ap, n_ap = aperture_map(g_c)
    rng = np.random.default_rng(4)
    v0, sg = rng.normal(0, 60, n_ap), rng.uniform(70, 160, n_ap)
    n_steps = 500
    cases = [dict(), dict(n_bundle=4, fourfold=True), dict(ap_map=ap, n_ap=n_ap, n_bundle=3, fourfold=True, density_mode=1),
             dict(ap_map=ap, n_ap=n_ap, n_bundle=2, fourfold=True, density_mode=1, gh=(v0, sg)), dict(ap_map=ap, n_ap=n_ap, gh=(v0, sg))]
    for kw in cases:
        grids = g_y if kw.get("density_mode") else g_c
        a = binding.sm_build_observable_library_rk32(pot, ics, n_steps, cfg["projections"], grids, want_diag=True, **TOL, **kw)
        o = smo.build_observable_library_rk32(CFG["potential"], ics, n_steps, cfg["projections"], grids, want_drift=True, **TOL, **kw)
        total = kw.get("n_bundle", 1) * (4 if kw.get("fourfold") else 1)
        key = "gh" if "gh" in kw else "losvd"
        for p in range(3):
            gp = a[key][p].cpu().numpy()
            if key == "gh":
                # the sums m >= 0 carry |alpha H_m| <= 0.4 per unit weight: same bound; edge samples move between apertures
                _row_l1_ok(gp, o["gh"][p], o["edge_w"][p] * 3, total, (kw.keys(), p))
                assert np.allclose(gp[..., 0].sum(1) + a["wout"][p].cpu().numpy(), total, atol=2e-5 * total)
            else:
                _row_l1_ok(gp, o["losvd"][p], o["edge_w"][p], total, (kw.keys(), p))
                assert np.allclose(gp.sum(1) + a["wout"][p].cpu().numpy(), total, atol=2e-5 * total)
        _row_l1_ok(a["dens"].cpu().numpy(), o["dens"], o["edge_w"][3], total, "dens")
        assert np.allclose(a["wout"].cpu().numpy(), o["wout"], atol=2 * o["edge_w"].max() + 2e-5 * total)
        assert a["t_end"].cpu().numpy() == pytest.approx(o["t_end"], rel=1e-9)
        d = a["diag"].cpu().numpy()
        assert d[:, 1].sum() == 0 and d[:, 0] == pytest.approx(o["drift"], rel=1e-6, abs=1e-12)
    # the plain call is the observable call without options
    plain = binding.sm_build_library_rk32(pot, ics, n_steps, cfg["projections"], g_c, **TOL)
    same = binding.sm_build_observable_library_rk32(pot, ics, n_steps, cfg["projections"], g_c, **TOL)
    for k in ("losvd", "dens", "wout", "t_end"):
        assert (plain[k] == same[k]).all().item(), k
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_build_observable_library_rk32(pot, ics, n_steps, cfg["projections"], g_c, n_bundle=5, **TOL)


def test_invalid_arguments_launch_nothing(cuda):
    static_bar = {"G": inputs.G_GALACTIC, "omega_p": 40.0, "phase0": 0.0, "components": [(inputs.FERRERS2, 0, [1e10, 4.0, 1.5, 0.5])]}
    pot = binding.sm_make_potential(static_bar)
    ics = np.array([[3.0, 0, 0, 0, 100.0, 0]])
    n0 = binding.sm_launch_count()
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_integrate_rk32(pot, ics, 10)           # a non-rotating triaxial component in a rotating frame
    ok = binding.sm_make_potential(CFG["potential"])
    for kw in (dict(n_steps=0), dict(n_steps=10, h0=0.0), dict(n_steps=10, atol_x=-1.0)):
        with pytest.raises(binding.SchwarmaxError):
            binding.sm_integrate_rk32(ok, ics, **kw)
    assert binding.sm_launch_count() == n0


def test_bench_rk32_and_paper_bar_modes_run_and_report(cuda):
    """bench.py --rk32 and --bar dehnen at reduced sizes: exit 0, one JSON line with the contract's keys, rows consistent."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    common = ["--n-orb", "1500", "--n-steps", "300", "--steps", "1", "--warmup", "1", "--no-cpu-baseline"]
    for mode, ok_key in ((["--rk32"], "rows_sum_to_one"), (["--rk32", "--bar", "dehnen"], "rows_sum_to_one"), (["--bar", "dehnen", "--no-e2e"], "row_sums_ok"),
                         (["--rk32", "--config", "3", "--n-trials", "5", "--apertures", "40"], "rows_sum_to_one")):
        r = subprocess.run([sys.executable, os.path.join(root, "bench.py")] + mode + common, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        line = json.loads(r.stdout.strip().splitlines()[-1])
        for k in ("metric", "value", "unit", "n_gpus", "ms_per_step", "roofline", "e2e", "gpu_launches", "clocks", "config", "dtype"):
            assert k in line, k
        assert line[ok_key] is True and line["gpu_launches"] > 0 and line["value"] > 0 and line["roofline"]["bound"] == "alu"
