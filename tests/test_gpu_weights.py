"""GPU parity of the weight solve (sm_solve_weights) against oracle/nnls.py, through the C ABI.

Tolerance: both sides are fp64; they differ in summation order and in how the linear
system is solved (explicit inverse by block Gauss-Jordan vs Cholesky), so one x-update differs by about
cond(G) * 2^-53 * |x| and the iteration (a non-expansive map) does not amplify it: 1e-9 * max|w| for cond(G) <~ 1e4.
"""
import numpy as np
import pytest

from paper_2607_00117_b200 import inputs

pytestmark = pytest.mark.gpu

RTOL = 1e-9


def oracle_system(p):
    from oracle import nnls as onnls
    n_orb = p["dens"].shape[0]
    blocks, tg, sg, o = [], [], [], 0
    for name, c0, st, nc in p["blocks"]:
        blocks.append(p[name].reshape(n_orb, -1)[:, c0::st][:, :nc])
        tg.append(p["target"][o:o + nc]); sg.append(p["sigma"][o:o + nc]); o += nc
    U, y, _ = onnls.stack_system(blocks, tg, sg, keep=p["keep"].astype(bool))
    return U, onnls.bootstrap(y, p["xi"])


def cuda_solve(p, lam, rho, n_iter, wtilde=None, use_keep=True, xi=True, want_chi2=False):
    import torch
    from paper_2607_00117_b200 import binding
    dev = {k: torch.as_tensor(p[k]).cuda() for k in ("dens", "gh")}
    blocks = [(dev[name], c0, st, nc) for name, c0, st, nc in p["blocks"]]
    out = binding.sm_solve_weights(blocks, p["target"], p["sigma"], lam, rho, n_iter, xi=p["xi"] if xi else None,
                                   keep=p["keep"] if use_keep else None, wtilde=wtilde, want_chi2=want_chi2)
    torch.cuda.synchronize()
    if want_chi2:
        n_blocks = len(p["blocks"])
        marg = binding.sm_marginal_chi2(out["chi2"], (1 << n_blocks) - 2)      # every block but the first (3-D density)
        return out["w"].cpu().numpy(), out["resid"].cpu().numpy(), out["chi2"].cpu().numpy(), marg.cpu().numpy()
    return out["w"].cpu().numpy(), out["resid"].cpu().numpy()


def test_gemm_building_block_against_numpy():
    import torch
    from paper_2607_00117_b200 import binding
    rng = np.random.default_rng(0)
    for (M, N, K) in [(1, 1, 1), (100, 257, 300), (129, 128, 17), (64, 300, 64), (300, 131, 1000)]:
        A = rng.standard_normal((M, K)); Bk = rng.standard_normal((N, K)); Bn = rng.standard_normal((K, N))
        C0 = rng.standard_normal((M, N))
        dA, dBk, dBn = (torch.as_tensor(x).cuda() for x in (A, Bk, Bn))
        tol = 1e-13 * K
        assert np.max(np.abs(binding.sm_debug_gemm_f64(dA, dBk, True).cpu().numpy() - A @ Bk.T)) < tol
        binding.sm_set_debug_flags(128)       # the register-tiled DFMA kernel instead of the FP64 matrix unit
        try:
            assert np.max(np.abs(binding.sm_debug_gemm_f64(dA, dBk, True).cpu().numpy() - A @ Bk.T)) < tol
        finally:
            binding.sm_set_debug_flags(0)
        assert np.max(np.abs(binding.sm_debug_gemm_f64(dA, dBn, False).cpu().numpy() - A @ Bn)) < tol
        got = binding.sm_debug_gemm_f64(dA, dBn, False, alpha=-1.0, beta=1.0, C_in=torch.as_tensor(C0).cuda()).cpu().numpy()
        assert np.max(np.abs(got - (C0 - A @ Bn))) < tol
        parts = binding.sm_debug_gemm_f64(dA, dBk, True, alpha=2.0, split_k=3).cpu().numpy()
        assert np.max(np.abs(parts.sum(axis=0) - 2.0 * A @ Bk.T)) < tol
    # operands that are views with a row pitch
    big = torch.as_tensor(rng.standard_normal((70, 90))).cuda()
    v = big[:, 10:75]
    assert np.max(np.abs(binding.sm_debug_gemm_f64(v, v, True).cpu().numpy() - (v @ v.T).cpu().numpy())) < 1e-11


@pytest.mark.parametrize("n", [1, 5, 64, 65, 200, 333])
def test_spd_inverse_building_block(n):
    import torch
    from paper_2607_00117_b200 import binding
    rng = np.random.default_rng(n)
    B = rng.standard_normal((n + 7, n))
    G = B.T @ B + 0.5 * np.eye(n)
    pad = np.zeros((n, n + 3)); pad[:, :n] = G
    d = torch.as_tensor(pad).cuda()
    binding.sm_debug_invert_spd(d[:, :n])
    inv = d.cpu().numpy()[:, :n]
    assert np.max(np.abs(inv @ G - np.eye(n))) < 1e-10 * np.linalg.cond(G)
    assert np.max(np.abs(inv - np.linalg.inv(G))) < 1e-12 * np.linalg.cond(G) * np.max(np.abs(inv))
    assert np.all(d.cpu().numpy()[:, n:] == 0)          # the padding is not touched


@pytest.mark.parametrize("n_orb,n_dens,n_ap,n_rhs,n_iter", [(300, 90, 25, 5, 60), (517, 301, 77, 100, 40), (130, 1, 1, 1, 25),
                                                                   (257, 40, 10, 130, 15)])
def test_weights_equal_the_oracle(n_orb, n_dens, n_ap, n_rhs, n_iter):
    from oracle import nnls as onnls
    p = inputs.weight_problem(n_orb, n_dens, n_ap, n_rhs, seed=3)
    U, Y = oracle_system(p)
    rho = 0.1 * float(np.mean(np.sum(U * U, axis=0)))
    wt = np.full(n_orb, 1.0 / n_orb)
    lam = 1e-3 * rho * n_orb * wt[0] ** 2          # regularisation of the same order as the data term
    w_ref, r_ref = onnls.admm_nnls(U, Y, lam, rho, n_iter, wtilde=wt)
    w, r, chi2, marg = cuda_solve(p, lam, rho, n_iter, wtilde=wt, want_chi2=True)
    # Eq. 5-6: chi^2 per block against the unperturbed data, and the bootstrap-marginalised model chi^2 without the density block
    y0 = onnls.bootstrap(Y[0] - p["xi"][0], np.zeros_like(p["xi"][:1]))[0]
    chi2_ref = onnls.chi2_blocks(U, y0, w_ref, [nc for _, _, _, nc in p["blocks"]])
    assert chi2.shape == chi2_ref.shape and np.allclose(chi2, chi2_ref, rtol=1e-7, atol=1e-9)
    cb = chi2_ref[:, 1:].sum(axis=1)
    assert abs(marg[0] - onnls.marginal_chi2(cb)) < 1e-7 * cb.min() and abs(marg[1] - cb.min()) < 1e-7 * cb.min()
    scale = np.max(np.abs(w_ref))
    assert scale > 0 and np.max(np.abs(w - w_ref)) < RTOL * scale
    assert np.all(w >= 0) and np.all(w[:, p["keep"] == 0] == 0)
    assert np.allclose(r, r_ref, rtol=1e-4, atol=1e-7 * scale * max(1.0, rho))
    # the support (which weights were clipped) is the same wherever the oracle is not within rounding of zero
    clear = np.abs(w_ref) > 1e-7 * scale
    assert np.array_equal((w > 0)[clear], (w_ref > 0)[clear])


def test_weights_without_options_and_one_iteration():
    from oracle import nnls as onnls
    p = inputs.weight_problem(200, 50, 20, 3, seed=9)
    p["keep"][:] = 1
    U, Y = oracle_system(p)
    rho = float(np.mean(np.sum(U * U, axis=0)))
    for n_iter in (1, 2):
        w_ref, _ = onnls.admm_nnls(U, Y[:1], 0.0, rho, n_iter)
        w, _ = cuda_solve(p, 0.0, rho, n_iter, use_keep=False, xi=False)
        assert w.shape == (1, 200) and np.max(np.abs(w - w_ref)) < RTOL * np.max(w_ref)


def test_all_orbits_dropped_gives_zero_weights_and_bad_arguments_fail():
    import torch
    from paper_2607_00117_b200 import binding
    p = inputs.weight_problem(70, 20, 8, 2, seed=4)
    p["keep"][:] = 0
    w, _ = cuda_solve(p, 1.0, 1.0, 5)
    assert np.all(w == 0)
    m = torch.zeros((4, 6), dtype=torch.float32, device="cuda")
    for kw in (dict(lam=-1.0, rho=1.0, n_iter=3), dict(lam=0.0, rho=0.0, n_iter=3), dict(lam=0.0, rho=1.0, n_iter=0)):
        with pytest.raises(binding.SchwarmaxError):
            binding.sm_solve_weights([(m,)], np.ones(6), np.ones(6), kw["lam"], kw["rho"], kw["n_iter"])
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_solve_weights([(m, 2, 3, 3)], np.ones(3), np.ones(3), 0.0, 1.0, 1)   # columns past the row pitch


def test_constraints_without_a_positive_tolerance_are_ignored():
    """include/schwarmax.h: a constraint whose tolerance d_sigma is not a positive finite number is ignored (its row of U and
    its entry of y are zero).  The solve with sigma = 0, -1, inf, nan on some constraints must equal the oracle's solve of the
    system with those constraints REMOVED, and its chi^2 blocks must not count them."""
    from oracle import nnls as onnls
    p = inputs.weight_problem(120, 30, 10, 3, seed=6)
    bad = np.array([2, 17, 31, 44, 75])
    q = dict(p, sigma=p["sigma"].copy())
    q["sigma"][bad] = [0.0, -1.0, np.inf, np.nan, 0.0]
    U, Y = oracle_system(p)
    keep_rows = np.setdiff1d(np.arange(U.shape[0]), bad)
    rho = 0.1 * float(np.mean(np.sum(U * U, axis=0)))
    w_ref, _ = onnls.admm_nnls(U[keep_rows], Y[:, keep_rows], 1e-3 * rho, rho, 40)
    w, _, chi2, _ = cuda_solve(q, 1e-3 * rho, rho, 40, want_chi2=True)
    assert np.all(np.isfinite(w)) and np.all(np.isfinite(chi2))
    assert np.max(np.abs(w - w_ref)) < RTOL * np.max(np.abs(w_ref))


def test_solution_of_a_full_size_problem_satisfies_kkt():
    """The size bench.py --weights times (7 500 bundles, 600 apertures, 100 bootstrap realisations), where the oracle
    would take minutes: properties that hold at any size -- feasibility, the KKT conditions of Eq. 4 to the level the
    reported ADMM residuals allow, and one realisation solved on its own reproducing its row of the batch."""
    import torch
    n_orb, n_dens, n_ap, n_rhs = 7500, 1500, 600, 100
    p = inputs.weight_problem(n_orb, n_dens, n_ap, n_rhs, seed=0)
    dev = {k: torch.as_tensor(p[k]).cuda() for k in ("dens", "gh")}
    sig = torch.as_tensor(p["sigma"]).cuda()
    cols = [dev[name].reshape(n_orb, -1)[:, c0::st][:, :nc].double() for name, c0, st, nc in p["blocks"]]
    Ut = torch.cat(cols, dim=1) / sig[None, :] * torch.as_tensor(p["keep"]).cuda()[:, None]
    Y = torch.as_tensor(p["target"] / p["sigma"]).cuda()[None, :] + torch.as_tensor(p["xi"]).cuda()
    rho = 0.1 * float((Ut * Ut).sum(dim=1).mean())
    lam = 1e-3 * rho * n_orb
    w, resid = cuda_solve(p, lam, rho, 300)
    assert np.all(w >= 0) and np.all(np.isfinite(w))
    wd = torch.as_tensor(w).cuda()
    grad = (wd @ Ut - Y) @ Ut.T + 2 * lam / n_orb * wd          # [n_rhs][n_orb]
    gscale = float((Y @ Ut.T).abs().max())
    # ADMM: grad Q(x) = -rho u + rho (z_prev - z) with u <= 0 and u z = 0, and grad Q(z) - grad Q(x) = (U^T U + D)(z - x):
    # the KKT violation of z is bounded by the dual residual plus ||U^T U + D|| times the primal residual
    v = torch.ones(n_orb, dtype=torch.float64, device="cuda")
    for _ in range(30):
        v = (v @ Ut) @ Ut.T
        norm_g = float(v.norm()); v = v / norm_g
    bound = 2 * ((norm_g + 2 * lam / n_orb) * resid[:, 0] + resid[:, 1]).max() + 1e-9 * gscale
    assert float((-grad).clamp(min=0).max()) < bound
    assert float((grad.abs() * (wd > 0)).max()) < bound
    # one realisation on its own reproduces its row of the batch
    p1 = dict(p); p1["xi"] = p["xi"][7:8]
    w1, _ = cuda_solve(p1, lam, rho, 300)
    assert np.array_equal(w1[0], w[7])


def test_library_to_weights_pipeline(smo, oracle_force):
    """The product chain end to end: the Gauss-Hermite library sm_build_gh_library writes (symmetrised bundles, cylindrical
    density cells) goes into sm_solve_weights in place, as strided views; the oracle chain (oracle library -> oracle ADMM)
    starts from the same initial conditions.  The two libraries agree to 2e-6 per sample in the Gauss-Hermite sums and
    exactly in the counts except for samples within rounding of a cell edge (none in this case: measured difference 1.6e-9),
    so the gate is 1e-6 rather than the 1e-9 of identical inputs."""
    import torch
    from oracle import nnls as onnls
    from paper_2607_00117_b200 import binding
    from test_oracle_bundles import aperture_map, cyl_grids
    cfg = inputs.CONFIGS[4]
    g = cyl_grids(cfg["grids"])
    n_bundle, n_rows = 3, 40
    ics = inputs.make_ics(cfg, oracle_force, n_orb=n_bundle * n_rows)
    ap, n_ap = aperture_map(g)
    rng = np.random.default_rng(5)
    v0, s = rng.normal(0, 60, n_ap), rng.uniform(70, 160, n_ap)
    args = (cfg["dt"], 600, cfg["stride"], cfg["projections"], g, ap, n_ap, v0, s)
    o = smo.build_gh_library(cfg["potential"], ics, *args, n_bundle=n_bundle, fourfold=True, density_mode=1)
    pot = binding.sm_make_potential(cfg["potential"])
    a = binding.sm_build_gh_library(pot, ics, *args, n_bundle=n_bundle, fourfold=True, density_mode=1)
    # stacking order of Eq. 3: 3-D mass, surface density, h_1..h_4 of projection 0
    o_gh = o["gh"][0].astype(np.float32).astype(np.float64)
    o_blocks = [o["dens"].astype(np.float64), o_gh[:, :, 0]] + [o_gh[:, :, 1 + m] for m in range(1, 5)]
    w_hidden = rng.random(n_rows) * (rng.random(n_rows) < 0.6)
    targets = [w_hidden @ b for b in o_blocks]
    s_sig = 0.01 * np.maximum(targets[1], 1e-3 * targets[1].max())
    sigmas = [0.01 * np.maximum(targets[0], 1e-3 * targets[0].max()), s_sig] + [2 * s_sig] * 4
    targets = [t + sg * rng.standard_normal(t.size) for t, sg in zip(targets, sigmas)]
    U, y, _ = onnls.stack_system(o_blocks, targets, sigmas)
    xi = rng.standard_normal((3, y.size)); xi[:, :o_blocks[0].shape[1]] = 0.0
    rho = 0.1 * float(np.mean(np.sum(U * U, axis=0)))
    lam = 1e-3 * rho * n_rows
    w_ref, _ = onnls.admm_nnls(U, onnls.bootstrap(y, xi), lam, rho, 200)
    gh0 = a["gh"][0]
    blocks = [(a["dens"],), (gh0, 0, 6, n_ap)] + [(gh0, 1 + m, 6, n_ap) for m in range(1, 5)]
    out = binding.sm_solve_weights(blocks, np.concatenate(targets), np.concatenate(sigmas), lam, rho, 200, xi=xi)
    w = out["w"].cpu().numpy()
    scale = np.max(w_ref)
    print("pipeline: max |w - w_ref| / max w =", np.max(np.abs(w - w_ref)) / scale, "near-edge rows", int((o["near_edge"].sum(0) > 0).sum()))
    assert np.max(np.abs(w - w_ref)) < 1e-6 * scale


def test_bench_model_and_weights_modes_run_and_report():
    """bench.py --model / --weights at reduced sizes: exit 0, one JSON line with the contract's keys, finite weights and chi^2."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    common = ["--steps", "1", "--warmup", "1", "--w-rhs", "4", "--w-iter", "12", "--no-cpu-baseline"]
    for mode, extra, ok_key in (("--model", ["--n-orb", "1200", "--n-steps", "400", "--apertures", "40"], "model_ok"),
                                ("--model", ["--rk32", "--n-orb", "1200", "--n-steps", "400", "--apertures", "40"], "model_ok"),
                                ("--weights", ["--n-orb", "300", "--apertures", "40", "--w-dens", "50"], "weights_ok")):
        r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), mode] + extra + common, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        line = json.loads(r.stdout.strip().splitlines()[-1])
        for k in ("metric", "value", "unit", "n_gpus", "ms_per_step", "roofline", "e2e", "gpu_launches", "clocks", "config", "dtype"):
            assert k in line, k
        assert line[ok_key] is True and line["gpu_launches"] > 0 and np.isfinite(line["chi2_model"])
        assert line["e2e"]["h2d_bytes_per_step"] > 0 and line["roofline"]["bound"] == "alu"
