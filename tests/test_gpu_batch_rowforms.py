"""Row a-8 for the paper's row forms (north_star item 4): sm_build_observable_library_batch and
sm_build_gh_library_batch -- symmetrised bundles, apertures, cylindrical cells and Gauss-Hermite sums for several trial
potentials in one integrator launch.  The oracle is the single-potential oracle called once per trial on that trial's
potential, viewing angles and ICs (config-3 recipe: BASELINE.json configs[3])."""
import numpy as np
import pytest

from paper_2607_00117_b200 import binding, inputs

from gpu_util import count_parity
from test_oracle_bundles import aperture_map, cyl_grids

pytestmark = pytest.mark.gpu

N_TRIALS, N_ORB, N_STEPS = 4, 96, 600


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def batch(oracle_force, torch_cuda):
    cfg = inputs.CONFIGS[3]
    draws = inputs.trial_draws(N_TRIALS, cfg["seed"])
    ics = np.stack([inputs.make_ics(cfg, oracle_force, n_orb=N_ORB, potential=d["potential"]) for d in draws])
    pot = binding.sm_make_potential_batch([d["potential"] for d in draws])
    return cfg, draws, ics, pot, [[d["projection"]] for d in draws]


def test_batched_gauss_hermite_library_matches_oracle_per_trial(smo, batch):
    """fp64: per trial, sample counts per aperture identical to the oracle on rows without near-edge samples, Gauss-Hermite sums
    within 2e-6 per sample, density counts identical -- plain rows and symmetrised bundles of 3 on cylindrical cells; per-trial
    ICs and shared ICs; the batch block of a trial is bit-identical to the single-trial call on that trial's potential."""
    cfg, draws, ics, pot, projs = batch
    g = cyl_grids(cfg["grids"])
    ap, n_ap = aperture_map(g)
    rng = np.random.default_rng(4)
    v0, s = rng.normal(0, 60, n_ap), rng.uniform(70, 160, n_ap)
    n_rec = N_STEPS // cfg["stride"]
    for n_bundle, fourfold, dmode, shared in ((1, False, 0, False), (3, True, 1, False), (3, True, 1, True)):
        src = ics[0] if shared else ics
        a = binding.sm_build_observable_library_batch(pot, src, cfg["dt"], N_STEPS, cfg["stride"], projs, g, ap, n_ap, n_bundle=n_bundle,
                                                      fourfold=fourfold, density_mode=dmode, gh=(v0, s))
        n_rows, total = N_ORB // n_bundle, n_bundle * (4 if fourfold else 1) * n_rec
        assert a["gh"].shape == (N_TRIALS, 1, n_rows, n_ap, 6) and a["dens"].shape[:2] == (N_TRIALS, n_rows)
        for t, d in enumerate(draws):
            it = ics[0] if shared else ics[t]
            o = smo.build_gh_library(d["potential"], it, cfg["dt"], N_STEPS, cfg["stride"], [d["projection"]], g, ap, n_ap, v0, s,
                                     n_bundle=n_bundle, fourfold=fourfold, density_mode=dmode)
            gh = a["gh"][t, 0].cpu().numpy().astype(np.float64)
            clean = o["near_edge"][0] == 0
            assert clean.sum() >= 0.7 * n_rows
            assert np.array_equal(gh[clean, :, 0], o["gh"][0, clean, :, 0]), t
            assert np.array_equal(gh[:, :, 0].sum(1) + a["nout"][t, 0].cpu().numpy(), np.full(n_rows, total))
            err = np.abs(gh[clean, :, 1:] - o["gh"][0, clean, :, 1:])
            assert np.all(err <= 2e-6 * o["gh"][0, clean, :, :1] + 1e-9), (t, err.max())
            assert np.abs(o["gh"][0, clean, :, 1:]).max() > 1.0
            assert count_parity(a["dens"][t].cpu().numpy(), o["dens"], o["near_edge"][1]) >= 0.7 * n_rows
            assert np.array_equal(a["dens"][t].sum(1).cpu().numpy() + a["nout"][t, 1].cpu().numpy(), np.full(n_rows, total))
            single = binding.sm_build_gh_library(binding.sm_make_potential(d["potential"]), it, cfg["dt"], N_STEPS, cfg["stride"],
                                                 [d["projection"]], g, ap, n_ap, v0, s, n_bundle=n_bundle, fourfold=fourfold, density_mode=dmode)
            assert (single["gh"][0] == a["gh"][t, 0]).all().item() and (single["dens"] == a["dens"][t]).all().item()
            assert (single["nout"] == a["nout"][t]).all().item()


def test_batched_aperture_rows_match_oracle_per_trial_and_trial_subrange(smo, batch):
    """The LOSVD row form (apertures x v_los, symmetrised bundles) per trial against the oracle in fp64; a trial sub-range
    [1, 3) gives the same blocks; fp32 batched (tables through L1, warp teams) equals the fp32 single-trial call bit for bit and
    keeps the row-sum invariant; the library-internal chunk loop (debug flag 1024: 1 MiB of staging) changes nothing."""
    cfg, draws, ics, pot, projs = batch
    g = cfg["grids"]
    ap, n_ap = aperture_map(g)
    n_rec = N_STEPS // cfg["stride"]
    args = (cfg["dt"], N_STEPS, cfg["stride"])
    kw = dict(n_bundle=3, fourfold=True)
    n_rows, total = N_ORB // 3, 12 * n_rec
    a = binding.sm_build_observable_library_batch(pot, ics, *args, projs, g, ap, n_ap, **kw)
    assert a["losvd"].shape == (N_TRIALS, 1, n_rows, n_ap * g["nv"])
    for t, d in enumerate(draws):
        o = smo.build_observable_library(d["potential"], ics[t], *args, [d["projection"]], g, ap, n_ap, **kw)
        assert count_parity(a["losvd"][t, 0].cpu().numpy(), o["losvd"][0], o["near_edge"][0]) >= 0.7 * n_rows
        assert count_parity(a["dens"][t].cpu().numpy(), o["dens"], o["near_edge"][1]) >= 0.7 * n_rows
        assert np.array_equal(a["losvd"][t, 0].sum(1).cpu().numpy() + a["nout"][t, 0].cpu().numpy(), np.full(n_rows, total))
    sub = binding.sm_build_observable_library_batch(pot, ics[1:3], *args, projs[1:3], g, ap, n_ap, trial0=1, n_trials=2, **kw)
    for k in ("losvd", "dens", "nout"):
        assert (sub[k] == a[k][1:3]).all().item(), k
    big = np.tile(ics, (1, 32, 1))               # 3 072 orbits per trial: two chunks of 1 536 under the 1 MiB staging cap
    whole = binding.sm_build_observable_library_batch(pot, big, *args, projs, g, ap, n_ap, **kw)
    prev = binding.sm_set_debug_flags(1024)
    try:
        chunked = binding.sm_build_observable_library_batch(pot, big, *args, projs, g, ap, n_ap, **kw)
    finally:
        binding.sm_set_debug_flags(prev)
    for k in ("losvd", "dens", "nout"):
        assert (chunked[k] == whole[k]).all().item(), k
        assert (whole[k][..., :n_rows, :] == a[k]).all().item() if k != "nout" else (whole[k][..., :n_rows] == a[k]).all().item(), k
    f32 = binding.sm_build_observable_library_batch(pot, ics, *args, projs, g, ap, n_ap, precision="f32", **kw)
    for t, d in enumerate(draws):
        single = binding.sm_build_observable_library(binding.sm_make_potential(d["potential"]), ics[t], *args, [d["projection"]], g, ap, n_ap,
                                                     precision="f32", **kw)
        assert (single["losvd"][0] == f32["losvd"][t, 0]).all().item() and (single["dens"] == f32["dens"][t]).all().item()
        assert np.array_equal(f32["losvd"][t, 0].sum(1).cpu().numpy() + f32["nout"][t, 0].cpu().numpy(), np.full(n_rows, total))
    with pytest.raises(binding.SchwarmaxError):   # the single-trial call refuses a batch potential
        binding.sm_build_observable_library(pot, ics[0], *args, projs[0], g, ap, n_ap)
    with pytest.raises(binding.SchwarmaxError):   # trial range outside the batch
        binding.sm_build_observable_library_batch(pot, ics, *args, projs, g, ap, n_ap, trial0=2, n_trials=4)


def test_adaptive_integrator_batched_trials_equal_the_single_trial_calls(smo, batch):
    """sm_build_observable_library_rk32_batch / sm_build_gh_library_rk32_batch: a CTA works on one trial at a time and moves through
    the trials; every per-orbit array holds n_trials x n_orb orbits.  Each trial's block must equal the single-trial call on that
    trial's potential BIT FOR BIT (fixed-point row sums are order-independent; same kernels) -- plain rows, and symmetrised bundles
    with apertures, cylindrical cells, Gauss-Hermite sums and the Jacobi diagnostic; per-trial and shared ICs; a trial sub-range; queue
    segments and orbit chunks (debug flags 8, 1024).  One trial is also compared with the oracle directly."""
    cfg, draws, ics, pot, projs = batch
    g = cyl_grids(cfg["grids"])
    ap, n_ap = aperture_map(g)
    rng = np.random.default_rng(4)
    v0, s = rng.normal(0, 60, n_ap), rng.uniform(70, 160, n_ap)
    n_att = 260
    singles = [binding.sm_make_potential(d["potential"]) for d in draws]
    cases = (dict(), dict(ap_map=ap, n_ap=n_ap, n_bundle=3, fourfold=True, density_mode=1, gh=(v0, s), want_diag=True),
             dict(ap_map=ap, n_ap=n_ap, n_bundle=2, fourfold=True, want_diag=True))
    for kw in cases:
        gr = g if kw.get("density_mode") else cfg["grids"]
        for shared, flags in ((False, 0), (True, 0), (False, 8), (False, 1024)):
            src = ics[0] if shared else ics
            prev = binding.sm_set_debug_flags(flags)
            try:
                b = binding.sm_build_observable_library_rk32_batch(pot, src, n_att, projs, gr, **kw)
            finally:
                binding.sm_set_debug_flags(prev)
            for t, d in enumerate(draws):
                one = binding.sm_build_observable_library_rk32(singles[t], ics[0] if shared else ics[t], n_att, [d["projection"]], gr, **kw)
                for k in ("gh" if "gh" in kw else "losvd", "dens", "wout", "t_end") + (("diag",) if kw.get("want_diag") else ()):
                    assert (b[k][t] == one[k]).all().item(), (k, t, shared, flags)
        sub = binding.sm_build_observable_library_rk32_batch(pot, ics[1:3], n_att, projs[1:3], gr, trial0=1, n_trials=2, **kw)
        full = binding.sm_build_observable_library_rk32_batch(pot, ics, n_att, projs, gr, **kw)
        for k in sub:
            if sub[k] is not None:
                assert (sub[k] == full[k][1:3]).all().item(), k
    # trial 2 of the plain batch against the oracle (weights to the edge weight + fp32 resolution, as the single-trial test does)
    b = binding.sm_build_observable_library_rk32_batch(pot, ics, n_att, projs, cfg["grids"])
    o = smo.build_observable_library_rk32(draws[2]["potential"], ics[2], n_att, [draws[2]["projection"]], cfg["grids"])
    l1 = np.abs(b["losvd"][2, 0].cpu().numpy().astype(np.float64) - o["losvd"][0]).sum(1)
    assert np.all(l1 <= 2 * o["edge_w"][0] + 2e-5), l1.max()
    assert b["t_end"][2].cpu().numpy() == pytest.approx(o["t_end"], rel=1e-9)
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_build_observable_library_rk32(pot, ics[0], n_att, projs[0], cfg["grids"])   # single-trial call, batch potential


def test_batched_row_forms_reject_bad_arguments_and_launch_nothing(batch):
    """Invalid arguments of the batched entry points return SM_ERR_* with a message and launch no kernel; empty libraries are legal."""
    import torch
    cfg, draws, ics, pot, projs = batch
    g = cfg["grids"]
    ap, n_ap = aperture_map(g)
    v0, s = np.zeros(n_ap), np.ones(n_ap)
    args = (cfg["dt"], N_STEPS, cfg["stride"])
    l0 = binding.sm_launch_count()
    bad = [
        lambda: binding.sm_build_observable_library_batch(pot, ics, *args, projs[:2], g, ap, n_ap),                       # projections for 2 of 4 trials
        lambda: binding.sm_build_observable_library_batch(pot, ics, *args, projs, g, ap, n_ap, n_bundle=5),              # 96 orbits are not bundles of 5
        lambda: binding.sm_build_observable_library_batch(pot, ics, *args, projs, g, None, 0, gh=(v0, s)),               # Gauss-Hermite rows need apertures
        lambda: binding.sm_build_observable_library_batch(pot, ics, *args, projs, g, ap, n_ap, density_mode=2),
        lambda: binding.sm_build_observable_library_batch(pot, ics, *args, projs, g, ap, n_ap, trial0=3, n_trials=2),     # past the end of the batch
        lambda: binding.sm_build_observable_library_batch(pot, ics, cfg["dt"], 0, 1, projs, g, ap, n_ap),                 # n_steps < 1
        lambda: binding.sm_build_observable_library_rk32_batch(pot, ics, 0, projs, g),                                    # no step attempts
        lambda: binding.sm_build_observable_library_rk32_batch(pot, ics, 100, projs, g, trial0=2, n_trials=3),
        lambda: binding.sm_build_observable_library_rk32_batch(pot, ics, 100, projs, g, n_bundle=7),
        lambda: binding.sm_build_observable_library_rk32_batch(pot, ics, 100, projs, g, h0=-1.0),
    ]
    for f in bad:
        with pytest.raises(binding.SchwarmaxError):
            f()
    assert binding.sm_launch_count() == l0
    empty = torch.zeros((N_TRIALS, 0, 6), dtype=torch.float64, device="cuda")
    out = binding.sm_build_observable_library_batch(pot, empty, *args, projs, g, ap, n_ap)
    assert out["losvd"].shape == (N_TRIALS, 1, 0, n_ap * g["nv"])
    out = binding.sm_build_observable_library_rk32_batch(pot, empty, 100, projs, g)
    assert out["t_end"].shape == (N_TRIALS, 0)
