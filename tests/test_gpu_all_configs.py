"""GPU parity tests (-m gpu) that close BASELINE.json `north_star` "matching the CPU oracle within the stated tolerances on
ALL FIVE configs": configs[2] at its own geometry and launch shape in both precisions, configs[3] in its own arithmetic
(fp32, batched potentials, per-trial ICs and angles), the fp32 variant with the plain 2e-2 aggregate gate on a sample large
enough for it, and the library-internal staging chunk loop.

Initial conditions of the 100 000-orbit runs take their circular speeds from the CUDA library's sm_eval_force (64 azimuths x
100 000 radii would cost the __float128 oracle 20 s); they are inputs, generated once and handed identically to both sides
(DESIGN.md 4).  Gates are those of DESIGN.md 6; every oracle-relative gate prints the numbers it compared."""
import numpy as np
import pytest

from paper_2607_00117_b200 import binding, inputs

from gpu_util import count_parity

pytestmark = pytest.mark.gpu

# An orbit is CERTIFIED for the per-orbit fp32 gate (L1 <= 2e-2) when the oracle's own answer is insensitive to input
# perturbations of the size of the fp32 rounding: BOTH oracle twins within 2e-3 of the oracle (a tenth of the gate.
# With n_rec = 1 000 samples per row ONE sample on the other side of a bin edge is an L1 of 2e-3, so few orbits qualify on the
# fine grids: the floors on the certified fraction only keep the gate from being vacuous, and the distribution gates -- median
# and 90th percentile of the per-orbit L1 against the twins' -- cover the other orbits).
CERT = 2e-3


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    return torch


def _device_force(pot):
    return lambda p, x: binding.sm_eval_force(pot, x, 0.0, want_phi=False).cpu().numpy()


def _rows_sum_ok(out, n_rec):
    ok = True
    for p in range(out["losvd"].shape[0]):
        ok = ok and bool((out["losvd"][p].sum(1) + out["nout"][p] == n_rec).all().item())
    return ok and bool((out["dens"].sum(1) + out["nout"][-1] == n_rec).all().item())


def _sample_indices(n, n_random, seed, block=512):
    """Group / warp / CTA boundaries of the bench launch shape plus random orbits."""
    fixed = [0, 1, 31, 32, 33, block - 1, block, block + 1, 2 * block - 1, 2 * block, 4095, 4096, n // 2, n - block, n - 33, n - 32, n - 2, n - 1]
    rng = np.random.default_rng(seed)
    return np.unique(np.concatenate([fixed, rng.integers(0, n, n_random)]))


def _l1_fractions(a, b):
    return np.abs(a / a.sum() - b / b.sum()).sum()


def test_config2_fp64_launch_shape_identical_counts(smo, torch_cuda):
    """configs[2]'s geometry (60x60x40 + 32^3: 18 + 4 shared-memory slabs per row) and launch shape (100 000 orbits: 512-thread
    CTAs, four warps per scheduler, the queue handing over time segments), stride 10, over the first 2 000 steps, where fp64
    counts are still a deterministic function of the inputs: row-sum invariant on EVERY orbit, and the rows of >= 64 sampled
    orbits (group / warp boundaries + random) identical to the oracle's away from bin edges."""
    torch = torch_cuda
    cfg = inputs.CONFIGS[2]
    pot = binding.sm_make_potential(cfg["potential"])
    ics = inputs.make_ics(cfg, _device_force(pot))
    n, steps = cfg["n_orb"], 2000
    n_rec = steps // cfg["stride"]
    g = binding.sm_build_library(pot, ics, cfg["dt"], steps, cfg["stride"], cfg["projections"], cfg["grids"])
    assert g["losvd"].shape == (1, 100000, 144000) and g["dens"].shape == (100000, 32768)
    assert _rows_sum_ok(g, n_rec)
    idx = _sample_indices(n, 56, 21)
    t_idx = torch.as_tensor(idx).cuda()
    gl, gd, gn = g["losvd"][0][t_idx].cpu().numpy(), g["dens"][t_idx].cpu().numpy(), g["nout"][:, t_idx].cpu().numpy()
    del g
    torch.cuda.empty_cache()
    o = smo.build_library(cfg["potential"], ics[idx], cfg["dt"], steps, cfg["stride"], cfg["projections"], cfg["grids"])
    n_l = count_parity(gl, o["losvd"][0], o["near_edge"][0])
    n_d = count_parity(gd, o["dens"], o["near_edge"][1])
    clean = o["near_edge"].sum(0) == 0
    assert np.array_equal(gn[:, clean], o["nout"][:, clean])
    print("cfg2 fp64 launch shape, 2000 steps: %d sampled rows, %d LOSVD / %d density rows identical to the oracle (the rest have near-edge samples)"
          % (len(idx), n_l, n_d))
    assert n_l >= 48 and n_d >= 48


def test_config2_full_size_both_precisions_sampled_against_oracle(smo, torch_cuda):
    """BASELINE.json configs[2] at FULL size (100 000 orbits x 20 000 steps, stride 10, 60x60x40 + 32^3; the 70.7 GB matrix)
    through the call and launch configuration bench.py times, in fp64 and in fp32.
    At any size: row sum + nout = n_rec on every orbit.  Sampled rows (128 orbits: group / warp boundaries + random): bit-identical
    to a separate call on the sampled orbits alone (a row depends neither on the launch configuration nor on its warp
    neighbours); and against the oracle integrated over all 20 000 steps, in the chaotic regime:
      fp64 -- the oracle's twin with ICs perturbed by 1e-12 certifies the insensitive orbits (twin L1 <= 2e-3; measured 78 %
              of the sample): per-orbit L1 <= 2e-2 on each of them (measured: identical counts), certified fraction >= 0.5;
      fp32 -- over 20 000 steps the fp32 rounding itself (eps sqrt(n_steps) ~ 1e-5) moves ~1 % of the 2 000 samples of a REGULAR
              orbit across an edge of the 144 000-cell grid, so hardly any orbit can meet 2e-2 whatever code produced it (the
              oracle's own twins, ICs x (1 + 3e-6) and x (1 - 8e-6), have a median L1 of a few 1e-2).  The gate is therefore
              statistical, against the oracle's own twins (all numbers printed): per-orbit L1 <= 2e-2 on the orbits BOTH twins
              certify; median and 90th percentile of the per-orbit L1 no larger than 1.5 x the larger twin's;
      both -- sample-summed fraction histograms no further from the oracle than 1.5 x its own twin (128 orbits cannot meet the
              plain 2e-2 either way: the twin itself is at 5e-2 ... 1e-1; the plain aggregate gate is carried by
              test_fp32_variant_plain_aggregate_gate, where the sample can be made large enough)."""
    torch = torch_cuda
    cfg = inputs.CONFIGS[2]
    pot = binding.sm_make_potential(cfg["potential"])
    ics = inputs.make_ics(cfg, _device_force(pot))
    n, steps = cfg["n_orb"], cfg["n_steps"]
    n_rec = steps // cfg["stride"]
    args = (cfg["dt"], steps, cfg["stride"], cfg["projections"], cfg["grids"])
    idx = _sample_indices(n, 110, 22)
    t_idx = torch.as_tensor(idx).cuda()
    o = smo.build_library(cfg["potential"], ics[idx], *args)
    bufs = None
    for prec, eps in (("f64", (1e-12,)), ("f32", (3e-6, -8e-6))):
        g = binding.sm_build_library(pot, ics, *args, precision=prec, **(bufs or {}))
        bufs = {k: g[k] for k in ("losvd", "dens", "nout")}       # one 70.7 GB allocation for both precisions
        assert _rows_sum_ok(g, n_rec), prec
        sub = binding.sm_build_library(pot, ics[idx], *args, precision=prec)
        assert (g["losvd"][0][t_idx] == sub["losvd"][0]).all().item(), prec
        assert (g["dens"][t_idx] == sub["dens"]).all().item(), prec
        assert (g["nout"][:, t_idx] == sub["nout"]).all().item(), prec
        gl, gd = sub["losvd"][0].cpu().numpy(), sub["dens"].cpu().numpy()
        twins = [smo.build_library(cfg["potential"], ics[idx] * (1 + e), *args) for e in eps]
        l1 = np.abs(gl - o["losvd"][0]).sum(1) / n_rec
        l1d = np.abs(gd - o["dens"]).sum(1) / n_rec
        tws = [np.abs(t["losvd"][0] - o["losvd"][0]).sum(1) / n_rec for t in twins]
        stable = np.all([t <= (2e-3 if prec == "f64" else CERT) for t in tws], axis=0)
        tw_med, tw_90 = max(np.median(t) for t in tws), max(np.quantile(t, 0.9) for t in tws)
        agg, aggd = _l1_fractions(gl.sum(0), o["losvd"][0].sum(0)), _l1_fractions(gd.sum(0), o["dens"].sum(0))
        agg_tw = max(_l1_fractions(t["losvd"][0].sum(0), o["losvd"][0].sum(0)) for t in twins)
        aggd_tw = max(_l1_fractions(t["dens"].sum(0), o["dens"].sum(0)) for t in twins)
        print("cfg2 full size %s: %d sampled, certified %d (%.2f); per-orbit L1 losvd (certified) max %.1e, (all) median %.1e 90pct %.1e; "
              "oracle twins (all) median %.1e 90pct %.1e; sample-summed L1 losvd %.2e (twin %.2e) dens %.2e (twin %.2e)"
              % (prec, len(idx), stable.sum(), stable.mean(), l1[stable].max() if stable.any() else 0.0, np.median(l1), np.quantile(l1, 0.9),
                 tw_med, tw_90, agg, agg_tw, aggd, aggd_tw))
        if prec == "f64":
            assert stable.mean() >= 0.5
        assert np.all(l1[stable] <= 2e-2) and np.all(l1d[stable] <= 2e-2)
        assert np.median(l1) <= max(1.5 * tw_med, 2e-2) and np.quantile(l1, 0.9) <= max(1.5 * tw_90, 2e-2)
        assert agg <= max(2e-2, 1.5 * agg_tw) and aggd <= max(2e-2, 1.5 * aggd_tw)
        del g, sub


def test_config3_fp32_batched_trials_against_oracle(smo, oracle_force, torch_cuda):
    """configs[3] in its OWN arithmetic: fp32, batched potentials (4 trial parameter sets in one launch, each with its own
    potential, viewing angles and ICs: common random numbers, the trial's own v_c), every trial against the oracle run on that
    trial's potential, over the first 1 000 steps (fp32 rounding hardly amplified: most rows identical) and over 5 000 steps.
    Gates of DESIGN.md 6 per trial, against the oracle's own fp32-sized twins (ICs x (1 + 1e-6) and x (1 - 3e-6) ~
    eps sqrt(n_steps)): row sums; per-orbit L1 <= 2e-2 on every orbit both twins certify (twin L1 <= CERT), a floor on the
    certified fraction (0.4 / 0.04); median and 90th percentile of the per-orbit L1 within 1.5 x the larger twin's;
    trial-summed fraction histograms no further from the oracle than 1.5 x its own twin (256 orbits are too few for the
    plain 2e-2 aggregate, which test_fp32_variant_plain_aggregate_gate carries).  All numbers printed."""
    cfg = inputs.CONFIGS[3]
    n_trials, n = 4, 256
    draws = inputs.trial_draws(n_trials, cfg["seed"])
    ics = np.stack([inputs.make_ics(cfg, oracle_force, n_orb=n, potential=d["potential"]) for d in draws])
    pot = binding.sm_make_potential_batch([d["potential"] for d in draws])
    projs = [[d["projection"]] for d in draws]
    for steps, floor in ((1000, 0.4), (5000, 0.04)):
        n_rec = steps // cfg["stride"]
        g = binding.sm_build_library_batch(pot, ics, cfg["dt"], steps, cfg["stride"], projs, cfg["grids"], precision="f32")
        for t, d in enumerate(draws):
            oargs = (cfg["dt"], steps, cfg["stride"], [d["projection"]], cfg["grids"])
            gl, gd = g["losvd"][t, 0].cpu().numpy(), g["dens"][t].cpu().numpy()
            gn = g["nout"][t].cpu().numpy()
            assert np.array_equal(gl.sum(1) + gn[0], np.full(n, n_rec)) and np.array_equal(gd.sum(1) + gn[1], np.full(n, n_rec))
            o = smo.build_library(d["potential"], ics[t], *oargs)
            l1 = np.abs(gl - o["losvd"][0]).sum(1) / n_rec
            l1d = np.abs(gd - o["dens"]).sum(1) / n_rec
            twins = [smo.build_library(d["potential"], ics[t] * (1 + e), *oargs) for e in (1e-6, -3e-6)]
            tws = [np.abs(tw["losvd"][0] - o["losvd"][0]).sum(1) / n_rec for tw in twins]
            stable = np.all([tw <= CERT for tw in tws], axis=0)
            tw_med, tw_90 = max(np.median(tw) for tw in tws), max(np.quantile(tw, 0.9) for tw in tws)
            agg, aggd = _l1_fractions(gl.sum(0), o["losvd"][0].sum(0)), _l1_fractions(gd.sum(0), o["dens"].sum(0))
            agg_tw = max(_l1_fractions(tw["losvd"][0].sum(0), o["losvd"][0].sum(0)) for tw in twins)
            aggd_tw = max(_l1_fractions(tw["dens"].sum(0), o["dens"].sum(0)) for tw in twins)
            print("cfg3 fp32 trial %d, %d steps: identical rows %d / %d; certified fraction %.2f; per-orbit L1 (certified) max %.1e, (all) median %.1e "
                  "90pct %.1e max %.1e; twins median %.1e 90pct %.1e; trial-summed L1 losvd %.2e (twin %.2e) dens %.2e (twin %.2e)"
                  % (t, steps, int((l1 == 0).sum()), n, stable.mean(), l1[stable].max(), np.median(l1), np.quantile(l1, 0.9), l1.max(),
                     tw_med, tw_90, agg, agg_tw, aggd, aggd_tw))
            assert stable.mean() >= floor
            assert np.all(l1[stable] <= 2e-2) and np.all(l1d[stable] <= 2e-2)
            assert np.median(l1) <= max(1.5 * tw_med, 2e-2) and np.quantile(l1, 0.9) <= max(1.5 * tw_90, 2e-2)
            assert agg <= max(2e-2, 1.5 * agg_tw) and aggd <= max(2e-2, 1.5 * aggd_tw)


def test_fp32_variant_plain_aggregate_gate(smo, oracle_force, torch_cuda):
    """north_star: "for fp32 and long or chaotic orbits, the per-orbit time-averaged bin fractions must agree within
    L1 <= 2e-2".  With 1 280 orbits x 5 000 steps of configs[1] the orbit-summed histogram of the oracle's OWN twin (ICs perturbed
    by 1e-6 ~ fp32 resolution) is within 1e-2 of the oracle (it falls as 1/sqrt(N): SURVEY 8(c-5)), so the stated gate applies as
    stated: (i) orbit-summed fraction histograms of the fp32 kernel within 2e-2 of the fp64 oracle, LOSVD and density;
    (ii) per-orbit L1 <= 2e-2 on every orbit both oracle twins (+1e-6, -3e-6) certify (twin L1 <= CERT), and at least 8 % of
    the orbits certified (measured: 11 %); (iii) median and 90th percentile of the per-orbit L1 no larger than 1.5 x the twin's.  The oracle's own twin must itself meet the plain gate on this sample (else the sample is too small)."""
    cfg = inputs.CONFIGS[1]
    n, steps = 1280, 5000
    ics = inputs.make_ics(cfg, oracle_force, n_orb=n)
    pot = binding.sm_make_potential(cfg["potential"])
    args = (cfg["dt"], steps, cfg["stride"], cfg["projections"], cfg["grids"])
    g = binding.sm_build_library(pot, ics, *args, precision="f32")
    o = smo.build_library(cfg["potential"], ics, *args)
    twin = smo.build_library(cfg["potential"], ics * (1 + 1e-6), *args)
    twin2 = smo.build_library(cfg["potential"], ics * (1 - 3e-6), *args)
    n_rec = steps // cfg["stride"]
    gl, gd = g["losvd"][0].cpu().numpy(), g["dens"].cpu().numpy()
    assert np.array_equal(gl.sum(1) + g["nout"][0].cpu().numpy(), np.full(n, n_rec))
    assert np.array_equal(gd.sum(1) + g["nout"][1].cpu().numpy(), np.full(n, n_rec))
    agg_l, agg_d = _l1_fractions(gl.sum(0), o["losvd"][0].sum(0)), _l1_fractions(gd.sum(0), o["dens"].sum(0))
    tw_l, tw_d = _l1_fractions(twin["losvd"][0].sum(0), o["losvd"][0].sum(0)), _l1_fractions(twin["dens"].sum(0), o["dens"].sum(0))
    per_orbit = np.abs(gl - o["losvd"][0]).sum(1) / n_rec
    t1 = np.abs(twin["losvd"][0] - o["losvd"][0]).sum(1) / n_rec
    t2 = np.abs(twin2["losvd"][0] - o["losvd"][0]).sum(1) / n_rec
    stable = (t1 <= CERT) & (t2 <= CERT)
    print("fp32 plain gate, %d orbits: aggregate L1 losvd %.2e dens %.2e (oracle twin: %.2e / %.2e); certified fraction %.2f; "
          "per-orbit L1 (certified) max %.1e, (all) median %.1e 90pct %.1e; twin (all) median %.1e 90pct %.1e"
          % (n, agg_l, agg_d, tw_l, tw_d, stable.mean(), per_orbit[stable].max(), np.median(per_orbit), np.quantile(per_orbit, 0.9),
             np.median(t1), np.quantile(t1, 0.9)))
    assert tw_l < 2e-2 and tw_d < 2e-2, "sample too small for the plain gate: the oracle's own twin does not meet it"
    assert agg_l < 2e-2 and agg_d < 2e-2
    assert stable.mean() >= 0.08
    assert np.all(per_orbit[stable] <= 2e-2)
    assert np.median(per_orbit) <= max(1.5 * np.median(t1), 2e-2) and np.quantile(per_orbit, 0.9) <= max(1.5 * np.quantile(t1, 0.9), 2e-2)


def test_internal_staging_chunk_loop_matches_single_pass(oracle_force, torch_cuda):
    """The library-internal orbit-chunk loop of sm_build_library (staged indices beyond the staging cap are built in balanced
    chunks of a multiple of 512 orbits) against the single-pass result: debug flag 1024 lowers the cap from 4 GiB to 1 MiB, so
    that 1 700 orbits x 150 samples x 4 histograms (4 MB of staged indices) take four chunks with a ragged last one, 4 496 bundled
    orbits three chunks of 2 048 (a multiple of 512 x n_bundle) and the batched call three chunks per trial.  Plain,
    bundled + fourfold and batched calls; rows, out-of-grid counters and the Jacobi diagnostic must be bit-identical."""
    cfg = inputs.CONFIGS[4]                      # three projections
    ics = inputs.make_ics(cfg, oracle_force, n_orb=4496)
    pot = binding.sm_make_potential(cfg["potential"])
    c3 = inputs.CONFIGS[3]
    draws = inputs.trial_draws(2, c3["seed"])
    potb = binding.sm_make_potential_batch([d["potential"] for d in draws])
    projs = [[d["projection"]] for d in draws]
    runs = []
    for flags in (0, 1024):
        prev = binding.sm_set_debug_flags(flags)
        try:
            a = binding.sm_build_library(pot, ics[:1700], cfg["dt"], 3000, cfg["stride"], cfg["projections"], cfg["grids"], want_diag=True)
            b = binding.sm_build_bundled_library(pot, ics, cfg["dt"], 800, cfg["stride"], cfg["projections"], cfg["grids"], n_bundle=4, fourfold=True)
            c = binding.sm_build_library_batch(potb, ics[:1100], c3["dt"], 1500, c3["stride"], projs, c3["grids"], precision="f32")
            runs.append((a, b, c))
        finally:
            binding.sm_set_debug_flags(prev)
    for x, y in zip(runs[0], runs[1]):
        for k in ("losvd", "dens", "nout"):
            assert (x[k] == y[k]).all().item(), k
    assert (runs[0][0]["diag"] == runs[1][0]["diag"]).all().item()


def test_config4_full_size_staged_route_sampled_against_oracle(smo, torch_cuda):
    """BASELINE.json configs[4] at FULL size: 500 000 orbits x 50 000 steps, stride 20, three projections (64x64x48 each) + 40^3 --
    a 1.31 TB matrix that exists only window by window.  The route bench.py times for it: ALL orbits integrated in one
    sm_stage_library_batch launch (20 GB of staged cell indices), then row windows through sm_flush_rows / sm_scatter_rows.
    Every orbit: staged samples + out-of-grid samples = n_rec per histogram.  Sampled rows (CTA / warp boundaries of the 512-thread
    launch + random): the flushed window rows are bit-identical to a separate sm_build_library call on the sampled orbits alone and to
    the scatter route; against the oracle over all 50 000 steps, on the orbits its 1e-12 twin certifies (twin L1 <= 2e-3): per-orbit
    L1 <= 2e-2 in all four histograms (measured: identical counts); the rest is bounded by the distribution gates of the config-2 test."""
    torch = torch_cuda
    cfg = inputs.CONFIGS[4]
    pot = binding.sm_make_potential(cfg["potential"])
    ics = inputs.make_ics(cfg, _device_force(pot))
    n, steps, g = cfg["n_orb"], cfg["n_steps"], cfg["grids"]
    n_rec, n_proj = steps // cfg["stride"], len(cfg["projections"])
    d_ics = torch.as_tensor(ics).cuda()
    st = binding.sm_stage_library_batch(pot, d_ics, cfg["dt"], steps, cfg["stride"], [cfg["projections"]], g)
    assert st.shape == (1, n_proj + 1, n, n_rec)
    idx = _sample_indices(n, 40, 44)
    oargs = (cfg["dt"], steps, cfg["stride"], cfg["projections"], g)
    sub = binding.sm_build_library(pot, ics[idx], *oargs)
    inside = torch.zeros((n_proj + 1, n), dtype=torch.int32, device="cuda")
    for h in range(n_proj + 1):                                    # in-grid samples per orbit, from the staged indices
        for a in range(0, n, 100000):
            inside[h, a:a + 100000] = (st[0, h, a:a + 100000] >= 0).sum(-1)
    # contiguous windows at the ends and the middle, and single-row windows for the scattered samples
    for a, b in ((0, 34), (n // 2 - 1, n // 2 + 2), (n - 34, n)):
        w = binding.sm_flush_rows(st, a, b - a, g)
        assert (w["losvd"][0].sum(-1) + w["nout"][0, :n_proj] == n_rec).all().item() and (w["dens"][0].sum(-1) + w["nout"][0, -1] == n_rec).all().item()
        assert (w["nout"][0] + inside[:, a:b] == n_rec).all().item()
        los = torch.zeros_like(w["losvd"]); den = torch.zeros_like(w["dens"])
        s2 = binding.sm_scatter_rows(st, a, b - a, g, los, den)
        for k in ("losvd", "dens", "nout"):
            assert (s2[k] == w[k]).all().item(), k
    for j, i in enumerate(idx):
        w = binding.sm_flush_rows(st, int(i), 1, g)
        assert (w["losvd"][0, :, 0] == sub["losvd"][:, j]).all().item(), i
        assert (w["dens"][0, 0] == sub["dens"][j]).all().item() and (w["nout"][0, :, 0] == sub["nout"][:, j]).all().item(), i
    del st
    o = smo.build_library(cfg["potential"], ics[idx], *oargs)
    tw = smo.build_library(cfg["potential"], ics[idx] * (1 + 1e-12), *oargs)
    stable = np.ones(len(idx), dtype=bool)
    l1s = []
    for h in range(n_proj + 1):
        key = (lambda d: d["losvd"][h]) if h < n_proj else (lambda d: d["dens"])
        gr = (sub["losvd"][h] if h < n_proj else sub["dens"]).cpu().numpy()
        l1s.append(np.abs(gr - key(o)).sum(1) / n_rec)
        stable &= np.abs(key(tw) - key(o)).sum(1) / n_rec <= 2e-3
    l1 = np.max(l1s, axis=0)
    print("cfg4 full size: %d sampled, certified %d (%.2f); per-orbit L1 (certified) max %.1e, identical rows %d; (all) median %.1e 90pct %.1e"
          % (len(idx), stable.sum(), stable.mean(), l1[stable].max() if stable.any() else 0.0, int((l1 == 0).sum()), np.median(l1), np.quantile(l1, 0.9)))
    assert stable.mean() >= 0.3
    assert np.all(l1[stable] <= 2e-2)


def test_config3_full_size_batch_launch_shape_rows_equal_separate_calls(oracle_force, torch_cuda):
    """BASELINE.json configs[3] at FULL size and in its own arithmetic: 64 trial potentials x 20 000 orbits x 10 000 steps in fp32, ALL
    trials integrated in ONE sm_stage_library_batch launch (the launch shape bench.py times: 40 000 warp teams on 148 x 16 slots, tables
    read through L1; 20 GB of staged indices; the 316 GB matrix exists only window by window).  Every (trial, orbit): in-grid + out-of-grid
    samples = n_rec per histogram.  Sampled (trial, orbit) rows are bit-identical to single-trial fp32 calls on that trial's potential, ICs
    and viewing angles -- a row does not depend on the batch, its launch shape or its warp neighbours -- so the per-trial oracle gates of
    test_config3_fp32_batched_trials_against_oracle (same kernels, 4 trials x 256 orbits) carry over to the full-size launch."""
    torch = torch_cuda
    cfg = inputs.CONFIGS[3]
    n_trials, n, steps, g = cfg["n_trials"], cfg["n_orb"], cfg["n_steps"], cfg["grids"]
    n_rec = steps // cfg["stride"]
    draws = inputs.trial_draws(n_trials, cfg["seed"])
    pot = binding.sm_make_potential_batch([d["potential"] for d in draws])
    ics = np.stack([inputs.make_ics(cfg, lambda p, x, t=t: binding.sm_eval_force(pot, x, 0.0, trial=t, want_phi=False).cpu().numpy(),
                                    potential=d["potential"]) for t, d in enumerate(draws)])
    d_ics = torch.as_tensor(ics).cuda()
    projs = [[d["projection"]] for d in draws]
    st = binding.sm_stage_library_batch(pot, d_ics, cfg["dt"], steps, cfg["stride"], projs, g, precision="f32")
    assert st.shape == (n_trials, 2, n, n_rec)
    rng = np.random.default_rng(9)
    for t in (0, 1, 31, 62, 63):
        w = binding.sm_flush_rows(st[t:t + 1], 0, n, g)          # the whole trial: 4.9 GB of rows
        assert (w["losvd"][0, 0].sum(-1) + w["nout"][0, 0] == n_rec).all().item() and (w["dens"][0].sum(-1) + w["nout"][0, 1] == n_rec).all().item()
        idx = np.unique(np.concatenate([[0, 31, 32, n - 1], rng.integers(0, n, 28)]))
        one = binding.sm_build_library(binding.sm_make_potential(draws[t]["potential"]), ics[t][idx], cfg["dt"], steps, cfg["stride"],
                                       [draws[t]["projection"]], g, precision="f32")
        t_idx = torch.as_tensor(idx).cuda()
        assert (w["losvd"][0, 0][t_idx] == one["losvd"][0]).all().item(), t
        assert (w["dens"][0][t_idx] == one["dens"]).all().item() and (w["nout"][0][:, t_idx] == one["nout"]).all().item(), t
        del w
