"""GPU parity tests (-m gpu): batched-potential mode, the fp32 variant, and edge cases."""
import numpy as np
import pytest

from paper_2607_00117_b200 import binding, inputs

from gpu_util import count_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    return torch


def _trial_ics(cfg, draws, force_fn, n_orb):
    return np.stack([inputs.make_ics(cfg, force_fn, n_orb=n_orb, potential=d["potential"]) for d in draws])


def test_batch_fp64_matches_oracle_per_trial(smo, oracle_force, torch_cuda):
    """Config-3 recipe (BASELINE.json configs[3]) with 3 trials x 96 orbits x 600 steps, run in fp64 so that
    counts must be identical; per-trial ICs (common random numbers, own v_c)."""
    cfg = inputs.CONFIGS[3]
    draws = inputs.trial_draws(3, cfg["seed"])
    ics = _trial_ics(cfg, draws, oracle_force, 96)
    pot = binding.sm_make_potential_batch([d["potential"] for d in draws])
    projs = [[d["projection"]] for d in draws]
    g = binding.sm_build_library_batch(pot, ics, cfg["dt"], 600, cfg["stride"], projs, cfg["grids"], precision="f64")
    for t, d in enumerate(draws):
        o = smo.build_library(d["potential"], ics[t], cfg["dt"], 600, cfg["stride"], [d["projection"]], cfg["grids"])
        assert count_parity(g["losvd"][t, 0].cpu().numpy(), o["losvd"][0], o["near_edge"][0]) > 80
        assert count_parity(g["dens"][t].cpu().numpy(), o["dens"], o["near_edge"][1]) > 80
    # a sub-range of trials with shared ICs reproduces the corresponding block
    sub = binding.sm_build_library_batch(pot, ics[1], cfg["dt"], 600, cfg["stride"], projs[1:3], cfg["grids"],
                                         precision="f64", trial0=1, n_trials=2)
    assert (sub["losvd"][0] == g["losvd"][1]).all().item()
    # trial index of the test hooks
    pts = np.random.default_rng(0).normal(size=(500, 3)) * [5, 5, 1]
    F = binding.sm_eval_force(pot, pts, 0.01, trial=2, want_phi=False).cpu().numpy()
    Fo = smo.eval_force(draws[2]["potential"], pts, 0.01, want_phi=False)
    assert np.max(np.linalg.norm(F - Fo, axis=1) / np.linalg.norm(Fo, axis=1)) < 1e-14


# (the fp32 statistical gates live in test_gpu_all_configs.py::test_fp32_variant_plain_aggregate_gate: 1 280 orbits, plain 2e-2)


def test_fp32_trajectories_short(smo, oracle_force, torch_cuda):
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=128)
    pot = binding.sm_make_potential(cfg["potential"])
    g = binding.sm_integrate_trajectories(pot, ics, cfg["dt"], 100, 100, precision="f32").cpu().numpy()
    o = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], 100, 100)
    rel = np.linalg.norm(g[0, :, :3] - o[0, :, :3], axis=1) / np.linalg.norm(o[0, :, :3], axis=1)
    assert np.median(rel) < 2e-5 and rel.max() < 2e-3


def test_edge_cases(smo, torch_cuda):
    torch = torch_cuda
    cfg = inputs.CONFIGS[0]
    pot = binding.sm_make_potential(cfg["potential"])
    ics = inputs.plummer_ics(37, 5)
    # stride not dividing n_steps: trailing steps integrated, not recorded
    g = binding.sm_build_library(pot, ics, 0.01, 103, 10, cfg["projections"], cfg["grids"])
    o = smo.build_library(cfg["potential"], ics, 0.01, 103, 10, cfg["projections"], cfg["grids"])
    assert count_parity(g["dens"].cpu().numpy(), o["dens"], o["near_edge"][1]) >= 30
    assert np.array_equal(g["dens"].sum(1).cpu().numpy() + g["nout"][1].cpu().numpy(), np.full(37, 10))
    # stride > n_steps: no recorded sample, rows are zero
    z = binding.sm_build_library(pot, ics, 0.01, 5, 10, cfg["projections"], cfg["grids"])
    assert z["losvd"].abs().sum().item() == 0 and z["dens"].abs().sum().item() == 0 and z["nout"].abs().sum().item() == 0
    # empty input
    e = binding.sm_build_library(pot, torch.empty((0, 6), dtype=torch.float64, device="cuda"), 0.01, 10, 1, cfg["projections"], cfg["grids"])
    assert e["losvd"].shape == (1, 0, 1500)
    # a single orbit, odd-sized grids (scalar store path), all samples out of range
    odd = dict(cfg["grids"], nx=7, ny=3, nv=5, dx=3, dy=5, dz=7)
    g1 = binding.sm_build_library(pot, ics[:1], 0.01, 50, 1, cfg["projections"], odd)
    o1 = smo.build_library(cfg["potential"], ics[:1], 0.01, 50, 1, cfg["projections"], odd)
    assert np.array_equal(g1["losvd"].cpu().numpy(), o1["losvd"]) or o1["near_edge"].sum() > 0
    far = dict(cfg["grids"], x0=100.0, x1=101.0, bx0=100.0, bx1=101.0)
    gf = binding.sm_build_library(pot, ics, 0.01, 20, 1, cfg["projections"], far)
    assert gf["losvd"].sum().item() == 0 and (gf["nout"] == 20).all().item()
    # non-finite state: counted as out of range, flagged in diag
    bad = ics.copy(); bad[3, 0] = np.nan
    gb = binding.sm_build_library(pot, bad, 0.01, 20, 1, cfg["projections"], cfg["grids"], want_diag=True)
    assert gb["nout"][:, 3].cpu().numpy().tolist() == [20, 20] and gb["diag"][3, 1].item() == 1.0
    # invalid arguments launch nothing and report an error
    for kw in (dict(dt=-0.01), dict(n_steps=0), dict(stride=0)):
        args = dict(dt=0.01, n_steps=10, stride=1); args.update(kw)
        with pytest.raises(binding.SchwarmaxError):
            binding.sm_build_library(pot, ics, args["dt"], args["n_steps"], args["stride"], cfg["projections"], cfg["grids"])
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_build_library(pot, ics, 0.01, 10, 1, cfg["projections"], dict(cfg["grids"], x1=-5.0))
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_build_library(pot, ics, 0.01, 10, 1, cfg["projections"] * 5, cfg["grids"])


def test_chunked_staging_matches_single_pass(torch_cuda, oracle_force):
    """Large n_rec x n_orb forces the internal orbit chunking (staging buffer cap); compare two chunkings by
    calling on sub-ranges through pointer offsets, as configs 3-4 are streamed."""
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=600)
    pot = binding.sm_make_potential(cfg["potential"])
    import torch
    d_ics = torch.as_tensor(ics).cuda()
    full = binding.sm_build_library(pot, d_ics, cfg["dt"], 300, 1, cfg["projections"], cfg["grids"])
    a = binding.sm_build_library(pot, d_ics[:256].contiguous(), cfg["dt"], 300, 1, cfg["projections"], cfg["grids"])
    b = binding.sm_build_library(pot, d_ics[256:].contiguous(), cfg["dt"], 300, 1, cfg["projections"], cfg["grids"])
    assert (full["losvd"][0, :256] == a["losvd"][0]).all().item() and (full["losvd"][0, 256:] == b["losvd"][0]).all().item()
    assert (full["dens"][256:] == b["dens"]).all().item()


def test_stage_then_flush_windows_equal_build_library(torch_cuda, oracle_force):
    """sm_stage_library_batch + sm_flush_rows (row windows, trial sub-ranges) must reproduce sm_build_library(_batch)
    bit for bit: it is the same path with the staged library owned by the caller."""
    torch = torch_cuda
    cfg = inputs.CONFIGS[4]                      # three projections
    ics = inputs.make_ics(cfg, oracle_force, n_orb=150)
    pot = binding.sm_make_potential(cfg["potential"])
    ref = binding.sm_build_library(pot, ics, cfg["dt"], 600, cfg["stride"], cfg["projections"], cfg["grids"])
    st = binding.sm_stage_library_batch(pot, ics, cfg["dt"], 600, cfg["stride"], [cfg["projections"]], cfg["grids"])
    assert st.shape == (1, 4, 150, 30)
    for a, b in ((0, 64), (64, 150), (149, 150)):
        w = binding.sm_flush_rows(st, a, b - a, cfg["grids"])
        assert (w["losvd"][0] == ref["losvd"][:, a:b]).all().item()
        assert (w["dens"][0] == ref["dens"][a:b]).all().item()
        assert (w["nout"][0] == ref["nout"][:, a:b]).all().item()
    # batched, fp32, per-trial ICs; flush one trial sub-range
    c3 = inputs.CONFIGS[3]
    draws = inputs.trial_draws(3, c3["seed"])
    ics3 = _trial_ics(c3, draws, oracle_force, 70)
    potb = binding.sm_make_potential_batch([d["potential"] for d in draws])
    projs = [[d["projection"]] for d in draws]
    refb = binding.sm_build_library_batch(potb, ics3, c3["dt"], 400, c3["stride"], projs, c3["grids"], precision="f32")
    stb = binding.sm_stage_library_batch(potb, ics3, c3["dt"], 400, c3["stride"], projs, c3["grids"], precision="f32")
    wb = binding.sm_flush_rows(stb[1:3].contiguous(), 10, 50, c3["grids"])
    assert (wb["losvd"] == refb["losvd"][1:3, :, 10:60]).all().item()
    assert (wb["dens"] == refb["dens"][1:3, 10:60]).all().item()
    assert (wb["nout"] == refb["nout"][1:3, :, 10:60]).all().item()
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_flush_rows(st, 100, 51, cfg["grids"])


def test_dma_zeroed_scatter_flush_equals_dense_flush(torch_cuda, oracle_force):
    """Outputs of at least 64 MB whose rows are sparse are zeroed by the copy engines on a library-owned side stream while
    the integrator runs, and only the non-zero cells are scattered afterwards; debug flag 4096 switches that off
    (dense slab flush after the integrator).  Both must give identical rows -- plain, batched and with the internal chunk loop,
    on rows that were full of garbage before the call -- and sm_scatter_rows into caller-zeroed rows must equal sm_flush_rows."""
    torch = torch_cuda
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=700)
    pot = binding.sm_make_potential(cfg["potential"])
    args = (cfg["dt"], 400, cfg["stride"], cfg["projections"], cfg["grids"])
    outs = []
    for flags in (0, 4096, 1024, 32768, 16):   # 32768: the store-loop fill in place of the bulk-copy-engine one; 16: orbits in the caller's order
        prev = binding.sm_set_debug_flags(flags)
        try:
            bufs = dict(losvd=torch.full((1, 700, 48000), 7.0, device="cuda"), dens=torch.full((700, 13824), -3.0, device="cuda"))
            a = binding.sm_build_library(pot, ics, *args, **bufs)
            b = binding.sm_build_library(pot, ics[:400], *args, precision="f32")
            torch.cuda.synchronize()
            outs.append((a, b))
        finally:
            binding.sm_set_debug_flags(prev)
    for o in outs[1:]:
        for x, y in zip(outs[0], o):
            for k in ("losvd", "dens", "nout"):
                assert (x[k] == y[k]).all().item(), k
    assert (outs[0][0]["losvd"][0].sum(1) + outs[0][0]["nout"][0] == 80).all().item()
    # the caller-zeroed two-call form, zeroing on a second stream as a streaming caller would
    st = binding.sm_stage_library_batch(pot, ics, *args[:3], [cfg["projections"]], cfg["grids"])
    ref = binding.sm_flush_rows(st, 100, 500, cfg["grids"])
    side = torch.cuda.Stream()
    los = torch.full((1, 1, 500, 48000), 5.0, device="cuda")
    den = torch.full((1, 500, 13824), 5.0, device="cuda")
    side.wait_stream(torch.cuda.current_stream())
    binding.sm_zero_async(los, stream=side)
    binding.sm_zero_async(den, stream=side)
    torch.cuda.current_stream().wait_stream(side)
    w = binding.sm_scatter_rows(st, 100, 500, cfg["grids"], los, den)
    for k in ("losvd", "dens", "nout"):
        assert (w[k] == ref[k]).all().item(), k


def test_orbit_order_does_not_change_results(torch_cuda, oracle_force):
    """The integrator hands its orbits to the warps in order of energy (order_*_kernel; debug flag 16 = the caller's order).  Orbits are
    independent, so rows, out-of-grid counts, Jacobi diagnostics and trajectories must be bit for bit the same either way: per-trial ICs
    in both precisions (every trial its own order), shared ICs, a count that is not a multiple of 32, the segment hand-over (flag 8)."""
    cfg = inputs.CONFIGS[3]
    draws = inputs.trial_draws(3, cfg["seed"])
    ics = _trial_ics(cfg, draws, oracle_force, 203)
    pot = binding.sm_make_potential_batch([d["potential"] for d in draws])
    projs = [[d["projection"]] for d in draws]
    cfg1 = inputs.CONFIGS[1]
    ics1 = inputs.make_ics(cfg1, oracle_force, n_orb=333)
    pot1 = binding.sm_make_potential(cfg1["potential"])

    def run(flags):
        prev = binding.sm_set_debug_flags(flags)
        try:
            out = [binding.sm_build_library_batch(pot, ics, cfg["dt"], 300, cfg["stride"], projs, cfg["grids"], precision=p) for p in ("f32", "f64")]
            out.append(binding.sm_build_library_batch(pot, ics[0], cfg["dt"], 300, cfg["stride"], projs, cfg["grids"], precision="f32"))
            out.append(binding.sm_build_library(pot1, ics1, cfg1["dt"], 400, cfg1["stride"], cfg1["projections"], cfg1["grids"], want_diag=True))
            traj = binding.sm_integrate_trajectories(pot1, ics1, cfg1["dt"], 200, 10)
            torch_cuda.cuda.synchronize()
            return out, traj
        finally:
            binding.sm_set_debug_flags(prev)
    ref, traj_ref = run(16)
    for flags in (0, 8):
        got, traj = run(flags)
        ref_f, traj_f = (ref, traj_ref) if flags == 0 else run(16 | 8)
        for a, b in zip(got, ref_f):
            for k in a:
                assert (a[k] == b[k]).all().item(), (flags, k)
        assert (traj == traj_f).all().item()
    assert (ref[0]["losvd"].sum(-1) + ref[0]["nout"][:, :1] == 60).all().item()


def test_zero_fill_kernels_zero_exactly_the_range(torch_cuda, oracle_force):
    """sm_zero_async with both fill kernels (bulk-copy engine: the default once an integrator launch has staged its table in shared
    memory; store loop: debug flag 32768): odd sizes, offsets that are not 16-byte aligned, sizes below and above one 16 KB block
    and above one block per SM; nothing outside the range is touched."""
    torch = torch_cuda
    cfg = inputs.CONFIGS[1]
    pot = binding.sm_make_potential(cfg["potential"])
    binding.sm_build_library(pot, inputs.make_ics(cfg, oracle_force, n_orb=64), cfg["dt"], 10, 5, cfg["projections"], cfg["grids"])
    for flags in (0, 32768):
        prev = binding.sm_set_debug_flags(flags)
        try:
            for off, n in ((0, 1), (1, 3), (3, 4099), (0, 4096), (5, 16384 * 148 // 4 + 7), (2, 3_000_001), (0, 0)):
                buf = torch.full((off + n + 9,), 3.0, device="cuda")
                if n:
                    binding.sm_zero_async(buf[off:off + n])
                torch.cuda.synchronize()
                assert (buf[off:off + n] == 0).all().item(), (flags, off, n)
                assert (buf[:off] == 3).all().item() and (buf[off + n:] == 3).all().item(), (flags, off, n)
        finally:
            binding.sm_set_debug_flags(prev)


def test_compact_rows_densify_to_the_dense_rows(smo, torch_cuda, oracle_force):
    """sm_flush_rows_compact: the non-zero cells of every row as (cell, count) pairs.  Scattering them into zero rows must give
    the rows of sm_flush_rows bit for bit (three projections, a row window, batched trials), the oracle's rows away from bin
    edges, total = the number of non-zero cells; a capacity that is too small is reported through total and writes nothing
    past the end."""
    torch = torch_cuda
    cfg = inputs.CONFIGS[4]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=150)
    pot = binding.sm_make_potential(cfg["potential"])
    g = cfg["grids"]
    nlos, nden = g["nx"] * g["ny"] * g["nv"], g["dx"] * g["dy"] * g["dz"]
    st = binding.sm_stage_library_batch(pot, ics, cfg["dt"], 2000, cfg["stride"], [cfg["projections"]], g)

    def densify(c, n_trials, n_hist, n_rows):
        rows = [[None] * n_hist for _ in range(n_trials)]
        total = int(c["total"].item())
        assert total == int(c["row_nnz"].sum().item()) and total <= c["cell"].numel()
        rid = torch.repeat_interleave(torch.arange(c["row_nnz"].numel(), device="cuda"), c["row_nnz"].view(-1).long())
        pos = torch.cat([torch.arange(s, s + n, device="cuda") for s, n in zip(c["row_start"].view(-1).tolist(), c["row_nnz"].view(-1).tolist())]) \
            if total else torch.empty(0, dtype=torch.long, device="cuda")
        assert torch.unique(pos).numel() == total                      # the runs do not overlap
        for t in range(n_trials):
            for h in range(n_hist):
                d = torch.zeros((n_rows, nlos if h < n_hist - 1 else nden), device="cuda")
                sel = (rid // n_rows) == t * n_hist + h
                d[rid[sel] % n_rows, c["cell"][pos[sel]].long()] = c["count"][pos[sel]]
                rows[t][h] = d
        return rows

    for a, n in ((0, 150), (37, 64)):
        ref = binding.sm_flush_rows(st, a, n, g)
        c = binding.sm_flush_rows_compact(st, a, n, g)
        d = densify(c, 1, 4, n)
        for p in range(3):
            assert (d[0][p] == ref["losvd"][0, p]).all().item()
        assert (d[0][3] == ref["dens"][0]).all().item()
        assert (c["nout"] == ref["nout"]).all().item()
        assert (c["count"][:int(c["total"].item())] > 0).all().item()
    o = smo.build_library(cfg["potential"], ics, cfg["dt"], 2000, cfg["stride"], cfg["projections"], g)
    assert count_parity(d[0][1][: 64].cpu().numpy(), o["losvd"][1][37:101], o["near_edge"][1][37:101]) >= 40
    # too small a capacity: total says what is needed, nothing is written past the end
    small = binding.sm_flush_rows_compact(st, 0, 150, g, capacity=1000)
    assert int(small["total"].item()) == int(binding.sm_flush_rows_compact(st, 0, 150, g)["total"].item()) > 1000
    # batched trials, fp32
    c3 = inputs.CONFIGS[3]
    draws = inputs.trial_draws(2, c3["seed"])
    ics3 = _trial_ics(c3, draws, oracle_force, 70)
    potb = binding.sm_make_potential_batch([d_["potential"] for d_ in draws])
    stb = binding.sm_stage_library_batch(potb, ics3, c3["dt"], 400, c3["stride"], [[d_["projection"]] for d_ in draws], c3["grids"], precision="f32")
    refb = binding.sm_flush_rows(stb, 5, 60, c3["grids"])
    gb = c3["grids"]
    nlos, nden = gb["nx"] * gb["ny"] * gb["nv"], gb["dx"] * gb["dy"] * gb["dz"]
    db = densify(binding.sm_flush_rows_compact(stb, 5, 60, gb), 2, 2, 60)
    for t in range(2):
        assert (db[t][0] == refb["losvd"][t, 0]).all().item() and (db[t][1] == refb["dens"][t]).all().item()
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_flush_rows_compact(st, 100, 51, g)


def test_symmetrised_bundles_match_oracle(smo, oracle_force, torch_cuda):
    """rows = bundles of n dithered realisations, every sample binned with the fourfold
    symmetrisation of PAPER.md:77-90 Table 1.  fp64 counts identical to the oracle on rows without near-edge samples;
    row sum + nout = n_bundle * 4 * n_rec in both precisions; bundling and symmetrisation also checked separately."""
    cfg = inputs.CONFIGS[4]                      # three projections
    ics = inputs.make_ics(cfg, oracle_force, n_orb=96)
    pot = binding.sm_make_potential(cfg["potential"])
    args = (cfg["dt"], 600, cfg["stride"], cfg["projections"], cfg["grids"])
    n_rec = 600 // cfg["stride"]
    for n_bundle, fourfold in ((4, True), (1, True), (3, False)):
        g = binding.sm_build_bundled_library(pot, ics, *args, n_bundle=n_bundle, fourfold=fourfold)
        o = smo.build_bundled_library(cfg["potential"], ics, *args, n_bundle=n_bundle, fourfold=fourfold)
        n_rows = 96 // n_bundle
        total = n_bundle * (4 if fourfold else 1) * n_rec
        for p in range(3):
            assert count_parity(g["losvd"][p].cpu().numpy(), o["losvd"][p], o["near_edge"][p]) >= 0.7 * n_rows
            assert np.array_equal(g["losvd"][p].sum(1).cpu().numpy() + g["nout"][p].cpu().numpy(), np.full(n_rows, total))
        assert count_parity(g["dens"].cpu().numpy(), o["dens"], o["near_edge"][3]) >= 0.7 * n_rows
        assert np.array_equal(g["dens"].sum(1).cpu().numpy() + g["nout"][3].cpu().numpy(), np.full(n_rows, total))
    # n_bundle = 1 without symmetrisation is sm_build_library
    plain = binding.sm_build_library(pot, ics, *args)
    same = binding.sm_build_bundled_library(pot, ics, *args, n_bundle=1, fourfold=False)
    for k in ("losvd", "dens", "nout"):
        assert (plain[k] == same[k]).all().item()
    # fp32 variant: invariants, and the segmented work queue reproduces the unsegmented rows
    a = binding.sm_build_bundled_library(pot, ics, *args, n_bundle=4, fourfold=True, precision="f32")
    prev = binding.sm_set_debug_flags(8)
    try:
        b = binding.sm_build_bundled_library(pot, ics, *args, n_bundle=4, fourfold=True, precision="f32")
    finally:
        binding.sm_set_debug_flags(prev)
    assert (a["losvd"] == b["losvd"]).all().item() and (a["dens"] == b["dens"]).all().item()
    assert np.array_equal(a["dens"].sum(1).cpu().numpy() + a["nout"][3].cpu().numpy(), np.full(24, 16 * n_rec))
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_build_bundled_library(pot, ics, *args, n_bundle=5, fourfold=True)


def test_aperture_regrouping_matches_oracle(smo, oracle_force, torch_cuda):
    """pixels regrouped on the fly into caller-defined apertures.  fp64 counts identical
    to the oracle (rows without near-edge samples), with and without symmetrised bundles; row sum + nout invariant; the
    identity map reproduces the pixel rows."""
    from test_oracle_bundles import aperture_map
    cfg = inputs.CONFIGS[4]
    g = cfg["grids"]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=90)
    pot = binding.sm_make_potential(cfg["potential"])
    ap, n_ap = aperture_map(g)
    args = (cfg["dt"], 600, cfg["stride"], cfg["projections"], g)
    n_rec = 600 // cfg["stride"]
    for n_bundle, fourfold in ((1, False), (3, True)):
        a = binding.sm_build_observable_library(pot, ics, *args, ap, n_ap, n_bundle=n_bundle, fourfold=fourfold)
        o = smo.build_observable_library(cfg["potential"], ics, *args, ap, n_ap, n_bundle=n_bundle, fourfold=fourfold)
        n_rows = 90 // n_bundle
        total = n_bundle * (4 if fourfold else 1) * n_rec
        assert a["losvd"].shape == (3, n_rows, n_ap * g["nv"])
        for p in range(3):
            assert count_parity(a["losvd"][p].cpu().numpy(), o["losvd"][p], o["near_edge"][p]) >= 0.7 * n_rows
            assert np.array_equal(a["losvd"][p].sum(1).cpu().numpy() + a["nout"][p].cpu().numpy(), np.full(n_rows, total))
        assert count_parity(a["dens"].cpu().numpy(), o["dens"], o["near_edge"][3]) >= 0.7 * n_rows
    ident = np.arange(g["nx"] * g["ny"], dtype=np.int32)
    same = binding.sm_build_observable_library(pot, ics, *args, ident, len(ident))
    plain = binding.sm_build_library(pot, ics, *args)
    for k in ("losvd", "dens", "nout"):
        assert (same[k] == plain[k]).all().item()
    f32 = binding.sm_build_observable_library(pot, ics, *args, ap, n_ap, n_bundle=2, fourfold=True, precision="f32")
    assert np.array_equal(f32["losvd"][0].sum(1).cpu().numpy() + f32["nout"][0].cpu().numpy(), np.full(45, 8 * n_rec))


def test_cylindrical_density_cells_match_oracle(smo, oracle_force, torch_cuda):
    """the 3-D mass matrix on cells uniform in (R, phi, z) (density_mode 1).  fp64 counts identical to the
    oracle on rows without near-edge samples, plain and with apertures + symmetrised bundles; invariants in fp32."""
    from test_oracle_bundles import aperture_map, cyl_grids
    cfg = inputs.CONFIGS[4]
    g = cyl_grids(cfg["grids"])
    ics = inputs.make_ics(cfg, oracle_force, n_orb=90)
    pot = binding.sm_make_potential(cfg["potential"])
    ap, n_ap = aperture_map(g)
    args = (cfg["dt"], 600, cfg["stride"], cfg["projections"], g)
    n_rec = 600 // cfg["stride"]
    for amap, na, n_bundle, fourfold in ((None, 0, 1, False), (ap, n_ap, 3, True)):
        a = binding.sm_build_observable_library(pot, ics, *args, amap, na, n_bundle=n_bundle, fourfold=fourfold, density_mode=1)
        o = smo.build_observable_library(cfg["potential"], ics, *args, amap, na, n_bundle=n_bundle, fourfold=fourfold, density_mode=1)
        n_rows = 90 // n_bundle
        total = n_bundle * (4 if fourfold else 1) * n_rec
        assert count_parity(a["dens"].cpu().numpy(), o["dens"], o["near_edge"][3]) >= 0.7 * n_rows
        assert np.array_equal(a["dens"].sum(1).cpu().numpy() + a["nout"][3].cpu().numpy(), np.full(n_rows, total))
        assert count_parity(a["losvd"][1].cpu().numpy(), o["losvd"][1], o["near_edge"][1]) >= 0.7 * n_rows
    f32 = binding.sm_build_observable_library(pot, ics, *args, None, 0, density_mode=1, precision="f32")
    assert np.array_equal(f32["dens"].sum(1).cpu().numpy() + f32["nout"][3].cpu().numpy(), np.full(90, n_rec))
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_build_observable_library(pot, ics, *args, None, 0, density_mode=2)


def test_gauss_hermite_library_matches_oracle(smo, oracle_force, torch_cuda):
    """Gauss-Hermite sums per aperture on the fly.  Sample counts per
    aperture identical to the oracle on rows without near-edge samples; the five Gauss-Hermite sums within 2e-6 per
    sample (fp32 evaluation of alpha*H_m on an fp32 v_los, 2^-32 fixed-point accumulation) -- plain, and with symmetrised
    bundles + cylindrical density cells; two calls give bit-identical rows (order-independent accumulation)."""
    from test_oracle_bundles import aperture_map, cyl_grids
    cfg = inputs.CONFIGS[4]
    g = cyl_grids(cfg["grids"])
    ics = inputs.make_ics(cfg, oracle_force, n_orb=90)
    pot = binding.sm_make_potential(cfg["potential"])
    ap, n_ap = aperture_map(g)
    rng = np.random.default_rng(4)
    v0, s = rng.normal(0, 60, n_ap), rng.uniform(70, 160, n_ap)
    args = (cfg["dt"], 600, cfg["stride"], cfg["projections"], g)
    n_rec = 600 // cfg["stride"]
    for n_bundle, fourfold, dmode in ((1, False, 0), (3, True, 1)):
        a = binding.sm_build_gh_library(pot, ics, *args, ap, n_ap, v0, s, n_bundle=n_bundle, fourfold=fourfold, density_mode=dmode)
        b = binding.sm_build_gh_library(pot, ics, *args, ap, n_ap, v0, s, n_bundle=n_bundle, fourfold=fourfold, density_mode=dmode)
        o = smo.build_gh_library(cfg["potential"], ics, *args, ap, n_ap, v0, s, n_bundle=n_bundle, fourfold=fourfold, density_mode=dmode)
        assert (a["gh"] == b["gh"]).all().item()
        n_rows = 90 // n_bundle
        total = n_bundle * (4 if fourfold else 1) * n_rec
        gh = a["gh"].cpu().numpy().astype(np.float64)
        assert gh.shape == (3, n_rows, n_ap, 6)
        for p in range(3):
            clean = o["near_edge"][p] == 0
            assert clean.sum() >= 0.7 * n_rows
            assert np.array_equal(gh[p, clean, :, 0], o["gh"][p, clean, :, 0])
            assert np.array_equal(gh[p, :, :, 0].sum(1) + a["nout"][p].cpu().numpy(), np.full(n_rows, total))
            err = np.abs(gh[p, clean, :, 1:] - o["gh"][p, clean, :, 1:])
            assert np.all(err <= 2e-6 * o["gh"][p, clean, :, :1] + 1e-9)
            assert np.abs(o["gh"][p, clean, :, 1:]).max() > 1.0
        assert count_parity(a["dens"].cpu().numpy(), o["dens"], o["near_edge"][3]) >= 0.7 * n_rows
    f32 = binding.sm_build_gh_library(pot, ics, *args, ap, n_ap, v0, s, precision="f32")
    assert np.array_equal(f32["gh"][0, :, :, 0].sum(1).cpu().numpy() + f32["nout"][0].cpu().numpy(), np.full(90, n_rec))
    with pytest.raises(binding.SchwarmaxError):
        binding.sm_build_gh_library(pot, ics, *args, ap, 5000, np.zeros(5000), np.ones(5000))


def test_two_host_threads_do_not_share_flags_timers_or_scratch(torch_cuda, oracle_force):
    """Library hygiene: debug flags and kernel timers are per host thread, scratch comes from a pool the library owns (the
    process's default pool keeps its release threshold), and two threads that make their own potentials and build libraries
    at the same time on their own streams get the results of a single-threaded run.  With more than one GPU visible the second
    thread uses the second device (per-device SM count, function attributes, side stream, pool)."""
    import threading
    import ctypes as C
    torch = torch_cuda
    cfg = inputs.CONFIGS[1]
    ics = inputs.make_ics(cfg, oracle_force, n_orb=320)
    args = (cfg["dt"], 300, cfg["stride"], cfg["projections"], cfg["grids"])
    ref = binding.sm_build_library(binding.sm_make_potential(cfg["potential"]), ics, *args)
    ref = {k: ref[k].cpu() for k in ("losvd", "dens", "nout")}
    n_dev = torch.cuda.device_count()
    out, err = {}, []

    def work(i):
        try:
            dev = i % n_dev
            torch.cuda.set_device(dev)
            assert binding.sm_set_debug_flags(4 if i == 0 else 0) == 0          # a fresh thread starts from 0
            with torch.cuda.stream(torch.cuda.Stream(device=dev)):
                pot = binding.sm_make_potential(cfg["potential"])
                d_ics = torch.as_tensor(ics).to("cuda:%d" % dev)
                for _ in range(3):
                    g = binding.sm_build_library(pot, d_ics, *args)
                torch.cuda.current_stream().synchronize()
                out[i] = {k: g[k].cpu() for k in ("losvd", "dens", "nout")}
            if i == 0:
                assert binding.sm_last_kernel_times()["integrate_ms"] > 0       # this thread's own timer
            else:
                with pytest.raises(binding.SchwarmaxError):
                    binding.sm_last_kernel_times()                              # timing was never enabled on this thread
            assert binding.sm_set_debug_flags(0) == (4 if i == 0 else 0)
        except Exception as ex:  # noqa: BLE001
            err.append((i, repr(ex)))

    th = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    [t.start() for t in th]
    [t.join() for t in th]
    assert not err, err
    for i in range(2):
        for k in ref:
            assert (out[i][k] == ref[k]).all().item(), (i, k)
    assert binding.sm_set_debug_flags(0) == 0                                    # the main thread's flags were never touched
