"""sm_stage_library_noalloc (include/schwarmax.h): the integrator on the library's static device scratch, for callers that may
not allocate.  It launches the same kernels as sm_stage_library_batch, so its staged cell indices must be IDENTICAL (integer
work: bit-exact, the bar every index test here uses), and the rows built from them identical too -- on two calls in a row, the
second of which finds the first one's leftovers in the shared scratch.  Collected last (zz): pytest -x stops at the first failure."""
import numpy as np
import pytest

from paper_2607_00117_b200 import binding, inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    return torch


def test_noalloc_stage_equals_pooled_stage_on_two_calls_in_a_row(torch_cuda, oracle_force):
    torch = torch_cuda
    cfg = inputs.CONFIGS[1]                     # barred potential: Ferrers table in shared memory, bar-phase table in scratch
    pot = binding.sm_make_potential(cfg["potential"])
    # 1st call: 9 000 orbits = 282 warp groups on 148 single-warp slots -> the queue cuts the time loop into segments and the orbit
    # state travels through the scratch; a ragged last warp.  2nd call: other ICs, other length, fp32, fewer orbits than slots
    # (one segment), straight after the first on the same stream.
    ics_a = torch.as_tensor(inputs.make_ics(cfg, oracle_force, n_orb=9000)).cuda()
    ics_b = torch.as_tensor(inputs.make_ics(dict(cfg, seed=cfg["seed"] + 7), oracle_force, n_orb=3001)).cuda()
    calls = ((ics_a, 1500, 5, "f64"), (ics_b, 901, 3, "f32"))
    refs = [binding.sm_stage_library_batch(pot, ics, cfg["dt"], n_steps, stride, [cfg["projections"]], cfg["grids"], precision=prec)[0].clone()
            for ics, n_steps, stride, prec in calls]
    outs = [torch.full((2, ics.shape[0], n_steps // stride), 12345, dtype=torch.int32, device="cuda") for ics, n_steps, stride, _ in calls]
    torch.cuda.synchronize()
    launches0, free0 = binding.sm_launch_count(), torch.cuda.mem_get_info()[0]
    for (ics, n_steps, stride, prec), out in zip(calls, outs):
        got = binding.sm_stage_library_noalloc(pot, ics, cfg["dt"], n_steps, stride, cfg["projections"], cfg["grids"], precision=prec, stage=out)
        assert got is out
    torch.cuda.synchronize()
    assert binding.sm_launch_count() - launches0 == 6          # set-up, phase table, integrator: this library's kernels did the work
    assert torch.cuda.mem_get_info()[0] >= free0               # no device memory was taken by the two calls
    for ref, out in zip(refs, outs):
        assert ref.shape == out.shape
        assert torch.equal(ref, out), "staged cell indices differ from sm_stage_library_batch"
    assert (outs[0] >= 0).float().mean().item() > 0.5         # the comparison is not one of empty libraries
    # and once more in the first shape, after the fp32 call has overwritten the scratch
    again = binding.sm_stage_library_noalloc(pot, ics_a, cfg["dt"], 1500, 5, cfg["projections"], cfg["grids"])
    assert torch.equal(again, refs[0])
    # rows from the staged indices (sm_flush_rows allocates nothing inside the library either)
    r0 = binding.sm_flush_rows(refs[0][None].contiguous(), 100, 300, cfg["grids"])
    r1 = binding.sm_flush_rows(again[None].contiguous(), 100, 300, cfg["grids"])
    for k in ("losvd", "dens", "nout"):
        assert torch.equal(r0[k], r1[k]), k
    assert (r1["dens"][0].sum(1) + r1["nout"][0, -1] == 300).all().item()


def test_noalloc_plummer_and_three_projections(torch_cuda, oracle_force):
    """Another potential class (config 0, no tables) and the three projections of config 4."""
    torch = torch_cuda
    for cid, n_orb, n_steps in ((0, 1000, 400), (4, 700, 800)):
        cfg = inputs.CONFIGS[cid]
        pot = binding.sm_make_potential(cfg["potential"])
        ics = inputs.make_ics(cfg, oracle_force, n_orb=n_orb)
        ref = binding.sm_stage_library_batch(pot, ics, cfg["dt"], n_steps, cfg["stride"], [cfg["projections"]], cfg["grids"])[0]
        got = binding.sm_stage_library_noalloc(pot, ics, cfg["dt"], n_steps, cfg["stride"], cfg["projections"], cfg["grids"])
        assert got.shape == (len(cfg["projections"]) + 1, n_orb, n_steps // cfg["stride"])
        assert torch.equal(ref, got), cid


def test_noalloc_rejects_sizes_beyond_the_static_scratch(torch_cuda):
    torch = torch_cuda
    cfg = inputs.CONFIGS[0]
    pot = binding.sm_make_potential(cfg["potential"])
    launches0 = binding.sm_launch_count()
    ics = torch.zeros((32769, 6), dtype=torch.float64, device="cuda")
    stage = torch.zeros((2, 32769, 1), dtype=torch.int32, device="cuda")
    with pytest.raises(binding.SchwarmaxError, match="SM_NOALLOC_MAX_ORB"):
        binding.sm_stage_library_noalloc(pot, ics, cfg["dt"], 10, 10, cfg["projections"], cfg["grids"], stage=stage)
    with pytest.raises(binding.SchwarmaxError, match="SM_NOALLOC_MAX_STEPS"):
        binding.sm_stage_library_noalloc(pot, ics[:64], cfg["dt"], 65535, 65535, cfg["projections"], cfg["grids"], stage=stage)
    assert binding.sm_launch_count() == launches0             # nothing was launched
    # the limits themselves are accepted: 32 768 orbits (1 024 warp groups, the whole state area) and 65 534 steps
    rng = np.random.default_rng(5)
    big = torch.as_tensor(rng.normal(size=(32768, 6)) * 0.5).cuda()
    ref = binding.sm_stage_library_batch(pot, big, cfg["dt"], 600, 10, [cfg["projections"]], cfg["grids"])[0]
    got = binding.sm_stage_library_noalloc(pot, big, cfg["dt"], 600, 10, cfg["projections"], cfg["grids"])
    assert torch.equal(ref, got)
    ref = binding.sm_stage_library_batch(pot, big[:40], cfg["dt"], 65534, 1000, [cfg["projections"]], cfg["grids"])[0]
    got = binding.sm_stage_library_noalloc(pot, big[:40], cfg["dt"], 65534, 1000, cfg["projections"], cfg["grids"])
    assert torch.equal(ref, got)
