"""CPU-side checks of the product's host logic (-m "not gpu"): the C-ABI library loads and exports every
symbol of include/schwarmax.h, and the host-compiled copy of the kernels' force code (tables + algebra)
agrees with the oracle.  No kernel runs here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2607_00117_b200 import binding, inputs
from paper_2607_00117_b200.build import build_library

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def so():
    return build_library()


def test_exports_every_declared_symbol(so):
    header = open(os.path.join(ROOT, "include", "schwarmax.h")).read()
    declared = set(re.findall(r"\b(sm_[a-z_0-9]+)\s*\(", header))
    declared -= {"sm_status", "sm_kind", "sm_precision"}
    assert {"sm_make_potential", "sm_build_library", "sm_build_library_batch"} <= declared
    lib = C.CDLL(so)
    for name in declared:
        assert hasattr(lib, name), name
    assert set(binding.EXPORTS) == declared
    assert binding.sm_version() >= 100


def test_struct_layouts_match_header():
    assert C.sizeof(binding.SmComponent) == 56
    assert C.sizeof(binding.SmPotentialDesc) == 24 + 8 + 8 * 56
    assert C.sizeof(binding.SmProjection) == 24
    assert C.sizeof(binding.SmGrids) == 16 + 48 + 16 + 48


def test_invalid_potentials_are_rejected_without_a_device(so):
    bad = [
        {"G": 1.0, "components": [(inputs.FERRERS2, 1, [1.0, 1.0, 2.0, 0.5])]},      # axes not a>b>c
        {"G": 1.0, "components": [(9, 0, [1.0, 1.0])]},                              # unknown kind
        {"G": 1.0, "components": [(inputs.NFW, 0, [1.0, 0.0])]},                     # r_s = 0
        {"G": -1.0, "components": [(inputs.PLUMMER, 0, [1.0, 1.0])]},                # G <= 0
        {"G": 1.0, "components": [(inputs.FERRERS2, 1, [1.0, 3.0, 2.0, 1.0]), (inputs.FERRERS2, 1, [1.0, 3.0, 2.0, 1.0])]},
    ]
    for spec in bad:
        with pytest.raises(binding.SchwarmaxError):
            binding.sm_make_potential(spec)


@pytest.mark.parametrize("scale", [None, [1.3, 0.7, 1.3, 0.7, 1.3, 0.7, 0.7, 1.3, 0.7], [0.7, 1.3, 0.7, 1.3, 0.7, 1.3, 1.3, 0.7, 1.3]])
def test_host_compiled_force_matches_oracle(smo, scale):
    pot = inputs.barred_potential(scale)
    rng = np.random.default_rng(7)
    pts = np.concatenate([rng.normal(size=(1500, 3)) * [6, 6, 1.2], rng.normal(size=(700, 3)) * [1.5, 0.6, 0.2],
                          rng.normal(size=(300, 3)) * [2, 1, 2], rng.normal(size=(200, 3)) * [40, 40, 10],
                          [[0, 0, 0], [1e-4, 0, 0], [4, 0, 0], [0, 1.5, 0], [0, 0, 0.5], [100, 3, 2], [0.3, 0.2, 1e-9]]])
    for t in (0.0, 0.0371):
        F, P = binding.sm_debug_host_force(pot, pts, t)
        Fo, Po = smo.eval_force(pot, pts, t)
        err = np.linalg.norm(F - Fo, axis=1) / np.maximum(np.linalg.norm(Fo, axis=1), 1e-300)
        err[0] = np.linalg.norm(F[-7] - Fo[-7])  # the origin: absolute
        assert np.max(err) < 1e-14
        assert np.median(err) < 5e-16
        assert np.max(np.abs(P / Po - 1)) < 3e-15
    F32, _ = binding.sm_debug_host_force(pot, pts, 0.0, "f32")
    Fo, _ = smo.eval_force(pot, pts, 0.0)
    nrm = np.linalg.norm(Fo, axis=1)
    ok = nrm > 0
    assert np.max(np.linalg.norm(F32 - Fo, axis=1)[ok] / nrm[ok]) < 2e-5


@pytest.mark.parametrize("comp", [None, (inputs.DEHNEN_T3, 1, [1e10, 0.8, 0.3, 4.0, 0.0]), (inputs.DEHNEN_V4, 1, [1e10, 0.5, 0.5, 2.0, -0.6]),
                                  (inputs.DEHNEN_T3, 1, [1e10, 0.0, 0.3, 4.0, 0.3])])
def test_host_compiled_needle_bars_match_oracle(smo, comp):
    """dehnen.cuh compiled for the host against the oracle's __float128 closed forms (Eq. 12, Appendix A):
    the paper's own stellar model (None), and single needle bars through every compile-time variant (T_3 / V_4, uniform
    and sloped needle).  A needle bar alone loses ~(r/L)^2 ulp to the differences of primitives."""
    pot = inputs.paper_bar_potential()
    if comp is not None:
        pot = dict(pot, components=[comp])
    rng = np.random.default_rng(11)
    pts = np.concatenate([rng.normal(size=(3000, 3)) * [6, 6, 1.2], rng.normal(size=(1000, 3)) * [2.0, 0.5, 0.3],
                          rng.normal(size=(300, 3)) * [30, 30, 8],
                          [[0, 0, 0], [4, 0, 0], [-4, 0, 0], [3.9, 1e-9, 0], [0, 0, 0.5], [60, 3, 2], [0.1, 0, 0]]])
    F, P = binding.sm_debug_host_force(pot, pts, 0.21)
    Fo, Po = smo.eval_force(pot, pts, 0.21)
    nrm = np.linalg.norm(Fo, axis=1)
    err = np.linalg.norm(F - Fo, axis=1) / nrm.clip(1e-3 * nrm.max())
    if comp is None:
        assert err.max() < 1e-13 and np.median(err) < 1e-15
        assert np.max(np.abs(P / Po - 1)) < 1e-14
    else:
        L = comp[2][3]
        assert np.all(err < 2e-14 * (1.0 + (np.linalg.norm(pts, axis=1) / L) ** 2).clip(1.0, 1e5))
        assert np.max(np.abs(P / Po - 1)) < 1e-11


def test_host_compiled_plummer_and_point_mass(smo):
    for b in (1.0, 0.0):
        pot = {"G": 1.0, "omega_p": 0.0, "phase0": 0.0, "components": [(inputs.PLUMMER, 0, [1.0, b])]}
        pts = np.random.default_rng(2).normal(size=(200, 3)) * 2 + 0.1
        F, P = binding.sm_debug_host_force(pot, pts)
        Fo, Po = smo.eval_force(pot, pts)
        assert F == pytest.approx(Fo, rel=2e-15)
        assert P == pytest.approx(Po, rel=2e-15)


@pytest.mark.parametrize("axes", [(4.0, 1.5, 0.5), (5.2, 1.05, 0.35), (2.8, 1.95, 0.65)])
def test_warm_started_lambda_converges_from_any_guess(smo, axes):
    """The kernels' fp32 Newton for the Ferrers lambda (ferrers.cuh) must reach |dlambda| < 1e-5 (c^2+lambda) -- what the
    force needs, DESIGN.md 5 -- from a cold start, from the integrator's warm start, and from arbitrarily bad guesses."""
    a, b, c = axes
    rng = np.random.default_rng(11)
    pts = np.concatenate([rng.normal(size=(20000, 3)) * [6, 6, 1.2], rng.normal(size=(10000, 3)) * [1.5, 0.6, 0.2],
                          rng.normal(size=(3000, 3)) * [40, 40, 10], rng.normal(size=(10000, 3)) * [3, 1, 0.4],
                          [[0, 0, 0], [a, 0, 0], [0, b, 0], [0, 0, c], [1e-3, 0, 0]]])
    exact = smo.ferrers_lambda(a, b, c, pts)
    C = c * c + exact
    guesses = {"cold": -np.ones(len(pts)), "zero": np.zeros(len(pts)), "warm": exact * (1 + 1e-3 * rng.normal(size=len(pts))),
               "half": exact * rng.uniform(0.5, 1.5, len(pts)), "x10": 10 * exact + 1, "huge": np.full(len(pts), 1e4)}
    for name, g in guesses.items():
        lam, iters = binding.sm_debug_host_lambda(a, b, c, pts, g)
        assert np.max(np.abs(lam - exact) / C) < 1e-5, name
        m2 = (pts ** 2 / np.array([a * a, b * b, c * c])).sum(1)
        assert np.all(lam[m2 < 1 - 1e-5] == 0), name     # inside the bar: exactly 0
        assert iters.max() <= 8, name
        if name == "warm":
            assert iters.mean() < 1.3 and iters.max() <= 3


def test_roofline_counts_are_those_of_the_current_kernels():
    """bench.py's roofline multiplies the executed-flop counts of profiles/kernel_counts.json (taken from ncu captures by
    `python -m paper_2607_00117_b200.ncu_summary`) by the work it timed: counts taken from older kernel sources would make
    `roofline.frac` silently wrong, so every entry carries a hash of the kernel sources and must match the tree."""
    import json
    from paper_2607_00117_b200 import ncu_summary
    with open(ncu_summary.COUNTS) as fh:
        counts = json.load(fh)
    assert "integrate_kernel/barred/f64" in counts and "integrate_kernel/barred/f32" in counts
    now = ncu_summary.csrc_sha16()
    stale = {k: v["csrc_sha16"] for k, v in counts.items() if k.startswith("integrate_kernel") and v["csrc_sha16"] != now}
    assert not stale, f"re-capture with ncu and ncu_summary.py: kernel sources are now {now}, counts were taken from {stale}"
    for k, v in counts.items():
        assert os.path.exists(os.path.join(os.path.dirname(ncu_summary.COUNTS), v["source"])), k


def test_potential_tables_built_on_two_threads_at_once_are_the_single_thread_tables():
    """sm_make_potential builds the Ferrers anchor tables on the host; a process may make potentials on several threads (one per
    GPU).  The table builder once kept its Chebyshev-to-monomial matrix in a static array that every call zeroed and refilled, so
    concurrent builds got coefficients that were off at rounding level or worse (seen as a flaky two-thread GPU test).  Forces from
    tables built on eight threads at the same time must equal the single-thread ones bit for bit (ctypes releases the GIL)."""
    import threading
    pot = inputs.CONFIGS[1]["potential"]
    rng = np.random.default_rng(3)
    pts = rng.normal(size=(64, 3)) * [6, 6, 1.2]
    ref, _ = binding.sm_debug_host_force(pot, pts)
    out, errs = {}, []

    def work(i):
        try:
            for _ in range(40):   # ~9 ms per build: the old static array failed ~50 of these 320 builds
                f, _ = binding.sm_debug_host_force(pot, pts)
                if not np.array_equal(f, ref):
                    errs.append((i, float(np.abs(f - ref).max())))
        except Exception as ex:  # noqa: BLE001
            errs.append((i, repr(ex)))

    th = [threading.Thread(target=work, args=(i,)) for i in range(8)]
    [t.start() for t in th]
    [t.join() for t in th]
    assert not errs, errs[:5]
