"""Pins of oracle/smo.py build_observable_library_rk32: the paper's observables (bundles, fourfold symmetrisation, aperture
regrouping, cylindrical density cells, Gauss-Hermite sums) on the samples of the paper's own
integrator with weights dt / t_total.  Nothing here calls the function's own formulas back: the pins are the plain
rows of build_library_rk32 (pinned in test_oracle_rk32.py) of mirrored / single / re-grouped inputs, numpy.histogramdd, and the
table of signs the paper prints (tests/golden/table1_fourfold.txt)."""
import os

import numpy as np
import pytest

from paper_2607_00117_b200 import inputs

CFG = inputs.CONFIGS[1]
G = dict(CFG["grids"], nx=12, ny=12, nv=8, dx=6, dy=6, dz=4)
PROJ = [(30 * inputs.DEG, 45 * inputs.DEG, 0.0), (0.3, 1.2, 2.0)]
N_STEPS = 240


@pytest.fixture(scope="module")
def ics(oracle_force):
    return inputs.make_ics(CFG, oracle_force, n_orb=24)


def table1():
    path = os.path.join(os.path.dirname(__file__), "golden", "table1_fourfold.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    return np.array([[int(v) for v in r[1:]] for r in rows])      # [4][6]


def test_weights_and_outside_weight_sum_to_the_number_of_copies(smo, ics):
    for n_bundle, fourfold in ((1, False), (3, True), (4, True)):
        o = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, G, n_bundle=n_bundle, fourfold=fourfold)
        total = n_bundle * (4 if fourfold else 1)
        for p in range(2):
            assert np.allclose(o["losvd"][p].sum(1) + o["wout"][p], total, rtol=0, atol=1e-12)
        assert np.allclose(o["dens"].sum(1) + o["wout"][2], total, rtol=0, atol=1e-12)
        assert o["losvd"].shape == (2, 24 // n_bundle, 12 * 12 * 8)


def test_plain_rows_are_those_of_build_library_rk32(smo, ics):
    a = smo.build_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, G)
    b = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, G)
    assert np.array_equal(a["losvd"], b["losvd"]) and np.array_equal(a["dens"], b["dens"]) and np.array_equal(a["wout"], b["wout"])


def test_fourfold_row_is_the_sum_of_the_rows_of_the_four_mirrored_initial_conditions(smo, ics):
    """the copies of Table 1 are orbits of the rotating barred potential themselves, so the symmetrised row of an
    orbit equals the sum of the PLAIN rows of its four mirrored initial conditions (signs from the stored table, applied at
    t = 0 where the bar lies along x).  The step-size controller sees |y| and e^2 only, so the mirrored orbits take the same
    steps; what is left is rounding amplified over 240 attempts."""
    signs = table1()
    assert signs.shape == (4, 6) and np.array_equal(signs[0], np.ones(6, dtype=int))
    sym = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, G, fourfold=True)
    acc_l, acc_d = 0.0, 0.0
    for s in signs:
        o = smo.build_library_rk32(CFG["potential"], ics * s[None, :], N_STEPS, PROJ, G)
        acc_l, acc_d = acc_l + o["losvd"], acc_d + o["dens"]
    # cells can differ only where a mirrored sample sits within rounding of a bin edge
    tol = 2 * sym["edge_w"].sum() + 1e-9
    assert np.abs(sym["losvd"] - acc_l).sum() <= tol and np.abs(sym["dens"] - acc_d).sum() <= tol
    assert np.abs(sym["losvd"] - acc_l).max() < 1e-9 or sym["edge_w"].sum() > 0
    # the symmetrised density is invariant under z -> -z and (x, y) -> (-x, -y) on this origin-symmetric grid
    d = sym["dens"].reshape(-1, G["dz"], G["dy"], G["dx"])
    assert np.allclose(d, d[:, ::-1], atol=1e-12) and np.allclose(d, d[:, :, ::-1, ::-1], atol=1e-12)


def test_bundle_row_is_the_sum_of_its_members_rows(smo, ics):
    one = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, G, fourfold=True)
    bun = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, G, n_bundle=4, fourfold=True)
    assert np.allclose(bun["losvd"], one["losvd"].reshape(2, 6, 4, -1).sum(2), rtol=0, atol=1e-13)
    assert np.allclose(bun["dens"], one["dens"].reshape(6, 4, -1).sum(1), rtol=0, atol=1e-13)
    assert np.allclose(bun["wout"], one["wout"].reshape(3, 6, 4).sum(2), rtol=0, atol=1e-13)


def test_aperture_regrouping_on_the_fly_equals_regrouping_the_pixel_rows(smo, ics):
    rng = np.random.default_rng(5)
    n_ap = 17
    ap = rng.integers(-1, n_ap + 1, G["nx"] * G["ny"]).astype(np.int32)     # -1 and n_ap: pixels without an aperture
    pix = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, G, n_bundle=2, fourfold=True)
    reg = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, G, ap, n_ap, n_bundle=2, fourfold=True)
    rows = pix["losvd"].reshape(2, 12, G["ny"] * G["nx"], G["nv"])
    want = np.zeros((2, 12, n_ap, G["nv"]))
    lost = np.zeros((2, 12))
    for px, a in enumerate(ap):
        if 0 <= a < n_ap:
            want[:, :, a] += rows[:, :, px]
        else:
            lost += rows[:, :, px].sum(-1)
    assert np.allclose(reg["losvd"].reshape(want.shape), want, rtol=0, atol=1e-13)
    assert np.allclose(reg["wout"][:2], pix["wout"][:2] + lost, rtol=0, atol=1e-12)
    assert np.array_equal(reg["dens"], pix["dens"])


def test_cylindrical_cells_by_weighted_histogramdd_of_the_samples(smo, ics):
    g = dict(G, dx=5, dy=8, dz=3, bx0=0.0, bx1=10.0, by0=0.0, by1=2 * np.pi, bz0=-3.0, bz1=3.0)
    o = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, g, density_mode=1)
    s, dtw, t_end = smo.integrate_rk32(CFG["potential"], ics, N_STEPS)
    for i in (0, 7, 23):
        R = np.hypot(s[:, i, 0], s[:, i, 1])
        phi = np.mod(np.arctan2(s[:, i, 1], s[:, i, 0]), 2 * np.pi)
        h, _ = np.histogramdd(np.stack([s[:, i, 2], phi, R], 1), bins=(3, 8, 5), range=((-3, 3), (0, 2 * np.pi), (0, 10)),
                              weights=dtw[:, i] / t_end[i])
        # histogramdd closes the last bin on the right; no sample sits exactly there
        assert np.abs(h.reshape(-1) - o["dens"][i]).sum() <= 2 * o["edge_w"][2, i] + 1e-12
    # the Cartesian block does not depend on the density mode
    c = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, g, density_mode=0)
    assert np.array_equal(c["losvd"], o["losvd"])


def test_gauss_hermite_sums_against_the_aperture_histogram(smo, ics):
    """[0] = the weight per aperture = the v-marginal of the aperture-histogram rows over a velocity range that holds every sample;
    [1 + m] = the limit of sum_bins weight x alpha H_m(bin centre) for 1 km/s bins (first-order bound per cell)."""
    rng = np.random.default_rng(6)
    n_ap = 9
    ap = rng.integers(0, n_ap, G["nx"] * G["ny"]).astype(np.int32)
    v0, sg = rng.normal(0, 40, n_ap), rng.uniform(80, 150, n_ap)
    fine = dict(G, nv=1600, v0=-800.0, v1=800.0)
    gh = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, fine, ap, n_ap, n_bundle=2, fourfold=True, gh=(v0, sg))
    hist = smo.build_observable_library_rk32(CFG["potential"], ics, N_STEPS, PROJ, fine, ap, n_ap, n_bundle=2, fourfold=True)
    h = hist["losvd"].reshape(2, 12, n_ap, 1600)
    assert np.allclose(gh["gh"][..., 0], h.sum(-1), rtol=0, atol=1e-12)
    centres = -800.0 + (np.arange(1600) + 0.5)
    for a in range(n_ap):
        t = smo.gh_terms((centres - v0[a]) / sg[a])                    # [1600][5]
        approx = h[:, :, a, :] @ t
        assert np.abs(approx - gh["gh"][:, :, a, 1:]).max() < 2e-3 * max(gh["gh"][:, :, a, 0].max(), 1e-30) + 1e-12
    assert np.abs(gh["gh"][..., 2:]).max() > 1e-2
    assert np.array_equal(gh["dens"], hist["dens"]) and np.allclose(gh["wout"][:2], hist["wout"][:2], atol=1e-12)


def test_jacobi_drift_output_is_the_papers_diagnostic(smo, ics):
    """Jacobi-energy errors of 1e-4 ... 1e-2 at rtol 1e-4, orbits above 1e-1 discarded.  drift = max over the
    accepted samples of |E_J - E_J(0)| / |E_J(0)|, E_J = v^2/2 + Phi - Omega_p L_z with the inertial velocity: recomputed here
    from the dumped samples with smo.jacobi, and in the paper's range."""
    o = smo.build_observable_library_rk32(CFG["potential"], ics, 600, PROJ, G, want_drift=True)
    s, dtw, _ = smo.integrate_rk32(CFG["potential"], ics, 600)
    ej0 = smo.jacobi(CFG["potential"], ics, 0.0)
    for i in (0, 5, 11):
        acc = dtw[:, i] > 0
        ej = smo.jacobi(CFG["potential"], s[acc, i], 0.0)             # bar-frame state at bar phase 0 = inertial state at t = 0
        assert o["drift"][i] == pytest.approx(np.max(np.abs(ej - ej0[i]) / abs(ej0[i])), rel=1e-12)
    assert 1e-5 < np.median(o["drift"]) < 1e-2 and o["drift"].max() < 1e-1
