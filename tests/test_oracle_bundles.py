"""Pins of the oracle's symmetrised orbit bundles (PAPER.md:71 dither bundles; Table 1), -m "not gpu".
The bundled function is checked against the already pinned plain path (oracle.smo.build_library) and the paper's table:
a plausible mistake in it (a wrong sign, a copy dropped, rows co-added across the wrong orbits) fails one of these."""
import os

import numpy as np
import pytest

from paper_2607_00117_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "table1_fourfold.txt")


def table1():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    return np.array([[float(v) for v in r[1:]] for r in rows])


@pytest.fixture(scope="module")
def setup(smo, oracle_force):
    cfg = inputs.CONFIGS[4]  # three projections, symmetric grids
    ics = inputs.make_ics(cfg, oracle_force, n_orb=12)
    return cfg, ics


def test_fourfold_row_equals_sum_of_plain_rows_of_the_mirrored_initial_conditions(smo, setup):
    """Table 1's copies are orbits of the rotating barred potential themselves, so the symmetrised row of
    an orbit must equal the sum of the PLAIN rows of the four initial conditions mirrored with the paper's signs."""
    cfg, ics = setup
    signs = table1()
    assert signs.shape == (4, 6)
    args = (cfg["dt"], 400, cfg["stride"], cfg["projections"], cfg["grids"])
    sym = smo.build_bundled_library(cfg["potential"], ics, *args, n_bundle=1, fourfold=True)
    acc = None
    for s in signs:
        o = smo.build_library(cfg["potential"], ics * s[None, :], *args)
        acc = {k: o[k].astype(np.float64) for k in ("losvd", "dens", "nout")} if acc is None else \
            {k: acc[k] + o[k] for k in acc}
    assert np.array_equal(sym["losvd"], acc["losvd"])
    assert np.array_equal(sym["dens"], acc["dens"])
    assert np.array_equal(sym["nout"], acc["nout"])
    n_rec = 400 // cfg["stride"]
    assert np.array_equal(sym["losvd"].sum(2) + sym["nout"][:3], np.full((3, 12), 4 * n_rec))
    assert np.array_equal(sym["dens"].sum(1) + sym["nout"][3], np.full(12, 4 * n_rec))


def test_bundle_row_is_the_sum_of_its_members(smo, setup):
    cfg, ics = setup
    args = (cfg["dt"], 300, cfg["stride"], cfg["projections"], cfg["grids"])
    plain = smo.build_library(cfg["potential"], ics, *args)
    b = smo.build_bundled_library(cfg["potential"], ics, *args, n_bundle=3, fourfold=False)
    assert b["losvd"].shape[1] == 4 and b["dens"].shape[0] == 4
    assert np.array_equal(b["losvd"], plain["losvd"].reshape(3, 4, 3, -1).sum(2))
    assert np.array_equal(b["dens"], plain["dens"].reshape(4, 3, -1).sum(1))
    assert np.array_equal(b["nout"], plain["nout"].reshape(4, 4, 3).sum(2))
    one = smo.build_bundled_library(cfg["potential"], ics, *args, n_bundle=1, fourfold=False)
    assert np.array_equal(one["losvd"], plain["losvd"]) and np.array_equal(one["dens"], plain["dens"])
    with pytest.raises(ValueError):
        smo.build_bundled_library(cfg["potential"], ics, *args, n_bundle=5, fourfold=False)  # 12 % 5 != 0


def test_symmetrised_density_is_invariant_under_the_mirror_maps(smo, setup):
    """On a grid that is symmetric about the origin the symmetrised density row is unchanged by z -> -z and by
    (x,y) -> (-x,-y) (cell index maps j -> n-1-j), for rows without samples on a bin edge."""
    cfg, ics = setup
    g = cfg["grids"]
    sym = smo.build_bundled_library(cfg["potential"], ics, cfg["dt"], 400, cfg["stride"], cfg["projections"], g, n_bundle=2, fourfold=True)
    d = sym["dens"].reshape(-1, g["dz"], g["dy"], g["dx"])
    clean = sym["near_edge"][3] == 0
    assert clean.sum() >= 4
    assert np.array_equal(d[clean], d[clean][:, ::-1, :, :])
    assert np.array_equal(d[clean], d[clean][:, :, ::-1, ::-1])
    plain = smo.build_bundled_library(cfg["potential"], ics, cfg["dt"], 400, cfg["stride"], cfg["projections"], g, n_bundle=2, fourfold=False)
    dp = plain["dens"].reshape(-1, g["dz"], g["dy"], g["dx"])
    assert not np.array_equal(dp, dp[:, ::-1, :, :])   # the unsymmetrised rows are not


def aperture_map(g, seed=0):
    """A Voronoi-like map for tests: pixels grouped into irregular apertures by nearest random generator, a border left out."""
    rng = np.random.default_rng(seed)
    n_ap = 23
    gen = rng.uniform(0, 1, (n_ap, 2)) * [g["nx"], g["ny"]]
    yy, xx = np.meshgrid(np.arange(g["ny"]) + 0.5, np.arange(g["nx"]) + 0.5, indexing="ij")
    d2 = (xx[..., None] - gen[:, 0]) ** 2 + (yy[..., None] - gen[:, 1]) ** 2
    m = d2.argmin(-1).astype(np.int32)
    m[:2, :] = -1; m[:, -3:] = -1          # pixels that belong to no aperture
    return m.reshape(-1), n_ap


def test_aperture_regrouping_equals_regrouping_the_pixel_rows(smo, setup):
    """collected in regular bins, then regrouped into the pre-defined apertures.  Regrouping on the fly must
    equal regrouping the plain pixel rows afterwards (cells of pixels with the same aperture added, pixels without an
    aperture dropped into nout) -- also for symmetrised bundles."""
    cfg, ics = setup
    g = cfg["grids"]
    ap, n_ap = aperture_map(g)
    args = (cfg["dt"], 400, cfg["stride"], cfg["projections"], g)
    for n_bundle, fourfold in ((1, False), (3, True)):
        pix = smo.build_bundled_library(cfg["potential"], ics, *args, n_bundle=n_bundle, fourfold=fourfold)
        obs = smo.build_observable_library(cfg["potential"], ics, *args, ap, n_ap, n_bundle=n_bundle, fourfold=fourfold)
        rows = pix["losvd"].reshape(3, -1, g["ny"] * g["nx"], g["nv"])
        want = np.zeros((3, rows.shape[1], n_ap, g["nv"]), dtype=np.float64)
        for a in range(n_ap):
            want[:, :, a] = rows[:, :, ap == a].sum(2)
        dropped = rows[:, :, ap < 0].sum((2, 3))
        assert np.array_equal(obs["losvd"].reshape(want.shape), want)
        assert np.array_equal(obs["nout"][:3], pix["nout"][:3] + dropped)
        assert np.array_equal(obs["dens"], pix["dens"]) and np.array_equal(obs["nout"][3], pix["nout"][3])
    ident = np.arange(g["nx"] * g["ny"], dtype=np.int32)   # identity map: nothing changes
    same = smo.build_observable_library(cfg["potential"], ics, *args, ident, len(ident))
    plain = smo.build_library(cfg["potential"], ics, *args)
    assert np.array_equal(same["losvd"], plain["losvd"]) and np.array_equal(same["nout"], plain["nout"])
    with pytest.raises(ValueError):
        smo.build_observable_library(cfg["potential"], ics, *args, ap, 5)   # map entries >= n_ap


def cyl_grids(g):
    """The paper's density grid: cells uniform in (R, phi, z), R in [0,10] kpc, z in [-3,3] kpc."""
    return dict(g, dx=10, dy=12, dz=5, bx0=0.0, bx1=10.0, by0=0.0, by1=2 * np.pi, bz0=-3.0, bz1=3.0)


def test_cylindrical_density_cells_by_bruteforce_rebinning(smo, setup):
    """density_mode 1 against numpy.histogramdd of (R, phi, z) computed from the oracle's own (pinned) trajectory dump;
    with the fourfold symmetrisation the row is invariant under phi -> phi + pi and z -> -z."""
    cfg, ics = setup
    g = cyl_grids(cfg["grids"])
    n_steps, stride = 400, 4
    out = smo.build_observable_library(cfg["potential"], ics, cfg["dt"], n_steps, stride, cfg["projections"], g, None, 0, density_mode=1)
    traj = smo.integrate_trajectories(cfg["potential"], ics, cfg["dt"], n_steps, stride)
    th = cfg["potential"]["omega_p"] * (np.arange(n_steps // stride) + 1) * stride * cfg["dt"]
    c, s = np.cos(th)[:, None], np.sin(th)[:, None]
    xb, yb, zb = c * traj[..., 0] + s * traj[..., 1], -s * traj[..., 0] + c * traj[..., 1], traj[..., 2]
    R, phi = np.hypot(xb, yb), np.mod(np.arctan2(yb, xb), 2 * np.pi)
    clean = out["near_edge"][3] == 0
    assert clean.sum() >= 8
    for i in np.flatnonzero(clean):
        h, _ = np.histogramdd(np.stack([zb[:, i], phi[:, i], R[:, i]], 1), bins=(g["dz"], g["dy"], g["dx"]),
                              range=((g["bz0"], g["bz1"]), (g["by0"], g["by1"]), (g["bx0"], g["bx1"])))
        # numpy closes the last bin on the right; the library's cells are half-open: such samples are near-edge ones
        assert np.array_equal(out["dens"][i].reshape(g["dz"], g["dy"], g["dx"]), h), i
    assert np.array_equal(out["dens"].sum(1) + out["nout"][3], np.full(len(ics), n_steps // stride))
    plain = smo.build_library(cfg["potential"], ics, cfg["dt"], n_steps, stride, cfg["projections"], g)
    assert np.array_equal(out["losvd"], plain["losvd"])        # the LOSVD block does not depend on the density mode
    sym = smo.build_observable_library(cfg["potential"], ics, cfg["dt"], n_steps, stride, cfg["projections"], g, None, 0,
                                       n_bundle=2, fourfold=True, density_mode=1)
    d = sym["dens"].reshape(-1, g["dz"], g["dy"], g["dx"])
    ok = sym["near_edge"][3] == 0
    assert ok.sum() >= 3
    assert np.array_equal(d[ok], np.roll(d[ok], g["dy"] // 2, axis=2))    # phi -> phi + pi
    assert np.array_equal(d[ok], d[ok][:, ::-1])                           # z -> -z


def test_gauss_hermite_terms_are_orthonormal(smo):
    """PAPER.md:110-114 cites van der Marel & Franx (1993) / Gerhard (1993) for the modified Hermite polynomials without
    printing them.  Their defining property pins normalisation and coefficients of the oracle's alpha(w) H_m(w):
    integral alpha^2 H_m H_n dw = delta_mn / (2 sqrt(pi)); hence a Gaussian LOSVD at (v0, s) has h_0 = 1, h_{m>=1} = 0."""
    w = np.linspace(-14, 14, 56001)
    t = smo.gh_terms(w)
    gram = np.trapezoid(t[:, :, None] * t[:, None, :], w, axis=0)
    assert np.allclose(gram, np.eye(5) / (2 * np.sqrt(np.pi)), atol=1e-12)
    assert np.allclose(t[:, 0], np.exp(-0.5 * w * w) / np.sqrt(2 * np.pi), rtol=1e-15)   # alpha itself
    par = np.array([1, -1, 1, -1, 1])                                                     # H_m(-w) = (-1)^m H_m(w)
    assert np.allclose(smo.gh_terms(-w), t * par, rtol=1e-14, atol=1e-300)
    assert np.allclose(t[28000, 1:] / t[28000, 0], [0, -1 / np.sqrt(2), 0, 3 / np.sqrt(24)])   # H_m(0)


def test_gauss_hermite_rows_against_the_pinned_histogram_path(smo, setup):
    """The per-sample Gauss-Hermite sums against the already pinned aperture LOSVD histogram: the sample counts per
    aperture are the v-marginal of the histogram rows (velocity range wide enough to hold every sample), and the m-th sum
    is the limit of sum_bins count * alpha H_m(w_centre) for fine velocity bins."""
    cfg, ics = setup
    g = dict(cfg["grids"], nv=2400, v0=-1200.0, v1=1200.0)
    ap, n_ap = aperture_map(g)
    rng = np.random.default_rng(4)
    v0, s = rng.normal(0, 60, n_ap), rng.uniform(70, 160, n_ap)
    args = (cfg["dt"], 400, cfg["stride"], cfg["projections"], g)
    for n_bundle, fourfold in ((1, False), (3, True)):
        gh = smo.build_gh_library(cfg["potential"], ics, *args, ap, n_ap, v0, s, n_bundle=n_bundle, fourfold=fourfold)
        hist = smo.build_observable_library(cfg["potential"], ics, *args, ap, n_ap, n_bundle=n_bundle, fourfold=fourfold)
        rows = hist["losvd"].reshape(3, -1, n_ap, g["nv"]).astype(np.float64)
        assert np.array_equal(gh["gh"][..., 0], rows.sum(-1))
        assert np.array_equal(gh["nout"], hist["nout"]) and np.array_equal(gh["dens"], hist["dens"])
        vc = g["v0"] + (np.arange(g["nv"]) + 0.5) * (g["v1"] - g["v0"]) / g["nv"]
        terms = np.stack([smo.gh_terms((vc - v0[a]) / s[a]) for a in range(n_ap)])      # [ap, nv, 5]
        binned = np.einsum("prav,avm->pram", rows, terms)
        # a sample sits anywhere in its 1 km/s bin: first-order error <= count * (bin/2s) * max|d(alpha H_m)/dw| per cell,
        # averaging out over many samples
        diff, count = gh["gh"][..., 1:] - binned, rows.sum(-1)[..., None]
        assert np.all(np.abs(diff) <= 5e-3 * count + 1e-12)
        assert np.all(np.abs(diff.sum((0, 1, 2))) / count.sum() < 3e-4)
        assert np.abs(gh["gh"][..., 1:]).max() > 1.0     # not trivially zero
    with pytest.raises(ValueError):
        smo.build_gh_library(cfg["potential"], ics, *args, ap, n_ap, v0, -s)
