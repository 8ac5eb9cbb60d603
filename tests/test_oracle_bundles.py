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
