"""Helpers shared by the -m gpu parity tests."""
import numpy as np


def count_parity(gpu_rows, ora_rows, near_edge):
    """Rows must be identical for orbits with no recorded sample within 1e-9 of a bin edge (north_star);
    for the others the L1 difference is bounded by two cells per near-edge sample.  Returns the number of
    orbits compared exactly."""
    gpu_rows = np.asarray(gpu_rows)
    clean = near_edge == 0
    assert np.array_equal(gpu_rows[clean], ora_rows[clean]), "bin counts differ on orbits without near-edge samples"
    l1 = np.abs(gpu_rows[~clean] - ora_rows[~clean]).sum(axis=1)
    assert np.all(l1 <= 2 * near_edge[~clean])
    return int(clean.sum())


def traj_rel_err(a, b, length_scale):
    """max over recorded steps of |dx|/max(|x|, 1e-3 L) and the same for v."""
    dx = np.linalg.norm(a[..., :3] - b[..., :3], axis=-1) / np.maximum(np.linalg.norm(b[..., :3], axis=-1), 1e-3 * length_scale)
    vs = np.median(np.linalg.norm(b[..., 3:], axis=-1))
    dv = np.linalg.norm(a[..., 3:] - b[..., 3:], axis=-1) / np.maximum(np.linalg.norm(b[..., 3:], axis=-1), 1e-3 * vs)
    return np.maximum(dx, dv).max(axis=0)
