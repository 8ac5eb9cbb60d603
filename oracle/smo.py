"""ctypes loader for the CPU oracle (libsm_oracle.so).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2607_00117_b200 (the CUDA product) and the
product imports nothing from here.
"""
import ctypes as C
import os

import numpy as np

from .build import build_oracle

PLUMMER, MIYAMOTO_NAGAI, NFW, FERRERS2, DEHNEN_T3, DEHNEN_V4 = 1, 2, 3, 4, 5, 6
W_ORDER = ["000", "100", "010", "001", "200", "020", "002", "110", "101", "011",
           "300", "030", "003", "210", "201", "120", "021", "102", "012", "111"]


class Component(C.Structure):
    _fields_ = [("kind", C.c_int), ("rotating", C.c_int), ("p", C.c_double * 6)]


class PotentialDesc(C.Structure):
    _fields_ = [("G", C.c_double), ("omega_p", C.c_double), ("phase0", C.c_double),
                ("n_comp", C.c_int), ("comp", Component * 8)]


class Projection(C.Structure):
    _fields_ = [("alpha", C.c_double), ("beta", C.c_double), ("gamma", C.c_double)]


class Grids(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nv", C.c_int),
                ("x0", C.c_double), ("x1", C.c_double), ("y0", C.c_double), ("y1", C.c_double),
                ("v0", C.c_double), ("v1", C.c_double),
                ("dx", C.c_int), ("dy", C.c_int), ("dz", C.c_int),
                ("bx0", C.c_double), ("bx1", C.c_double), ("by0", C.c_double), ("by1", C.c_double),
                ("bz0", C.c_double), ("bz1", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle())
        for name in ("smo_eval_force", "smo_integrate_trajectories", "smo_build_library", "smo_ferrers_lambda",
                     "smo_ferrers_W", "smo_project", "smo_jacobi", "smo_num_threads", "smo_integrate_rk32"):
            getattr(_lib, name).restype = C.c_int
    return _lib


def make_desc(spec):
    """spec: dict(G, omega_p, phase0=0, components=[(kind, rotating, [params...]), ...])."""
    d = PotentialDesc()
    d.G, d.omega_p, d.phase0 = spec["G"], spec.get("omega_p", 0.0), spec.get("phase0", 0.0)
    comps = spec["components"]
    d.n_comp = len(comps)
    for i, (kind, rot, p) in enumerate(comps):
        d.comp[i].kind, d.comp[i].rotating = int(kind), int(rot)
        for j, v in enumerate(p):
            d.comp[i].p[j] = float(v)
    return d


def make_grids(g):
    out = Grids()
    for k, v in g.items():
        setattr(out, k, v)
    return out


def _dp(a):
    return a.ctypes.data_as(C.c_void_p)


def _chk(rc, what):
    if rc != 0:
        raise ValueError(f"{what} failed with code {rc}")


def eval_force(spec, xyz, t=0.0, want_phi=True):
    xyz = np.ascontiguousarray(xyz, dtype=np.float64).reshape(-1, 3)
    F = np.empty_like(xyz)
    Phi = np.empty(len(xyz)) if want_phi else None
    d = make_desc(spec)
    _chk(lib().smo_eval_force(C.byref(d), _dp(xyz), C.c_int64(len(xyz)), C.c_double(t), _dp(F),
                              _dp(Phi) if want_phi else None), "smo_eval_force")
    return (F, Phi) if want_phi else F


def integrate_trajectories(spec, ics, dt, n_steps, stride=1, state_prec=0):
    ics = np.ascontiguousarray(ics, dtype=np.float64).reshape(-1, 6)
    n_rec = n_steps // stride
    traj = np.empty((n_rec, len(ics), 6))
    d = make_desc(spec)
    _chk(lib().smo_integrate_trajectories(C.byref(d), _dp(ics), C.c_int64(len(ics)), C.c_double(dt),
                                          C.c_int64(n_steps), C.c_int32(stride), C.c_int(state_prec), _dp(traj)),
         "smo_integrate_trajectories")
    return traj


def integrate_rk32(spec, ics, n_steps, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3):
    """The paper's adaptive Bogacki-Shampine RK3(2) in the rotating frame.
    -> samples[n_steps, n, 6] (bar-axes position, inertial velocity on bar axes), dt_w[n_steps, n], t_end[n]."""
    ics = np.ascontiguousarray(ics, dtype=np.float64).reshape(-1, 6)
    n = len(ics)
    samples, dt_w, t_end = np.empty((n_steps, n, 6)), np.empty((n_steps, n)), np.empty(n)
    d = make_desc(spec)
    _chk(lib().smo_integrate_rk32(C.byref(d), _dp(ics), C.c_int64(n), C.c_int64(n_steps), C.c_double(rtol), C.c_double(atol_x),
                                  C.c_double(atol_v), C.c_double(h0), _dp(samples), _dp(dt_w), _dp(t_end)), "smo_integrate_rk32")
    return samples, dt_w, t_end


def build_library_rk32(spec, ics, n_steps, projections, grids, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3):
    """delta-t-weighted matrices of the paper's integrator ("each sample along the orbit is reweighted linearly by its
    corresponding integration time step size ... the weight of each sample is dt/t_total"), written out with numpy on the samples of
    integrate_rk32: bin rule and layouts as build_library (floor((u - lo) * n/(hi - lo)), half-open; LOSVD (iy*nx+ix)*nv+iv, density
    (iz*dy+iy)*dx+ix, density in the bar frame), projection of PAPER.md:96-100 Eq. 1 with R = Rz(gamma) Rx(beta) Rz(alpha).
    -> dict(losvd[n_proj,n,nlos], dens[n,nden], wout[n_proj+1,n], edge_w[n_proj+1,n], t_end[n]) in float64; edge_w = the weight of the
    samples that lie within 1e-9 bin widths of a bin edge (their cell is a coin toss between two correct codes)."""
    samples, dtw, t_end = integrate_rk32(spec, ics, n_steps, rtol, atol_x, atol_v, h0)
    n = samples.shape[1]
    g = grids
    nlos, nden = g["nx"] * g["ny"] * g["nv"], g["dx"] * g["dy"] * g["dz"]
    losvd = np.zeros((len(projections), n, nlos))
    dens = np.zeros((n, nden))
    wout = np.zeros((len(projections) + 1, n))
    edge_w = np.zeros((len(projections) + 1, n))
    w = dtw / t_end[None, :]                                   # [n_steps, n]
    orb = np.broadcast_to(np.arange(n)[None, :], w.shape)

    def cells(u, lo, hi, nb):
        f = (u - lo) * (nb / (hi - lo))
        ok = (f >= 0) & (f < nb)
        near = np.abs(f - np.rint(f)) < 1e-9
        return np.where(ok, np.floor(f), 0).astype(np.int64), ok, near

    def scatter(rows, out_row, edge_row, idx, ok, near):
        np.add.at(rows, (orb[ok], idx[ok]), w[ok])
        np.add.at(out_row, orb[~ok], w[~ok])
        np.add.at(edge_row, orb[near], w[near])

    x, y, z, vx, vy, vz = (samples[..., j] for j in range(6))
    jx, okx, ex = cells(x, g["bx0"], g["bx1"], g["dx"])
    jy, oky, ey = cells(y, g["by0"], g["by1"], g["dy"])
    jz, okz, ez = cells(z, g["bz0"], g["bz1"], g["dz"])
    scatter(dens, wout[-1], edge_w[-1], (jz * g["dy"] + jy) * g["dx"] + jx, okx & oky & okz, ex | ey | ez)
    for p, (al, be, ga) in enumerate(projections):
        ca, sa, cb, sb, cg, sg = np.cos(al), np.sin(al), np.cos(be), np.sin(be), np.cos(ga), np.sin(ga)
        x1, y1 = x * ca - y * sa, x * sa + y * ca              # Rz(alpha)
        y2 = y1 * cb - z * sb                                  # Rx(beta), image-plane row
        X, Y = x1 * cg - y2 * sg, x1 * sg + y2 * cg            # Rz(gamma)
        vlos = (vx * sa + vy * ca) * sb + vz * cb              # z' row of Rx(beta) Rz(alpha) applied to v
        ix, ok1, e1 = cells(X, g["x0"], g["x1"], g["nx"])
        iy, ok2, e2 = cells(Y, g["y0"], g["y1"], g["ny"])
        iv, ok3, e3 = cells(vlos, g["v0"], g["v1"], g["nv"])
        scatter(losvd[p], wout[p], edge_w[p], (iy * g["nx"] + ix) * g["nv"] + iv, ok1 & ok2 & ok3, e1 | e2 | e3)
    return dict(losvd=losvd, dens=dens, wout=wout, edge_w=edge_w, t_end=t_end)


# PAPER.md:77-84 Table 1: the four copies of a sample (signs of x, y, z; the velocity signs are the same three)
FOURFOLD_SIGNS = ((1, 1, 1), (1, 1, -1), (-1, -1, 1), (-1, -1, -1))


def build_observable_library_rk32(spec, ics, n_steps, projections, grids, ap_map=None, n_ap=0, n_bundle=1, fourfold=False,
                                  density_mode=0, gh=None, rtol=1e-4, atol_x=1e-4, atol_v=1e-4, h0=1e-3, want_drift=False):
    """The paper's OWN pipeline on the paper's own integrator: samples of integrate_rk32, each with
    weight dt / t_total of ITS orbit; rows = bundles of n_bundle consecutive orbits, every sample
    binned with the copies of Table 1 when `fourfold` (copies taken of the bar-frame sample, R18);
    image pixels regrouped into apertures by ap_map[ny*nx] (< 0 or >= n_ap: no aperture); density cells Cartesian
    (density_mode 0) or uniform in (R, phi in [0, 2 pi), z) (density_mode 1); with gh = (v0[n_ap], s[n_ap]) the
    velocity axis is not binned and every aperture gets [sum of w, sum of w alpha(u) H_m(u), m = 0..4], u = (v_los - v0)/s
    (Eq. 2, R17; gh_terms is the pinned alpha H_m).  Bin rule, layouts and projection as
    build_library_rk32.  Plain numpy loops over copies and projections, float64.
    -> dict(losvd[n_proj, n_rows, n_cells] or gh[n_proj, n_rows, n_ap, 6], dens[n_rows, nden], wout[n_proj+1, n_rows],
            edge_w[n_proj+1, n_rows], t_end[n], drift[n] (max relative Jacobi-integral error over the accepted samples))."""
    samples, dtw, t_end = integrate_rk32(spec, ics, n_steps, rtol, atol_x, atol_v, h0)
    n = samples.shape[1]
    if n % n_bundle:
        raise ValueError("n_orb must be a multiple of n_bundle")
    n_rows = n // n_bundle
    g = grids
    npix, nv, nden = g["nx"] * g["ny"], g["nv"], g["dx"] * g["dy"] * g["dz"]
    if ap_map is not None:
        ap_map = np.asarray(ap_map, dtype=np.int64).reshape(-1)
    elif gh is not None:
        raise ValueError("Gauss-Hermite rows need an aperture map")
    n_img = n_ap if ap_map is not None else npix
    n_proj = len(projections)
    out_los = np.zeros((n_proj, n_rows, n_img, 6)) if gh is not None else np.zeros((n_proj, n_rows, n_img * nv))
    dens = np.zeros((n_rows, nden))
    wout = np.zeros((n_proj + 1, n_rows))
    edge_w = np.zeros((n_proj + 1, n_rows))
    w = dtw / t_end[None, :]                                   # [n_steps, n]: rejected attempts have weight 0
    row = np.broadcast_to((np.arange(n) // n_bundle)[None, :], w.shape)

    def cells(u, lo, hi, nb):
        f = (u - lo) * (nb / (hi - lo))
        ok = (f >= 0) & (f < nb)
        near = np.abs(f - np.rint(f)) < 1e-9
        return np.where(ok, np.floor(f), 0).astype(np.int64), ok, near

    for sx, sy, sz in (FOURFOLD_SIGNS if fourfold else FOURFOLD_SIGNS[:1]):
        x, y, z = sx * samples[..., 0], sy * samples[..., 1], sz * samples[..., 2]
        vx, vy, vz = sx * samples[..., 3], sy * samples[..., 4], sz * samples[..., 5]
        if density_mode == 1:
            phi = np.arctan2(y, x)
            phi = np.where(phi < 0, phi + 2 * np.pi, phi)
            d0, d1 = np.sqrt(x * x + y * y), phi
        else:
            d0, d1 = x, y
        j0, ok0, e0 = cells(d0, g["bx0"], g["bx1"], g["dx"])
        j1, ok1, e1 = cells(d1, g["by0"], g["by1"], g["dy"])
        j2, ok2, e2 = cells(z, g["bz0"], g["bz1"], g["dz"])
        ok, near = ok0 & ok1 & ok2, e0 | e1 | e2
        np.add.at(dens, (row[ok], ((j2 * g["dy"] + j1) * g["dx"] + j0)[ok]), w[ok])
        np.add.at(wout[-1], row[~ok], w[~ok])
        np.add.at(edge_w[-1], row[near], w[near])
        for p, (al, be, ga) in enumerate(projections):
            ca, sa, cb, sb, cg, sg = np.cos(al), np.sin(al), np.cos(be), np.sin(be), np.cos(ga), np.sin(ga)
            x1, y1 = x * ca - y * sa, x * sa + y * ca
            y2 = y1 * cb - z * sb
            X, Y = x1 * cg - y2 * sg, x1 * sg + y2 * cg
            vlos = (vx * sa + vy * ca) * sb + vz * cb
            ix, okx, ex = cells(X, g["x0"], g["x1"], g["nx"])
            iy, oky, ey = cells(Y, g["y0"], g["y1"], g["ny"])
            ok, near = okx & oky, ex | ey
            img = iy * g["nx"] + ix
            if ap_map is not None:
                a_ = np.where(ok, ap_map[np.where(ok, img, 0)], -1)
                ok = ok & (a_ >= 0) & (a_ < n_ap)
                img = np.where(ok, a_, 0)
            if gh is None:
                iv, okv, ev = cells(vlos, g["v0"], g["v1"], nv)
                ok, near = ok & okv, near | ev
                np.add.at(out_los[p], (row[ok], (img * nv + iv)[ok]), w[ok])
            else:
                v0, s_ = np.asarray(gh[0], dtype=np.float64), np.asarray(gh[1], dtype=np.float64)
                u = (vlos[ok] - v0[img[ok]]) / s_[img[ok]]
                terms = gh_terms(u)                            # [.., 5] alpha(u) H_m(u), m = 0..4 (pinned in test_oracle_bundles)
                np.add.at(out_los[p][..., 0], (row[ok], img[ok]), w[ok])
                for m in range(5):
                    np.add.at(out_los[p][..., 1 + m], (row[ok], img[ok]), w[ok] * terms[:, m])
            np.add.at(wout[p], row[~ok], w[~ok])
            np.add.at(edge_w[p], row[near], w[near])
    res = dict(dens=dens, wout=wout, edge_w=edge_w, t_end=t_end)
    res["gh" if gh is not None else "losvd"] = out_los
    if want_drift:
        # Jacobi integral of every accepted sample (inertial velocity on bar axes: E_J = v^2/2 + Phi - Omega_p L_z, smo_jacobi at t = 0
        # with phase0 = 0 evaluates exactly that on bar-frame states); orbits above 1e-1 are discarded
        spec0 = dict(spec, phase0=0.0)
        ej0 = jacobi(spec, ics, 0.0)
        drift = np.zeros(n)
        for k in range(n_steps):
            acc = dtw[k] > 0
            if acc.any():
                ej = jacobi(spec0, samples[k][acc], 0.0)
                drift[acc] = np.maximum(drift[acc], np.abs(ej - ej0[acc]) / np.abs(ej0[acc]))
        res["drift"] = drift
    return res


def build_library(spec, ics, dt, n_steps, stride, projections, grids, state_prec=0, want_diag=False):
    """Returns dict(losvd[n_proj,n_orb,nlos], dens[n_orb,nden], nout[n_proj+1,n_orb], near_edge, diag)."""
    ics = np.ascontiguousarray(ics, dtype=np.float64).reshape(-1, 6)
    n = len(ics)
    g = make_grids(grids)
    nlos, nden = g.nx * g.ny * g.nv, g.dx * g.dy * g.dz
    P = (Projection * len(projections))(*[Projection(*p) for p in projections])
    losvd = np.empty((len(projections), n, nlos), dtype=np.float32)
    dens = np.empty((n, nden), dtype=np.float32)
    nout = np.empty((len(projections) + 1, n), dtype=np.int32)
    near = np.empty_like(nout)
    diag = np.empty((n, 2)) if want_diag else None
    d = make_desc(spec)
    _chk(lib().smo_build_library(C.byref(d), _dp(ics), C.c_int64(n), C.c_double(dt), C.c_int64(n_steps),
                                 C.c_int32(stride), P, C.c_int(len(projections)), C.byref(g), C.c_int(state_prec),
                                 _dp(losvd), _dp(dens), _dp(nout), _dp(diag) if want_diag else None, _dp(near)),
         "smo_build_library")
    return dict(losvd=losvd, dens=dens, nout=nout, near_edge=near, diag=diag)


def build_bundled_library(spec, ics, dt, n_steps, stride, projections, grids, n_bundle=1, fourfold=True):
    """Symmetrised orbit bundles -> dict(losvd[n_proj,n_rows,nlos], dens[n_rows,nden], nout[n_proj+1,n_rows], near_edge)."""
    ics = np.ascontiguousarray(ics, dtype=np.float64).reshape(-1, 6)
    n = len(ics)
    n_rows = n // n_bundle
    g = make_grids(grids)
    nlos, nden = g.nx * g.ny * g.nv, g.dx * g.dy * g.dz
    P = (Projection * len(projections))(*[Projection(*p) for p in projections])
    losvd = np.empty((len(projections), n_rows, nlos), dtype=np.float32)
    dens = np.empty((n_rows, nden), dtype=np.float32)
    nout = np.empty((len(projections) + 1, n_rows), dtype=np.int32)
    near = np.empty_like(nout)
    d = make_desc(spec)
    _chk(lib().smo_build_bundled_library(C.byref(d), _dp(ics), C.c_int64(n), C.c_double(dt), C.c_int64(n_steps),
                                         C.c_int32(stride), P, C.c_int(len(projections)), C.byref(g), C.c_int32(n_bundle),
                                         C.c_int(int(fourfold)), _dp(losvd), _dp(dens), _dp(nout), _dp(near)),
         "smo_build_bundled_library")
    return dict(losvd=losvd, dens=dens, nout=nout, near_edge=near)


def build_observable_library(spec, ics, dt, n_steps, stride, projections, grids, ap_map, n_ap, n_bundle=1, fourfold=False,
                             density_mode=0):
    """Aperture-regrouped rows -> dict(losvd[n_proj,n_rows,n_ap*nv], dens, nout, near_edge); ap_map[ny*nx] int32, < 0 = no aperture."""
    ics = np.ascontiguousarray(ics, dtype=np.float64).reshape(-1, 6)
    n = len(ics)
    n_rows = n // n_bundle
    g = make_grids(grids)
    if ap_map is not None:
        ap_map = np.ascontiguousarray(ap_map, dtype=np.int32).reshape(-1)
        if len(ap_map) != g.nx * g.ny:
            raise ValueError("ap_map must have ny*nx entries")
    nlos, nden = (n_ap if ap_map is not None else g.nx * g.ny) * g.nv, g.dx * g.dy * g.dz
    P = (Projection * len(projections))(*[Projection(*p) for p in projections])
    losvd = np.empty((len(projections), n_rows, nlos), dtype=np.float32)
    dens = np.empty((n_rows, nden), dtype=np.float32)
    nout = np.empty((len(projections) + 1, n_rows), dtype=np.int32)
    near = np.empty_like(nout)
    d = make_desc(spec)
    _chk(lib().smo_build_observable_library(C.byref(d), _dp(ics), C.c_int64(n), C.c_double(dt), C.c_int64(n_steps),
                                            C.c_int32(stride), P, C.c_int(len(projections)), C.byref(g), C.c_int32(n_bundle),
                                            C.c_int(int(fourfold)), _dp(ap_map) if ap_map is not None else None, C.c_int32(n_ap),
                                            C.c_int(density_mode), _dp(losvd), _dp(dens), _dp(nout), _dp(near)),
         "smo_build_observable_library")
    return dict(losvd=losvd, dens=dens, nout=nout, near_edge=near)


def gh_terms(w):
    w = np.ascontiguousarray(w, dtype=np.float64).reshape(-1)
    out = np.empty((len(w), 5))
    _chk(lib().smo_gh_terms(_dp(w), C.c_int64(len(w)), _dp(out)), "smo_gh_terms")
    return out


def build_gh_library(spec, ics, dt, n_steps, stride, projections, grids, ap_map, n_ap, v0, s, n_bundle=1, fourfold=False,
                     density_mode=0):
    """Gauss-Hermite matrices -> dict(gh[n_proj,n_rows,n_ap,6] float64, dens, nout, near_edge)."""
    ics = np.ascontiguousarray(ics, dtype=np.float64).reshape(-1, 6)
    n = len(ics)
    n_rows = n // n_bundle
    g = make_grids(grids)
    ap_map = np.ascontiguousarray(ap_map, dtype=np.int32).reshape(-1)
    v0 = np.ascontiguousarray(v0, dtype=np.float64).reshape(-1)
    s = np.ascontiguousarray(s, dtype=np.float64).reshape(-1)
    if len(ap_map) != g.nx * g.ny or len(v0) != n_ap or len(s) != n_ap:
        raise ValueError("ap_map needs ny*nx entries, v0 and s need n_ap")
    P = (Projection * len(projections))(*[Projection(*p) for p in projections])
    gh = np.empty((len(projections), n_rows, n_ap, 6))
    dens = np.empty((n_rows, g.dx * g.dy * g.dz), dtype=np.float32)
    nout = np.empty((len(projections) + 1, n_rows), dtype=np.int32)
    near = np.empty_like(nout)
    d = make_desc(spec)
    _chk(lib().smo_build_gh_library(C.byref(d), _dp(ics), C.c_int64(n), C.c_double(dt), C.c_int64(n_steps), C.c_int32(stride),
                                    P, C.c_int(len(projections)), C.byref(g), C.c_int32(n_bundle), C.c_int(int(fourfold)),
                                    _dp(ap_map), C.c_int32(n_ap), _dp(v0), _dp(s), C.c_int(density_mode), _dp(gh), _dp(dens),
                                    _dp(nout), _dp(near)), "smo_build_gh_library")
    return dict(gh=gh, dens=dens, nout=nout, near_edge=near)


def ferrers_lambda(a, b, c, xyz):
    xyz = np.ascontiguousarray(xyz, dtype=np.float64).reshape(-1, 3)
    lam = np.empty(len(xyz))
    _chk(lib().smo_ferrers_lambda(C.c_double(a), C.c_double(b), C.c_double(c), _dp(xyz), C.c_int64(len(xyz)), _dp(lam)),
         "smo_ferrers_lambda")
    return lam


def ferrers_W(a, b, c, lam):
    W = np.empty(20)
    _chk(lib().smo_ferrers_W(C.c_double(a), C.c_double(b), C.c_double(c), C.c_double(lam), _dp(W)), "smo_ferrers_W")
    return dict(zip(W_ORDER, W))


def project(angles, xb, vb):
    p = Projection(*angles)
    xb = np.ascontiguousarray(xb, dtype=np.float64)
    vb = np.ascontiguousarray(vb, dtype=np.float64)
    out = np.empty(3)
    _chk(lib().smo_project(C.byref(p), _dp(xb), _dp(vb), _dp(out)), "smo_project")
    return out


def jacobi(spec, state, t=0.0):
    state = np.ascontiguousarray(state, dtype=np.float64).reshape(-1, 6)
    ej = np.empty(len(state))
    d = make_desc(spec)
    _chk(lib().smo_jacobi(C.byref(d), _dp(state), C.c_int64(len(state)), C.c_double(t), _dp(ej)), "smo_jacobi")
    return ej


def num_threads():
    return lib().smo_num_threads()
