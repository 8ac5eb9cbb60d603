"""Seeded synthetic inputs and the five workload definitions of BASELINE.json `configs`.

This module serves BOTH the CUDA product's tests/bench and the CPU oracle, so it holds none of
the method's arithmetic: no force, no integrator, no projection, no binning.  Where an input
recipe needs the circular speed of the trial potential (BASELINE.json configs[1]: "circular
velocity times (1+N(0,0.1))"), the caller passes a force callback; tests pass the oracle's,
bench.py passes the CUDA library's.  Recipes follow DESIGN.md "Input recipe".

A potential is a plain dict: {"G", "omega_p", "phase0", "components": [(kind, rotating, [p...])]}
with kind 1=Plummer{M,b}, 2=Miyamoto-Nagai{M,a,b}, 3=NFW{rho_s,r_s}, 4=Ferrers n=2{M,a,b,c}.
"""
import math

import numpy as np

PLUMMER, MIYAMOTO_NAGAI, NFW, FERRERS2, DEHNEN_T3, DEHNEN_V4 = 1, 2, 3, 4, 5, 6
G_GALACTIC = 4.30091e-6  # kpc (km/s)^2 / Msun, BASELINE.json configs[1]
DEG = math.pi / 180.0


def plummer_potential():
    return {"G": 1.0, "omega_p": 0.0, "phase0": 0.0, "components": [(PLUMMER, 0, [1.0, 1.0])]}


def barred_potential(scale=None, omega_scale=1.0):
    """Config-1 potential (BASELINE.json configs[1]).  scale: optional 10 multipliers in the order
    disc M,a,b; bar M,a,b,c; halo rho_s,r_s (omega_p has its own) used by the config-3 trials."""
    s = [1.0] * 9 if scale is None else list(scale)
    return {"G": G_GALACTIC, "omega_p": 40.0 * omega_scale, "phase0": 0.0,
            "components": [(MIYAMOTO_NAGAI, 0, [5e10 * s[0], 3.0 * s[1], 0.3 * s[2]]),
                           (FERRERS2, 1, [1e10 * s[3], 4.0 * s[4], 1.5 * s[5], 0.5 * s[6]]),
                           (NFW, 0, [1e7 * s[7], 15.0 * s[8]])]}


def paper_bar_potential(M_b=1e10, L_b=4.0, M_d=5e10, R_d=3.0, H_d=0.3, omega_p=40.0):
    """The paper's own stellar model: Miyamoto-Nagai disc + Dehnen & Aly (2023) long bar T_3
    (eta = 1, (a, b, L) = (L_b/5, b_d, L_b)) + boxy/peanut bulge V_4 (eta = 0, (a, b, L) = (0.5, 0.5, 0.1) kpc), with the
    NFW halo of BASELINE.json configs[1].  The paper ties the two bar masses and calls M_b "the total bar mass": each
    component carries M_b/2 here (reading R21); the fitted values are not printed, so M_b, L_b, Omega_p are
    configs[1]'s bar mass, bar half-length and pattern speed."""
    return {"G": G_GALACTIC, "omega_p": omega_p, "phase0": 0.0,
            "components": [(MIYAMOTO_NAGAI, 0, [M_d, R_d, H_d]),
                           (DEHNEN_T3, 1, [0.5 * M_b, L_b / 5.0, H_d, L_b, 1.0]),
                           (DEHNEN_V4, 1, [0.5 * M_b, 0.5, 0.5, 0.1, 0.0]),
                           (NFW, 0, [1e7, 15.0])]}


def _grids(n_pix, n_v, n_dens, half_xy, half_v, half_d):
    return {"nx": n_pix, "ny": n_pix, "nv": n_v, "x0": -half_xy, "x1": half_xy, "y0": -half_xy, "y1": half_xy,
            "v0": -half_v, "v1": half_v, "dx": n_dens, "dy": n_dens, "dz": n_dens,
            "bx0": -half_d, "bx1": half_d, "by0": -half_d, "by1": half_d, "bz0": -half_d, "bz1": half_d}


# (alpha, beta, gamma): bar angle to the line of nodes -> alpha, inclination -> beta,
# position angle -> gamma; gamma = 0 where BASELINE.json does not state it.
CONFIGS = {
    0: dict(name="cfg0_plummer_tiny", potential=plummer_potential(), ics="plummer", n_orb=1000, dt=0.01,
            n_steps=1000, stride=1, projections=[(0.0, 60 * DEG, 0.0)], grids=_grids(10, 15, 10, 5.0, 1.5, 5.0),
            precision="f64", seed=0),
    1: dict(name="cfg1_barred", potential=barred_potential(), ics="disc", n_orb=20000, dt=1e-3, n_steps=10000,
            stride=5, projections=[(30 * DEG, 45 * DEG, 0.0)], grids=_grids(40, 30, 24, 10.0, 450.0, 12.0),
            precision="f64", seed=1),
    2: dict(name="cfg2_library", potential=barred_potential(), ics="disc", n_orb=100000, dt=1e-3, n_steps=20000,
            stride=10, projections=[(30 * DEG, 45 * DEG, 0.0)], grids=_grids(60, 40, 32, 10.0, 450.0, 12.0),
            precision="f64+f32", seed=2),
    3: dict(name="cfg3_mcmc_batch", potential=barred_potential(), ics="disc", n_orb=20000, n_trials=64, dt=1e-3,
            n_steps=10000, stride=5, projections=[(30 * DEG, 45 * DEG, 0.0)],
            grids=_grids(40, 30, 24, 10.0, 450.0, 12.0), precision="f32", seed=3),
    4: dict(name="cfg4_stress", potential=barred_potential(), ics="disc", n_orb=500000, dt=1e-3, n_steps=50000,
            stride=20, projections=[(30 * DEG, b * DEG, 0.0) for b in (20, 50, 80)],
            grids=_grids(64, 48, 40, 10.0, 450.0, 12.0), precision="f64", seed=4),
}


def plummer_ics(n, seed):
    """Config 0: r = (u^(-2/3)-1)^(-1/2), isotropic directions; speed v = q*sqrt(2)*(1+r^2)^(-1/4)
    with q drawn by rejection under g(q) = q^2 (1-q^2)^(7/2) <= 0.1 (the standard Plummer recipe)."""
    rng = np.random.default_rng(seed)
    u = rng.uniform(1e-10, 1.0, n)
    r = 1.0 / np.sqrt(u ** (-2.0 / 3.0) - 1.0 + 1e-300)

    def iso(m):
        ct = rng.uniform(-1.0, 1.0, m)
        ph = rng.uniform(0.0, 2 * math.pi, m)
        st = np.sqrt(1.0 - ct * ct)
        return np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)

    pos = r[:, None] * iso(n)
    q = np.empty(n)
    todo = np.arange(n)
    while len(todo):
        x1 = rng.uniform(0.0, 1.0, len(todo))
        x2 = rng.uniform(0.0, 0.1, len(todo))
        ok = x2 < x1 * x1 * (1.0 - x1 * x1) ** 3.5
        q[todo[ok]] = x1[ok]
        todo = todo[~ok]
    speed = q * math.sqrt(2.0) * (1.0 + r * r) ** -0.25
    vel = speed[:, None] * iso(n)
    return np.ascontiguousarray(np.concatenate([pos, vel], axis=1))


def disc_deviates(n, seed, R_d=3.0, z0=0.3):
    """Positions R ~ Gamma(2,R_d) (exponential disc), phi ~ U(0,2pi), z ~ sech^2(z/z0), and four
    standard-normal deviates per orbit; the velocity scale comes later from v_c(R)."""
    rng = np.random.default_rng(seed)
    u1 = rng.uniform(1e-12, 1.0, n)
    u2 = rng.uniform(1e-12, 1.0, n)
    phi = rng.uniform(0.0, 2 * math.pi, n)
    uz = rng.uniform(1e-9, 1.0 - 1e-9, n)
    g = rng.standard_normal((4, n))
    return {"R": -R_d * np.log(u1 * u2), "phi": phi, "z": z0 * np.arctanh(2.0 * uz - 1.0), "g": g}


N_AZIMUTH = 64


def vc_probe_points(R):
    """Points (len(R)*64, 3) at z=0 on 64 mid-point azimuths for the axisymmetrised circular speed."""
    az = 2 * math.pi * (np.arange(N_AZIMUTH) + 0.5) / N_AZIMUTH
    x = R[:, None] * np.cos(az)[None, :]
    y = R[:, None] * np.sin(az)[None, :]
    return np.ascontiguousarray(np.stack([x, y, np.zeros_like(x)], axis=-1).reshape(-1, 3))


def vc_from_forces(R, pts, F):
    """v_c^2(R) = -R <F_R>_phi with the bar at theta = 0 ('axisymmetrised version')."""
    FR = (pts[:, 0] * F[:, 0] + pts[:, 1] * F[:, 1]).reshape(len(R), N_AZIMUTH) / R[:, None]
    return np.sqrt(np.maximum(-R * FR.mean(axis=1), 0.0))


def disc_ics(dev, vc, sigma=(30.0, 30.0, 20.0), frac=0.1):
    R, phi, z, g = dev["R"], dev["phi"], dev["z"], dev["g"]
    vR = sigma[0] * g[0]
    vphi = vc * (1.0 + frac * g[1]) + sigma[1] * g[2]
    vz = sigma[2] * g[3]
    c, s = np.cos(phi), np.sin(phi)
    return np.ascontiguousarray(np.stack([R * c, R * s, z, vR * c - vphi * s, vR * s + vphi * c, vz], axis=1))


def make_ics(cfg, force_fn, n_orb=None, potential=None):
    """ICs [n,6] for a config.  force_fn(potential_dict, xyz[n,3]) -> F[n,3] at t=0 (used only for
    v_c of disc configs).  n_orb truncates the SAME seeded stream (first n orbits)."""
    n = cfg["n_orb"]
    if cfg["ics"] == "plummer":
        ics = plummer_ics(n, cfg["seed"])
        return ics[:n_orb] if n_orb else ics
    dev = disc_deviates(n, cfg["seed"])
    if n_orb:
        dev = {"R": dev["R"][:n_orb], "phi": dev["phi"][:n_orb], "z": dev["z"][:n_orb], "g": dev["g"][:, :n_orb]}
    pot = potential if potential is not None else cfg["potential"]
    pts = vc_probe_points(dev["R"])
    vc = vc_from_forces(dev["R"], pts, force_fn(pot, pts))
    return disc_ics(dev, vc)


def trial_draws(n_trials, seed):
    """Config 3: per trial, 9 potential multipliers + omega_p multiplier ~ U(0.7,1.3), beta and alpha
    multipliers ~ U(0.7,1.3) around 45 and 30 deg, gamma ~ U(0,pi); one stream, trial-major."""
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(n_trials):
        m = rng.uniform(0.7, 1.3, 10)
        ang = rng.uniform(0.7, 1.3, 2)
        gam = rng.uniform(0.0, math.pi)
        # order of m: disc M,a,b; bar M,a,b,c,Omega_p; halo rho_s,r_s
        scale = [m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[8], m[9]]
        out.append({"potential": barred_potential(scale, omega_scale=m[7]),
                    "projection": (30 * DEG * ang[1], 45 * DEG * ang[0], gam)})
    return out


def aperture_map(grids, n_ap, seed=0):
    """Synthetic stand-in for a pre-defined Voronoi binning ("~600 apertures"): every image pixel is
    assigned to the nearest of n_ap seeded generators, denser towards the centre as adaptive binning is -> int32 [ny*nx]."""
    rng = np.random.default_rng(seed)
    nx, ny = grids["nx"], grids["ny"]
    r = np.sqrt(rng.uniform(0, 1, n_ap)) ** 1.5 * 0.72
    phi = rng.uniform(0, 2 * math.pi, n_ap)
    gx, gy = (0.5 + r * np.cos(phi)) * nx, (0.5 + r * np.sin(phi)) * ny
    yy, xx = np.meshgrid(np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    d2 = (xx[..., None] - gx) ** 2 + (yy[..., None] - gy) ** 2
    return d2.argmin(-1).astype(np.int32).reshape(-1)


def weight_problem(n_orb, n_dens, n_ap, n_rhs, seed=0, fill=0.08):
    """Seeded stand-in for the inputs of the weight solve: library-shaped matrices and mock targets.

    The paper's targets come from its mock galaxy, which is not available; here they are the model of a hidden
    non-negative weight vector (half of the orbits unused), so a good fit exists.  Returns a dict of numpy arrays:
      dens [n_orb][n_dens] f32     counts; every orbit visits about `fill` of the cells (sparse rows, like a library)
      gh   [n_orb][n_ap][6] f32    the sm_build_gh_library layout: [0] counts, [1] the m = 0 sum, [2..5] the m = 1..4 sums
      blocks                       the stacking order of Eq. 3 as (array name, col0, col_stride, n_cols): density, surface
                                   density, h_1..h_4
      target, sigma [n_con]        observed values and tolerances: 1 % of the target for the two density blocks
                                   (PAPER.md:125), for h_m 2 % of the aperture's surface-density target (floored)
      xi [n_rhs][n_con]            unit normal bootstrap draws, zero on the 3-D density rows; row 0 is zero
      keep [n_orb] u8              the drift cut: about 0.1 % of the orbits dropped
    """
    rng = np.random.default_rng([seed, n_orb, n_dens, n_ap])
    dens = (rng.random((n_orb, n_dens)) < fill) * rng.integers(1, 200, (n_orb, n_dens))
    cnt = (rng.random((n_orb, n_ap)) < fill) * rng.integers(1, 400, (n_orb, n_ap))
    gh = np.zeros((n_orb, n_ap, 6), dtype=np.float32)
    gh[:, :, 0] = cnt
    gh[:, :, 1] = cnt * (0.25 + 0.05 * rng.random((n_orb, n_ap)))
    for m in range(1, 5):
        gh[:, :, 1 + m] = cnt * (0.1 / m) * rng.standard_normal((n_orb, n_ap))
    dens = dens.astype(np.float32)
    w_true = rng.random(n_orb) * (rng.random(n_orb) < 0.5) / n_orb
    blocks = [("dens", 0, 1, n_dens), ("gh", 0, 6, n_ap)] + [("gh", 1 + m, 6, n_ap) for m in range(1, 5)]
    t_dens = w_true @ dens.astype(np.float64)
    t_gh = np.einsum("i,iac->ca", w_true, gh.astype(np.float64))     # [6][n_ap]
    target = np.concatenate([t_dens, t_gh[0]] + [t_gh[1 + m] for m in range(1, 5)])
    floor_d, floor_s = 1e-3 * t_dens.max(), 1e-3 * t_gh[0].max()
    s_sigma = 0.01 * np.maximum(t_gh[0], floor_s)
    sigma = np.concatenate([0.01 * np.maximum(t_dens, floor_d), s_sigma] + [2.0 * s_sigma] * 4)
    xi = rng.standard_normal((n_rhs, target.size))
    xi[:, :n_dens] = 0.0
    xi[0] = 0.0
    target = target + sigma * np.concatenate([np.zeros(n_dens), rng.standard_normal(5 * n_ap)])   # the mock data are noisy
    keep = (rng.random(n_orb) >= 1e-3).astype(np.uint8)
    return {"dens": dens, "gh": gh, "blocks": blocks, "target": target, "sigma": sigma, "xi": xi, "keep": keep,
            "n_con": int(target.size)}
