"""Pins for the oracle's force field (-m "not gpu").

Each pin is independent of the oracle's own formulas: mpmath quadrature of the DEFINING
integrals (not the Carlson/recursion route the oracle takes), numerical differentiation of the
paper's potentials (Eq.8, Eq.10), Poisson's equation, far-field limits, and the stored
reference values of tests/golden/config1_force_pins.txt.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

from paper_2607_00117_b200 import inputs

mp.mp.dps = 30
G = inputs.G_GALACTIC
A_, B_, C_ = 4.0, 1.5, 0.5
MBAR = 1e10
POT1 = inputs.CONFIGS[1]["potential"]


def single(comp, omega_p=0.0):
    return {"G": G, "omega_p": omega_p, "phase0": 0.0, "components": [comp]}


MN = single(POT1["components"][0])
FER = single((inputs.FERRERS2, 0, [MBAR, A_, B_, C_]))
HALO = single(POT1["components"][2])


def mp_lambda(x, y, z):
    a2, b2, c2 = mp.mpf(A_) ** 2, mp.mpf(B_) ** 2, mp.mpf(C_) ** 2
    X, Y, Z = mp.mpf(x) ** 2, mp.mpf(y) ** 2, mp.mpf(z) ** 2
    if X / a2 + Y / b2 + Z / c2 <= 1:
        return mp.mpf(0)
    f = lambda u: X / (a2 + u) + Y / (b2 + u) + Z / (c2 + u) - 1
    lo, hi = mp.mpf(0), X + Y + Z  # f(lo) > 0 > f(hi)
    return mp.findroot(f, (lo, hi), solver="anderson", tol=1e-40, maxsteps=200)


def mp_ferrers(x, y, z):
    """Phi and F straight from the homoeoid integrals (Binney & Tremaine 2008 eq. 2.140 form):
    Phi = -(pi G abc rho_c/3) int_lam^inf (1-m^2(u))^3 du/Delta ; dPhi/dx_i = 2 pi G abc rho_c x_i
    int_lam^inf (1-m^2(u))^2 du/((a_i^2+u) Delta), rho_c = 105 M/(32 pi abc)."""
    a2, b2, c2 = mp.mpf(A_) ** 2, mp.mpf(B_) ** 2, mp.mpf(C_) ** 2
    x, y, z = mp.mpf(x), mp.mpf(y), mp.mpf(z)
    lam = mp_lambda(x, y, z)
    rho_c = 105 * mp.mpf(MBAR) / (32 * mp.pi * A_ * B_ * C_)
    K = mp.pi * mp.mpf(G) * A_ * B_ * C_ * rho_c
    D = lambda u: mp.sqrt((a2 + u) * (b2 + u) * (c2 + u))
    m2 = lambda u: x * x / (a2 + u) + y * y / (b2 + u) + z * z / (c2 + u)
    brk = [lam, lam + 1, lam + 10, lam + 100, lam + 1e4, mp.inf]
    phi = -(K / 3) * mp.quad(lambda u: (1 - m2(u)) ** 3 / D(u), brk)
    F = [-2 * K * xi * mp.quad(lambda u: (1 - m2(u)) ** 2 / ((ai + u) * D(u)), brk)
         for xi, ai in ((x, a2), (y, b2), (z, c2))]
    return lam, phi, F


FERRERS_POINTS = [(1, 0.5, 0.1), (5, 2, 1), (10, -7, 0.3), (0.3, -0.2, 0.05), (3.9, 0.1, 0.02), (4.05, 0.0, 0.0),
                  (0, 1.6, 0), (0.0, 0.0, 0.7), (-2.5, 1.0, -0.3), (30, -20, 10), (80, 5, 2), (0.5, 0.4, 0.45)]


@pytest.mark.parametrize("pt", FERRERS_POINTS)
def test_ferrers_force_vs_defining_integral(smo, pt):
    lam, phi, F = mp_ferrers(*pt)
    Fo, Po = smo.eval_force(FER, [pt])
    lo = smo.ferrers_lambda(A_, B_, C_, [pt])[0]
    assert lo == pytest.approx(float(lam), rel=1e-14, abs=1e-15)
    assert Po[0] == pytest.approx(float(phi), rel=2e-15)
    scale = max(abs(float(f)) for f in F)
    for j in range(3):
        assert abs(Fo[0, j] - float(F[j])) <= 3e-15 * scale


@pytest.mark.parametrize("lam", [0.0, 0.37, 5.0, 200.0, 2000.0])
def test_ferrers_W_vs_quadrature(smo, lam):
    a2, b2, c2 = mp.mpf(A_) ** 2, mp.mpf(B_) ** 2, mp.mpf(C_) ** 2
    W = smo.ferrers_W(A_, B_, C_, lam)
    L = mp.mpf(lam)
    for key, val in W.items():
        i, j, k = (int(ch) for ch in key)
        f = lambda u: 1 / (mp.sqrt((a2 + u) * (b2 + u) * (c2 + u)) * (a2 + u) ** i * (b2 + u) ** j * (c2 + u) ** k)
        ref = mp.quad(f, [L, L + 1, L + 10, L + 100, L + 1e4, mp.inf])
        assert val == pytest.approx(float(ref), rel=3e-16), key


def test_golden_pins(smo):
    path = os.path.join(os.path.dirname(__file__), "golden", "config1_force_pins.txt")
    pots = {"MN": MN, "NFW": HALO, "FERRERS": FER}
    n = 0
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        name, *vals = line.split()
        x, y, z, phi, fx, fy, fz = map(float, vals)
        F, P = smo.eval_force(pots[name], [[x, y, z]])
        assert P[0] == pytest.approx(phi, rel=2e-14)
        assert F[0] == pytest.approx([fx, fy, fz], rel=2e-14)
        n += 1
    assert n == 9
    _, P0 = smo.eval_force(FER, [[0, 0, 0]])
    assert P0[0] == pytest.approx(-50271.6906051041, rel=2e-14)
    assert smo.ferrers_lambda(A_, B_, C_, [[5, 2, 1], [10, -7, 0.3]]) == pytest.approx(
        [17.6447035812083, 137.907356967128], rel=1e-14)


def test_paper_eq8_eq10_gradients(smo):
    """F = -grad Phi with Phi typed from PAPER.md Eq.8 (NFW, M_DM = 4 pi rho_s r_s^3) and Eq.10 (MN)."""
    GMd, a, b = mp.mpf(G) * 5e10, 3, mp.mpf("0.3")
    GMh, rs = mp.mpf(G) * 4 * mp.pi * 1e7 * 15 ** 3, 15
    phi_mn = lambda x, y, z: -GMd / mp.sqrt(x * x + y * y + (a + mp.sqrt(z * z + b * b)) ** 2)
    phi_nfw = lambda x, y, z: -GMh * mp.log(1 + mp.sqrt(x * x + y * y + z * z) / rs) / mp.sqrt(x * x + y * y + z * z)
    rng = np.random.default_rng(5)
    pts = rng.normal(size=(12, 3)) * [6, 6, 1.5]
    pts[0] = [1e-3, 2e-3, -1e-3]  # small radius: the cancellation-prone NFW regime
    pts[1] = [0.02, 0.0, 0.01]
    for pot, phi in ((MN, phi_mn), (HALO, phi_nfw)):
        F, P = smo.eval_force(pot, pts)
        for i, p in enumerate(pts):
            ref = [-mp.diff(phi, tuple(p), n=tuple(int(k == j) for k in range(3))) for j in range(3)]
            assert P[i] == pytest.approx(float(phi(*p)), rel=2e-15)
            s = max(abs(float(r)) for r in ref)
            assert np.max(np.abs(F[i] - np.array([float(r) for r in ref]))) <= 3e-15 * s


def test_circular_speeds_closed_form(smo):
    R = np.array([3.0, 8.0, 20.0])
    pts = np.stack([R, 0 * R, 0 * R], axis=1)
    vc_mn = np.sqrt(-R * smo.eval_force(MN, pts)[0][:, 0])
    vc_h = np.sqrt(-R * smo.eval_force(HALO, pts)[0][:, 0])
    # v_c^2 = R dPhi/dR: MN  GM R^2/(R^2+(a+b)^2)^{3/2};  NFW  GM_DM [ln(1+X)-X/(1+X)]/R
    ref_mn = np.sqrt(G * 5e10 * R ** 2 / (R ** 2 + 3.3 ** 2) ** 1.5)
    X = R / 15.0
    ref_h = np.sqrt(G * 4 * math.pi * 1e7 * 15.0 ** 3 * (np.log1p(X) - X / (1 + X)) / R)
    assert vc_mn == pytest.approx(ref_mn, rel=1e-14)
    assert vc_h == pytest.approx(ref_h, rel=1e-13)
    assert vc_mn == pytest.approx([147.710152626, 145.726083668, 101.62510243], rel=1e-10)
    assert vc_h == pytest.approx([97.5632777548, 134.735624508, 158.620267469], rel=1e-10)
    # Plummer G=M=b=1 (BASELINE.json configs[0])
    Fp, Pp = smo.eval_force(inputs.plummer_potential(), [[1.0, 0, 0], [0, 0, 0]])
    assert math.sqrt(-Fp[0, 0]) == pytest.approx(0.594603557501361, rel=1e-14)
    assert Pp[1] == pytest.approx(-1.0, rel=1e-15)
    # azimuthally averaged total v_c used by the IC recipe
    pts = inputs.vc_probe_points(R)
    vc = inputs.vc_from_forces(R, pts, smo.eval_force(POT1, pts, want_phi=False))
    assert vc == pytest.approx([222.36, 211.89, 194.03], abs=6e-3)


def test_ferrers_poisson_and_far_field(smo):
    """div F = -4 pi G rho inside the bar (rho = rho_c (1-m^2)^2), 0 outside; F -> -GM x/r^3 far away."""
    h = 2e-3
    rho_c = 105 * MBAR / (32 * math.pi * A_ * B_ * C_)
    for pt in [(0.5, 0.3, 0.1), (2.0, -0.5, 0.2), (0, 0, 0), (3.0, 0.2, -0.1), (5.0, 1.0, 0.5), (1.0, 2.0, 0.0)]:
        p = np.array(pt, float)
        stencil = np.array([p + s * h * e for e in np.eye(3) for s in (2, 1, -1, -2)])
        F = smo.eval_force(FER, stencil, want_phi=False).reshape(3, 4, 3)
        div = sum((-F[j, 0, j] + 8 * F[j, 1, j] - 8 * F[j, 2, j] + F[j, 3, j]) / (12 * h) for j in range(3))
        m2 = p[0] ** 2 / A_ ** 2 + p[1] ** 2 / B_ ** 2 + p[2] ** 2 / C_ ** 2
        rho = rho_c * (1 - m2) ** 2 if m2 < 1 else 0.0
        assert div == pytest.approx(-4 * math.pi * G * rho, rel=1e-7, abs=1e-7 * 4 * math.pi * G * rho_c)
    far = np.array([[300.0, -200.0, 100.0]])
    F = smo.eval_force(FER, far, want_phi=False)[0]
    r = np.linalg.norm(far)
    assert F == pytest.approx(-G * MBAR * far[0] / r ** 3, rel=2e-4)  # quadrupole ~ (a/r)^2
    # reflection symmetries of a triaxial bar (Table 1 relies on them)
    base = np.array([1.3, -0.7, 0.2])
    F0 = smo.eval_force(FER, [base], want_phi=False)[0]
    for sgn in ([1, 1, -1], [-1, -1, 1], [-1, 1, 1]):
        Fs = smo.eval_force(FER, [base * sgn], want_phi=False)[0]
        assert np.array_equal(Fs, F0 * sgn)


def test_force_is_minus_grad_phi_total_rotating(smo):
    """Total config-1 force at t != 0 (bar rotated by Omega_p t) against central differences of the oracle's Phi,
    and against rotating the t=0 field by hand."""
    t = 0.0137
    rng = np.random.default_rng(11)
    pts = rng.normal(size=(8, 3)) * [5, 5, 1]
    h = 1e-4
    F, _ = smo.eval_force(POT1, pts, t)
    for j in range(3):
        e = np.zeros(3); e[j] = h
        Pp = smo.eval_force(POT1, pts + e, t)[1]
        Pm = smo.eval_force(POT1, pts - e, t)[1]
        Pp2 = smo.eval_force(POT1, pts + 2 * e, t)[1]
        Pm2 = smo.eval_force(POT1, pts - 2 * e, t)[1]
        grad = (-Pp2 + 8 * Pp - 8 * Pm + Pm2) / (12 * h)
        assert F[:, j] == pytest.approx(-grad, rel=1e-7, abs=1e-5)
    th = 40.0 * t
    c, s = math.cos(th), math.sin(th)
    Rm = np.array([[c, s, 0], [-s, c, 0], [0, 0, 1]])  # inertial -> bar frame
    bar_only = single((inputs.FERRERS2, 1, [MBAR, A_, B_, C_]), omega_p=40.0)
    Fb_t = smo.eval_force(bar_only, pts, t, want_phi=False)
    Fb_0 = smo.eval_force(FER, pts @ Rm.T, 0.0, want_phi=False) @ Rm
    assert Fb_t == pytest.approx(Fb_0, rel=1e-13, abs=1e-11)
