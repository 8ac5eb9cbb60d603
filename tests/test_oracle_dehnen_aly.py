"""Pins for the oracle's Dehnen & Aly (2023) needle bars T_3 and V_4 (-m "not gpu").

The oracle evaluates the closed form of the needle convolution (elementary antiderivatives).  The pins take other routes:
mpmath quadrature of the DEFINING integral PAPER.md:217 Eq. 12 with the coefficients of PAPER.md:489-495 Appendix A;
Poisson's equation against the paper's printed DENSITIES (an independent set of printed coefficients) convolved with the
same needle; numerical differentiation of the potential; the limits L -> 0 (parent pair), a -> 0 (Plummer), r -> infinity
(monopole of mass M_b); the reflection symmetries of PAPER.md:77-90.
"""
import mpmath as mp
import numpy as np
import pytest

from paper_2607_00117_b200 import inputs

mp.mp.dps = 30
G = inputs.G_GALACTIC
M = 5e9
T3P = dict(a=0.8, b=0.3, L=4.0, eta=1.0)     # (a, b, L)_T3 = (L_b/5, b_d, L_b), eta = 1
V4P = dict(a=0.5, b=0.5, L=0.1, eta=0.0)     # (a, b, L)_V4 = (0.5, 0.5, 0.1) kpc, eta = 0
GEN = dict(a=0.7, b=0.4, L=1.3, eta=-0.6)    # a generic needle, both eta terms active


def spec(kind, p, M_=M):
    return {"G": G, "omega_p": 0.0, "phase0": 0.0, "components": [(kind, 0, [M_, p["a"], p["b"], p["L"], p["eta"]])]}


def needle(u, L, eta):
    return (1 + eta * (1 - 2 * abs(u) / L)) / (2 * L)


def parent_phi(kind, R2, z, a, b):
    """Appendix A as printed, with R^2 = R2 + Z^2 (R2 = cylindrical radius squared)."""
    zeta = mp.sqrt(z * z + b * b); Z = a + zeta; Rc = mp.sqrt(R2 + Z * Z)
    if kind == inputs.DEHNEN_T3:
        return -(1 / Rc + a * (Z - a / 3) / Rc ** 3 + a * a * Z * Z / Rc ** 5)
    return -(1 / Rc + (a * (Z - 2 * a / 5) + b * b / 2) / Rc ** 3
             + 3 * a * (a * Z * (2 * Z - a) / 5 + b * b / 2 * (Z - a / 5)) / Rc ** 5
             + a * a * Z * Z * (a * Z + 3 * b * b) / Rc ** 7 + 7 * a ** 3 * b * b * Z ** 4 / (2 * Rc ** 9 * zeta))


def parent_rho(kind, R2, z, a, b):
    """The printed densities (per unit mass)."""
    zeta = mp.sqrt(z * z + b * b); Z = a + zeta; Rc = mp.sqrt(R2 + Z * Z)
    if kind == inputs.DEHNEN_T3:
        return b * b / (4 * mp.pi) * (3 / Rc ** 5 + 5 * a * Z * Z * (3 * zeta ** 2 - 2 * a * zeta + a * a) / (Rc ** 7 * zeta ** 3)
                                      + 35 * a * a * Z ** 4 / (Rc ** 9 * zeta ** 2))
    return 3 * b ** 4 / (8 * mp.pi) * (5 / Rc ** 7
                                       + 7 * a * Z * Z * (5 * zeta ** 4 - 4 * a * zeta ** 3 + 3 * a * a * zeta ** 2 - 2 * a ** 3 * zeta + a ** 4) / (Rc ** 9 * zeta ** 5)
                                       + 63 * a * a * Z ** 4 * (2 * zeta ** 2 - 2 * a * zeta + a * a) / (Rc ** 11 * zeta ** 4)
                                       + 231 * a ** 3 * Z ** 6 / (Rc ** 13 * zeta ** 3))


def convolved(fn, kind, pt, p):
    """int_{x-L}^{x+L} f(x-x') fn(x'^2+y^2, z) dx' : Eq. 12 applied to the whole expression (it is linear in R^-n)."""
    x, y, z = (mp.mpf(v) for v in pt)
    a, b, L, eta = (mp.mpf(p[k]) for k in ("a", "b", "L", "eta"))
    brk = sorted({x - L, x, x + L, mp.mpf(0)} & {v for v in (x - L, x, x + L, mp.mpf(0)) if x - L <= v <= x + L})
    return mp.quad(lambda xp: needle(x - xp, L, eta) * fn(kind, xp * xp + y * y, z, a, b), brk)


POINTS = [(1.0, 0.5, 0.1), (3.9, 0.2, 0.05), (5.0, 2.0, 1.0), (0.0, 0.0, 0.0), (0.0, 1.2, -0.4), (-2.5, 1.0, -0.3),
          (4.0, 0.0, 0.0), (10.0, -7.0, 0.3), (0.05, 0.02, 0.6), (30.0, -20.0, 10.0)]
CASES = [(inputs.DEHNEN_T3, T3P), (inputs.DEHNEN_V4, V4P), (inputs.DEHNEN_T3, GEN), (inputs.DEHNEN_V4, GEN)]


@pytest.mark.parametrize("kind,p", CASES)
def test_potential_vs_defining_integral(smo, kind, p):
    F, Phi = smo.eval_force(spec(kind, p), POINTS)
    for pt, ph in zip(POINTS, Phi):
        ref = float(G * M * convolved(parent_phi, kind, pt, p))
        assert ph == pytest.approx(ref, rel=2e-14), (kind, pt)


@pytest.mark.parametrize("kind,p", CASES)
def test_force_is_minus_gradient_and_poisson_with_the_printed_density(smo, kind, p):
    """F = -grad Phi by differentiating the DEFINING integral with mpmath, and div F = -4 pi G rho with the paper's printed
    rho convolved with the needle (4th-order central differences of the oracle's F, h = 0.01: truncation ~1e-8)."""
    pts = [pt for pt in POINTS if pt != (4.0, 0.0, 0.0) or p["L"] != 4.0][:7]
    F, _ = smo.eval_force(spec(kind, p), pts)
    for pt, f in zip(pts, F):
        for ax in range(3):
            def phi_ax(t, ax=ax, pt=pt):
                q = list(pt); q[ax] = t
                return G * M * convolved(parent_phi, kind, q, p)
            ref = -float(mp.diff(phi_ax, mp.mpf(pt[ax]), h=mp.mpf("1e-8")))
            assert f[ax] == pytest.approx(ref, rel=1e-10, abs=1e-9 * float(np.linalg.norm(f)) + 1e-300), (kind, pt, ax)
    h = 0.01
    for pt in pts[:5]:
        if p["L"] == 4.0 and abs(abs(pt[0]) - 4.0) < 0.2:
            continue
        div = 0.0
        for ax in range(3):
            sten = []
            for k in (-2, -1, 1, 2):
                q = list(pt); q[ax] += k * h; sten.append(q)
            Fs, _ = smo.eval_force(spec(kind, p), sten)
            div += (Fs[0][ax] - 8 * Fs[1][ax] + 8 * Fs[2][ax] - Fs[3][ax]) / (12 * h)
        rho = float(M * convolved(parent_rho, kind, pt, p))
        assert div == pytest.approx(-4 * np.pi * G * rho, rel=3e-6), (kind, pt)


@pytest.mark.parametrize("kind", [inputs.DEHNEN_T3, inputs.DEHNEN_V4])
def test_short_needle_is_the_parent_pair(smo, kind):
    """L -> 0: I_n -> R^-n, whatever eta (the replacement R^-n -> I_n)."""
    p = dict(a=0.8, b=0.3, L=1e-5, eta=0.7)
    _, Phi = smo.eval_force(spec(kind, p), POINTS)
    for pt, ph in zip(POINTS, Phi):
        ref = float(G * M * parent_phi(kind, mp.mpf(pt[0]) ** 2 + mp.mpf(pt[1]) ** 2, mp.mpf(pt[2]), mp.mpf(p["a"]), mp.mpf(p["b"])))
        assert ph == pytest.approx(ref, rel=1e-9)


def test_t3_without_disc_scale_and_needle_is_plummer(smo):
    """a = 0, L -> 0: Phi_T3 = -GM/sqrt(R^2 + z^2 + b^2), the oracle's (separately pinned) Plummer sphere."""
    p = dict(a=0.0, b=0.6, L=1e-6, eta=1.0)
    F, Phi = smo.eval_force(spec(inputs.DEHNEN_T3, p), POINTS)
    Fp, Pp = smo.eval_force({"G": G, "omega_p": 0.0, "phase0": 0.0, "components": [(inputs.PLUMMER, 0, [M, 0.6])]}, POINTS)
    assert np.allclose(Phi, Pp, rtol=1e-10, atol=0)
    assert np.allclose(F, Fp, rtol=1e-9, atol=1e-9 * np.abs(Fp).max())


@pytest.mark.parametrize("kind,p", CASES)
def test_far_field_monopole_and_symmetries(smo, kind, p):
    far = np.array([[3e4, 1e4, -2e4], [0.0, 5e4, 0.0]])
    F, Phi = smo.eval_force(spec(kind, p), far)
    r = np.linalg.norm(far, axis=1)
    assert np.allclose(Phi, -G * M / r, rtol=3e-4)
    assert np.allclose(F, -G * M * far / r[:, None] ** 3, rtol=1e-3, atol=1e-3 * G * M / r.min() ** 2)
    pt = np.array([1.7, -0.9, 0.35])
    signs = np.array([[1, 1, 1], [-1, 1, 1], [1, -1, 1], [1, 1, -1], [-1, -1, -1]], dtype=float)
    F, Phi = smo.eval_force(spec(kind, p), signs * pt)
    assert np.allclose(Phi, Phi[0], rtol=1e-15)
    assert np.allclose(F, signs * F[0], rtol=1e-13)
    # total mass M: Gauss's law is covered by the monopole; the centre is an equilibrium
    F0, _ = smo.eval_force(spec(kind, p), [[0.0, 0.0, 0.0]])
    assert np.all(np.abs(F0) < 1e-12 * G * M)


def test_rotating_needle_bar_conserves_the_jacobi_integral(smo):
    """The paper's stellar model (disc + T3 + V4 rotating at Omega_p + halo) through the oracle's KDK loop: the Jacobi
    integral drifts at second order in dt (PAPER.md:86 quotes 1e-4..1e-2 for its own integrator)."""
    pot = inputs.paper_bar_potential()
    ics = np.array([[3.0, 0.5, 0.1, -20.0, 190.0, 15.0], [2.0, -1.0, 0.3, 60.0, 150.0, -10.0], [5.0, 1.0, -0.2, 30.0, 200.0, 20.0]])
    drift = []
    for dt, n in ((1e-3, 1000), (5e-4, 2000)):
        tr = smo.integrate_trajectories(pot, ics, dt, n, stride=n // 50)
        t = dt * (n // 50) * np.arange(1, 51)
        ej0 = smo.jacobi(pot, ics, 0.0)
        ej = np.array([smo.jacobi(pot, tr[k], t[k]) for k in range(50)])
        drift.append(np.abs(ej - ej0).max(axis=0) / np.abs(ej0))
    assert np.all(drift[1] < 1e-3) and np.all(drift[1] > 0)
    ratio = drift[0] / drift[1]
    assert np.all((ratio > 3.0) & (ratio < 5.0)), ratio
