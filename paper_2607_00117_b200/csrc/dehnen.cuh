// dehnen.cuh -- the paper's own bar: Dehnen & Aly (2023) needle bars T_3 (long bar) and V_4 (boxy/peanut
// bulge), Eq. 12 and PAPER.md:485-497 Appendix A.  The axisymmetric parent (Appendix A) is a sum
// of terms c_n(Z, zeta) R^-n, n odd, with Z = a + zeta, zeta = sqrt(z^2 + b^2); the barred model replaces
//     R^-n  ->  I_n(x,y,Z) = int_{x-L}^{x+L} f(x-x') (x'^2 + s^2)^(-n/2) dx',   s^2 = y^2 + Z^2,
//     f(u) = [1 + eta (1 - 2|u|/L)] / (2L)                                                      (Eq. 12).
// f is linear on either side of u = 0, so I_n is a combination of the two elementary primitives of r^-n and
// t r^-n (r^2 = t^2 + s^2) taken at the three abscissae t = x-L, x, x+L:
//     P_n(t) = int r^-n dt:   P_1 = asinh(t/s),  n s^2 P_{n+2} = t r^-n + (n-1) P_n      (integration by parts)
//     Q_n(t) = int t r^-n dt: Q_1 = r,           Q_n = -r^(2-n)/(n-2)  (n >= 3)
// With d1 g = g(x+L) - g(x-L) and d2 g = g(x+L) + g(x-L) - 2 g(x):
//     2L I_n   = (1+eta) d1 P_n + (2 eta/L) (x d2 P_n - d2 Q_n)
//     dI_n/dx  = (1-eta)/(2L) d1 r^-n + (eta/L^2) d2 P_n
//     dI_n/dy  = -n y I_{n+2},    dI_n/dZ = -n Z I_{n+2}.
// The recurrence for P_n only adds terms of the sign of t (no cancellation); the differences d1, d2 lose
// ~(r/L)^2 of the 53 bits far outside the needle, where the bar is a small part of the total force, but far too
// much of a 24-bit mantissa: the needle integrals are therefore evaluated in fp64 in BOTH arithmetic variants of
// the integrator; T only carries the position in and the force out.
#pragma once
#include "force.cuh"

namespace smx {

enum { K_DEHNEN_T3 = 5, K_DEHNEN_V4 = 6 };

// ln(w) for w >= 1, branch-free: w = 2^e m with m in (sqrt(1/2), sqrt(2)], ln m = 2 atanh(s), s = (m-1)/(m+1) (m - 1 is exact),
// series and ln 2 split as in nfw_g (force.cuh).  The absolute error is ~1e-16: P_1 only enters through the differences d1, d2.
SMX_HD double log_ge1(double w) {
    int e; double m;
    split_sqrt2(w, e, m);
    const double s = (m - 1.0) * rcp_t(m + 1.0);
    const double z = s * s;
    double P = LogC<double>::p(LogC<double>::NP - 1);
#pragma unroll
    for (int i = LogC<double>::NP - 2; i >= 0; --i) P = fma(P, z, LogC<double>::p(i));
    const double s2 = s + s;
    const double ef = (double)e;
    return fma(ef, LogC<double>::ln2_hi(), fma(ef, LogC<double>::ln2_lo(), fma(s2 * z, P, s2)));
}

// the primitives at one abscissa t: P[j] = P_{2j+1}(t), k[j] = r^-(2j+1); *r_out = r.  cs[j] = 1/(n s^2), cm[j] = (n-1)/(n s^2),
// n = 2j+1 (shared by the abscissae of one evaluation).  P_1 = asinh(t/s) = sign(t) ln((|t| + r)/s); P_3 = t r^-1 / s^2.
template <int NJ>
SMX_HD void needle_primitives(double t, double s2, double rs /*1/s*/, const double* cs, const double* cm, double* P, double* k, double* r_out) {
    const double r2 = fma(t, t, s2);
    const double u = rsqrt_t(r2), u2 = u * u;
    const double r = r2 * u;
    const double as = log_ge1((fabs(t) + r) * rs);
    P[0] = t < 0.0 ? -as : as;
    k[0] = u;
    *r_out = r;
#pragma unroll
    for (int j = 0; j + 1 < NJ; ++j) {
        P[j + 1] = j == 0 ? (t * u) * cs[0] : fma(t * cs[j], k[j], cm[j] * P[j]);
        k[j + 1] = k[j] * u2;
    }
}

// NTERM terms of the parent (3: T_3, 5: V_4).  c = {GM, a, b^2, L, e1 = (1+eta)/(2L), e2 = eta/L^2}.  ETA = false: a uniform needle (eta = 0,
// the paper's V_4 bulge): the terms in d2 vanish and with them the primitives at t = x.
template <int NTERM, bool PHI, bool ETA>
SMX_HD void needle_bar(const double* c, double x, double y, double z, double& fx, double& fy, double& fz, double& phi) {
    constexpr int NJ = NTERM + 1;
    const double GM = c[0], a = c[1], b2 = c[2], L = c[3], e1 = c[4], e2 = c[5];
    const double z2b = fma(z, z, b2);
    const double rzeta = rsqrt_t(z2b), zeta = z2b * rzeta;
    const double Z = a + zeta;
    const double s2 = fma(y, y, Z * Z);
    const double rs = rsqrt_t(s2), rs2 = rs * rs;
    double cs[NJ - 1], cm[NJ - 1];
#pragma unroll
    for (int j = 0; j + 1 < NJ; ++j) { cs[j] = rs2 * (1.0 / (2 * j + 1)); cm[j] = rs2 * ((2.0 * j) / (2 * j + 1)); }
    double Pm[NJ], P0[NJ], Pp[NJ], km[NJ], k0[NJ], kp[NJ], rm, r0, rp;
    needle_primitives<NJ>(x - L, s2, rs, cs, cm, Pm, km, &rm);
    if constexpr (ETA) needle_primitives<NJ>(x, s2, rs, cs, cm, P0, k0, &r0);
    needle_primitives<NJ>(x + L, s2, rs, cs, cm, Pp, kp, &rp);
    double I[NJ], Ix[NTERM];
    const double e3 = ETA ? fma(-e2, L, e1) : e1;  // (1-eta)/(2L)
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        const int n = 2 * j + 1;
        const double d1P = Pp[j] - Pm[j];
        if constexpr (ETA) {
            const double d2P = (Pp[j] - P0[j]) + (Pm[j] - P0[j]);
            double d2Q;  // Q_1 = r = r^2 r^-1;  Q_n = -r^-(n-2)/(n-2)
            if (j == 0) {
                d2Q = (rp - r0) + (rm - r0);
            } else {
                d2Q = ((k0[j - 1] - kp[j - 1]) + (k0[j - 1] - km[j - 1])) * (1.0 / (n - 2));
            }
            I[j] = fma(e1, d1P, e2 * fma(x, d2P, -d2Q));
            if (j < NTERM) Ix[j] = fma(e3, kp[j] - km[j], e2 * d2P);
        } else {
            I[j] = e1 * d1P;
            if (j < NTERM) Ix[j] = e3 * (kp[j] - km[j]);
        }
    }
    // coefficients of the parent pair (Appendix A) and their derivatives with respect to zeta (Z = a + zeta)
    double cn[NTERM], dn[NTERM];
    cn[0] = 1.0; dn[0] = 0.0;
    if constexpr (NTERM == 3) {
        cn[1] = a * (Z - a * (1.0 / 3.0));  dn[1] = a;
        cn[2] = a * a * Z * Z;              dn[2] = 2.0 * a * a * Z;
    } else {
        const double Z2 = Z * Z, a2 = a * a;
        cn[1] = fma(a, Z - 0.4 * a, 0.5 * b2);                                   dn[1] = a;
        cn[2] = 3.0 * a * fma(0.2 * a * Z, 2.0 * Z - a, 0.5 * b2 * (Z - 0.2 * a));
        dn[2] = 3.0 * a * fma(0.2 * a, 4.0 * Z - a, 0.5 * b2);
        cn[3] = a2 * Z2 * fma(a, Z, 3.0 * b2);                                   dn[3] = a2 * Z * fma(3.0 * a, Z, 6.0 * b2);
        const double g = 3.5 * a2 * a * b2 * rzeta;                              // 7 a^3 b^2 / (2 zeta)
        cn[4] = g * Z2 * Z2;                                                      dn[4] = g * Z2 * Z * (4.0 - Z * rzeta);
    }
    double S = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
#pragma unroll
    for (int j = 0; j < NTERM; ++j) {
        const double n = (double)(2 * j + 1);
        if (PHI) S = fma(cn[j], I[j], S);
        gx = fma(cn[j], Ix[j], gx);
        gy = fma(-n * cn[j], I[j + 1], gy);
        gz = fma(dn[j], I[j], fma(-n * Z * cn[j], I[j + 1], gz));
    }
    // Phi = -GM S, F = -grad Phi; d zeta / dz = z / zeta
    fx += GM * gx;
    fy += GM * gy * y;
    fz += GM * gz * (z * rzeta);
    if (PHI) phi -= GM * S;
}

// one compile-time variant, arithmetic type T in and out (the specialised kernel of the paper's model)
template <typename T, int NTERM, bool PHI, bool ETA>
SMX_HD void needle_bar_T(const CompS<T>& c, T x, T y, T z, T& fx, T& fy, T& fz, T& phi) {
    double cc[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) cc[i] = (double)c.c[i];
    double gx = 0.0, gy = 0.0, gz = 0.0, ph = 0.0;
    needle_bar<NTERM, PHI, ETA>(cc, (double)x, (double)y, (double)z, gx, gy, gz, ph);
    fx += (T)gx; fy += (T)gy; fz += (T)gz;
    if (PHI) phi += (T)ph;
}

template <typename T, bool PHI>
SMX_HD void dehnen_aly(const CompS<T>& c, T x, T y, T z, T& fx, T& fy, T& fz, T& phi) {
    double cc[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) cc[i] = (double)c.c[i];
    double gx = 0.0, gy = 0.0, gz = 0.0, ph = 0.0;
    const bool uniform = cc[5] == 0.0;
    if (c.kind == K_DEHNEN_T3) {
        if (uniform) needle_bar<3, PHI, false>(cc, (double)x, (double)y, (double)z, gx, gy, gz, ph);
        else needle_bar<3, PHI, true>(cc, (double)x, (double)y, (double)z, gx, gy, gz, ph);
    } else {
        if (uniform) needle_bar<5, PHI, false>(cc, (double)x, (double)y, (double)z, gx, gy, gz, ph);
        else needle_bar<5, PHI, true>(cc, (double)x, (double)y, (double)z, gx, gy, gz, ph);
    }
    fx += (T)gx; fy += (T)gy; fz += (T)gz;
    if (PHI) phi += (T)ph;
}

}  // namespace smx
