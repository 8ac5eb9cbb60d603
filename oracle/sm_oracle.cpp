// sm_oracle.cpp -- CPU ORACLE (TEST INFRASTRUCTURE ONLY; see sm_oracle.h).
//
// Plain and slow on purpose.  No blocking, no fusion, no tables: every force is the analytic
// expression evaluated in __float128 and rounded once; the integrator, projection and binning
// are the loops of DESIGN.md "Algorithm" written out in the order stated there.
// Shares no code with paper_2607_00117_b200/csrc.  Build: see oracle/build.py
// (g++ -O2 -ffp-contract=off -fopenmp -std=gnu++17 ... -lquadmath).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): mpmath quadrature of the defining Ferrers
// integrals, Laplacian = 4 pi G rho, closed-form circular speeds (Eq.8, Eq.10),
// Kepler period/ellipse, dt^2 scaling, energy / Jacobi conservation, row sums, brute-force
// re-binning with numpy.  No function here is "parity unpinned".
#include "sm_oracle.h"
#include <quadmath.h>
#include <cmath>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef __float128 Q;

namespace {

struct Q3 { Q x, y, z; };

// ---------------------------------------------------------------- Carlson symmetric integrals
// R_F(x,y,z) = 1/2 int_0^inf dt / sqrt((t+x)(t+y)(t+z));  duplication theorem (Carlson 1979).
Q carlson_rf(Q x, Q y, Q z) {
    const Q tol = 1e-6Q;  // truncation error of the 5th-order series ~ tol^6
    Q mu, dx, dy, dz;
    for (int it = 0; it < 200; ++it) {
        Q sx = sqrtq(x), sy = sqrtq(y), sz = sqrtq(z);
        Q lam = sx * sy + sy * sz + sz * sx;
        x = (x + lam) / 4; y = (y + lam) / 4; z = (z + lam) / 4;
        mu = (x + y + z) / 3;
        dx = (mu - x) / mu; dy = (mu - y) / mu; dz = (mu - z) / mu;
        if (fmaxq(fmaxq(fabsq(dx), fabsq(dy)), fabsq(dz)) < tol) break;
    }
    Q e2 = dx * dy - dz * dz, e3 = dx * dy * dz;
    return (1 - e2 / 10 + e3 / 14 + e2 * e2 / 24 - 3 * e2 * e3 / 44) / sqrtq(mu);
}
// R_D(x,y,z) = 3/2 int_0^inf dt / (sqrt((t+x)(t+y)) (t+z)^{3/2}).
Q carlson_rd(Q x, Q y, Q z) {
    const Q tol = 1e-6Q;
    Q sum = 0, fac = 1, mu, dx, dy, dz;
    for (int it = 0; it < 200; ++it) {
        Q sx = sqrtq(x), sy = sqrtq(y), sz = sqrtq(z);
        Q lam = sx * sy + sy * sz + sz * sx;
        sum += fac / (sz * (z + lam));
        fac /= 4;
        x = (x + lam) / 4; y = (y + lam) / 4; z = (z + lam) / 4;
        mu = (x + y + 3 * z) / 5;
        dx = (mu - x) / mu; dy = (mu - y) / mu; dz = (mu - z) / mu;
        if (fmaxq(fmaxq(fabsq(dx), fabsq(dy)), fabsq(dz)) < tol) break;
    }
    Q ea = dx * dy, eb = dz * dz, ec = ea - eb, ed = ea - 6 * eb, ee = ed + 2 * ec;
    Q s = 1 + ed * (-3 / 14.0Q + (9 / 88.0Q) * ed - (9 / 52.0Q) * dz * ee)
            + dz * (ee / 6 + dz * (-(9 / 22.0Q) * ec + dz * (3 / 26.0Q) * ea));
    return 3 * sum + fac * s / (mu * sqrtq(mu));
}

// ---------------------------------------------------------------- Ferrers n=2
// lambda: 0 inside (m^2(0) <= 1), else the positive root of m^2(lambda) = 1,
// m^2(u) = x^2/(a^2+u) + y^2/(b^2+u) + z^2/(c^2+u).  f(u) = m^2(u)-1 is decreasing and convex
// for u > -c^2, so Newton started left of the root (u0 = max(0, r^2-a^2), f(u0) >= 0)
// increases monotonically to it.
Q ferrers_lambda(Q a2, Q b2, Q c2, Q X, Q Y, Q Z) {
    if (X / a2 + Y / b2 + Z / c2 <= 1) return 0;
    Q u = X + Y + Z - a2;
    if (u < 0) u = 0;
    for (int it = 0; it < 300; ++it) {
        Q A = a2 + u, B = b2 + u, C = c2 + u;
        Q f = X / A + Y / B + Z / C - 1;
        Q fp = -(X / (A * A) + Y / (B * B) + Z / (C * C));
        Q du = -f / fp;
        u += du;
        if (fabsq(du) <= 1e-32Q * (u + a2)) break;
    }
    return u < 0 ? (Q)0 : u;
}

enum { I000, I100, I010, I001, I200, I020, I002, I110, I101, I011,
       I300, I030, I003, I210, I201, I120, I021, I102, I012, I111 };

// W_ijk(lambda) = int_lambda^inf du / (Delta (a^2+u)^i (b^2+u)^j (c^2+u)^k).
void ferrers_W(Q a2, Q b2, Q c2, Q lam, Q* W) {
    Q A = a2 + lam, B = b2 + lam, C = c2 + lam;
    Q p = a2 - b2, q = a2 - c2, r = b2 - c2;
    Q E = 2 / sqrtq(A * B * C);
    W[I000] = 2 * carlson_rf(A, B, C);
    W[I100] = (2 / 3.0Q) * carlson_rd(B, C, A);
    W[I001] = (2 / 3.0Q) * carlson_rd(A, B, C);
    W[I010] = E - W[I100] - W[I001];                 // W100+W010+W001 = 2/sqrt(ABC)
    // partial fractions: 1/B-1/A = p/(AB), 1/C-1/A = q/(AC), 1/C-1/B = r/(BC)
    W[I110] = (W[I010] - W[I100]) / p;
    W[I101] = (W[I001] - W[I100]) / q;
    W[I011] = (W[I001] - W[I010]) / r;
    // (2i+1)W_{i+1,j,k} + (2j+1)W_{i,j+1,k} + (2k+1)W_{i,j,k+1} = 2/(sqrt(ABC) A^i B^j C^k)
    W[I200] = (E / A - W[I110] - W[I101]) / 3;
    W[I020] = (E / B - W[I110] - W[I011]) / 3;
    W[I002] = (E / C - W[I101] - W[I011]) / 3;
    W[I210] = (W[I110] - W[I200]) / p;
    W[I120] = (W[I020] - W[I110]) / p;
    W[I201] = (W[I101] - W[I200]) / q;
    W[I102] = (W[I002] - W[I101]) / q;
    W[I021] = (W[I011] - W[I020]) / r;
    W[I012] = (W[I002] - W[I011]) / r;
    W[I111] = (W[I011] - W[I101]) / p;
    W[I300] = (E / (A * A) - W[I210] - W[I201]) / 5;
    W[I030] = (E / (B * B) - W[I120] - W[I021]) / 5;
    W[I003] = (E / (C * C) - W[I102] - W[I012]) / 5;
}

// rho = rho_c (1-m^2)^2, rho_c = 105 M / (32 pi a b c);
// dPhi/dx_i = 2 pi G a b c rho_c x_i int_lambda^inf (1-m^2(u))^2 du / ((a_i^2+u) Delta(u)),
// Phi = -(pi G a b c rho_c / 3) int_lambda^inf (1-m^2(u))^3 du / Delta(u).
void ferrers_force(Q GM, Q a, Q b, Q c, Q3 xb, Q3* F, Q* Phi) {
    Q a2 = a * a, b2 = b * b, c2 = c * c;
    Q X = xb.x * xb.x, Y = xb.y * xb.y, Z = xb.z * xb.z;
    Q lam = ferrers_lambda(a2, b2, c2, X, Y, Z);
    Q W[20];
    ferrers_W(a2, b2, c2, lam, W);
    Q K = 105 * GM / 16;  // 2 pi G a b c rho_c
    Q gx = W[I100] - 2 * (X * W[I200] + Y * W[I110] + Z * W[I101]) + X * X * W[I300] + Y * Y * W[I120]
         + Z * Z * W[I102] + 2 * X * Y * W[I210] + 2 * X * Z * W[I201] + 2 * Y * Z * W[I111];
    Q gy = W[I010] - 2 * (X * W[I110] + Y * W[I020] + Z * W[I011]) + X * X * W[I210] + Y * Y * W[I030]
         + Z * Z * W[I012] + 2 * X * Y * W[I120] + 2 * X * Z * W[I111] + 2 * Y * Z * W[I021];
    Q gz = W[I001] - 2 * (X * W[I101] + Y * W[I011] + Z * W[I002]) + X * X * W[I201] + Y * Y * W[I021]
         + Z * Z * W[I003] + 2 * X * Y * W[I111] + 2 * X * Z * W[I102] + 2 * Y * Z * W[I012];
    F->x = -K * xb.x * gx; F->y = -K * xb.y * gy; F->z = -K * xb.z * gz;
    if (Phi) {
        Q S1 = X * W[I100] + Y * W[I010] + Z * W[I001];
        Q S2 = X * X * W[I200] + Y * Y * W[I020] + Z * Z * W[I002]
             + 2 * (X * Y * W[I110] + X * Z * W[I101] + Y * Z * W[I011]);
        Q S3 = X * X * X * W[I300] + Y * Y * Y * W[I030] + Z * Z * Z * W[I003]
             + 3 * (X * X * Y * W[I210] + X * X * Z * W[I201] + X * Y * Y * W[I120] + Y * Y * Z * W[I021]
                    + X * Z * Z * W[I102] + Y * Z * Z * W[I012])
             + 6 * X * Y * Z * W[I111];
        *Phi = -(K / 6) * (W[I000] - 3 * S1 + 3 * S2 - S3);
    }
}

// ---------------------------------------------------------------- the other components
// Plummer: Phi = -GM/sqrt(r^2+b^2) (b = 0: point mass).
void plummer_force(Q GM, Q b, Q3 x, Q3* F, Q* Phi) {
    Q s2 = x.x * x.x + x.y * x.y + x.z * x.z + b * b;
    Q s = sqrtq(s2);
    Q f = -GM / (s2 * s);
    F->x = f * x.x; F->y = f * x.y; F->z = f * x.z;
    if (Phi) *Phi = -GM / s;
}
// Miyamoto-Nagai, Eq.10: Phi = -GM / sqrt(R^2 + (a + sqrt(z^2+b^2))^2).
void mn_force(Q GM, Q a, Q b, Q3 x, Q3* F, Q* Phi) {
    Q zeta = sqrtq(x.z * x.z + b * b);
    Q D = a + zeta;
    Q s2 = x.x * x.x + x.y * x.y + D * D;
    Q s = sqrtq(s2);
    Q f = -GM / (s2 * s);
    F->x = f * x.x; F->y = f * x.y; F->z = f * x.z * D / zeta;
    if (Phi) *Phi = -GM / s;
}
// NFW, Eq.8 with M_DM = 4 pi rho_s r_s^3: Phi = -G M_DM ln(1+r/r_s)/r,
// F = -G M_DM [ln(1+X) - X/(1+X)] / r^3 * x,  X = r/r_s;  F(0) = 0, Phi(0) = -G M_DM / r_s.
void nfw_force(Q G, Q rho_s, Q r_s, Q3 x, Q3* F, Q* Phi) {
    Q GMdm = G * 4 * M_PIq * rho_s * r_s * r_s * r_s;
    Q r = sqrtq(x.x * x.x + x.y * x.y + x.z * x.z);
    if (r == 0) { F->x = F->y = F->z = 0; if (Phi) *Phi = -GMdm / r_s; return; }
    Q Xr = r / r_s;
    Q L = log1pq(Xr);
    Q f = -GMdm * (L - Xr / (1 + Xr)) / (r * r * r);
    F->x = f * x.x; F->y = f * x.y; F->z = f * x.z;
    if (Phi) *Phi = -GMdm * L / r;
}

// ---------------------------------------------------------------- Dehnen & Aly (2023) needle bars
// PAPER.md:211-237 Eq. 12 and PAPER.md:485-497 Appendix A.  The barred model is the axisymmetric
// parent pair with every R^{-n} (R^2 = x^2 + y^2 + Z^2, Z = a + zeta, zeta = sqrt(z^2 + b^2))
// replaced by the needle convolution
//     I_n(x,y,Z;L,eta) = int_{x-L}^{x+L} f(x-x') dx' / (x'^2 + y^2 + Z^2)^{n/2},
//     f(u) = [1 + eta (1 - 2|u|/L)] / (2L)  for |u| < L.
// With s^2 = y^2 + Z^2, r(t) = sqrt(t^2 + s^2), k_n(t) = r^{-n}, and the elementary antiderivatives
//     A_n(t) = int k_n dt :  A_1 = asinh(t/s),  A_{n+2} = [t r^{-n} + (n-1) A_n] / (n s^2)
//     B_n(t) = int t k_n dt: B_1 = r,           B_n = -r^{2-n}/(n-2)   (n >= 3)
// the integral splits at x' = x (where |x-x'| changes branch):
//     I_n = { (1+eta) [A_n(x+L) - A_n(x-L)]
//             - (2 eta/L) ( x [2A_n(x) - A_n(x-L) - A_n(x+L)] + B_n(x+L) + B_n(x-L) - 2B_n(x) ) } / (2L)
//     dI_n/dx = (1-eta)/(2L) [k_n(x+L) - k_n(x-L)] - (eta/L^2) [2A_n(x) - A_n(x-L) - A_n(x+L)]
//     dI_n/dy = -n y I_{n+2},   dI_n/dZ = -n Z I_{n+2}        (differentiate under the integral)
// n is odd, 1..11.  L -> 0 gives back R^{-n} (the parent model).  Everything in __float128: the differences
// of antiderivatives lose (r/L)^2 digits at most, far below the 33 carried.
void needle_A(Q t, Q s2, Q* A /*[6]: n=1,3,..,11*/, Q* k /*[6]*/) {
    Q r2 = t * t + s2, r = sqrtq(r2), s = sqrtq(s2);
    Q rn = 1 / r;                       // r^{-n}, n = 1
    A[0] = asinhq(t / s);
    k[0] = rn;
    for (int j = 0; j < 5; ++j) {       // n = 2j+1 -> n+2
        int n = 2 * j + 1;
        A[j + 1] = (t * rn + (n - 1) * A[j]) / (n * s2);
        rn /= r2;
        k[j + 1] = rn;
    }
}
Q needle_B(Q t, Q s2, int n) {
    Q r2 = t * t + s2;
    if (n == 1) return sqrtq(r2);
    return -powq(r2, (Q)(2 - n) / 2) / (n - 2);
}
// I[j], dIdx[j] for n = 2j+1, j = 0..5
void needle_I(Q x, Q y, Q Z, Q L, Q eta, Q* I, Q* dIdx) {
    Q s2 = y * y + Z * Z;
    Q Am[6], A0[6], Ap[6], km[6], k0[6], kp[6];
    needle_A(x - L, s2, Am, km);
    needle_A(x, s2, A0, k0);
    needle_A(x + L, s2, Ap, kp);
    for (int j = 0; j < 6; ++j) {
        int n = 2 * j + 1;
        Q D = Ap[j] - Am[j];
        Q S = 2 * A0[j] - Am[j] - Ap[j];
        Q BB = needle_B(x + L, s2, n) + needle_B(x - L, s2, n) - 2 * needle_B(x, s2, n);
        I[j] = ((1 + eta) * D - (2 * eta / L) * (x * S + BB)) / (2 * L);
        dIdx[j] = (1 - eta) / (2 * L) * (kp[j] - km[j]) - (eta / (L * L)) * S;
    }
}
// Phi = -GM sum_n c_n(Z,zeta) I_n.  model 3: T_3 (Appendix A Eq. A1), model 4: V_4 (second pair).
// c[j], dc[j] = d c_n / d zeta (Z = a + zeta, so d/dzeta acts on Z and on the explicit zeta).
void dehnen_aly_force(int model, Q GM, Q a, Q b, Q L, Q eta, Q3 x, Q3* F, Q* Phi) {
    Q zeta = sqrtq(x.z * x.z + b * b), Z = a + zeta;
    Q c[5] = {0, 0, 0, 0, 0}, dc[5] = {0, 0, 0, 0, 0};
    int nterm;
    if (model == 3) {
        nterm = 3;
        c[0] = 1;
        c[1] = a * (Z - a / 3);                     dc[1] = a;
        c[2] = a * a * Z * Z;                       dc[2] = 2 * a * a * Z;
    } else {
        nterm = 5;
        Q b2 = b * b;
        c[0] = 1;
        c[1] = a * (Z - 2 * a / 5) + b2 / 2;        dc[1] = a;
        c[2] = 3 * a * (a * Z * (2 * Z - a) / 5 + b2 / 2 * (Z - a / 5));
        dc[2] = 3 * a * (a * (4 * Z - a) / 5 + b2 / 2);
        c[3] = a * a * Z * Z * (a * Z + 3 * b2);    dc[3] = a * a * (3 * a * Z * Z + 6 * b2 * Z);
        c[4] = 7 * a * a * a * b2 * Z * Z * Z * Z / (2 * zeta);
        dc[4] = 7 * a * a * a * b2 / 2 * (4 * Z * Z * Z / zeta - Z * Z * Z * Z / (zeta * zeta));
    }
    Q I[6], dIdx[6];
    needle_I(x.x, x.y, Z, L, eta, I, dIdx);
    Q P = 0, gx = 0, gy = 0, gzeta = 0;             // gradient of sum c_n I_n
    for (int j = 0; j < nterm; ++j) {
        int n = 2 * j + 1;
        P += c[j] * I[j];
        gx += c[j] * dIdx[j];
        gy += c[j] * (-n * x.y * I[j + 1]);
        gzeta += dc[j] * I[j] + c[j] * (-n * Z * I[j + 1]);
    }
    // Phi = -GM P  =>  F = -grad Phi = +GM grad P;  d zeta/dz = z/zeta
    F->x = GM * gx; F->y = GM * gy; F->z = GM * gzeta * x.z / zeta;
    if (Phi) *Phi = -GM * P;
}

void component_force(const smo_potential_desc* d, const smo_component* c, Q3 x, Q3* F, Q* Phi) {
    Q G = d->G;
    switch (c->kind) {
        case SMO_PLUMMER: plummer_force(G * (Q)c->p[0], c->p[1], x, F, Phi); break;
        case SMO_MIYAMOTO_NAGAI: mn_force(G * (Q)c->p[0], c->p[1], c->p[2], x, F, Phi); break;
        case SMO_NFW: nfw_force(G, c->p[0], c->p[1], x, F, Phi); break;
        case SMO_FERRERS2: ferrers_force(G * (Q)c->p[0], c->p[1], c->p[2], c->p[3], x, F, Phi); break;
        case SMO_DEHNEN_T3: dehnen_aly_force(3, G * (Q)c->p[0], c->p[1], c->p[2], c->p[3], c->p[4], x, F, Phi); break;
        case SMO_DEHNEN_V4: dehnen_aly_force(4, G * (Q)c->p[0], c->p[1], c->p[2], c->p[3], c->p[4], x, F, Phi); break;
        default: F->x = F->y = F->z = 0; if (Phi) *Phi = 0;
    }
}

// acc(x,t): static components at x; rotating components at x_b = Rz(-theta) x, rotated back.
// theta = Omega_p*t + phase0 is formed in double (the method's precision); everything after
// that is __float128.
void total_force(const smo_potential_desc* d, Q3 x, double t, Q3* F, Q* Phi) {
    Q3 Fs = {0, 0, 0};
    Q P = 0;
    bool any_rot = false;
    for (int i = 0; i < d->n_comp; ++i) {
        if (d->comp[i].rotating) { any_rot = true; continue; }
        Q3 f; Q ph;
        component_force(d, &d->comp[i], x, &f, Phi ? &ph : nullptr);
        Fs.x += f.x; Fs.y += f.y; Fs.z += f.z;
        if (Phi) P += ph;
    }
    if (any_rot) {
        double theta = d->omega_p * t + d->phase0;
        Q c = cosq((Q)theta), s = sinq((Q)theta);
        Q3 xb = { c * x.x + s * x.y, -s * x.x + c * x.y, x.z };
        Q3 Fb = {0, 0, 0};
        for (int i = 0; i < d->n_comp; ++i) {
            if (!d->comp[i].rotating) continue;
            Q3 f; Q ph;
            component_force(d, &d->comp[i], xb, &f, Phi ? &ph : nullptr);
            Fb.x += f.x; Fb.y += f.y; Fb.z += f.z;
            if (Phi) P += ph;
        }
        Fs.x += c * Fb.x - s * Fb.y;
        Fs.y += s * Fb.x + c * Fb.y;
        Fs.z += Fb.z;
    }
    *F = Fs;
    if (Phi) *Phi = P;
}

int check_desc(const smo_potential_desc* d) {
    if (!d || d->n_comp < 1 || d->n_comp > 8) return -1;
    for (int i = 0; i < d->n_comp; ++i) {
        const smo_component& c = d->comp[i];
        if (c.kind == SMO_FERRERS2 && !(c.p[1] > c.p[2] && c.p[2] > c.p[3] && c.p[3] > 0)) return -1;
        if ((c.kind == SMO_DEHNEN_T3 || c.kind == SMO_DEHNEN_V4) &&
            !(c.p[1] >= 0 && c.p[2] > 0 && c.p[3] > 0 && c.p[4] >= -1 && c.p[4] <= 1)) return -1;
        if (c.kind < 1 || c.kind > 6) return -1;
    }
    return 0;
}

template <class R>
struct Orbit {
    R x[3], v[3], a[3];
    const smo_potential_desc* d;
    void accel(double t) {
        Q3 F; Q3 xq = { (Q)x[0], (Q)x[1], (Q)x[2] };
        total_force(d, xq, t, &F, nullptr);
        a[0] = (R)F.x; a[1] = (R)F.y; a[2] = (R)F.z;
    }
    void init(const double* ic) {
        for (int j = 0; j < 3; ++j) { x[j] = ic[j]; v[j] = ic[3 + j]; }
        accel(0.0);
    }
    // one kick-drift-kick step ending at t_k = k*dt (north_star item 2)
    void step(double dt, int64_t k) {
        R h = (R)dt / 2;
        for (int j = 0; j < 3; ++j) v[j] = v[j] + h * a[j];
        for (int j = 0; j < 3; ++j) x[j] = x[j] + (R)dt * v[j];
        double t = (double)k * dt;
        accel(t);
        for (int j = 0; j < 3; ++j) v[j] = v[j] + h * a[j];
    }
};

struct RotM { double ca, sa, cb, sb, cg, sg; };

// R = Rz(gamma) Rx(beta) Rz(alpha), active, right-handed (Eq.1):
// out = { x', y', v_z' }.
void project(const RotM& m, const double* xb, const double* vb, double* out) {
    double x1 = xb[0] * m.ca - xb[1] * m.sa;
    double y1 = xb[0] * m.sa + xb[1] * m.ca;
    double y2 = y1 * m.cb - xb[2] * m.sb;
    out[0] = x1 * m.cg - y2 * m.sg;
    out[1] = x1 * m.sg + y2 * m.cg;
    double vy1 = vb[0] * m.sa + vb[1] * m.ca;
    out[2] = vy1 * m.sb + vb[2] * m.cb;
}

// bin index of u on [lo,hi) with n bins: floor((u-lo)*n/(hi-lo)); -1 if outside or NaN.
inline int bin1(double u, double lo, double inv, int n, bool* edge) {
    double w = (u - lo) * inv;
    if (std::isfinite(w) && std::fabs(w - std::nearbyint(w)) < 1e-9) *edge = true;
    if (!(w >= 0.0) || !(w < (double)n)) return -1;
    return (int)std::floor(w);
}

double jacobi(const smo_potential_desc* d, const double* s, double t) {
    Q3 F; Q P; Q3 xq = { (Q)s[0], (Q)s[1], (Q)s[2] };
    total_force(d, xq, t, &F, &P);
    Q v2 = (Q)s[3] * s[3] + (Q)s[4] * s[4] + (Q)s[5] * s[5];
    Q Lz = (Q)s[0] * s[4] - (Q)s[1] * s[3];
    return (double)(v2 / 2 + P - (Q)d->omega_p * Lz);
}

template <class R>
int build_library_t(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt,
                    int64_t n_steps, int32_t stride, const smo_projection* proj, int n_proj,
                    const smo_grids* g, float* losvd, float* dens, int32_t* nout, double* diag,
                    int32_t* near_edge) {
    const int64_t nlos = (int64_t)g->nx * g->ny * g->nv, nden = (int64_t)g->dx * g->dy * g->dz;
    std::vector<RotM> rm(n_proj);
    for (int p = 0; p < n_proj; ++p)
        rm[p] = { std::cos(proj[p].alpha), std::sin(proj[p].alpha), std::cos(proj[p].beta),
                  std::sin(proj[p].beta), std::cos(proj[p].gamma), std::sin(proj[p].gamma) };
    const double ivx = g->nx / (g->x1 - g->x0), ivy = g->ny / (g->y1 - g->y0), ivv = g->nv / (g->v1 - g->v0);
    const double idx = g->dx / (g->bx1 - g->bx0), idy = g->dy / (g->by1 - g->by0), idz = g->dz / (g->bz1 - g->bz0);
#pragma omp parallel for schedule(dynamic)
    for (int64_t i = 0; i < n_orb; ++i) {
        for (int p = 0; p < n_proj; ++p) std::memset(losvd + ((int64_t)p * n_orb + i) * nlos, 0, sizeof(float) * nlos);
        std::memset(dens + i * nden, 0, sizeof(float) * nden);
        std::vector<int32_t> no(n_proj + 1, 0), ne(n_proj + 1, 0);
        Orbit<R> o; o.d = d; o.init(ics + 6 * i);
        double ej0 = 0, drift = 0; int bad = 0;
        if (diag) { double s0[6]; for (int j = 0; j < 6; ++j) s0[j] = ics[6 * i + j]; ej0 = jacobi(d, s0, 0.0); }
        for (int64_t k = 1; k <= n_steps; ++k) {
            o.step(dt, k);
            if (k % stride) continue;
            double t = (double)k * dt;
            double s[6] = { (double)o.x[0], (double)o.x[1], (double)o.x[2], (double)o.v[0], (double)o.v[1], (double)o.v[2] };
            // sample -> bar frame: x_b = Rz(-theta) x, v_b = Rz(-theta) v (inertial velocity
            // resolved on bar axes)
            double theta = d->omega_p * t + d->phase0;
            double c = std::cos(theta), sn = std::sin(theta);
            double xb[3] = { c * s[0] + sn * s[1], -sn * s[0] + c * s[1], s[2] };
            double vb[3] = { c * s[3] + sn * s[4], -sn * s[3] + c * s[4], s[5] };
            bool e = false;
            int jx = bin1(xb[0], g->bx0, idx, g->dx, &e), jy = bin1(xb[1], g->by0, idy, g->dy, &e),
                jz = bin1(xb[2], g->bz0, idz, g->dz, &e);
            if (jx >= 0 && jy >= 0 && jz >= 0) dens[i * nden + ((int64_t)jz * g->dy + jy) * g->dx + jx] += 1.0f;
            else no[n_proj]++;
            if (e) ne[n_proj]++;
            for (int p = 0; p < n_proj; ++p) {
                double out[3]; project(rm[p], xb, vb, out);
                bool e2 = false;
                int ix = bin1(out[0], g->x0, ivx, g->nx, &e2), iy = bin1(out[1], g->y0, ivy, g->ny, &e2),
                    iv = bin1(out[2], g->v0, ivv, g->nv, &e2);
                if (ix >= 0 && iy >= 0 && iv >= 0)
                    losvd[((int64_t)p * n_orb + i) * nlos + ((int64_t)iy * g->nx + ix) * g->nv + iv] += 1.0f;
                else no[p]++;
                if (e2) ne[p]++;
            }
            if (diag) {
                bool fin = true; for (int j = 0; j < 6; ++j) fin = fin && std::isfinite(s[j]);
                if (!fin) bad = 1;
                else { double ej = jacobi(d, s, t); double r = std::fabs(ej - ej0) / std::fabs(ej0); if (r > drift) drift = r; }
            }
        }
        for (int p = 0; p <= n_proj; ++p) {
            if (nout) nout[(int64_t)p * n_orb + i] = no[p];
            if (near_edge) near_edge[(int64_t)p * n_orb + i] = ne[p];
        }
        if (diag) { diag[2 * i] = drift; diag[2 * i + 1] = bad; }
    }
    return 0;
}

template <class R>
int integrate_t(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt,
                int64_t n_steps, int32_t stride, double* traj) {
#pragma omp parallel for schedule(dynamic)
    for (int64_t i = 0; i < n_orb; ++i) {
        Orbit<R> o; o.d = d; o.init(ics + 6 * i);
        for (int64_t k = 1; k <= n_steps; ++k) {
            o.step(dt, k);
            if (k % stride) continue;
            double* out = traj + ((k / stride - 1) * n_orb + i) * 6;
            for (int j = 0; j < 3; ++j) { out[j] = (double)o.x[j]; out[3 + j] = (double)o.v[j]; }
        }
    }
    return 0;
}

// ---------------------------------------------------------------- the paper's own integrator
// "a simpler third-order adaptive-timestep Runge-Kutta method (Bogacki & Shampine 1989) with a relative tolerance of
// 1e-4 ... the integration is done with a fixed number of steps ... performed in the reference frame of the galactic
// bar ... The velocities in the bar rest frame are transformed back to the inertial frame after the orbital integration"
// and every sample is weighted by its step size dt.  State y = (x_b, u): position on bar axes and
// velocity IN the rotating frame,
//     dx_b/dt = u,    du/dt = F(x_b) - 2 Omega x u - Omega x (Omega x x_b),   Omega = Omega_p e_z
//                           = F + (2 Omega_p u_y + Omega_p^2 x_b,  -2 Omega_p u_x + Omega_p^2 y_b,  0).
// Bogacki-Shampine 3(2) pair with first-same-as-last:
//     k1 = f(y);  k2 = f(y + h/2 k1);  k3 = f(y + 3h/4 k2);  y' = y + h (2/9 k1 + 1/3 k2 + 4/9 k3);  k4 = f(y');
//     e = h (-5/72 k1 + 1/12 k2 + 1/9 k3 - 1/8 k4)       (third-order minus embedded second-order solution).
// Step control (reading R23; the paper prints only the tolerance): err = rms_i e_i / (atol_i + rtol max(|y_i|,|y'_i|));
// accept iff err <= 1; h <- h min(5, max(0.2, 0.9 err^(-1/3))).  Every attempt uses up one of the n_steps; a rejected attempt
// leaves the state where it was and carries weight 0.  rtol <= 0: fixed steps h0 (no control), for the order pins.
// Sample k = state after attempt k, positions on bar axes, velocity = inertial velocity on bar axes u + Omega x x_b (reading R1).
struct RotState { double y[6]; };
void rot_rhs(const smo_potential_desc* d0, double omega, const double* y, double* f) {
    Q3 F; Q3 xq = { (Q)y[0], (Q)y[1], (Q)y[2] };
    total_force(d0, xq, 0.0, &F, nullptr);       // d0: the same components with the bar at rest along x (theta = 0)
    f[0] = y[3]; f[1] = y[4]; f[2] = y[5];
    f[3] = (double)F.x + 2 * omega * y[4] + omega * omega * y[0];
    f[4] = (double)F.y - 2 * omega * y[3] + omega * omega * y[1];
    f[5] = (double)F.z;
}

int check_run(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt, int64_t n_steps, int32_t stride) {
    if (check_desc(d) || !ics || n_orb < 0 || !(dt > 0) || !std::isfinite(dt) || n_steps < 1 || stride < 1) return -1;
    return 0;
}

}  // namespace

extern "C" {

int smo_eval_force(const smo_potential_desc* d, const double* xyz, int64_t n, double t, double* F, double* Phi) {
    if (check_desc(d) || !xyz || !F || n < 0) return -1;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        Q3 x = { (Q)xyz[3 * i], (Q)xyz[3 * i + 1], (Q)xyz[3 * i + 2] }, f; Q P;
        total_force(d, x, t, &f, Phi ? &P : nullptr);
        F[3 * i] = (double)f.x; F[3 * i + 1] = (double)f.y; F[3 * i + 2] = (double)f.z;
        if (Phi) Phi[i] = (double)P;
    }
    return 0;
}

int smo_integrate_trajectories(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt,
                               int64_t n_steps, int32_t stride, int state_prec, double* traj) {
    if (check_run(d, ics, n_orb, dt, n_steps, stride) || !traj) return -1;
    return state_prec ? integrate_t<long double>(d, ics, n_orb, dt, n_steps, stride, traj)
                      : integrate_t<double>(d, ics, n_orb, dt, n_steps, stride, traj);
}

int smo_integrate_rk32(const smo_potential_desc* d, const double* ics, int64_t n_orb, int64_t n_steps, double rtol,
                       double atol_x, double atol_v, double h0, double* samples, double* dt_w, double* t_end) {
    if (check_desc(d) || !ics || n_orb < 0 || n_steps < 1 || !(h0 > 0) || !std::isfinite(h0) || !samples || !dt_w) return -1;
    if (rtol > 0 && (!(atol_x >= 0) || !(atol_v >= 0))) return -1;
    // the rotating-frame equations need every non-rotating component to be axisymmetric about z
    smo_potential_desc d0 = *d; d0.omega_p = 0.0; d0.phase0 = 0.0;
    for (int i = 0; i < d->n_comp; ++i)
        if (!d->comp[i].rotating && d->omega_p != 0.0 && d->comp[i].kind > SMO_NFW) return -1;
    const double om = d->omega_p, c0 = std::cos(d->phase0), s0 = std::sin(d->phase0);
#pragma omp parallel for schedule(dynamic)
    for (int64_t i = 0; i < n_orb; ++i) {
        const double* ic = ics + 6 * i;
        double y[6], k1[6], k2[6], k3[6], k4[6], yt[6], yn[6];
        // inertial ICs at t = 0 -> bar axes, then u = v_b - Omega x x_b
        y[0] = c0 * ic[0] + s0 * ic[1]; y[1] = -s0 * ic[0] + c0 * ic[1]; y[2] = ic[2];
        y[3] = c0 * ic[3] + s0 * ic[4] + om * y[1]; y[4] = -s0 * ic[3] + c0 * ic[4] - om * y[0]; y[5] = ic[5];
        double h = h0, t = 0.0;
        rot_rhs(&d0, om, y, k1);
        for (int64_t k = 0; k < n_steps; ++k) {
            for (int j = 0; j < 6; ++j) yt[j] = y[j] + h * (0.5 * k1[j]);
            rot_rhs(&d0, om, yt, k2);
            for (int j = 0; j < 6; ++j) yt[j] = y[j] + h * (0.75 * k2[j]);
            rot_rhs(&d0, om, yt, k3);
            for (int j = 0; j < 6; ++j) yn[j] = y[j] + h * ((2.0 / 9.0) * k1[j] + (1.0 / 3.0) * k2[j] + (4.0 / 9.0) * k3[j]);
            rot_rhs(&d0, om, yn, k4);
            bool accept = true;
            double h_next = h;
            if (rtol > 0) {
                double sum = 0;
                for (int j = 0; j < 6; ++j) {
                    double e = h * ((-5.0 / 72.0) * k1[j] + (1.0 / 12.0) * k2[j] + (1.0 / 9.0) * k3[j] - (1.0 / 8.0) * k4[j]);
                    double sc = (j < 3 ? atol_x : atol_v) + rtol * std::fmax(std::fabs(y[j]), std::fabs(yn[j]));
                    sum += (e / sc) * (e / sc);
                }
                double err = std::sqrt(sum / 6.0);
                accept = err <= 1.0;                     // NaN rejects
                double fac = err > 0 ? 0.9 * std::pow(err, -1.0 / 3.0) : (err == 0 ? 5.0 : 0.2);   // NaN estimate: shrink (reading R23)
                if (!(fac >= 0.2)) fac = 0.2;
                if (fac > 5.0) fac = 5.0;
                h_next = h * fac;
            }
            double w = 0.0;
            if (accept) {
                for (int j = 0; j < 6; ++j) { y[j] = yn[j]; k1[j] = k4[j]; }
                t += h; w = h;
            }
            h = h_next;
            double* out = samples + (k * n_orb + i) * 6;
            out[0] = y[0]; out[1] = y[1]; out[2] = y[2];
            out[3] = y[3] - om * y[1]; out[4] = y[4] + om * y[0]; out[5] = y[5];
            dt_w[k * n_orb + i] = w;
        }
        if (t_end) t_end[i] = t;
    }
    return 0;
}

int smo_build_library(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt, int64_t n_steps,
                      int32_t stride, const smo_projection* proj, int n_proj, const smo_grids* g, int state_prec,
                      float* losvd, float* dens, int32_t* nout, double* diag, int32_t* near_edge) {
    if (check_run(d, ics, n_orb, dt, n_steps, stride) || !proj || n_proj < 1 || !g || !losvd || !dens) return -1;
    if (g->nx < 1 || g->ny < 1 || g->nv < 1 || g->dx < 1 || g->dy < 1 || g->dz < 1) return -1;
    if (!(g->x1 > g->x0) || !(g->y1 > g->y0) || !(g->v1 > g->v0) || !(g->bx1 > g->bx0) || !(g->by1 > g->by0) || !(g->bz1 > g->bz0)) return -1;
    return state_prec ? build_library_t<long double>(d, ics, n_orb, dt, n_steps, stride, proj, n_proj, g, losvd, dens, nout, diag, near_edge)
                      : build_library_t<double>(d, ics, n_orb, dt, n_steps, stride, proj, n_proj, g, losvd, dens, nout, diag, near_edge);
}

// Symmetrised orbit bundles (PAPER.md:71 dither bundles, Table 1 fourfold symmetrisation): row r co-adds
// the n_bundle consecutive orbits r*n_bundle .. r*n_bundle+n_bundle-1, and (fourfold != 0) every recorded bar-frame
// sample is binned four times with the sign flips of Table 1:
//   copy 1 (x,y,z; vx,vy,vz)   copy 2 (x,y,-z; vx,vy,-vz)   copy 3 (-x,-y,z; -vx,-vy,vz)   copy 4 (-x,-y,-z; -vx,-vy,-vz).
// Aperture regrouping ("The orbits are collected first in regular bins and then regrouped into Voronoi bins
// according to the pre-defined binning strategy"): ap_map[iy*nx+ix] is the aperture of image pixel (ix,iy), < 0 = the pixel
// belongs to no aperture (such samples are dropped and counted in nout like out-of-grid ones); the LOSVD row then holds
// n_ap*nv cells, index ap*nv+iv.  ap_map == NULL: no regrouping.
// density_mode 1: the 3-D mass matrix on cells uniform in (R, phi, z) ("we divide the 3D cylindrical space
// into N_dens bins uniformly spaced in (R, phi, z) direction"): the grid's (bx, by, bz) ranges and (dx, dy, dz) counts
// then mean R, phi in [0, 2 pi), z; index (jz*dy + jphi)*dx + jR.
int smo_build_observable_library(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt, int64_t n_steps,
                                 int32_t stride, const smo_projection* proj, int n_proj, const smo_grids* g, int32_t n_bundle,
                                 int fourfold, const int32_t* ap_map, int32_t n_ap, int density_mode, float* losvd, float* dens,
                                 int32_t* nout, int32_t* near_edge) {
    if (check_run(d, ics, n_orb, dt, n_steps, stride) || !proj || n_proj < 1 || !g || !losvd || !dens) return -1;
    if (density_mode != 0 && density_mode != 1) return -1;
    if (n_bundle < 1 || n_orb % n_bundle) return -1;
    if (g->nx < 1 || g->ny < 1 || g->nv < 1 || g->dx < 1 || g->dy < 1 || g->dz < 1) return -1;
    if (ap_map) {
        if (n_ap < 1) return -1;
        for (int64_t i = 0; i < (int64_t)g->nx * g->ny; ++i) if (ap_map[i] >= n_ap) return -1;
    }
    const int64_t n_rows = n_orb / n_bundle;
    const int64_t nlos = ap_map ? (int64_t)n_ap * g->nv : (int64_t)g->nx * g->ny * g->nv, nden = (int64_t)g->dx * g->dy * g->dz;
    std::vector<RotM> rm(n_proj);
    for (int p = 0; p < n_proj; ++p)
        rm[p] = { std::cos(proj[p].alpha), std::sin(proj[p].alpha), std::cos(proj[p].beta),
                  std::sin(proj[p].beta), std::cos(proj[p].gamma), std::sin(proj[p].gamma) };
    const double ivx = g->nx / (g->x1 - g->x0), ivy = g->ny / (g->y1 - g->y0), ivv = g->nv / (g->v1 - g->v0);
    const double idx = g->dx / (g->bx1 - g->bx0), idy = g->dy / (g->by1 - g->by0), idz = g->dz / (g->bz1 - g->bz0);
    static const double SGN[4][2] = { {1, 1}, {1, -1}, {-1, 1}, {-1, -1} };  // {sign of (x,y,vx,vy), sign of (z,vz)}
    const int n_copy = fourfold ? 4 : 1;
#pragma omp parallel for schedule(dynamic)
    for (int64_t r = 0; r < n_rows; ++r) {
        for (int p = 0; p < n_proj; ++p) std::memset(losvd + ((int64_t)p * n_rows + r) * nlos, 0, sizeof(float) * nlos);
        std::memset(dens + r * nden, 0, sizeof(float) * nden);
        std::vector<int32_t> no(n_proj + 1, 0), ne(n_proj + 1, 0);
        for (int64_t i = r * n_bundle; i < (r + 1) * n_bundle; ++i) {
            Orbit<double> o; o.d = d; o.init(ics + 6 * i);
            for (int64_t k = 1; k <= n_steps; ++k) {
                o.step(dt, k);
                if (k % stride) continue;
                double t = (double)k * dt;
                double theta = d->omega_p * t + d->phase0;
                double c = std::cos(theta), sn = std::sin(theta);
                double xb0[3] = { c * o.x[0] + sn * o.x[1], -sn * o.x[0] + c * o.x[1], o.x[2] };
                double vb0[3] = { c * o.v[0] + sn * o.v[1], -sn * o.v[0] + c * o.v[1], o.v[2] };
                for (int m = 0; m < n_copy; ++m) {
                    double xb[3] = { SGN[m][0] * xb0[0], SGN[m][0] * xb0[1], SGN[m][1] * xb0[2] };
                    double vb[3] = { SGN[m][0] * vb0[0], SGN[m][0] * vb0[1], SGN[m][1] * vb0[2] };
                    bool e = false;
                    // density cell: Cartesian (x_b, y_b, z_b), or (density_mode 1) the paper's cylindrical cells uniform in
                    // (R, phi, z) of the bar frame, phi = atan2(y_b, x_b) taken in [0, 2 pi)
                    double u0 = xb[0], u1 = xb[1];
                    if (density_mode == 1) {
                        u0 = std::sqrt(xb[0] * xb[0] + xb[1] * xb[1]);
                        u1 = std::atan2(xb[1], xb[0]);
                        if (u1 < 0) u1 += 2 * M_PI;
                    }
                    int jx = bin1(u0, g->bx0, idx, g->dx, &e), jy = bin1(u1, g->by0, idy, g->dy, &e),
                        jz = bin1(xb[2], g->bz0, idz, g->dz, &e);
                    if (jx >= 0 && jy >= 0 && jz >= 0) dens[r * nden + ((int64_t)jz * g->dy + jy) * g->dx + jx] += 1.0f;
                    else no[n_proj]++;
                    if (e) ne[n_proj]++;
                    for (int p = 0; p < n_proj; ++p) {
                        double out[3]; project(rm[p], xb, vb, out);
                        bool e2 = false;
                        int ix = bin1(out[0], g->x0, ivx, g->nx, &e2), iy = bin1(out[1], g->y0, ivy, g->ny, &e2),
                            iv = bin1(out[2], g->v0, ivv, g->nv, &e2);
                        int64_t cell = -1;
                        if (ix >= 0 && iy >= 0 && iv >= 0) {
                            const int64_t pix = (int64_t)iy * g->nx + ix;
                            if (!ap_map) cell = pix * g->nv + iv;
                            else if (ap_map[pix] >= 0) cell = (int64_t)ap_map[pix] * g->nv + iv;
                        }
                        if (cell >= 0) losvd[((int64_t)p * n_rows + r) * nlos + cell] += 1.0f;
                        else no[p]++;
                        if (e2) ne[p]++;
                    }
                }
            }
        }
        for (int p = 0; p <= n_proj; ++p) {
            if (nout) nout[(int64_t)p * n_rows + r] = no[p];
            if (near_edge) near_edge[(int64_t)p * n_rows + r] = ne[p];
        }
    }
    return 0;
}

// Gauss-Hermite terms of one sample (Eq.2): alpha(w) H_m(w), m = 0..4, with alpha(w) = exp(-w^2/2)/sqrt(2 pi)
// and the modified Hermite polynomials of van der Marel & Franx (1993) / Gerhard (1993), which the paper cites without
// printing them (reading R17):
//   H0 = 1, H1 = sqrt(2) w, H2 = (2w^2-1)/sqrt(2), H3 = (2 sqrt(2) w^3 - 3 sqrt(2) w)/sqrt(6), H4 = (4w^4-12w^2+3)/sqrt(24),
// orthonormal in the sense  integral alpha(w)^2 H_m(w) H_n(w) dw = delta_mn / (2 sqrt(pi)).
static void gh_terms(double w, double* t) {
    const double al = std::exp(-0.5 * w * w) / std::sqrt(2.0 * M_PI);
    const double w2 = w * w;
    t[0] = al;
    t[1] = al * std::sqrt(2.0) * w;
    t[2] = al * (2.0 * w2 - 1.0) / std::sqrt(2.0);
    t[3] = al * (2.0 * std::sqrt(2.0) * w2 * w - 3.0 * std::sqrt(2.0) * w) / std::sqrt(6.0);
    t[4] = al * (4.0 * w2 * w2 - 12.0 * w2 + 3.0) / std::sqrt(24.0);
}

int smo_gh_terms(const double* w, int64_t n, double* out5) {
    for (int64_t i = 0; i < n; ++i) gh_terms(w[i], out5 + 5 * i);
    return 0;
}

// Gauss-Hermite observable matrices on the fly ("we compute h_m of every orbit i in every 2D aperture n";
// PAPER.md:108 for the surface density): per row, projection and aperture n, over the recorded samples k whose image pixel
// belongs to aperture n (ALL line-of-sight velocities),
//   gh[..][n][0]   = number of samples                       (the surface-density matrix before normalisation)
//   gh[..][n][1+m] = sum_k alpha(w_k) H_m(w_k), m = 0..4,    w_k = (v_los,k - v0[n]) / s[n]
// so that h_m of the row's LOSVD in aperture n is (2 sqrt(pi)/gamma) gh[1+m]/gh[0] for a LOSVD of unit mass (the caller
// normalises).  Bundles, fourfold symmetrisation and density cells as in smo_build_observable_library; the velocity axis of
// the grids is not used.
int smo_build_gh_library(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt, int64_t n_steps,
                         int32_t stride, const smo_projection* proj, int n_proj, const smo_grids* g, int32_t n_bundle,
                         int fourfold, const int32_t* ap_map, int32_t n_ap, const double* v0, const double* sw, int density_mode,
                         double* gh, float* dens, int32_t* nout, int32_t* near_edge) {
    if (check_run(d, ics, n_orb, dt, n_steps, stride) || !proj || n_proj < 1 || !g || !gh || !dens || !ap_map || !v0 || !sw) return -1;
    if (n_bundle < 1 || n_orb % n_bundle || n_ap < 1) return -1;
    if (density_mode != 0 && density_mode != 1) return -1;
    for (int64_t i = 0; i < (int64_t)g->nx * g->ny; ++i) if (ap_map[i] >= n_ap) return -1;
    for (int i = 0; i < n_ap; ++i) if (!(sw[i] > 0)) return -1;
    const int64_t n_rows = n_orb / n_bundle;
    const int64_t nden = (int64_t)g->dx * g->dy * g->dz, ngh = (int64_t)n_ap * 6;
    std::vector<RotM> rm(n_proj);
    for (int p = 0; p < n_proj; ++p)
        rm[p] = { std::cos(proj[p].alpha), std::sin(proj[p].alpha), std::cos(proj[p].beta),
                  std::sin(proj[p].beta), std::cos(proj[p].gamma), std::sin(proj[p].gamma) };
    const double ivx = g->nx / (g->x1 - g->x0), ivy = g->ny / (g->y1 - g->y0);
    const double idx = g->dx / (g->bx1 - g->bx0), idy = g->dy / (g->by1 - g->by0), idz = g->dz / (g->bz1 - g->bz0);
    static const double SGN[4][2] = { {1, 1}, {1, -1}, {-1, 1}, {-1, -1} };
    const int n_copy = fourfold ? 4 : 1;
#pragma omp parallel for schedule(dynamic)
    for (int64_t r = 0; r < n_rows; ++r) {
        for (int p = 0; p < n_proj; ++p) for (int64_t q = 0; q < ngh; ++q) gh[((int64_t)p * n_rows + r) * ngh + q] = 0.0;
        std::memset(dens + r * nden, 0, sizeof(float) * nden);
        std::vector<int32_t> no(n_proj + 1, 0), ne(n_proj + 1, 0);
        for (int64_t i = r * n_bundle; i < (r + 1) * n_bundle; ++i) {
            Orbit<double> o; o.d = d; o.init(ics + 6 * i);
            for (int64_t k = 1; k <= n_steps; ++k) {
                o.step(dt, k);
                if (k % stride) continue;
                double t = (double)k * dt;
                double theta = d->omega_p * t + d->phase0;
                double c = std::cos(theta), sn = std::sin(theta);
                double xb0[3] = { c * o.x[0] + sn * o.x[1], -sn * o.x[0] + c * o.x[1], o.x[2] };
                double vb0[3] = { c * o.v[0] + sn * o.v[1], -sn * o.v[0] + c * o.v[1], o.v[2] };
                for (int m = 0; m < n_copy; ++m) {
                    double xb[3] = { SGN[m][0] * xb0[0], SGN[m][0] * xb0[1], SGN[m][1] * xb0[2] };
                    double vb[3] = { SGN[m][0] * vb0[0], SGN[m][0] * vb0[1], SGN[m][1] * vb0[2] };
                    bool e = false;
                    double u0 = xb[0], u1 = xb[1];
                    if (density_mode == 1) {
                        u0 = std::sqrt(xb[0] * xb[0] + xb[1] * xb[1]);
                        u1 = std::atan2(xb[1], xb[0]);
                        if (u1 < 0) u1 += 2 * M_PI;
                    }
                    int jx = bin1(u0, g->bx0, idx, g->dx, &e), jy = bin1(u1, g->by0, idy, g->dy, &e),
                        jz = bin1(xb[2], g->bz0, idz, g->dz, &e);
                    if (jx >= 0 && jy >= 0 && jz >= 0) dens[r * nden + ((int64_t)jz * g->dy + jy) * g->dx + jx] += 1.0f;
                    else no[n_proj]++;
                    if (e) ne[n_proj]++;
                    for (int p = 0; p < n_proj; ++p) {
                        double out[3]; project(rm[p], xb, vb, out);
                        bool e2 = false;
                        int ix = bin1(out[0], g->x0, ivx, g->nx, &e2), iy = bin1(out[1], g->y0, ivy, g->ny, &e2);
                        int ap = (ix >= 0 && iy >= 0) ? ap_map[(int64_t)iy * g->nx + ix] : -1;
                        if (ap >= 0) {
                            double tm[5];
                            gh_terms((out[2] - v0[ap]) / sw[ap], tm);
                            double* row = gh + ((int64_t)p * n_rows + r) * ngh + (int64_t)ap * 6;
                            row[0] += 1.0;
                            for (int q = 0; q < 5; ++q) row[1 + q] += tm[q];
                        } else no[p]++;
                        if (e2) ne[p]++;
                    }
                }
            }
        }
        for (int p = 0; p <= n_proj; ++p) {
            if (nout) nout[(int64_t)p * n_rows + r] = no[p];
            if (near_edge) near_edge[(int64_t)p * n_rows + r] = ne[p];
        }
    }
    return 0;
}

int smo_build_bundled_library(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt, int64_t n_steps,
                              int32_t stride, const smo_projection* proj, int n_proj, const smo_grids* g, int32_t n_bundle,
                              int fourfold, float* losvd, float* dens, int32_t* nout, int32_t* near_edge) {
    return smo_build_observable_library(d, ics, n_orb, dt, n_steps, stride, proj, n_proj, g, n_bundle, fourfold, nullptr, 0, 0,
                                        losvd, dens, nout, near_edge);
}

int smo_ferrers_lambda(double a, double b, double c, const double* xyz, int64_t n, double* lam) {
    if (!(a > b && b > c && c > 0)) return -1;
    for (int64_t i = 0; i < n; ++i)
        lam[i] = (double)ferrers_lambda((Q)a * a, (Q)b * b, (Q)c * c, (Q)xyz[3 * i] * xyz[3 * i],
                                        (Q)xyz[3 * i + 1] * xyz[3 * i + 1], (Q)xyz[3 * i + 2] * xyz[3 * i + 2]);
    return 0;
}

int smo_ferrers_W(double a, double b, double c, double lam, double* W20) {
    if (!(a > b && b > c && c > 0) || lam < 0) return -1;
    Q W[20];
    ferrers_W((Q)a * a, (Q)b * b, (Q)c * c, (Q)lam, W);
    for (int i = 0; i < 20; ++i) W20[i] = (double)W[i];
    return 0;
}

int smo_project(const smo_projection* p, const double* xb, const double* vb, double* out3) {
    RotM m = { std::cos(p->alpha), std::sin(p->alpha), std::cos(p->beta), std::sin(p->beta), std::cos(p->gamma), std::sin(p->gamma) };
    project(m, xb, vb, out3);
    return 0;
}

int smo_jacobi(const smo_potential_desc* d, const double* state, int64_t n, double t, double* EJ) {
    if (check_desc(d)) return -1;
    for (int64_t i = 0; i < n; ++i) EJ[i] = jacobi(d, state + 6 * i, t);
    return 0;
}

int smo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
