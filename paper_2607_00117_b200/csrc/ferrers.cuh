// ferrers.cuh -- Ferrers n=2 bar force (and potential) from the tabulated anchor integrals.
//
//   rho = rho_c (1-m^2)^2,  rho_c = 105 M/(32 pi abc),  m^2(u) = x^2/A + y^2/B + z^2/C,
//   A=a^2+u, B=b^2+u, C=c^2+u, Delta = sqrt(ABC), lambda = positive root of m^2(lambda)=1 (0 inside);
//   F_i = -K x_i int_lambda^inf (1-m^2(u))^2 du /(A_i Delta),  K = 2 pi G abc rho_c = 105 GM/16.
// Expanding (1-m^2)^2 gives F in terms of W_ijk(lambda) = int_lambda^inf du/(Delta A^i B^j C^k).
// Steps:
//   1. lambda by clamped, warm-started Newton in fp32 (the force is stationary in lambda to second order:
//      dF ~ dlambda^3, so fp32 accuracy is far more than enough);
//   2. anchors W210, W201, W021, W111 from the piecewise polynomials in C = c^2+lambda;
//   3. the other 15 W_ijk from the exact identities
//        (2i+1)W_{i+1,j,k} + (2j+1)W_{i,j+1,k} + (2k+1)W_{i,j,k+1} = 2/(Delta A^i B^j C^k)
//        W_{i,j+1,k} = W_{i+1,j,k} + p W_{i+1,j+1,k},  W_{i,j,k+1} = W_{i+1,j,k} + q W_{i+1,j,k+1}
//      arranged so that error amplification stays below ~10 everywhere;
//   4. the degree-2 polynomial in (x^2, y^2, z^2).
#pragma once
#include "force.cuh"

namespace smx {

// lambda in fp32: Newton on psi(u) = 1/m^2(u) - 1, which is increasing and concave for u > -c^2 and
// nearly linear both close to the pole u = -c^2 and in the far field.  For a concave increasing function the
// Newton iterate lies left of the root after the first step from ANY start, and then converges monotonically;
// plain Newton on m^2-1 crawls near the pole.  The iterate is clamped at 0, so points inside the ellipsoid
// (m^2(0) <= 1) end at exactly 0.
//   guess >= 0: warm start (the integrator passes the value extrapolated from the previous two steps, which is
//   within ~1e-3 of the root: one or two iterations);  guess < 0: cold start from a weighted-radius estimate.
// The loop ends when EVERY lane of the warp made a step <= FERRERS_LAMBDA_TOL (c^2+lambda): the error left after
// such a step is of order tol^2 (quadratic convergence), i.e. < 1e-5 (c^2+lambda), which the force needs.
// All 32 lanes of the warp must call this together (the kernels keep out-of-range lanes alive).
constexpr int FERRERS_NEWTON_MAXIT = 16;
constexpr float FERRERS_LAMBDA_TOL = 1.5e-3f;
SMX_HD float ferrers_lambda32(float a2, float b2, float c2, float X, float Y, float Z, float guess, int* iters = nullptr) {
    float r2 = X + Y + Z;
    float cold = r2 > 0.0f ? fmaxf(0.0f, r2 - (a2 * X + b2 * Y + c2 * Z) * frcp(r2)) : 0.0f;
    float lam = guess >= 0.0f ? guess : cold;
    int it = 0;
    for (; it < FERRERS_NEWTON_MAXIT; ++it) {
        float iA = frcp(a2 + lam), iB = frcp(b2 + lam), iC = frcp(c2 + lam);
        float tA = X * iA, tB = Y * iB, tC = Z * iC;
        float m2 = tA + tB + tC;
        float s2 = tA * iA + tB * iB + tC * iC;  // -d(m^2)/du
        float step = s2 > 0.0f ? (m2 - 1.0f) * m2 * frcp(s2) : -lam;  // s2 == 0 only at the centre: lambda = 0
        float nl = fmaxf(0.0f, lam + step);
        bool conv = fabsf(nl - lam) <= FERRERS_LAMBDA_TOL * (c2 + nl);
        lam = nl;
#ifdef __CUDA_ARCH__
        if (__all_sync(0xFFFFFFFFu, conv)) { ++it; break; }
#else
        if (conv) { ++it; break; }
#endif
    }
    if (iters) *iters = it;
    return lam;
}

// anchors W210, W201, W021, W111 (and W000 if PHI) at C = c^2 + lambda
template <typename T, bool PHI>
SMX_HD void ferrers_anchors(const PotS<T>& P, const T* tab, T A, T C, T* w) {
    constexpr int NC = FT<T>::NCOEF;
    constexpr int ROW = FT<T>::ROW;
    T tau;
    int j = ft_key(C, P.ft_ls, &tau) - P.ft_key0;
    if (j < P.ft_nint) {
        j = j < 0 ? 0 : j;
        const T* row = tab + j * ROW;
#pragma unroll
        for (int f = 0; f < FT_NANCHOR; ++f) {
            T s = row[f * NC + NC - 1];
#pragma unroll
            for (int k = NC - 2; k >= 0; --k) s = fma_t(s, tau, row[f * NC + k]);
            w[f] = s;
        }
        if (PHI) {
            const T* r0 = P.tab0 + (long long)j * NC;
            T s = r0[NC - 1];
#pragma unroll
            for (int k = NC - 2; k >= 0; --k) s = fma_t(s, tau, r0[k]);
            w[FT_NANCHOR] = s;
        }
    } else {  // far field: W_f = S^(n_f+1/2) sum_m far[f][m] S^m, S = 1/A
        T rS = rsqrt_t(A);
        T S = rS * rS;
        T S3 = S * S * S * rS;
#pragma unroll
        for (int f = 0; f < (PHI ? FT_NFUNC : FT_NANCHOR); ++f) {
            T s = P.far[f][FT_NFAR - 1];
#pragma unroll
            for (int m = FT_NFAR - 2; m >= 0; --m) s = fma_t(s, S, P.far[f][m]);
            w[f] = s * (f < FT_NANCHOR ? S3 : rS);
        }
    }
}

template <typename T, bool PHI>
SMX_HD void ferrers(const PotS<T>& P, const T* tab, const CompS<T>& c, T x, T y, T z, T& fx, T& fy, T& fz, T& phi, float& lam_io) {
    const T K = c.c[0], a2 = c.c[1], b2 = c.c[2], c2 = c.c[3], p = c.c[4], q = c.c[5];
    const T X = x * x, Y = y * y, Z = z * z;
    // lam_io: in = warm-start guess (< 0: none), out = the lambda found
    lam_io = ferrers_lambda32((float)a2, (float)b2, (float)c2, (float)X, (float)Y, (float)Z, lam_io);
    const T lam = (T)lam_io;
    const T A = a2 + lam, B = b2 + lam, C = c2 + lam;
    T w[FT_NFUNC];
    ferrers_anchors<T, PHI>(P, tab, A, C, w);
    const T W210 = w[0], W201 = w[1], W021 = w[2], W111 = w[3];
    // elementary terms 2/(Delta A^i B^j C^k)
    const T rsq = rsqrt_t(A * B * C);
    const T E = (T)2 * rsq, inv = rsq * rsq;
    const T iA = B * C * inv, iB = A * C * inv, iC = A * B * inv;
    const T eA = E * iA, eB = E * iB, eC = E * iC;
    const T third = (T)(1.0 / 3.0), fifth = (T)0.2;
    // level 3
    const T W120 = fma_t(fma_t(eA, iB, -W111), third, -W210);
    const T W102 = fma_t(fma_t(eA, iC, -W111), third, -W201);
    const T W012 = fma_t(fma_t(eB, iC, -W111), third, -W021);
    const T W300 = (fma_t(eA, iA, -W210) - W201) * fifth;
    const T W030 = (fma_t(eB, iB, -W120) - W021) * fifth;
    const T W003 = (fma_t(eC, iC, -W102) - W012) * fifth;
    // level 2
    const T W200 = fma_t(-q, W201, fma_t(-p, W210, eA)) * fifth;
    const T W110 = fma_t(p, W210, W200);
    const T W101 = fma_t(q, W201, W200);
    const T W020 = fma_t(p, W120, W110);
    const T W011 = fma_t(q, W111, W110);
    const T W002 = fma_t(q, W102, W101);
    // level 1
    const T W100 = fma_t(-q, W101, fma_t(-p, W110, E)) * third;
    const T W010 = fma_t(p, W110, W100);
    const T W001 = fma_t(q, W101, W100);
    // (1-m^2)^2 / A_i expanded
    const T XX = X * X, YY = Y * Y, ZZ = Z * Z, XY = (T)2 * X * Y, XZ = (T)2 * X * Z, YZ = (T)2 * Y * Z;
    T gx = fma_t((T)-2, fma_t(X, W200, fma_t(Y, W110, Z * W101)), W100);
    gx = fma_t(XX, W300, fma_t(YY, W120, fma_t(ZZ, W102, fma_t(XY, W210, fma_t(XZ, W201, fma_t(YZ, W111, gx))))));
    T gy = fma_t((T)-2, fma_t(X, W110, fma_t(Y, W020, Z * W011)), W010);
    gy = fma_t(XX, W210, fma_t(YY, W030, fma_t(ZZ, W012, fma_t(XY, W120, fma_t(XZ, W111, fma_t(YZ, W021, gy))))));
    T gz = fma_t((T)-2, fma_t(X, W101, fma_t(Y, W011, Z * W002)), W001);
    gz = fma_t(XX, W201, fma_t(YY, W021, fma_t(ZZ, W003, fma_t(XY, W111, fma_t(XZ, W102, fma_t(YZ, W012, gz))))));
    fx -= K * x * gx; fy -= K * y * gy; fz -= K * z * gz;
    if (PHI) {
        // Phi = -(K/6) int (1-m^2)^3 du/Delta = -(K/6)[W000 - 3 S1 + 3 S2 - S3]
        const T W000 = w[FT_NANCHOR];
        T S1 = X * W100 + Y * W010 + Z * W001;
        T S2 = XX * W200 + YY * W020 + ZZ * W002 + XY * W110 + XZ * W101 + YZ * W011;
        T S3 = XX * X * W300 + YY * Y * W030 + ZZ * Z * W003
             + (T)3 * (XX * Y * W210 + XX * Z * W201 + X * YY * W120 + YY * Z * W021 + X * ZZ * W102 + Y * ZZ * W012)
             + (T)6 * X * Y * Z * W111;
        phi -= K * (T)(1.0 / 6.0) * (W000 - (T)3 * S1 + (T)3 * S2 - S3);
    }
}

// ---------------------------------------------------------------- total field
template <typename T, bool PHI>
SMX_HD void comp_force(const PotS<T>& P, const T* tab, const CompS<T>& c, T x, T y, T z, T& fx, T& fy, T& fz, T& phi, float& lam_io) {
    switch (c.kind) {
        case K_PLUMMER: plummer<T, PHI>(c, x, y, z, fx, fy, fz, phi); break;
        case K_MN: miyamoto_nagai<T, PHI>(c, x, y, z, fx, fy, fz, phi); break;
        case K_NFW: nfw<T, PHI>(c, x, y, z, fx, fy, fz, phi); break;
        case K_FERRERS: ferrers<T, PHI>(P, tab, c, x, y, z, fx, fy, fz, phi, lam_io); break;
        default: break;
    }
}

// a = F(x, t) with (cs, sn) = (cos, sin) of the bar angle Omega_p t + phase0:
// static components at x; rotating ones at x_b = Rz(-theta) x, rotated back.
// POT selects a specialised body (same arithmetic, no component loop); `tab` = Ferrers anchor table.
template <typename T, bool PHI, int POT>
SMX_HD void total_force(const PotS<T>& P, const T* tab, T x, T y, T z, T cs, T sn, T& ax, T& ay, T& az, T& phi, float& lam_io) {
    ax = ay = az = (T)0;
    if (PHI) phi = (T)0;
    if (POT == POT_PLUMMER) {
        plummer<T, PHI>(P.comp[0], x, y, z, ax, ay, az, phi);
    } else if (POT == POT_BARRED) {
        miyamoto_nagai<T, PHI>(P.comp[P.i_mn], x, y, z, ax, ay, az, phi);
        nfw<T, PHI>(P.comp[P.i_nfw], x, y, z, ax, ay, az, phi);
        T xb = fma_t(cs, x, sn * y), yb = fma_t(cs, y, -sn * x);
        T bx = (T)0, by = (T)0, bz = (T)0;
        ferrers<T, PHI>(P, tab, P.comp[P.i_fer], xb, yb, z, bx, by, bz, phi, lam_io);
        ax += fma_t(cs, bx, -sn * by);
        ay += fma_t(sn, bx, cs * by);
        az += bz;
    } else {
        for (int i = 0; i < P.n_comp; ++i)
            if (!P.comp[i].rotating) comp_force<T, PHI>(P, tab, P.comp[i], x, y, z, ax, ay, az, phi, lam_io);
        if (P.has_rot) {
            T xb = fma_t(cs, x, sn * y), yb = fma_t(cs, y, -sn * x);
            T bx = (T)0, by = (T)0, bz = (T)0;
            for (int i = 0; i < P.n_comp; ++i)
                if (P.comp[i].rotating) comp_force<T, PHI>(P, tab, P.comp[i], xb, yb, z, bx, by, bz, phi, lam_io);
            ax += fma_t(cs, bx, -sn * by);
            ay += fma_t(sn, bx, cs * by);
            az += bz;
        }
    }
}

}  // namespace smx
