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
#include "dehnen.cuh"
#include "force.cuh"

namespace smx {

// lambda in fp32: root of psi(u) = 1/m^2(u) - 1, which is increasing and concave for u > -c^2 and nearly linear both
// close to the pole u = -c^2 and in the far field (plain Newton on m^2 - 1 crawls near the pole).  With M = m^2(u),
// s2 = sum X_i/A_i^2 = -M', s3 = sum X_i/A_i^3 = M''/2:
//   Newton on psi   du = (M-1) M / s2                  monotone from the left after the first step from ANY start
//   Halley on psi   du = (M-1) s2 / (s2^2 - (M-1) s3)  cubic convergence; used when its denominator is safely positive
// (the two agree to first order at the root).  The iterate is clamped at 0, so points inside the ellipsoid (M(0) <= 1)
// end at exactly 0.
//   guess >= 0: warm start (the integrator passes the quadratic extrapolation of the previous three steps, within
//   ~1e-3..1e-2 of the root: ONE Halley step leaves ~1e-7);  guess < 0: cold start from a weighted-radius estimate.
// The loop ends when EVERY lane of the warp made a step <= FERRERS_LAMBDA_TOL (c^2+lambda): the error left after such
// a step is O(tol^2) even for the Newton fallback, i.e. < 1e-5 (c^2+lambda), which the force needs.
// All 32 lanes of the warp must call this together (the kernels keep out-of-range lanes alive).
constexpr int FERRERS_NEWTON_MAXIT = 16;
constexpr float FERRERS_LAMBDA_TOL = 8.0e-3f;

#ifdef __CUDA_ARCH__
#define SMX_ALL(pred) __all_sync(0xFFFFFFFFu, (pred))
#define SMX_ANY(pred) __any_sync(0xFFFFFFFFu, (pred))
#else
#define SMX_ALL(pred) (pred)
#define SMX_ANY(pred) (pred)
#endif

// one clamped step; conv = the step was <= tol (c^2 + lambda) and of Halley type (or the iterate sits at the clamp)
SMX_HD float ferrers_lambda_step(float a2, float b2, float c2, float X, float Y, float Z, float lam, bool& conv) {
    float iA = frcp(a2 + lam), iB = frcp(b2 + lam), iC = frcp(c2 + lam);
    float tA = X * iA, tB = Y * iB, tC = Z * iC;
    float m2 = tA + tB + tC;
    float uA = tA * iA, uB = tB * iB, uC = tC * iC;
    float s2 = uA + uB + uC;                      // -d(m^2)/du
    float s3 = uA * iA + uB * iB + uC * iC;       // (1/2) d2(m^2)/du2
    float d = m2 - 1.0f;
    float den_h = s2 * s2 - d * s3;
    bool halley = den_h > 0.5f * s2 * s2;         // always true near the root (d -> 0) and for d < 0
    float num = halley ? d * s2 : d * m2;
    float den = halley ? den_h : s2;
    float step = s2 > 0.0f ? num * frcp(den) : -lam;  // s2 == 0 only at the centre: lambda = 0
    float nl = fmaxf(0.0f, lam + step);
    float moved = fabsf(nl - lam);
    // after a Halley step of relative size t the error is O(t^3); after a Newton step O(t^2): ask more of the latter
    conv = moved <= (halley ? FERRERS_LAMBDA_TOL : 0.5f * FERRERS_LAMBDA_TOL) * (c2 + nl);
    return nl;
}

// COLD_OK = false: the caller guarantees guess >= 0 (the integrator's time loop, which starts every orbit from a separate
// cold solve): without the cold-start vote and branch the extrapolation, the rotation into the bar frame and the first
// iteration form ONE basic block with the disc and halo forces, which the scheduler then interleaves with the iteration.
template <bool COLD_OK = true>
SMX_HD float ferrers_lambda32(float a2, float b2, float c2, float X, float Y, float Z, float guess, int* iters = nullptr) {
    float lam = guess;
    if (COLD_OK && SMX_ANY(guess < 0.0f)) {  // cold start (first step of an orbit, test hooks): weighted-radius estimate
        float r2 = X + Y + Z;
        float cold = r2 > 0.0f ? fmaxf(0.0f, r2 - (a2 * X + b2 * Y + c2 * Z) * frcp(r2)) : 0.0f;
        lam = guess >= 0.0f ? guess : cold;
    }
    bool conv;
    // one unconditional iteration (what the integrator's extrapolated warm start needs): straight-line code that the
    // scheduler interleaves with the disc and halo chains; further iterations only while some lane of the warp moves
    lam = ferrers_lambda_step(a2, b2, c2, X, Y, Z, lam, conv);
    int it = 1;
    while (!SMX_ALL(conv) && it < FERRERS_NEWTON_MAXIT) {
        // a lane that has converged keeps its value, so that an orbit's result never depends on its warp neighbours
        bool c2nd;
        const float nl = ferrers_lambda_step(a2, b2, c2, X, Y, Z, lam, c2nd);
        lam = conv ? lam : nl;
        conv = conv || c2nd;
        ++it;
    }
    if (iters) *iters = it;
    return lam;
}

// Loop-invariant description of the Ferrers component, held in registers by the integrator.
// SH = true: `tab_sh` is the 32-bit shared-memory address of the anchor table and rows are read with ld.shared
// (the generic pointer made the compiler re-derive the shared window base, an S2R, in every step).
template <typename T, bool SH>
struct FerrersCtx {
    T K, a2, b2, c2, p, q;
    float fa2, fb2, fc2;
    int key0, nint;
    const T* tab;       // anchor rows [interval][ROW]
    unsigned tab_sh;    // the same as a shared-memory address (SH)
    const T* tab0;      // W000 rows (potential only)
    const T* far;       // far-field series [FT_NFUNC][FT_NFAR]
};

template <typename T, bool SH>
SMX_HD FerrersCtx<T, SH> make_ferrers_ctx(const PotS<T>& P, const T* tab, const CompS<T>& c) {
    FerrersCtx<T, SH> f;
    f.K = c.c[0]; f.a2 = c.c[1]; f.b2 = c.c[2]; f.c2 = c.c[3]; f.p = c.c[4]; f.q = c.c[5];
    f.fa2 = (float)f.a2; f.fb2 = (float)f.b2; f.fc2 = (float)f.c2;
    f.key0 = P.ft_key0; f.nint = P.ft_nint;
    f.tab = tab; f.tab0 = P.tab0; f.far = &P.far[0][0];
    f.tab_sh = 0;
#ifdef __CUDA_ARCH__
    if (SH) {
        unsigned a = (unsigned)__cvta_generic_to_shared(tab);
        asm volatile("mov.u32 %0, %1;" : "=r"(f.tab_sh) : "r"(a));  // opaque: keeps the address in a register
    }
#endif
    return f;
}

// The four anchors on interval j at tau, fp64 path.  Row = 20 doubles [f][k<5] + 12 floats [f][k-5<3], 13 16-byte
// loads: W_f = sum_{k<5} c_k tau^k (fp64 Horner) + tau^5 (c5 + c6 tau + c7 tau^2) (fp32 Horner; |tail| < 1.1e-9 W).
template <bool SH>
SMX_HD void eval_anchor_row(const FerrersCtx<double, SH>& F, int j, double tau, double* w) {
    double d[FT_NANCHOR * FT_ND];
    float t[FT_NANCHOR * FT_NF];
    bool loaded = false;
#ifdef __CUDA_ARCH__
    if (SH) {
        const unsigned a = F.tab_sh + (unsigned)j * (FT_ROW64 * 8);
#pragma unroll
        for (int i = 0; i < FT_NANCHOR * FT_ND; i += 2)
            asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(d[i]), "=d"(d[i + 1]) : "r"(a + i * 8));
#pragma unroll
        for (int i = 0; i < FT_NANCHOR * FT_NF; i += 4)
            asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(t[i]), "=f"(t[i + 1]), "=f"(t[i + 2]), "=f"(t[i + 3])
                : "r"(a + FT_NANCHOR * FT_ND * 8 + i * 4));
        loaded = true;
    }
#endif
    if (!loaded) {
        const double* row = F.tab + (long long)j * FT_ROW64;
        const float* tail = reinterpret_cast<const float*>(row + FT_NANCHOR * FT_ND);
#pragma unroll
        for (int i = 0; i < FT_NANCHOR * FT_ND; ++i) d[i] = row[i];
#pragma unroll
        for (int i = 0; i < FT_NANCHOR * FT_NF; ++i) t[i] = tail[i];
    }
    const float tf = (float)tau;
    const double t2 = tau * tau, t5 = t2 * t2 * tau;
#pragma unroll
    for (int f = 0; f < FT_NANCHOR; ++f) {
        float tl = t[f * FT_NF + FT_NF - 1];
#pragma unroll
        for (int k = FT_NF - 2; k >= 0; --k) tl = tl * tf + t[f * FT_NF + k];
        double s = d[f * FT_ND + FT_ND - 1];
#pragma unroll
        for (int k = FT_ND - 2; k >= 0; --k) s = fma_t(s, tau, d[f * FT_ND + k]);
        w[f] = fma_t(t5, (double)tl, s);
    }
}
// fp32 path: 20 floats [f][k<5], five 16-byte loads
template <bool SH>
SMX_HD void eval_anchor_row(const FerrersCtx<float, SH>& F, int j, float tau, float* w) {
    float r[FT_ROW32];
    const float4* row = reinterpret_cast<const float4*>(F.tab + (long long)j * FT_ROW32);
#pragma unroll
    for (int i = 0; i < FT_ROW32 / 4; ++i) {
        const float4 v = row[i];
        r[4 * i] = v.x; r[4 * i + 1] = v.y; r[4 * i + 2] = v.z; r[4 * i + 3] = v.w;
    }
#pragma unroll
    for (int f = 0; f < FT_NANCHOR; ++f) {
        float s = r[f * FT_NCOEF32 + FT_NCOEF32 - 1];
#pragma unroll
        for (int k = FT_NCOEF32 - 2; k >= 0; --k) s = fma_t(s, tau, r[f * FT_NCOEF32 + k]);
        w[f] = s;
    }
}

// anchors W210, W201, W021, W111 (and W000 if PHI) at C = c^2 + lambda
template <typename T, bool PHI, bool SH>
SMX_HD void ferrers_anchors(const FerrersCtx<T, SH>& F, T A, T C, T* w) {
    T tau;
    const int jraw = ft_key(C, &tau) - F.key0;
    const bool far = jraw >= F.nint;
    // the table path is straight-line code for every lane (clamped row, discarded where far) ...
    const int j = jraw < 0 ? 0 : (far ? F.nint - 1 : jraw);
    eval_anchor_row<SH>(F, j, tau, w);
    if (PHI) {  // W000: eight doubles per interval, global memory (potential / Jacobi diagnostic only, fp64 only)
        const T* r0 = F.tab0 + (long long)j * FT_NC0;
        T s = r0[FT_NC0 - 1];
#pragma unroll
        for (int k = FT_NC0 - 2; k >= 0; --k) s = fma_t(s, tau, r0[k]);
        w[FT_NANCHOR] = s;
    }
    // ... and the far field (C >= 2^FT_E1, r > ~32 kpc) is a rare warp-uniform branch after it:
    // W_f = S^(n_f+1/2) sum_m far[f][m] S^m, S = 1/A
    if (SMX_ANY(far)) {
        T rS = rsqrt_t(A);
        T S = rS * rS;
        T S3 = S * S * S * rS;
#pragma unroll
        for (int f = 0; f < (PHI ? FT_NFUNC : FT_NANCHOR); ++f) {
            T s = F.far[f * FT_NFAR + FT_NFAR - 1];
#pragma unroll
            for (int m = FT_NFAR - 2; m >= 0; --m) s = fma_t(s, S, F.far[f * FT_NFAR + m]);
            s *= (f < FT_NANCHOR ? S3 : rS);
            w[f] = far ? s : w[f];
        }
    }
}

template <typename T, bool PHI, bool SH, bool COLD_OK = true>
SMX_HD void ferrers(const FerrersCtx<T, SH>& F, T x, T y, T z, T& fx, T& fy, T& fz, T& phi, float& lam_io) {
    const T p = F.p, q = F.q;
    const T X = x * x, Y = y * y, Z = z * z;
    // lam_io: in = warm-start guess (< 0: none), out = the lambda found
    lam_io = ferrers_lambda32<COLD_OK>(F.fa2, F.fb2, F.fc2, (float)X, (float)Y, (float)Z, lam_io);
    const T lam = (T)lam_io;
    const T A = F.a2 + lam, B = F.b2 + lam, C = F.c2 + lam;
    T w[FT_NFUNC];
    ferrers_anchors<T, PHI, SH>(F, A, C, w);
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
    // (1-m^2)^2 / A_i expanded; three short independent sums per component instead of one nine-deep FMA chain
    const T XX = X * X, YY = Y * Y, ZZ = Z * Z, XY = (T)2 * X * Y, XZ = (T)2 * X * Z, YZ = (T)2 * Y * Z;
    const T gx = (fma_t(XX, W300, fma_t(YY, W120, ZZ * W102)) + fma_t(XY, W210, fma_t(XZ, W201, YZ * W111)))
               + fma_t((T)-2, fma_t(X, W200, fma_t(Y, W110, Z * W101)), W100);
    const T gy = (fma_t(XX, W210, fma_t(YY, W030, ZZ * W012)) + fma_t(XY, W120, fma_t(XZ, W111, YZ * W021)))
               + fma_t((T)-2, fma_t(X, W110, fma_t(Y, W020, Z * W011)), W010);
    const T gz = (fma_t(XX, W201, fma_t(YY, W021, ZZ * W003)) + fma_t(XY, W111, fma_t(XZ, W102, YZ * W012)))
               + fma_t((T)-2, fma_t(X, W101, fma_t(Y, W011, Z * W002)), W001);
    fx -= F.K * x * gx; fy -= F.K * y * gy; fz -= F.K * z * gz;
    if (PHI) {
        // Phi = -(K/6) int (1-m^2)^3 du/Delta = -(K/6)[W000 - 3 S1 + 3 S2 - S3]
        const T W000 = w[FT_NANCHOR];
        T S1 = X * W100 + Y * W010 + Z * W001;
        T S2 = XX * W200 + YY * W020 + ZZ * W002 + XY * W110 + XZ * W101 + YZ * W011;
        T S3 = XX * X * W300 + YY * Y * W030 + ZZ * Z * W003
             + (T)3 * (XX * Y * W210 + XX * Z * W201 + X * YY * W120 + YY * Z * W021 + X * ZZ * W102 + Y * ZZ * W012)
             + (T)6 * X * Y * Z * W111;
        phi -= F.K * (T)(1.0 / 6.0) * (W000 - (T)3 * S1 + (T)3 * S2 - S3);
    }
}

// ---------------------------------------------------------------- total field
template <typename T, bool PHI>
SMX_HD void comp_force(const PotS<T>& P, const T* tab, const CompS<T>& c, T x, T y, T z, T& fx, T& fy, T& fz, T& phi, float& lam_io) {
    switch (c.kind) {
        case K_PLUMMER: plummer<T, PHI>(c, x, y, z, fx, fy, fz, phi); break;
        case K_MN: miyamoto_nagai<T, PHI>(c, x, y, z, fx, fy, fz, phi); break;
        case K_NFW: nfw<T, PHI>(c, x, y, z, fx, fy, fz, phi); break;
        case K_FERRERS: {
            const FerrersCtx<T, false> F = make_ferrers_ctx<T, false>(P, tab, c);
            ferrers<T, PHI, false>(F, x, y, z, fx, fy, fz, phi, lam_io);
            break;
        }
        case K_DEHNEN_T3:
        case K_DEHNEN_V4: dehnen_aly<T, PHI>(c, x, y, z, fx, fy, fz, phi); break;
        default: break;
    }
}

// a = F(x, t) with (cs, sn) = (cos, sin) of the bar angle Omega_p t + phase0:
// static components at x; rotating ones at x_b = Rz(-theta) x, rotated back.
// POT selects a specialised body (same arithmetic, no component loop); `tab` = Ferrers anchor table;
// FB = the Ferrers invariants prepared once by the caller (used by POT_BARRED only).
template <typename T, bool PHI, int POT, bool SH, bool COLD_OK = true>
SMX_HD void total_force(const PotS<T>& P, const T* tab, const FerrersCtx<T, SH>& FB, T x, T y, T z, T cs, T sn,
                        T& ax, T& ay, T& az, T& phi, float& lam_io) {
    ax = ay = az = (T)0;
    if (PHI) phi = (T)0;
    if (POT == POT_PLUMMER) {
        plummer<T, PHI>(P.comp[0], x, y, z, ax, ay, az, phi);
    } else if (POT == POT_BARRED) {
        T xb = fma_t(cs, x, sn * y), yb = fma_t(cs, y, -sn * x);
        T bx = (T)0, by = (T)0, bz = (T)0;
        // disc and halo in front of the bar: they do not depend on lambda, and in this order their FP64 chains share a
        // basic block with the fp32 lambda iteration (a latency-bound chain of its own), see ferrers_lambda32
        miyamoto_nagai<T, PHI>(P.comp[P.i_mn], x, y, z, ax, ay, az, phi);
        nfw<T, PHI>(P.comp[P.i_nfw], x, y, z, ax, ay, az, phi);
        ferrers<T, PHI, SH, COLD_OK>(FB, xb, yb, z, bx, by, bz, phi, lam_io);
        ax += fma_t(cs, bx, -sn * by);
        ay += fma_t(sn, bx, cs * by);
        az += bz;
    } else if (POT == POT_NEEDLE) {
        // one basic block: the two needle bars, the disc and the halo are independent chains the scheduler interleaves
        T xb = fma_t(cs, x, sn * y), yb = fma_t(cs, y, -sn * x);
        T bx = (T)0, by = (T)0, bz = (T)0;
        needle_bar_T<T, 3, PHI, true>(P.comp[P.i_fer], xb, yb, z, bx, by, bz, phi);
        needle_bar_T<T, 5, PHI, false>(P.comp[P.i_v4], xb, yb, z, bx, by, bz, phi);
        miyamoto_nagai<T, PHI>(P.comp[P.i_mn], x, y, z, ax, ay, az, phi);
        nfw<T, PHI>(P.comp[P.i_nfw], x, y, z, ax, ay, az, phi);
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
template <typename T, bool PHI, int POT>
SMX_HD void total_force(const PotS<T>& P, const T* tab, T x, T y, T z, T cs, T sn, T& ax, T& ay, T& az, T& phi, float& lam_io) {
    FerrersCtx<T, false> FB{};
    if (POT == POT_BARRED) FB = make_ferrers_ctx<T, false>(P, tab, P.comp[P.i_fer]);
    total_force<T, PHI, POT, false>(P, tab, FB, x, y, z, cs, sn, ax, ay, az, phi, lam_io);
}

}  // namespace smx
