// force.cuh -- analytic force field of the trial potential, FMA-dense, templated on the arithmetic
// type T (double / float).  __host__ __device__ so that the same code can be exercised on the host
// by sm_debug_host_force (CPU-side tests); the product path runs it in the CUDA kernels only.
//
// Components (include/schwarmax.h): Plummer; Miyamoto-Nagai (Eq.10); NFW
// (Eq.8); Ferrers n=2 bar (BASELINE.json configs[1]).
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>

#include "ferrers_table.h"

#ifdef __CUDACC__
#define SMX_HD __host__ __device__ __forceinline__
#else
#define SMX_HD inline
#endif

namespace smx {

constexpr int MAX_COMP = 8;
enum { K_PLUMMER = 1, K_MN = 2, K_NFW = 3, K_FERRERS = 4 };
// potential classes with a specialised kernel: exactly {static MN, static NFW, rotating Ferrers} / one static Plummer
// POT_NEEDLE: the paper's stellar model {static MN, static NFW, rotating sloped T_3 needle bar, rotating uniform V_4 needle bar}
enum { POT_GENERIC = 0, POT_BARRED = 1, POT_PLUMMER = 2, POT_NEEDLE = 3 };

// Per-trial device-side description, built on the host in fp64.
struct CompDev {
    int kind, rotating;
    double c[6];  // Plummer {GM,b^2}  MN {GM,a,b^2}  NFW {G*M_DM, 1/r_s, r_s}  Ferrers {K=105GM/16, a^2, b^2, c^2, p=a^2-b^2, q=a^2-c^2}
                  // Dehnen-Aly T_3 / V_4 {GM, a, b^2, L, (1+eta)/(2L), eta/L^2}
};
struct PotDev {
    double omega_p, phase0;
    int n_comp, has_rot, has_ferrers;
    int pot_class, i_mn, i_nfw, i_fer;  // POT_BARRED: indices of the three components; POT_NEEDLE: i_fer = the T_3 bar
    int i_v4;                           // POT_NEEDLE: the V_4 bar
    int ft_key0, ft_nint;          // Ferrers table geometry of the fp64-path table (keys with FT_LS64)
    int ft32_key0, ft32_nint;      // and of the fp32-path table (keys with FT_LS32)
    long long ft_off64, ft_off32;  // offsets of this trial's table in the fp64 / fp32 coefficient buffers (elements)
    long long ft_off0;             // offset of this trial's W000 table (elements)
    CompDev comp[MAX_COMP];
    double far[FT_NFUNC][FT_NFAR];
};

// The same, converted to the kernel's arithmetic type and resident in shared memory.
template <typename T>
struct CompS { int kind, rotating; T c[6]; };
template <typename T>
struct PotS {
    int n_comp, has_rot, has_ferrers;
    int pot_class, i_mn, i_nfw, i_fer, i_v4;
    int ft_key0, ft_nint;   // geometry of the table of type T
    CompS<T> comp[MAX_COMP];
    T far[FT_NFUNC][FT_NFAR];
    const T* tab;   // Ferrers anchor coefficients [interval][ROW] = 4 x NCOEF (+ padding) (shared memory in the hot kernels)
    const T* tab0;  // W000 coefficients [interval][NCOEF] (global; potential only, fp64 only)
};

template <typename T> struct FT;
// LS = log2(sub-intervals per octave); ROW = pitch of one interval's anchor block in elements of T.  Lanes of a warp
// sit in different intervals, so the pitch decides the shared-memory bank pattern of the 16-byte row loads: 52 words
// (fp64 path, 208 B) and 20 words (fp32 path) are both = 20 mod 32, which spreads consecutive intervals over all eight
// 4-bank groups (a 320-byte pitch, = 16 mod 32, put every lane on one of two groups: 16-way conflicts, profiles/r1a).
template <> struct FT<double> { static constexpr int LS = FT_LS64; static constexpr int ROW = FT_ROW64; };
template <> struct FT<float> { static constexpr int LS = FT_LS32; static constexpr int ROW = FT_ROW32; };

// ---------------------------------------------------------------- small helpers
// 1/sqrt(x) and 1/x for positive normal x: hardware seed (MUFU.RSQ64H / MUFU.RCP64H, ~2^-20) plus one
// third-order correction (truncation ~2^-60), branch-free -- the library routines carry a slow-path call.
SMX_HD double rsqrt_t(double x) {
#ifdef __CUDA_ARCH__
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double t = x * y;
    double e = fma(-t, y, 1.0);
    double q = e * fma(0.375, e, 0.5);
    return fma(y, q, y);
#else
    return 1.0 / std::sqrt(x);
#endif
}
SMX_HD double rcp_t(double x) {
#ifdef __CUDA_ARCH__
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    double q = fma(e, e, e);
    y = fma(y, q, y);
    e = fma(-x, y, 1.0);  // one more linear step: the seed is only ~20 bits, e^3 alone leaves ~2^-60
    return fma(y, e, y);
#else
    return 1.0 / x;
#endif
}
SMX_HD float rsqrt_t(float x) {
#ifdef __CUDA_ARCH__
    return rsqrtf(x);
#else
    return 1.0f / std::sqrt(x);
#endif
}
SMX_HD float rcp_t(float x) {
#ifdef __CUDA_ARCH__
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
#else
    return 1.0f / x;
#endif
}
SMX_HD float frcp(float x) { return rcp_t(x); }

// NFW kernel g(X) = ln(1+X) - X/(1+X), X = r/r_s >= 0, branch-free and FMA-only after two reciprocals (the library
// log carries special-case branches that split the step into basic blocks), and ln(1+X) itself for the potential.
//   w = 1+X = 2^e m, m in (sqrt(1/2), sqrt(2)];  s = (m-1)/(m+1);  ln m = 2 atanh(s) = 2s + 2 s^3 P(s^2),
//   P(z) = sum_n z^n/(2n+3) (|s| <= 0.1716: truncated after z^8, the first omitted term is 2.3e-17 of ln m).
//   e = 0 (X < 0.414):  s = X/(2+X) formed from X itself, and 2s - X/(1+X) = s X/(1+X) EXACTLY, so
//                       g = s X/w + 2 s^3 P: all terms positive, full relative accuracy down to X -> 0 (g ~ X^2/2);
//   e >= 1:             g = e ln2 + 2 s^3 P + (2s - X/w), a cancellation of at most ~6x.
// ln2 is split so that e ln2_hi is exact (ln2_hi has 29 significant bits).
#ifdef __CUDACC__
// the fp64 series coefficients live in constant memory: DFMA reads a constant-bank operand directly, whereas a
// 64-bit immediate costs two UMOV issue slots each time it is (re)materialised
__constant__ double c_logp[11] = {1.0 / 3, 1.0 / 5, 1.0 / 7, 1.0 / 9, 1.0 / 11, 1.0 / 13, 1.0 / 15, 1.0 / 17, 1.0 / 19,
                                  0.6931471787393093, 1.8206359985041462e-09};
#endif
template <typename T> struct LogC;
template <> struct LogC<double> {
    static constexpr int NP = 9;
    SMX_HD static double p(int i) {
#ifdef __CUDA_ARCH__
        return c_logp[i];
#else
        constexpr double c[NP] = {1.0 / 3, 1.0 / 5, 1.0 / 7, 1.0 / 9, 1.0 / 11, 1.0 / 13, 1.0 / 15, 1.0 / 17, 1.0 / 19};
        return c[i];
#endif
    }
#ifdef __CUDA_ARCH__
    SMX_HD static double ln2_hi() { return c_logp[9]; }
    SMX_HD static double ln2_lo() { return c_logp[10]; }
#else
    SMX_HD static double ln2_hi() { return 0.6931471787393093; }
    SMX_HD static double ln2_lo() { return 1.8206359985041462e-09; }
#endif
};
template <> struct LogC<float> {
    static constexpr int NP = 4;
    SMX_HD static float p(int i) {
        constexpr float c[NP] = {1.0f / 3, 1.0f / 5, 1.0f / 7, 1.0f / 9};
        return c[i];
    }
    SMX_HD static float ln2_hi() { return 0.693145751953125f; }
    SMX_HD static float ln2_lo() { return 1.42860682e-06f; }
};
// exponent e and mantissa m of w = 2^e m with m in (sqrt(1/2), sqrt(2)]
SMX_HD void split_sqrt2(double w, int& e, double& m) {
#ifdef __CUDA_ARCH__
    int hi = __double2hiint(w), lo = __double2loint(w);
#else
    uint64_t bits; std::memcpy(&bits, &w, 8); int hi = (int)(bits >> 32), lo = (int)(uint32_t)bits;
#endif
    e = (hi >> 20) - 1023;
    int mh = (hi & 0x000FFFFF) | 0x3FF00000;             // m in [1,2)
    const int big = mh > 0x3FF6A09E;                      // m > sqrt(2) (high-word compare is enough)
    mh -= big << 20; e += big;                            // m/2, e+1
#ifdef __CUDA_ARCH__
    m = __hiloint2double(mh, lo);
#else
    uint64_t mb = ((uint64_t)(uint32_t)mh << 32) | (uint32_t)lo; std::memcpy(&m, &mb, 8);
#endif
}
SMX_HD void split_sqrt2(float w, int& e, float& m) {
#ifdef __CUDA_ARCH__
    int bits = __float_as_int(w);
#else
    int bits; std::memcpy(&bits, &w, 4);
#endif
    e = (bits >> 23) - 127;
    int mb = (bits & 0x007FFFFF) | 0x3F800000;
    const int big = mb > 0x3FB504F3;
    mb -= big << 23; e += big;
#ifdef __CUDA_ARCH__
    m = __int_as_float(mb);
#else
    std::memcpy(&m, &mb, 4);
#endif
}
// -> g(X); *L = ln(1+X) when WANT_L
template <typename T, bool WANT_L>
SMX_HD T nfw_g(T X, T* L) {
    const T w = (T)1 + X;
    const T rw = rcp_t(w);
    int e; T m;
    split_sqrt2(w, e, m);
    const bool small = e == 0;
    const T num = small ? X : m - (T)1, den = small ? (T)2 + X : m + (T)1;
    const T s = num * rcp_t(den);
    const T z = s * s;
    T P = LogC<T>::p(LogC<T>::NP - 1);
#pragma unroll
    for (int i = LogC<T>::NP - 2; i >= 0; --i) P = P * z + LogC<T>::p(i);
    const T tail = (T)2 * s * z * P;                       // 2 s^3 P(s^2)
    const T xw = X * rw;
    const T bracket = small ? s * xw : (T)2 * s - xw;      // 2s - X/(1+X)
    const T ef = (T)e;
    if (WANT_L) *L = ef * LogC<T>::ln2_hi() + (ef * LogC<T>::ln2_lo() + ((T)2 * s + tail));
    return ef * LogC<T>::ln2_hi() + (ef * LogC<T>::ln2_lo() + (tail + bracket));
}
template <typename T> SMX_HD T fma_t(T a, T b, T c) { return a * b + c; }  // contracted to FMA by nvcc

// interval key of C > 0 from its binary representation; *tau in [-1,1) within the interval
SMX_HD int ft_key(double C, double* tau) {
    constexpr int ls = FT_LS64;
#ifdef __CUDA_ARCH__
    int hi = __double2hiint(C);
#else
    uint64_t bits; std::memcpy(&bits, &C, 8); int hi = (int)(bits >> 32);
#endif
    int shift = 20 - ls;
    int key = hi >> shift;
    int eb = hi >> 20;
#ifdef __CUDA_ARCH__
    double L = __hiloint2double(key << shift, 0);
    double sc = __hiloint2double((2047 + ls - eb) << 20, 0);  // 2^(1+ls-(eb-1023))
#else
    uint64_t lb = (uint64_t)(uint32_t)(key << shift) << 32; double L; std::memcpy(&L, &lb, 8);
    uint64_t sb = (uint64_t)(uint32_t)((2047 + ls - eb) << 20) << 32; double sc; std::memcpy(&sc, &sb, 8);
#endif
    *tau = (C - L) * sc - 1.0;
    return key;
}
SMX_HD int ft_key(float C, float* tau) {
    constexpr int ls = FT_LS32;
#ifdef __CUDA_ARCH__
    int bits = __float_as_int(C);
#else
    int bits; std::memcpy(&bits, &C, 4);
#endif
    int shift = 23 - ls;
    int key = bits >> shift;
    int eb = bits >> 23;
    int lbits = key << shift, sbits = (255 + ls - eb) << 23;  // 2^(1+ls-(eb-127))
#ifdef __CUDA_ARCH__
    float L = __int_as_float(lbits), sc = __int_as_float(sbits);
#else
    float L, sc; std::memcpy(&L, &lbits, 4); std::memcpy(&sc, &sbits, 4);
#endif
    *tau = (C - L) * sc - 1.0f;
    return key + (896 << ls);  // same numbering as the fp64 keys
}

// ---------------------------------------------------------------- spherical / axisymmetric components
template <typename T, bool PHI>
SMX_HD void plummer(const CompS<T>& c, T x, T y, T z, T& fx, T& fy, T& fz, T& phi) {
    T s2 = fma_t(x, x, fma_t(y, y, fma_t(z, z, c.c[1])));
    T rs = rsqrt_t(s2);
    T g = c.c[0] * rs;
    T f = -g * rs * rs;
    fx += f * x; fy += f * y; fz += f * z;
    if (PHI) phi -= g;
}

template <typename T, bool PHI>
SMX_HD void miyamoto_nagai(const CompS<T>& c, T x, T y, T z, T& fx, T& fy, T& fz, T& phi) {
    T z2b = fma_t(z, z, c.c[2]);
    T rz = rsqrt_t(z2b);
    T D = fma_t(z2b, rz, c.c[1]);  // a + sqrt(z^2+b^2)
    T s2 = fma_t(x, x, fma_t(y, y, D * D));
    T rs = rsqrt_t(s2);
    T g = c.c[0] * rs;
    T f = -g * rs * rs;
    fx += f * x; fy += f * y; fz += f * z * (D * rz);
    if (PHI) phi -= g;
}

template <typename T, bool PHI>
SMX_HD void nfw(const CompS<T>& c, T x, T y, T z, T& fx, T& fy, T& fz, T& phi) {
    T r2 = fma_t(x, x, fma_t(y, y, z * z));
    T rs = r2 > (T)0 ? rsqrt_t(r2) : (T)0;
    T r = r2 * rs;
    T X = r * c.c[1];
    T L = (T)0;
    T g = nfw_g<T, PHI>(X, &L);
    T f = -c.c[0] * g * rs * rs * rs;   // -G M_DM g(X)/r^3; at r = 0: rs = 0 and the force vanishes
    fx += f * x; fy += f * y; fz += f * z;
    if (PHI) phi -= (r2 > (T)0) ? c.c[0] * L * rs : c.c[0] * c.c[1];
}

}  // namespace smx
