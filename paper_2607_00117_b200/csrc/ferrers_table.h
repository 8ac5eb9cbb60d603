// ferrers_table.h -- host-side construction of the per-potential Ferrers (n=2) tables.
//
// The bar force needs 19 integrals W_ijk(lambda) = int_lambda^inf du /(Delta A^i B^j C^k)
// (A=a^2+u, B=b^2+u, C=c^2+u, Delta=sqrt(ABC)); for ONE potential they are functions of the
// single scalar lambda.  Four "anchor" functions of level i+j+k=3 are tabulated as piecewise
// polynomials in C = c^2+lambda on intervals cut from the binary representation of C
// (2^LS equal sub-intervals per octave); the other 15 follow from positive-term recurrences
// (see DESIGN.md "Ferrers force").  A fifth function, W000, is tabulated for the potential.
//
// Two tables are built per potential:
//   fp64 path  2^6 sub-intervals per octave, degree 7.  A row is what one lane reads per force evaluation, and the
//              shared-memory bandwidth of those reads bounds the kernel when the GPU is full, so the row is made as
//              small as the accuracy allows: the monomial coefficients k = 0..4 are doubles, k = 5..7 are floats
//              (|c_k/c_0| < 1.1e-9 for k >= 5 on these intervals, so their fp32 rounding is < 7e-17 of W) and the
//              tail c5 + c6 tau + c7 tau^2 is evaluated in fp32: 208 bytes per row instead of 320.
//   fp32 path  2^4 sub-intervals per octave, degree 4, floats: 80 bytes per row.
//
// Construction (independent of the CPU oracle, which uses Carlson duplication in __float128):
// dW/dlambda = -1/(Delta A^i B^j C^k) is elementary, so on every interval the Chebyshev series of
// the integrand is integrated term by term, and the constants of integration are accumulated from
// the far end inward, starting from the convergent far-field series in S = 1/A.  long double.
#pragma once
#include <vector>

namespace smx {

constexpr int FT_NFUNC = 5;    // W210, W201, W021, W111, W000
constexpr int FT_NANCHOR = 4;  // the first four feed the force
constexpr int FT_LS64 = 6;     // fp64 path: log2(sub-intervals per octave)
constexpr int FT_ND = 5;       // fp64 path: coefficients k = 0..4 stored as doubles
constexpr int FT_NF = 3;       // fp64 path: coefficients k = 5..7 stored as floats
constexpr int FT_ROW64 = (FT_NANCHOR * FT_ND * 8 + FT_NANCHOR * FT_NF * 4) / 8;  // row pitch in doubles (26 = 208 B)
constexpr int FT_NC0 = FT_ND + FT_NF;  // W000: all eight coefficients as doubles (global memory, potential only)
constexpr int FT_LS32 = 4;     // fp32 path
constexpr int FT_NCOEF32 = 5;
constexpr int FT_ROW32 = FT_NANCHOR * FT_NCOEF32;  // 20 floats = 80 B
constexpr int FT_NFAR = 12;    // far-field series terms
constexpr int FT_E1 = 10;      // tables cover C < 2^FT_E1 (lambda < ~1000, r < ~32 kpc); beyond it the far-field series

struct FerrersTable {
    double a2, b2, c2;
    int key0_64, n_int64;  // first interval key (hi32(C) >> (20-LS64)) and interval count of the fp64-path table
    int key0_32, n_int32;  // the same for the fp32-path table (fp64 key numbering with LS32)
    double fit_err;        // max over intervals/functions of the relative truncation estimate (fp64 path)
    // rows64[j*FT_ROW64 ...]: doubles [f][k<5] (20), then floats [f][k-5<3] (12, stored in 6 double slots);
    // W_f(C) = sum_k c_k tau^k, tau in [-1,1) on interval j
    std::vector<double> rows64;
    std::vector<double> coef0;   // W000: [j][FT_NC0]
    std::vector<float> rows32;   // [j][f][k<5]
    // far[f][m]: W_f = S^(n_f+1/2) * sum_m far[f][m] S^m, S = 1/(a^2+lambda), n_f = 3,3,3,3,0
    double far[FT_NFUNC][FT_NFAR];
};

// Builds the tables for semi-axes a>b>c>0.  Returns false on invalid axes.
bool build_ferrers_table(double a, double b, double c, FerrersTable* out);

}  // namespace smx
