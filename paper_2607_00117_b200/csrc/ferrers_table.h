// ferrers_table.h -- host-side construction of the per-potential Ferrers (n=2) tables.
//
// The bar force needs 19 integrals W_ijk(lambda) = int_lambda^inf du /(Delta A^i B^j C^k)
// (A=a^2+u, B=b^2+u, C=c^2+u, Delta=sqrt(ABC)); for ONE potential they are functions of the
// single scalar lambda.  Four "anchor" functions of level i+j+k=3 are tabulated as piecewise
// polynomials in C = c^2+lambda on intervals cut from the binary representation of C
// (2^LS equal sub-intervals per octave); the other 15 follow from positive-term recurrences
// (see DESIGN.md "Ferrers force").  A fifth function, W000, is tabulated for the potential.
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
constexpr int FT_NCOEF = 10;   // monomial coefficients per function per interval (fp64 path)
constexpr int FT_NCOEF32 = 5;  // fp32 path
constexpr int FT_NFAR = 12;    // far-field series terms
constexpr int FT_LS = 4;     // log2(sub-intervals per octave) of every table the library builds
constexpr int FT_E1 = 11;      // table covers C < 2^FT_E1; beyond it the far-field series is used

struct FerrersTable {
    double a2, b2, c2;
    int ls;        // log2(sub-intervals per octave)
    int key0;      // (hi32(C) >> (20-ls)) of the first interval
    int n_int;     // number of intervals
    double fit_err;  // max over intervals/functions of the relative truncation estimate
    // coef[(j*FT_NFUNC + f)*FT_NCOEF + k]: W_f(C) = sum_k coef_k tau^k, tau in [-1,1] on interval j
    std::vector<double> coef;
    // coef32[(j*FT_NANCHOR + f)*FT_NCOEF32 + k], same for the fp32 path (anchors only)
    std::vector<float> coef32;
    // far[f][m]: W_f = S^(n_f+1/2) * sum_m far[f][m] S^m, S = 1/(a^2+lambda), n_f = 3,3,3,3,0
    double far[FT_NFUNC][FT_NFAR];
};

// Builds the table for semi-axes a>b>c>0.  Returns false on invalid axes.
bool build_ferrers_table(double a, double b, double c, int ls, FerrersTable* out);

// Host mirror of the device evaluation (same interval logic), for CPU-side tests:
// out5 = {W210, W201, W021, W111, W000} at lambda >= 0.
void eval_ferrers_table_host(const FerrersTable& t, double lambda, double* out5);

}  // namespace smx
