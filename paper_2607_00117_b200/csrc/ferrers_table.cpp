// ferrers_table.cpp -- see ferrers_table.h.  Plain host C++ (long double), no CUDA.
#include "ferrers_table.h"

#include <cmath>
#include <cstdint>
#include <cstring>

namespace smx {
namespace {

typedef long double LD;
const int FIJK[FT_NFUNC][3] = {{2, 1, 0}, {2, 0, 1}, {0, 2, 1}, {1, 1, 1}, {0, 0, 0}};
constexpr int NCHEB = 24;

inline int key_of(double C, int ls) {
    uint64_t bits;
    std::memcpy(&bits, &C, 8);
    return (int)((uint32_t)(bits >> 32) >> (20 - ls));
}

LD ipow(LD x, int n) { LD r = 1; for (int i = 0; i < n; ++i) r *= x; return r; }

// coefficients g_m / (n+1/2+m) of the far-field series in S = 1/A
void far_series(LD p, LD q, int i, int j, int k, int nterm, LD* out) {
    int n = i + j + k;
    LD aj = j + 0.5L, ak = k + 0.5L;
    std::vector<LD> cj(nterm), ck(nterm);
    cj[0] = ck[0] = 1;
    for (int l = 1; l < nterm; ++l) {
        cj[l] = cj[l - 1] * (aj + l - 1) / l * p;   // (1-ps)^(-aj)
        ck[l] = ck[l - 1] * (ak + l - 1) / l * q;   // (1-qs)^(-ak)
    }
    for (int m = 0; m < nterm; ++m) {
        LD g = 0;
        for (int l = 0; l <= m; ++l) g += cj[l] * ck[m - l];
        out[m] = g / (n + 0.5L + m);
    }
}

}  // namespace

bool build_ferrers_table(double a, double b, double c, int ls, FerrersTable* t) {
    if (!(a > b && b > c && c > 0) || ls < 2 || ls > 7) return false;
    t->a2 = a * a; t->b2 = b * b; t->c2 = c * c; t->ls = ls;
    const LD q = (LD)t->a2 - (LD)t->c2, r = (LD)t->b2 - (LD)t->c2, p = (LD)t->a2 - (LD)t->b2;
    t->key0 = key_of(t->c2, ls);
    const int key1 = (FT_E1 + 1023) << ls;
    t->n_int = key1 - t->key0;
    if (t->n_int < 1) return false;
    t->coef.assign((size_t)t->n_int * FT_NFUNC * FT_NCOEF, 0.0);
    t->coef32.assign((size_t)t->n_int * FT_NANCHOR * FT_NCOEF32, 0.0f);
    t->fit_err = 0;

    // Chebyshev T_n -> monomial coefficients
    static LD tc[NCHEB + 1][NCHEB + 1];
    for (int n = 0; n <= NCHEB; ++n) for (int k = 0; k <= NCHEB; ++k) tc[n][k] = 0;
    tc[0][0] = 1; tc[1][1] = 1;
    for (int n = 2; n <= NCHEB; ++n)
        for (int k = 0; k <= n; ++k) tc[n][k] = (k ? 2 * tc[n - 1][k - 1] : 0) - tc[n - 2][k];
    LD node[NCHEB], cosmn[NCHEB][NCHEB];
    const LD PI = acosl(-1.0L);
    for (int m = 0; m < NCHEB; ++m) {
        node[m] = cosl(PI * (m + 0.5L) / NCHEB);
        for (int n = 0; n < NCHEB; ++n) cosmn[n][m] = cosl(PI * n * (m + 0.5L) / NCHEB);
    }

    for (int f = 0; f < FT_NFUNC; ++f) {
        const int i = FIJK[f][0], j = FIJK[f][1], k = FIJK[f][2], n = i + j + k;
        LD fs[40];
        far_series(p, q, i, j, k, 40, fs);
        for (int m = 0; m < FT_NFAR; ++m) t->far[f][m] = (double)fs[m];
        // value at the right end of the table, C = 2^FT_E1
        LD Cend = ldexpl(1.0L, FT_E1), S = 1 / (Cend + q), WR = 0;
        for (int m = 39; m >= 0; --m) WR = WR * S + fs[m];
        WR *= ipow(S, n) * sqrtl(S);
        for (int jj = t->n_int - 1; jj >= 0; --jj) {
            const int key = t->key0 + jj, eb = key >> ls, sub = key & ((1 << ls) - 1);
            const LD L = ldexpl(1.0L + (LD)sub / (1 << ls), eb - 1023), w = ldexpl(1.0L, eb - 1023 - ls);
            const LD mid = L + w / 2, hw = w / 2;
            LD h[NCHEB], an[NCHEB + 2], bn[NCHEB + 1], wn[NCHEB + 1];
            for (int m = 0; m < NCHEB; ++m) {
                LD C = mid + hw * node[m], A = C + q, B = C + r;
                h[m] = 1 / (sqrtl(A * B * C) * ipow(A, i) * ipow(B, j) * ipow(C, k));
            }
            for (int nn = 0; nn < NCHEB; ++nn) {
                LD s = 0;
                for (int m = 0; m < NCHEB; ++m) s += h[m] * cosmn[nn][m];
                an[nn] = 2 * s / NCHEB;
            }
            an[NCHEB] = an[NCHEB + 1] = 0;
            LD sumb = 0;
            for (int nn = 1; nn <= NCHEB; ++nn) { bn[nn] = (an[nn - 1] - an[nn + 1]) / (2 * nn); sumb += bn[nn]; }
            wn[0] = WR + hw * sumb;
            for (int nn = 1; nn <= NCHEB; ++nn) wn[nn] = -hw * bn[nn];
            // truncate, estimate, convert to monomials
            LD tail = 0;
            for (int nn = FT_NCOEF; nn <= NCHEB; ++nn) tail += fabsl(wn[nn]);
            double rel = (double)(tail / WR);
            if (rel > t->fit_err) t->fit_err = rel;
            for (int kk = 0; kk < FT_NCOEF; ++kk) {
                LD cmon = 0;
                for (int nn = kk; nn < FT_NCOEF; ++nn) cmon += wn[nn] * tc[nn][kk];
                t->coef[((size_t)jj * FT_NFUNC + f) * FT_NCOEF + kk] = (double)cmon;
            }
            if (f < FT_NANCHOR)
                for (int kk = 0; kk < FT_NCOEF32; ++kk) {
                    LD cmon = 0;
                    for (int nn = kk; nn < FT_NCOEF32; ++nn) cmon += wn[nn] * tc[nn][kk];
                    t->coef32[((size_t)jj * FT_NANCHOR + f) * FT_NCOEF32 + kk] = (float)cmon;
                }
            LD WL = 0;
            for (int nn = NCHEB; nn >= 0; --nn) WL += (nn & 1) ? -wn[nn] : wn[nn];
            WR = WL;
        }
    }
    return true;
}

void eval_ferrers_table_host(const FerrersTable& t, double lambda, double* out) {
    const double C = t.c2 + lambda;
    const int key = key_of(C, t.ls);
    const int j = key - t.key0;
    static const int NF[FT_NFUNC] = {3, 3, 3, 3, 0};
    if (j >= t.n_int) {
        const double S = 1.0 / (t.a2 + lambda), rS = std::sqrt(S);
        for (int f = 0; f < FT_NFUNC; ++f) {
            double s = 0;
            for (int m = FT_NFAR - 1; m >= 0; --m) s = s * S + t.far[f][m];
            double pre = rS;
            for (int e = 0; e < NF[f]; ++e) pre *= S;
            out[f] = s * pre;
        }
        return;
    }
    const int eb = key >> t.ls, sub = key & ((1 << t.ls) - 1);
    const double L = std::ldexp(1.0 + (double)sub / (1 << t.ls), eb - 1023);
    const double tau = (C - L) * std::ldexp(1.0, 1 + t.ls - (eb - 1023)) - 1.0;
    for (int f = 0; f < FT_NFUNC; ++f) {
        const double* c = &t.coef[((size_t)(j < 0 ? 0 : j) * FT_NFUNC + f) * FT_NCOEF];
        double s = c[FT_NCOEF - 1];
        for (int k = FT_NCOEF - 2; k >= 0; --k) s = s * tau + c[k];
        out[f] = s;
    }
}

}  // namespace smx
