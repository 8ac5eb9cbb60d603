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

// One pass over all intervals of one table geometry (2^ls sub-intervals per octave): for every function f and interval
// jj (from the far end inward) hands the monomial coefficients c[0..ncoef) of W_f on that interval to sink(f, jj, c),
// and returns the largest relative truncation estimate.
template <class Sink>
double build_level(const FerrersTable& t, int ls, int key0, int n_int, int ncoef, int n_func, Sink sink) {
    const LD q = (LD)t.a2 - (LD)t.c2, r = (LD)t.b2 - (LD)t.c2, p = (LD)t.a2 - (LD)t.b2;
    // Chebyshev T_n -> monomial coefficients
    // (a function-local table filled once by a thread-safe static initialiser: it used to be a plain static array zeroed and
    // refilled by every call, so two host threads making potentials at the same time corrupted each other's coefficients)
    struct ChebToMono {
        LD c[NCHEB + 1][NCHEB + 1];
        ChebToMono() {
            for (int n = 0; n <= NCHEB; ++n) for (int k = 0; k <= NCHEB; ++k) c[n][k] = 0;
            c[0][0] = 1; c[1][1] = 1;
            for (int n = 2; n <= NCHEB; ++n)
                for (int k = 0; k <= n; ++k) c[n][k] = (k ? 2 * c[n - 1][k - 1] : 0) - c[n - 2][k];
        }
    };
    static const ChebToMono cheb;
    const LD (*tc)[NCHEB + 1] = cheb.c;
    LD node[NCHEB], cosmn[NCHEB][NCHEB];
    const LD PI = acosl(-1.0L);
    for (int m = 0; m < NCHEB; ++m) {
        node[m] = cosl(PI * (m + 0.5L) / NCHEB);
        for (int n = 0; n < NCHEB; ++n) cosmn[n][m] = cosl(PI * n * (m + 0.5L) / NCHEB);
    }
    double fit_err = 0;
    for (int f = 0; f < n_func; ++f) {
        const int i = FIJK[f][0], j = FIJK[f][1], k = FIJK[f][2], n = i + j + k;
        LD fs[40];
        far_series(p, q, i, j, k, 40, fs);
        // value at the right end of the table, C = 2^FT_E1
        LD Cend = ldexpl(1.0L, FT_E1), S = 1 / (Cend + q), WR = 0;
        for (int m = 39; m >= 0; --m) WR = WR * S + fs[m];
        WR *= ipow(S, n) * sqrtl(S);
        for (int jj = n_int - 1; jj >= 0; --jj) {
            const int key = key0 + jj, eb = key >> ls, sub = key & ((1 << ls) - 1);
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
            for (int nn = ncoef; nn <= NCHEB; ++nn) tail += fabsl(wn[nn]);
            double rel = (double)(tail / WR);
            if (rel > fit_err) fit_err = rel;
            LD cm[NCHEB + 1];
            for (int kk = 0; kk < ncoef; ++kk) {
                LD cmon = 0;
                for (int nn = kk; nn < ncoef; ++nn) cmon += wn[nn] * tc[nn][kk];
                cm[kk] = cmon;
            }
            sink(f, jj, cm);
            LD WL = 0;
            for (int nn = NCHEB; nn >= 0; --nn) WL += (nn & 1) ? -wn[nn] : wn[nn];
            WR = WL;
        }
    }
    return fit_err;
}

}  // namespace

bool build_ferrers_table(double a, double b, double c, FerrersTable* t) {
    if (!(a > b && b > c && c > 0)) return false;
    t->a2 = a * a; t->b2 = b * b; t->c2 = c * c;
    const LD q = (LD)t->a2 - (LD)t->c2, p = (LD)t->a2 - (LD)t->b2;
    t->key0_64 = key_of(t->c2, FT_LS64);
    t->n_int64 = ((FT_E1 + 1023) << FT_LS64) - t->key0_64;
    t->key0_32 = key_of(t->c2, FT_LS32);
    t->n_int32 = ((FT_E1 + 1023) << FT_LS32) - t->key0_32;
    if (t->n_int64 < 1 || t->n_int32 < 1) return false;
    for (int f = 0; f < FT_NFUNC; ++f) {
        LD fs[FT_NFAR];
        far_series(p, q, FIJK[f][0], FIJK[f][1], FIJK[f][2], FT_NFAR, fs);
        for (int m = 0; m < FT_NFAR; ++m) t->far[f][m] = (double)fs[m];
    }
    t->rows64.assign((size_t)t->n_int64 * FT_ROW64, 0.0);
    t->coef0.assign((size_t)t->n_int64 * FT_NC0, 0.0);
    t->rows32.assign((size_t)t->n_int32 * FT_ROW32, 0.0f);
    t->fit_err = build_level(*t, FT_LS64, t->key0_64, t->n_int64, FT_ND + FT_NF, FT_NFUNC, [&](int f, int jj, const LD* cm) {
        if (f == FT_NANCHOR) {
            for (int k = 0; k < FT_NC0; ++k) t->coef0[(size_t)jj * FT_NC0 + k] = (double)cm[k];
            return;
        }
        double* row = &t->rows64[(size_t)jj * FT_ROW64];
        float* tail = reinterpret_cast<float*>(row + FT_NANCHOR * FT_ND);
        for (int k = 0; k < FT_ND; ++k) row[f * FT_ND + k] = (double)cm[k];
        for (int k = 0; k < FT_NF; ++k) tail[f * FT_NF + k] = (float)cm[FT_ND + k];
    });
    build_level(*t, FT_LS32, t->key0_32, t->n_int32, FT_NCOEF32, FT_NANCHOR, [&](int f, int jj, const LD* cm) {
        for (int k = 0; k < FT_NCOEF32; ++k) t->rows32[(size_t)jj * FT_ROW32 + f * FT_NCOEF32 + k] = (float)cm[k];
    });
    return true;
}

}  // namespace smx
