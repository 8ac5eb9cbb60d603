// sm_oracle.cpp -- CPU ORACLE (TEST INFRASTRUCTURE ONLY; see sm_oracle.h).
//
// Plain and slow on purpose.  No blocking, no fusion, no tables: every force is the analytic
// expression (sm_oracle_forces.inc) evaluated in __float128 and rounded once (a second, plain-double compilation of the same
// expressions exists only to time a CPU baseline: state_prec = 2); the integrator, projection and binning
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

// The forces are written once (sm_oracle_forces.inc) and compiled for two arithmetic types.
namespace fq {   // the parity oracle: __float128
typedef __float128 Q;
#define Q_LIT(x) x##Q
#define Q_NEWTON_TOL 1e-32Q
#define Q_PI M_PIq
#define Q_SQRT sqrtq
#define Q_FABS fabsq
#define Q_FMAX fmaxq
#define Q_LOG1P log1pq
#define Q_POW powq
#define Q_ASINH asinhq
#define Q_COS cosq
#define Q_SIN sinq
#include "sm_oracle_forces.inc"
#undef Q_LIT
#undef Q_NEWTON_TOL
#undef Q_PI
#undef Q_SQRT
#undef Q_FABS
#undef Q_FMAX
#undef Q_LOG1P
#undef Q_POW
#undef Q_ASINH
#undef Q_COS
#undef Q_SIN
}  // namespace fq
namespace fd {   // plain double: timing only (state_prec = 2)
typedef double Q;
#define Q_LIT(x) x
#define Q_NEWTON_TOL 4e-16
#define Q_PI M_PI
#define Q_SQRT std::sqrt
#define Q_FABS std::fabs
#define Q_FMAX std::fmax
#define Q_LOG1P std::log1p
#define Q_POW std::pow
#define Q_ASINH std::asinh
#define Q_COS std::cos
#define Q_SIN std::sin
#include "sm_oracle_forces.inc"
#undef Q_LIT
#undef Q_NEWTON_TOL
#undef Q_PI
#undef Q_SQRT
#undef Q_FABS
#undef Q_FMAX
#undef Q_LOG1P
#undef Q_POW
#undef Q_ASINH
#undef Q_COS
#undef Q_SIN
}  // namespace fd

typedef fq::Q Q;
using fq::Q3;
using fq::carlson_rf; using fq::carlson_rd; using fq::ferrers_lambda; using fq::ferrers_W; using fq::ferrers_force; using fq::total_force;
using fq::component_force; using fq::dehnen_aly_force; using fq::needle_I;

namespace {

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

// DBL = false: forces in __float128 (the parity oracle).  DBL = true: the same force expressions in plain double (namespace fd) --
// state_prec = 2, used only to TIME a CPU baseline free of software quad arithmetic; no parity test compares against it.
template <class R, bool DBL = false>
struct Orbit {
    R x[3], v[3], a[3];
    const smo_potential_desc* d;
    void accel(double t) {
        if (DBL) {
            fd::Q3 F; fd::Q3 xd = { (double)x[0], (double)x[1], (double)x[2] };
            fd::total_force(d, xd, t, &F, nullptr);
            a[0] = (R)F.x; a[1] = (R)F.y; a[2] = (R)F.z;
            return;
        }
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

template <class R, bool DBL = false>
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
        Orbit<R, DBL> o; o.d = d; o.init(ics + 6 * i);
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

template <class R, bool DBL = false>
int integrate_t(const smo_potential_desc* d, const double* ics, int64_t n_orb, double dt,
                int64_t n_steps, int32_t stride, double* traj) {
#pragma omp parallel for schedule(dynamic)
    for (int64_t i = 0; i < n_orb; ++i) {
        Orbit<R, DBL> o; o.d = d; o.init(ics + 6 * i);
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
    if (state_prec == 2) return integrate_t<double, true>(d, ics, n_orb, dt, n_steps, stride, traj);
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
    if (state_prec == 2) return build_library_t<double, true>(d, ics, n_orb, dt, n_steps, stride, proj, n_proj, g, losvd, dens, nout, diag, near_edge);
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
