/* sm_oracle.h -- CPU ORACLE for orbit-library construction (TEST INFRASTRUCTURE ONLY).
 *
 * This header belongs to the oracle: a plain, slow, obviously-correct CPU restatement of
 * the hot path of arXiv 2607.00117 (SchwarMAX) as fixed by BASELINE.json `north_star`.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.  It shares NO code with the CUDA product (paper_2607_00117_b200/csrc,
 * include/schwarmax.h): the structs below are re-declared here on purpose.
 *
 * What the path computes (citations: PAPER.md = /root/reference/PAPER.md):
 *   - potentials: NFW halo PAPER.md:185-188 Eq.8; Miyamoto-Nagai disc PAPER.md:203-205 Eq.10;
 *     Plummer sphere and Ferrers n=2 bar per BASELINE.json configs[0], configs[1] (textbook
 *     forms, Binney & Tremaine 2008 sec. 2.5; see DESIGN.md "Readings" R3);
 *   - fixed-step kick-drift-kick leapfrog in the inertial frame with bar angle
 *     theta = Omega_p*t (BASELINE.json north_star item 2; the paper's own integrator,
 *     PAPER.md:75, is replaced by mandate);
 *   - recorded samples moved to the bar frame (velocities stay inertial),
 *     projected by R = Rz(gamma) Rx(beta) Rz(alpha) (Eq.1), image plane
 *     (X,Y) = (x',y'), v_los = v_z';
 *   - binned into an aperture x v_los histogram and a 3-D density grid
 *     (PAPER.md:104-108), one dense float row per orbit.
 *
 * All pointers are HOST pointers owned by the caller.  Return 0 on success, <0 on error.
 */
#ifndef SM_ORACLE_H
#define SM_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { SMO_PLUMMER = 1, SMO_MIYAMOTO_NAGAI = 2, SMO_NFW = 3, SMO_FERRERS2 = 4, SMO_DEHNEN_T3 = 5, SMO_DEHNEN_V4 = 6 };

/* p[]: Plummer{M,b}  MN{M,a,b}  NFW{rho_s,r_s}  Ferrers2{M,a,b,c} (a>b>c>0).
 * Dehnen & Aly (2023) needle bars T_3 / V_4 (Eq.12, Appendix A): {M,a,b,L,eta},
 * a >= 0, b > 0, L > 0, -1 <= eta <= 1; the needle lies along the component's x axis.
 * rotating != 0: the component is fixed in the bar frame (angle Omega_p*t + phase0). */
typedef struct { int kind; int rotating; double p[6]; } smo_component;
typedef struct { double G, omega_p, phase0; int n_comp; smo_component comp[8]; } smo_potential_desc;
typedef struct { double alpha, beta, gamma; } smo_projection; /* radians */
typedef struct {
    int nx, ny, nv; double x0, x1, y0, y1, v0, v1;     /* LOSVD block: index (iy*nx+ix)*nv+iv */
    int dx, dy, dz; double bx0, bx1, by0, by1, bz0, bz1; /* density:   index (iz*dy+iy)*dx+ix */
} smo_grids;

/* state_prec: 0 = orbit state (x,v) carried in double, 1 = in long double (sensitivity floor); forces evaluated in __float128 and
 * rounded to the state type.  2 = state AND forces in plain double: the same force expressions compiled for double, for TIMING a CPU
 * baseline that is not slowed down by software quad arithmetic (bench.py); parity tests never compare against it. */

/* Force F[n][3] (= -grad Phi, inertial components) and potential Phi[n] (may be NULL) at
 * inertial positions xyz[n][3] and time t. */
int smo_eval_force(const smo_potential_desc*, const double* xyz, int64_t n, double t,
                   double* F, double* Phi);

/* KDK leapfrog; traj[n_rec][n_orb][6] (inertial x,y,z,vx,vy,vz) after steps stride,2*stride,...
 * n_rec = n_steps/stride (integer division). */
int smo_integrate_trajectories(const smo_potential_desc*, const double* ics, int64_t n_orb,
                               double dt, int64_t n_steps, int32_t stride, int state_prec,
                               double* traj);

/* The paper's own integrator: adaptive Bogacki-Shampine RK3(2) in the bar's rotating frame, a fixed number
 * of step attempts (a rejected attempt leaves the state in place and has weight 0); rtol <= 0: fixed steps h0.  ics are inertial at t = 0.
 * samples[n_steps][n_orb][6] = position on bar axes and INERTIAL velocity on bar axes after each attempt; dt_w[n_steps][n_orb] = the
 * accepted step size (the paper's sample weight delta-t), 0 if rejected; t_end[n_orb] = total integrated time (may be NULL).
 * Step control: DESIGN.md reading R23. */
int smo_integrate_rk32(const smo_potential_desc*, const double* ics, int64_t n_orb, int64_t n_steps, double rtol,
                       double atol_x, double atol_v, double h0, double* samples, double* dt_w, double* t_end);

/* Full path.  losvd[n_proj][n_orb][nx*ny*nv], dens[n_orb][dx*dy*dz] raw counts as float;
 * nout[n_proj+1][n_orb] out-of-grid sample counts (last block = density grid), may be NULL;
 * diag[n_orb][2] = {max relative Jacobi-integral drift over recorded samples, 0/1 non-finite flag},
 * may be NULL;  near_edge[n_proj+1][n_orb] = number of recorded samples with a coordinate
 * within 1e-9 bin widths of a bin edge (north_star: such samples are excluded from the
 * identical-count comparison), may be NULL. */
int smo_build_library(const smo_potential_desc*, const double* ics, int64_t n_orb,
                      double dt, int64_t n_steps, int32_t stride,
                      const smo_projection* proj, int n_proj, const smo_grids*,
                      int state_prec, float* losvd, float* dens, int32_t* nout, double* diag,
                      int32_t* near_edge);

/* Symmetrised orbit bundles (n dithered realisations "treated as one orbit bundle"; Table 1:
 * three mirror copies of each orbit "co-added and treated as a single symmetrised orbit bundle").  Row r co-adds orbits
 * r*n_bundle .. (r+1)*n_bundle-1 (n_orb must be a multiple of n_bundle); fourfold != 0 bins every recorded bar-frame
 * sample four times with the sign flips of Table 1.  losvd[n_proj][n_orb/n_bundle][nx*ny*nv], dens[n_orb/n_bundle][..],
 * nout / near_edge [n_proj+1][n_orb/n_bundle]; row sum + nout = n_bundle * (fourfold ? 4 : 1) * n_rec. */
int smo_build_bundled_library(const smo_potential_desc*, const double* ics, int64_t n_orb, double dt, int64_t n_steps,
                              int32_t stride, const smo_projection* proj, int n_proj, const smo_grids*, int32_t n_bundle,
                              int fourfold, float* losvd, float* dens, int32_t* nout, int32_t* near_edge);

/* The same with aperture regrouping: ap_map[ny*nx] gives the aperture (0..n_ap-1, or < 0 for none) of every
 * image pixel; the LOSVD row holds n_ap*nv cells, index ap*nv+iv; samples on pixels without an aperture count in nout.
 * ap_map == NULL: plain pixels (then identical to smo_build_bundled_library).
 * density_mode 0: Cartesian bar-frame density cells; 1: the paper's cylindrical cells, the grid's b* ranges and
 * d* counts meaning (R, phi in [0,2pi), z), phi = atan2(y_b, x_b), index (jz*dy+jphi)*dx+jR. */
int smo_build_observable_library(const smo_potential_desc*, const double* ics, int64_t n_orb, double dt, int64_t n_steps,
                                 int32_t stride, const smo_projection* proj, int n_proj, const smo_grids*, int32_t n_bundle,
                                 int fourfold, const int32_t* ap_map, int32_t n_ap, int density_mode, float* losvd, float* dens,
                                 int32_t* nout, int32_t* near_edge);

/* Gauss-Hermite observable matrices on the fly (Eq.2; v0, s per aperture as in PAPER.md:175).  Per row,
 * projection and aperture n, over the recorded samples whose image pixel belongs to aperture n (all velocities):
 *   gh[n_proj][n_rows][n_ap][6] (double): [0] = number of samples (surface-density matrix),
 *   [1+m] = sum_k alpha(w_k) H_m(w_k), m = 0..4, w_k = (v_los,k - v0[n])/s[n], alpha(w) = exp(-w^2/2)/sqrt(2 pi),
 *   H_m = the modified Hermite polynomials of van der Marel & Franx (1993) / Gerhard (1993) (not printed in the paper).
 * dens / nout / near_edge / n_bundle / fourfold / density_mode as in smo_build_observable_library. */
int smo_build_gh_library(const smo_potential_desc*, const double* ics, int64_t n_orb, double dt, int64_t n_steps,
                         int32_t stride, const smo_projection* proj, int n_proj, const smo_grids*, int32_t n_bundle,
                         int fourfold, const int32_t* ap_map, int32_t n_ap, const double* v0, const double* s, int density_mode,
                         double* gh, float* dens, int32_t* nout, int32_t* near_edge);
/* alpha(w) H_m(w), m = 0..4, for n values of w: out5[n][5]. */
int smo_gh_terms(const double* w, int64_t n, double* out5);

/* Test hooks for pinning the Ferrers pieces: lambda(x) and the 20 integrals
 * W_ijk(lambda) = int_lambda^inf du / (Delta(u) (a^2+u)^i (b^2+u)^j (c^2+u)^k), i+j+k<=3, in the
 * order 000 100 010 001 200 020 002 110 101 011 300 030 003 210 201 120 021 102 012 111. */
int smo_ferrers_lambda(double a, double b, double c, const double* xyz, int64_t n, double* lam);
int smo_ferrers_W(double a, double b, double c, double lam, double* W20);
/* Projection of one (x_b, v_b) pair: out = {X, Y, v_los}. */
int smo_project(const smo_projection*, const double* xb, const double* vb, double* out3);
/* Jacobi integral E_J = v^2/2 + Phi(x,t) - Omega_p (x vy - y vx) for inertial state[n][6]. */
int smo_jacobi(const smo_potential_desc*, const double* state, int64_t n, double t, double* EJ);
int smo_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
