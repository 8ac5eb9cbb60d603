/* schwarmax.h -- C ABI of the B200-native orbit-library builder (libschwarmax.so).
 *
 * One hot path of arXiv 2607.00117 (SchwarMAX), as fixed by BASELINE.json `north_star`:
 * integrate N independent orbits in a disc + rotating bar + halo potential, move every recorded
 * sample to the bar frame, sky-project it and bin it into a per-orbit (aperture x v_los)
 * histogram and a 3-D density grid -- the orbit-observable matrix the weight solve consumes
 * (sections 2.2.2-2.2.4).  Everything below runs in hand-written CUDA kernels
 * for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *  - `d_*` pointers are DEVICE memory owned by the caller; everything else is HOST memory.
 *  - Calls enqueue work on `cuda_stream` (a cudaStream_t passed as void*, NULL = default stream)
 *    and return without synchronising, except where stated.  The caller synchronises the stream.
 *  - Outputs are fully overwritten; no pre-zeroing is required.
 *  - Every function returns an sm_status; nothing throws across the ABI.  sm_last_error() gives a
 *    thread-local message for the last failure.  Invalid arguments launch nothing.
 *  - Calls may be made from several host threads and on several devices of one process: the device is the calling thread's
 *    current CUDA device; debug flags and kernel timers are per thread; scratch memory comes from a stream-ordered pool the
 *    library owns on each device (the process's default pool is not touched); an sm_potential belongs to the device it was made on.
 *  - Units are whatever G is expressed in (configs: kpc, km/s, Msun; time unit kpc/(km/s)).
 */
#ifndef SCHWARMAX_H
#define SCHWARMAX_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef enum { SM_OK = 0, SM_ERR_INVALID_ARG = -1, SM_ERR_UNSUPPORTED = -2, SM_ERR_CUDA = -3, SM_ERR_NOMEM = -4 } sm_status;

/* Potential components.
 *  SM_PLUMMER         p = {M, b}            Phi = -GM/sqrt(r^2+b^2); b = 0 is a point mass (BASELINE.json configs[0])
 *  SM_MIYAMOTO_NAGAI  p = {M, a, b}         PAPER.md:203-205 Eq.10 (a,b = the paper's R_d, H_d)
 *  SM_NFW             p = {rho_s, r_s}      PAPER.md:185-188 Eq.8 with M_DM = 4 pi rho_s r_s^3
 *  SM_FERRERS2        p = {M, a, b, c}      Ferrers n=2 ellipsoid rho = rho_c (1-m^2)^2, a>b>c>0 (BASELINE.json configs[1])
 *  SM_DEHNEN_T3/_V4   p = {M, a, b, L, eta}   Dehnen & Aly (2023) needle bars, the paper's own bar: the parent pairs T_3 / V_4
 *                     of PAPER.md:485-497 Appendix A with every R^-n replaced by the needle integral I_n of PAPER.md:211-219
 *                     Eq.12 (half-length L > 0 along the component's x axis, slope -1 <= eta <= 1; a >= 0, b > 0).  The
 *                     needle integrals are evaluated in fp64 in both precisions (their closed forms are differences).
 * rotating != 0: the component is fixed in the bar frame, which is rotated about z by
 * theta(t) = omega_p*t + phase0 with respect to the inertial frame. */
typedef enum { SM_PLUMMER = 1, SM_MIYAMOTO_NAGAI = 2, SM_NFW = 3, SM_FERRERS2 = 4, SM_DEHNEN_T3 = 5, SM_DEHNEN_V4 = 6 } sm_kind;
typedef struct { int kind; int rotating; double p[6]; } sm_component;
typedef struct { double G, omega_p, phase0; int n_comp; sm_component comp[8]; } sm_potential_desc;

/* Arithmetic of the integrator and of the projection/binning decisions.
 *  SM_F64: fp64 state, force, projection and bin decision.
 *  SM_F32: fp32 state, force, projection and bin decision; the bar phase is formed in fp64.
 * Histogram cells are fp32 counts in both (exact: a cell never exceeds n_rec <= 2^24), so
 * BASELINE.json configs[4] ("fp64 integration and fp32 accumulation") is SM_F64. */
typedef enum { SM_F64 = 0, SM_F32 = 1 } sm_precision;

/* Sky projection, Eq.1: R = Rz(gamma) Rx(beta) Rz(alpha), active right-handed;
 * image plane (X,Y) = (x',y'), v_los = v_z'.  Radians. */
typedef struct { double alpha, beta, gamma; } sm_projection;

/* Histogram geometry.  LOSVD block (shared by all projections): nx*ny*nv cells over
 * [x0,x1) x [y0,y1) x [v0,v1), flat index (iy*nx+ix)*nv+iv.  Density grid in the bar frame:
 * dx*dy*dz cells over [bx0,bx1) x [by0,by1) x [bz0,bz1), flat index (iz*dy+iy)*dx+ix.
 * Bin of u on [lo,hi) with n bins: floor((u-lo)*(n/(hi-lo))); samples outside (or NaN) are
 * dropped and counted in d_nout. */
typedef struct {
    int nx, ny, nv; double x0, x1, y0, y1, v0, v1;
    int dx, dy, dz; double bx0, bx1, by0, by1, bz0, bz1;
} sm_grids;

typedef struct sm_potential sm_potential; /* opaque; owns device-side constant tables */

/* Build `n_trials` potentials (n_trials = 1 for a single model) from host descriptors desc[n_trials].
 * Precomputes the per-potential tables (Ferrers W_ijk(lambda) piecewise polynomials)
 * on the host in extended precision, uploads them, and SYNCHRONISES.  Fails with SM_ERR_INVALID_ARG
 * on bad kinds, non-positive scale lengths, Ferrers axes not a>b>c>0, more than one Ferrers
 * component per potential, or n_comp outside [1,8]. */
int sm_make_potential(const sm_potential_desc* desc, sm_potential** out);
int sm_make_potential_batch(const sm_potential_desc* desc, int n_trials, sm_potential** out);
void sm_free_potential(sm_potential*);

/* The hot path.
 *  d_ics    [n_orb][6]  x,y,z,vx,vy,vz, inertial frame, t = 0 (fp64 also for SM_F32)
 *  dt, n_steps, stride  kick-drift-kick leapfrog with t_k = k*dt; samples recorded after steps
 *                        stride, 2*stride, ...; n_rec = n_steps/stride (integer division)
 *  proj     [n_proj]    host; 1 <= n_proj <= 4
 *  d_losvd  [n_proj][n_orb][nx*ny*nv]  fp32 counts
 *  d_dens   [n_orb][dx*dy*dz]          fp32 counts
 *  d_nout   [n_proj+1][n_orb] int32 out-of-grid counts (last block: density grid); may be NULL
 *  d_diag   [n_orb][2] {max relative Jacobi-integral drift over recorded samples, non-finite flag};
 *           may be NULL (costs one potential evaluation per recorded sample when given; SM_F64 only)
 * Row sums satisfy sum(row) + nout = n_rec for every orbit and histogram.  Orbit sub-ranges are
 * expressed by offsetting d_ics and sizing the outputs for the sub-range.  The potential must
 * hold exactly one trial. */
int sm_build_library(const sm_potential*, const double* d_ics, int64_t n_orb, double dt, int64_t n_steps,
                     int32_t stride, const sm_projection* proj, int n_proj, const sm_grids*, int precision,
                     float* d_losvd, float* d_dens, int32_t* d_nout, double* d_diag, void* cuda_stream);

/* Batched-potential mode (north_star item 4): trials [trial0, trial0+n_trials)
 * of a batch potential in ONE integrator launch.
 *  d_ics    [n_trials][n_orb][6] if ics_per_trial != 0, else [n_orb][6] shared by all trials
 *  proj     [n_trials][n_proj] host
 *  d_losvd  [n_trials][n_proj][n_orb][nlos], d_dens [n_trials][n_orb][nden], d_nout [n_trials][n_proj+1][n_orb] */
int sm_build_library_batch(const sm_potential* batch, int trial0, int n_trials, const double* d_ics,
                           int ics_per_trial, int64_t n_orb, double dt, int64_t n_steps, int32_t stride,
                           const sm_projection* proj, int n_proj, const sm_grids*, int precision,
                           float* d_losvd, float* d_dens, int32_t* d_nout, void* cuda_stream);

/* Symmetrised orbit bundles: the same path with rows = bundles.
 *  n_bundle  consecutive orbits co-added into one row: PAPER.md:71, the n dithered realisations of an initial condition are
 *            "treated as one orbit bundle"; n_orb must be a multiple of n_bundle; the caller supplies the realisations.
 *  fourfold  != 0: every recorded bar-frame sample is binned four times with the sign flips of PAPER.md:77-90 Table 1,
 *            (x,y,z;vx,vy,vz) (x,y,-z;vx,vy,-vz) (-x,-y,z;-vx,-vy,vz) (-x,-y,-z;-vx,-vy,-vz): "three mirror copies ... co-added".
 * d_losvd [n_proj][n_orb/n_bundle][nx*ny*nv], d_dens [n_orb/n_bundle][dx*dy*dz], d_nout [n_proj+1][n_orb/n_bundle] (may be NULL);
 * row sum + nout = n_bundle * (fourfold ? 4 : 1) * n_rec, which must not exceed 2^24.  Single-trial potentials; batches: sm_build_observable_library_batch. */
int sm_build_bundled_library(const sm_potential*, const double* d_ics, int64_t n_orb, double dt, int64_t n_steps,
                             int32_t stride, const sm_projection* proj, int n_proj, const sm_grids*, int precision,
                             int32_t n_bundle, int fourfold, float* d_losvd, float* d_dens, int32_t* d_nout, void* cuda_stream);

/* The same with aperture regrouping on the fly ("collected first in regular bins and
 * then regrouped into Voronoi bins according to the pre-defined binning strategy"): d_ap_map[ny*nx] (DEVICE, int32, caller-owned)
 * gives the aperture 0..n_ap-1 of image pixel (ix,iy) at [iy*nx+ix], or < 0 when the pixel belongs to no aperture (such
 * samples count in d_nout, as do map entries >= n_ap).  The LOSVD row then has n_ap*nv cells, index ap*nv+iv:
 * d_losvd [n_proj][n_orb/n_bundle][n_ap*nv].  d_ap_map == NULL: plain pixels (= sm_build_bundled_library).
 * density_mode 0: Cartesian bar-frame density cells (sm_grids as documented above); 1: the paper's 3-D mass matrix on cells
 * uniform in (R, phi, z): dx, dy, dz then count the R, phi, z cells over [bx0,bx1) x [by0,by1) x [bz0,bz1) with
 * R = sqrt(x_b^2+y_b^2) and phi = atan2(y_b, x_b) taken in [0, 2 pi); flat index (jz*dy + jphi)*dx + jR. */
int sm_build_observable_library(const sm_potential*, const double* d_ics, int64_t n_orb, double dt, int64_t n_steps,
                                int32_t stride, const sm_projection* proj, int n_proj, const sm_grids*, int precision,
                                int32_t n_bundle, int fourfold, const int32_t* d_ap_map, int32_t n_ap, int density_mode,
                                float* d_losvd, float* d_dens, int32_t* d_nout, void* cuda_stream);

/* Gauss-Hermite observable matrices on the fly (Eq.2: "we compute h_m of every orbit i
 * in every 2D aperture n"): instead of the v_los histogram, per row, projection and aperture n the six sums over the recorded
 * samples whose image pixel belongs to aperture n (all velocities; the velocity axis of sm_grids is not used):
 *   d_gh [n_proj][n_orb/n_bundle][n_ap][6] fp32:  [0] = number of samples (surface-density matrix),
 *   [1+m] = sum_k alpha(w_k) H_m(w_k), m = 0..4,  w_k = (v_los,k - d_v0[n]) / d_s[n],  alpha(w) = exp(-w^2/2)/sqrt(2 pi),
 *   H_m = the modified Hermite polynomials of van der Marel & Franx (1993) / Gerhard (1993), which the paper cites without
 *   printing: H0 = 1, H1 = sqrt2 w, H2 = (2w^2-1)/sqrt2, H3 = (2 sqrt2 w^3 - 3 sqrt2 w)/sqrt6, H4 = (4w^4-12w^2+3)/sqrt24.
 * The caller normalises (h_m of a unit-mass LOSVD = 2 sqrt(pi)/gamma * [1+m]/[0]).  d_v0, d_s [n_ap] DEVICE doubles, the
 * pre-defined centre and width of each aperture's reference Gaussian; d_ap_map as above (required, n_ap <= 4000).
 * Sums are accumulated in 64-bit fixed point (2^-32), so rows do not depend on the order of additions.  d_dens, d_nout,
 * n_bundle, fourfold, density_mode as in sm_build_observable_library. */
int sm_build_gh_library(const sm_potential*, const double* d_ics, int64_t n_orb, double dt, int64_t n_steps, int32_t stride,
                        const sm_projection* proj, int n_proj, const sm_grids*, int precision, int32_t n_bundle, int fourfold,
                        const int32_t* d_ap_map, int32_t n_ap, const double* d_v0, const double* d_s, int density_mode,
                        float* d_gh, float* d_dens, int32_t* d_nout, void* cuda_stream);

/* Row a-8 for the paper's row forms (north_star item 4; 48 000 model evaluations): the bundled / aperture /
 * cylindrical / Gauss-Hermite libraries of trials [trial0, trial0+n_trials) of a batch potential in ONE integrator launch.
 * Trial arguments as in sm_build_library_batch (d_ics [n_orb][6] shared or [n_trials][n_orb][6]; proj [n_trials][n_proj] host);
 * row-form arguments as in the single-trial calls; the aperture map and the reference Gaussians (d_v0, d_s) are those of the
 * DATA and therefore shared by all trials.  Outputs carry a leading trial axis:
 *   d_losvd [n_trials][n_proj][n_orb/n_bundle][cells], d_gh [n_trials][n_proj][n_orb/n_bundle][n_ap][6],
 *   d_dens [n_trials][n_orb/n_bundle][dx*dy*dz], d_nout [n_trials][n_proj+1][n_orb/n_bundle] (may be NULL).
 * Each trial's block equals what the single-trial call gives for that trial's potential, angles and ICs (same kernels). */
int sm_build_observable_library_batch(const sm_potential* batch, int trial0, int n_trials, const double* d_ics, int ics_per_trial,
                                      int64_t n_orb, double dt, int64_t n_steps, int32_t stride, const sm_projection* proj, int n_proj,
                                      const sm_grids*, int precision, int32_t n_bundle, int fourfold, const int32_t* d_ap_map,
                                      int32_t n_ap, int density_mode, float* d_losvd, float* d_dens, int32_t* d_nout, void* cuda_stream);
int sm_build_gh_library_batch(const sm_potential* batch, int trial0, int n_trials, const double* d_ics, int ics_per_trial, int64_t n_orb,
                              double dt, int64_t n_steps, int32_t stride, const sm_projection* proj, int n_proj, const sm_grids*,
                              int precision, int32_t n_bundle, int fourfold, const int32_t* d_ap_map, int32_t n_ap, const double* d_v0,
                              const double* d_s, int density_mode, float* d_gh, float* d_dens, int32_t* d_nout, void* cuda_stream);

/* The same path in two calls, for callers that want to own the compact staged library (what sm_build_library does
 * internally).  A dense row is 0.25 ... 2.6 MB per orbit, the staged form 16 ... 40 KB: with rows larger than HBM / n_orb
 * (BASELINE.json configs[3], configs[4]) the caller integrates ALL orbits in one launch -- which is what fills the GPU --
 * and then flushes row windows through a ring of dense buffers.
 *  sm_stage_library_batch  rows a-1..a-6: integrates trials [trial0, trial0+n_trials) x n_orb orbits and writes one cell
 *      index per recorded sample and histogram, d_stage [n_trials][n_proj+1][n_orb][n_rec] uint32 (n_rec = n_steps/stride;
 *      histogram n_proj = density grid; 0xFFFFFFFF = sample outside the grid).  Other arguments as sm_build_library_batch
 *      (a single-trial potential with n_trials = 1 is the unbatched case).
 *  sm_flush_rows           row a-7: dense fp32 rows of orbits [orb0, orb0+n_rows) of every trial of a staged library:
 *      d_losvd [n_trials][n_proj][n_rows][nlos], d_dens [n_trials][n_rows][nden], d_nout [n_trials][n_proj+1][n_rows] (may be NULL).
 *      A trial sub-range is expressed by offsetting d_stage by whole trials. */
int sm_stage_library_batch(const sm_potential* batch, int trial0, int n_trials, const double* d_ics, int ics_per_trial,
                           int64_t n_orb, double dt, int64_t n_steps, int32_t stride, const sm_projection* proj,
                           int n_proj, const sm_grids*, int precision, uint32_t* d_stage, void* cuda_stream);
int sm_flush_rows(const uint32_t* d_stage, int n_trials, int n_proj, int64_t n_orb, int64_t n_rec, int64_t orb0,
                  int64_t n_rows, const sm_grids*, float* d_losvd, float* d_dens, int32_t* d_nout, void* cuda_stream);

/* sm_flush_rows into rows the CALLER has zeroed: only the non-zero cells are written (rows are ~98 % zeros: a few hundred
 * distinct cells out of 10^4 ... 10^5), from a shared-memory hash histogram per row (warp-aggregated shared atomics).  The
 * caller zeroes the window -- sm_zero_async on another stream -- while the integrator runs, which takes
 * the dense HBM-bound write off the critical path (sm_build_library does the same internally).  Same arguments and layouts as
 * sm_flush_rows; d_losvd and d_dens must be all-zero on entry, d_nout is overwritten. */
int sm_scatter_rows(const uint32_t* d_stage, int n_trials, int n_proj, int64_t n_orb, int64_t n_rec, int64_t orb0,
                    int64_t n_rows, const sm_grids*, float* d_losvd, float* d_dens, int32_t* d_nout, void* cuda_stream);
/* Row a-7 in COMPACT form: rows are ~98 % zeros (a median of ~470 distinct LOSVD cells out of 48 000 per orbit), and a
 * host consumer of the dense form pays PCIe for the zeros.  Same staged library and row window as sm_flush_rows; for every
 * (trial, histogram, row) the non-zero cells as (cell index, count) pairs:
 *   d_cell [capacity] u32, d_count [capacity] f32    the entries; row r = (trial*(n_proj+1) + hist)*n_rows + i occupies
 *   d_row_start[r] .. d_row_start[r] + d_row_nnz[r]  (runs are handed out by an atomic cursor: rows are NOT in order in the
 *                                                    entry arrays, and the entries of a row are in no particular order)
 *   d_total [1] u64   entries needed in all (zeroed by the call).  If it exceeds `capacity`, the entries past the end were
 *                     dropped: call again with larger arrays.  capacity = n_trials*(n_proj+1)*n_rows*n_rec always suffices.
 *   d_nout  as in sm_flush_rows (may be NULL).
 * Scattering count into a zero row at cell gives exactly the row sm_flush_rows writes.  n_rec <= 4096. */
int sm_flush_rows_compact(const uint32_t* d_stage, int n_trials, int n_proj, int64_t n_orb, int64_t n_rec, int64_t orb0,
                          int64_t n_rows, const sm_grids*, int64_t capacity, uint32_t* d_cell, float* d_count,
                          int64_t* d_row_start, int32_t* d_row_nnz, int32_t* d_nout, uint64_t* d_total, void* cuda_stream);

/* Zero n_bytes of device memory on cuda_stream with a kernel whose footprint fits BESIDE the persistent integrator, which
 * cudaMemsetAsync and device-to-device copies do not (they are SM kernels too and wait for it): one warp per SM that feeds the SM's
 * bulk-copy engine from a zeroed 16 KB shared-memory block (7.2 TB/s alone on a B200, ~3.3 TB/s beside the fp64 integrator), or,
 * where the integrator launches of the device read their tables through L1 (fp32 batches), one CTA of 128 threads per SM with a
 * paced store loop. */
int sm_zero_async(void* d_ptr, uint64_t n_bytes, void* cuda_stream);

/* Rows a-1..a-6 WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): sm_stage_library_batch for ONE trial (`trial`) of a potential, ICs [n_orb][6], d_stage
 * [n_proj+1][n_orb][n_rec] uint32 as there, same staged indices bit for bit (same kernels).  All of the integrator's scratch
 * (work-queue counters, projection constants, bar-phase table, orbit state between queue segments) lives in one static
 * device array of SM_NOALLOC_SCRATCH_BYTES (4 MiB + 128 KiB + 256 B) that every GPU that loads the library holds until the process exits;
 * the call makes no cudaMalloc / cudaMallocAsync / cudaFree, creates no pool, stream or event, copies nothing from the host, and
 * runs three kernels on cuda_stream without synchronising.  (The first call on a device looks the array's address up with
 * cudaGetSymbolAddress, which may load the module: make that call outside a capture.)
 * Limits: n_orb <= SM_NOALLOC_MAX_ORB and n_steps <= SM_NOALLOC_MAX_STEPS, else SM_ERR_UNSUPPORTED with a message that names the
 * limit and nothing is launched; larger libraries go through it by orbit range (d_ics + 6*i0, a staging buffer per range) or
 * through sm_stage_library_batch.  No Jacobi diagnostic, no bundles / apertures (plain rows only).
 * SHARED STATE: every call on one device uses the same array and finds the last call's contents there; each call clears what
 * must start at zero, so calls in stream order are independent, but calls that OVERLAP on one GPU (different streams or
 * host threads without an ordering between them) race on the scratch and give wrong results.  Rows: sm_flush_rows /
 * sm_scatter_rows / sm_flush_rows_compact on the staged indices, which allocate nothing either. */
#define SM_NOALLOC_MAX_ORB 32768
#define SM_NOALLOC_MAX_STEPS 65534
#define SM_NOALLOC_SCRATCH_BYTES 4325632
int sm_stage_library_noalloc(const sm_potential*, int trial, const double* d_ics, int64_t n_orb, double dt, int64_t n_steps,
                             int32_t stride, const sm_projection* proj, int n_proj, const sm_grids*, int precision,
                             uint32_t* d_stage, void* cuda_stream);

/* Orbital weights (Sect. 2.3): non-negative least squares on the stacked library
 * matrix by ADMM, all bootstrap realisations at once.
 *
 *   Q(w) = 1/2 ||U w - y||^2 + (lambda/N_orb) sum_i (w_i/wtilde_i)^2,  w >= 0          (PAPER.md:122 Eq. 3, :129 Eq. 4)
 *
 * "U is constructed by stacking all the matrices (m_{i,n}, Sigma_{i,n}, h_{m,i,n})": each sm_weight_block
 * is a strided view of a matrix an sm_build_* call wrote, element (i, c) = d_rows[i*row_pitch + col0 + c*col_stride]
 * (e.g. the Gauss-Hermite matrix [rows][n_ap][6] gives Sigma as col0 = 0, col_stride = 6 and h_m as col0 = 1+m); the
 * constraint index runs over the blocks in the order given, n_con = sum n_cols.  U[n][i] = element / d_sigma[n],
 * y_b[n] = d_target[n] / d_sigma[n] + d_xi[b][n]: d_sigma is the tolerance of constraint n (0.01 m*_n, 0.01 Sigma*_n,
 * Delta h*_{m,n}; a constraint whose tolerance is not a positive finite number is IGNORED: its row of U and its entry of y are zero), d_xi the unit-normal bootstrap draws of PAPER.md:136 ("perturbing them according to
 * their measurement uncertainties"), drawn by the caller, zero on the 3-D density rows; NULL = no perturbation.  "All
 * realisations share ... the same system matrix U, only the data vector y changes": one factorisation, n_rhs right-hand sides.
 *  d_keep    [n_orb] bytes or NULL: 0 drops the orbit (weight exactly 0) -- the Jacobi-drift cut of PAPER.md:86 applied to
 *            sm_build_library's d_diag.   d_wtilde [n_orb] > 0 or NULL (= 1, Eq. 4 as printed).
 *  ADMM (scaled form, reading R19): z = u = 0; n_iter times
 *            x = (U^T U + diag(2 lambda/(N_orb wtilde_i^2)) + rho I)^-1 (U^T y + rho (z - u));  z' = max(0, x + u);  u += x - z'.
 *  d_w       [n_rhs][n_orb] the clipped iterate z after n_iter iterations (>= 0).
 *  d_resid   [n_rhs][2] or NULL: ||x - z||_2 and rho ||z - z_prev||_2 of the last iteration.
 *  d_chi2    [n_rhs][n_blocks] or NULL: per realisation and block, sum over the block's constraints of
 *            ((sum_i w_i U_n,i) - d_target[n]/d_sigma[n])^2 -- the chi^2 terms of Eq. 3 against the UNPERTURBED data (DESIGN.md
 *            reading R20); Eq. 5 is the sum over the surface-density and Gauss-Hermite blocks.
 * All pointers except `blocks` are DEVICE pointers, fp64 unless stated, caller-owned; the call allocates its workspace
 * (8 n_orb (n_con + n_orb) bytes and small terms) from the stream's memory pool and is asynchronous on cuda_stream.
 * rho > 0, lambda >= 0, n_iter >= 1, 1 <= n_rhs <= 4096, 1 <= n_orb <= 65535, n_con >= 1.  fp64 throughout; sums are taken in a fixed
 * order, so results are reproducible from run to run. */
typedef struct sm_weight_block {
    const float* d_rows;
    int64_t row_pitch;
    int32_t col0, col_stride, n_cols;
} sm_weight_block;
int sm_solve_weights(const sm_weight_block* blocks, int n_blocks, int32_t n_orb, const double* d_target,
                     const double* d_sigma, const double* d_xi, int32_t n_rhs, const uint8_t* d_keep,
                     const double* d_wtilde, double lambda, double rho, int32_t n_iter, double* d_w, double* d_resid,
                     double* d_chi2, void* cuda_stream);

/* Model likelihood (Eq. 5-6): chi2_b = sum over the blocks k with bit k of block_mask set of d_chi2[b][k]
 * (the paper's choice "excludes chi^2_dens": leave the 3-D density block out of the mask), marginalised over the bootstrap
 * realisations as d_out[0] = chi2_min - 2 ln[(1/n_rhs) sum_b exp((chi2_min - chi2_b)/2)], d_out[1] = chi2_min.  Eq. 6 prints
 * "ln[sum_b exp((chi2_min - chi2_b)/2)] + const"; this is that quantity as -2 ln of the mean likelihood (reading R20), so that
 * equal chi2_b give chi2_b.  d_chi2 [n_rhs][n_blocks], d_out [2]: DEVICE fp64.  n_blocks <= 16. */
int sm_marginal_chi2(const double* d_chi2, int32_t n_rhs, int n_blocks, uint32_t block_mask, double* d_out, void* cuda_stream);

/* The paper's own integrator (reading R23): adaptive Bogacki-Shampine RK3(2) in the bar's
 * rotating frame, n_steps step ATTEMPTS per orbit (a rejected attempt leaves the state in place and has weight 0), relative
 * tolerance rtol (the paper: 1e-4; rtol <= 0: fixed steps h0), absolute tolerances atol_x / atol_v on positions / velocities, first
 * step h0.  fp64.  d_ics [n_orb][6] inertial at t = 0.  Every non-rotating component must be axisymmetric when omega_p or phase0 is
 * non-zero (SM_ERR_UNSUPPORTED otherwise).
 *  d_samples [n_steps][n_orb][6]  state after each attempt: position on bar axes, INERTIAL velocity on bar axes; may be NULL
 *  d_dtw     [n_steps][n_orb]     accepted step size of each attempt (the paper's sample weight delta-t), 0 if rejected; may be NULL
 *  d_tend    [n_orb]              total integrated time; may be NULL */
int sm_integrate_rk32(const sm_potential*, const double* d_ics, int64_t n_orb, int64_t n_steps, double rtol, double atol_x,
                      double atol_v, double h0, double* d_samples, double* d_dtw, double* d_tend, void* cuda_stream);

/* The same integrator into the orbit-observable matrices: every sample is sky-projected and binned as in sm_build_library, with
 * weight delta-t / t_total instead of 1.  d_losvd [n_proj][n_orb][nx*ny*nv], d_dens [n_orb][dx*dy*dz]: fp32 time
 * fractions (a row and its entry of d_wout sum to 1 up to fp32 rounding); d_wout [n_proj+1][n_orb] = the fraction of the time spent
 * outside each grid, may be NULL; d_tend [n_orb] may be NULL.  Asynchronous on cuda_stream like every other call (scratch:
 * 4 (n_proj + 2) n_orb n_steps bytes from the library's stream-ordered pool, in orbit chunks beyond 4 GiB).  Cell sums are
 * accumulated in 2^-32 fixed point, so rows do not depend on the order of additions. */
int sm_build_library_rk32(const sm_potential*, const double* d_ics, int64_t n_orb, int64_t n_steps, double rtol, double atol_x,
                          double atol_v, double h0, const sm_projection* proj, int n_proj, const sm_grids*, float* d_losvd,
                          float* d_dens, float* d_wout, double* d_tend, void* cuda_stream);

/* The paper's own pipeline on the paper's own integrator: the weighted rows with the row forms
 * of sm_build_observable_library / sm_build_gh_library -- bundles of n_bundle consecutive orbits (every member weighted by ITS
 * t_total), the fourfold copies of Table 1, pixels regrouped by d_ap_map into n_ap apertures, Cartesian or cylindrical density
 * cells; or, for the _gh call, per aperture {sum of w, sum of w alpha(u) H_m(u), m = 0..4}, u = (v_los - d_v0)/d_s.
 *  d_losvd [n_proj][n_orb/n_bundle][n_cells]  (n_cells = nx*ny*nv, or n_ap*nv with a map)   d_gh [n_proj][n_orb/n_bundle][n_ap][6]
 *  d_dens  [n_orb/n_bundle][dx*dy*dz]         d_wout [n_proj+1][n_orb/n_bundle] (may be NULL): row + wout = n_bundle (x 4 if fourfold)
 *  d_tend  [n_orb] (may be NULL)
 *  d_diag  [n_orb][2] (may be NULL): {max over the accepted samples of |E_J - E_J(0)| / |E_J(0)|, non-finite flag}, the Jacobi-
 *          integral error of PAPER.md:86 ("typical 1e-4 ... 1e-2; orbits above 1e-1 are discarded"): threshold it into the d_keep
 *          mask of sm_solve_weights.  Costs one potential evaluation per attempt.
 * Other arguments as in sm_build_library_rk32 and sm_build_observable_library / sm_build_gh_library. */
int sm_build_observable_library_rk32(const sm_potential*, const double* d_ics, int64_t n_orb, int64_t n_steps, double rtol,
                                     double atol_x, double atol_v, double h0, const sm_projection* proj, int n_proj, const sm_grids*,
                                     int32_t n_bundle, int fourfold, const int32_t* d_ap_map, int32_t n_ap, int density_mode,
                                     float* d_losvd, float* d_dens, float* d_wout, double* d_tend, double* d_diag, void* cuda_stream);
int sm_build_gh_library_rk32(const sm_potential*, const double* d_ics, int64_t n_orb, int64_t n_steps, double rtol, double atol_x,
                             double atol_v, double h0, const sm_projection* proj, int n_proj, const sm_grids*, int32_t n_bundle,
                             int fourfold, const int32_t* d_ap_map, int32_t n_ap, const double* d_v0, const double* d_s, int density_mode,
                             float* d_gh, float* d_dens, float* d_wout, double* d_tend, double* d_diag, void* cuda_stream);

/* Batched potentials for the adaptive path (row a-8 on the paper's own pipeline): trials [trial0, trial0+n_trials) of a batch
 * potential in one integrator launch per orbit chunk.  A CTA holds one trial's table at a time and moves through the trials, so the GPU fills
 * with n_trials x n_orb orbits even where one trial alone would leave it latency-bound.  d_ics [n_orb][6] shared or [n_trials][n_orb][6]
 * (ics_per_trial != 0); proj [n_trials][n_proj] host; aperture map and reference Gaussians shared.  Outputs with a leading trial axis:
 * d_losvd [n_trials][n_proj][rows][cells] / d_gh [n_trials][n_proj][rows][n_ap][6], d_dens [n_trials][rows][dx*dy*dz],
 * d_wout [n_trials][n_proj+1][rows], d_tend [n_trials][n_orb], d_diag [n_trials][n_orb][2] (the last three may be NULL).
 * Each trial's block is bit-identical to the single-trial call on that trial's potential (fixed-point sums, same kernels). */
int sm_build_observable_library_rk32_batch(const sm_potential* batch, int trial0, int n_trials, const double* d_ics, int ics_per_trial, int64_t n_orb,
                                           int64_t n_steps, double rtol, double atol_x, double atol_v, double h0, const sm_projection* proj,
                                           int n_proj, const sm_grids*, int32_t n_bundle, int fourfold, const int32_t* d_ap_map, int32_t n_ap,
                                           int density_mode, float* d_losvd, float* d_dens, float* d_wout, double* d_tend, double* d_diag,
                                           void* cuda_stream);
int sm_build_gh_library_rk32_batch(const sm_potential* batch, int trial0, int n_trials, const double* d_ics, int ics_per_trial, int64_t n_orb,
                                   int64_t n_steps, double rtol, double atol_x, double atol_v, double h0, const sm_projection* proj, int n_proj,
                                   const sm_grids*, int32_t n_bundle, int fourfold, const int32_t* d_ap_map, int32_t n_ap, const double* d_v0,
                                   const double* d_s, int density_mode, float* d_gh, float* d_dens, float* d_wout, double* d_tend,
                                   double* d_diag, void* cuda_stream);

/* Test hooks (the parity gates of north_star need them).
 * Force F[n][3] = -grad Phi (inertial components) and Phi[n] (may be NULL) at inertial positions
 * d_xyz[n][3], time t, for trial `trial` of the potential.  Outputs are fp64 in both precisions. */
int sm_eval_force(const sm_potential*, int trial, const double* d_xyz, int64_t n, double t, int precision,
                  double* d_F, double* d_Phi, void* cuda_stream);
/* Trajectory dump: d_traj[n_rec][n_orb][6], inertial, same integrator as sm_build_library. */
int sm_integrate_trajectories(const sm_potential*, int trial, const double* d_ics, int64_t n_orb, double dt,
                              int64_t n_steps, int32_t stride, int precision, double* d_traj, void* cuda_stream);

/* The two building blocks of sm_solve_weights on their own (fp64, device pointers, asynchronous on cuda_stream):
 * C[m][n] = alpha * sum_k A[m][k] * (b_kmajor ? B[n][k] : B[k][n]) + beta * C[m][n] with row pitches lda, ldb, ldc in
 * elements (beta != 0 needs alpha != 0); split_k > 1 writes split_k partial products, slab s at d_C + s*M*ldc (beta ignored); and the in-place
 * inverse of a symmetric positive definite matrix d_A [n][lda], n <= 65535 (symmetric block sweep without pivoting; only the
 * lower triangle is read, the full inverse is written). */
int sm_debug_gemm_f64(int b_kmajor, int M, int N, int K, double alpha, const double* d_A, int64_t lda, const double* d_B,
                      int64_t ldb, double beta, double* d_C, int64_t ldc, int split_k, void* cuda_stream);
int sm_debug_invert_spd(double* d_A, int64_t lda, int n, void* cuda_stream);

/* A/B switches for measurement: bit 0 = skip recording/binning/flush
 * (integrator only; final states are written to the staging buffer to keep the work alive),
 * bit 1 = flush rows with global atomics into a pre-zeroed row instead of the shared-memory slab path,
 * bit 2 = record CUDA events around the kernels (see sm_last_kernel_times),
 * bit 3 = run the integrator's work queue with at most 3 CTAs and segments of 3 strides (exercises the
 * segment hand-over on small test inputs; results must not change),
 * bit 5 = always flush rows through the dense shared-memory slab (one pass over the samples per 8 192-cell slab),
 * bit 6 = always through the sparse shared-memory hash histogram (one pass over the samples, non-zero cells patched into
 * the zero row); by default the library takes the slab unless its replays would read more than half the row's cells
 * (bundles),
 * bit 7 = sm_solve_weights / sm_debug_gemm_f64 run K-major contractions on the register-tiled DFMA kernel instead of the FP64
 * matrix unit (mma.sync m8n8k4).
 * 256: integrate with the generic component-loop kernel even where a specialised one exists (Plummer / Ferrers-barred /
 * needle-barred potential classes): same arithmetic per component, contracted differently, so results agree at rounding level.
 * 512: sm_build_library_rk32 builds its weighted rows as the first version did (zero the row, fp32 atomics on the global row) instead of
 * the fixed-point shared-memory hash (A/B; plain rows only).
 * 4096: sm_build_* calls do not zero their outputs on a side stream while the integrator runs; the rows are then written
 * whole by the dense slab / sparse kernels after it, as sm_flush_rows does.
 * 2048: the integrator hands out work per CTA instead of per warp (the form it must take for several fp64 trials in one launch).
 * 1024: the library-owned staging buffer of the sm_build_* calls is capped at 1 MiB instead of 4 GiB, so that small test inputs
 * go through the orbit-chunk loop (results must not change).
 * 16384: launches of at most 256 threads per CTA (fewer than ~38 000 orbits) use the register-capped integrator instantiation of the
 * large launches instead of their own (A/B; same source, results must not change).
 * 16: the integrator hands the orbits to its warps in the order the caller gave instead of in order of energy (A/B; results must not
 * change: orbits are independent, the order only decides which orbits share a warp).
 * 8192: the scatter of sm_scatter_rows / sm_flush_rows_compact runs 256-thread CTAs even where the library expects an integrator of
 * another stream on the SMs (A/B; by default 128-thread CTAs, which fit beside it).
 * 32768: every zero fill (the outputs of the sm_build_* calls, sm_zero_async) runs the paced store loop instead of the bulk-copy-engine
 * kernel (A/B).  Bits 16-23 (sleep in ns), 24-27 (stores per thread between sleeps; store loop only) and 28-30 (store loop: log2 of
 * threads / 32; bulk-copy kernel: block = 4 KB << x, at most 16 KB) override the fill's pacing (A/B, profiles/r2b, r2k, r2l).
 * The flags belong to the calling HOST THREAD (thread-local; a process may drive several GPUs from several threads); default 0.
 * Returns the thread's previous value. */
int sm_set_debug_flags(int flags);

/* Device time of the work of the last sm_build_* / sm_stage_library_batch / sm_flush_rows / sm_build_library_rk32 call made with
 * debug flag 4 set: ms4 = {bar-phase table, integrator (summed over orbit chunks), row build / scatter, zero fill of the outputs
 * on the library's side stream (concurrent with the integrator; 0 when the dense flush was used)} in milliseconds,
 * from CUDA events recorded around each on its stream.  Synchronises on those events. */
int sm_last_kernel_times(double* ms4);

/* The same for the last sm_solve_weights call: ms4 = {assembling U^T, y, the Gram matrix and U^T y; the inverse; the
 * whole iteration loop; the x-update launches of iterations 0, 16, 32, ... alone (each bracketed by its own events,
 * so [3] / ceil(n_iter/16) is the average duration of one launch of the dominant kernel)}. */
int sm_last_solve_times(double* ms4);

/* Peak-FMA microbenchmark used as the roofline denominator: runs `iters` dependent-chain-free
 * FMAs per thread over a full grid, returns achieved FLOP/s (FMA = 2) in *flops.  Synchronises. */
int sm_measure_fma_peak(int precision, int iters, double* flops);

/* Host-only test hooks (no CUDA call, never on the product path): the kernels' force algebra and their fp32 lambda iteration
 * compiled for the host, so that the -m "not gpu" tests can exercise the table construction and the iteration without a GPU.
 *  sm_debug_host_force   F[n][3] (and Phi[n], may be NULL) at host points xyz[n][3], time t, for a host descriptor.
 *  sm_debug_host_lambda  the Ferrers lambda of points xyz[n][3] for semi-axes a > b > c from warm-start guesses guess[n]
 *                        (< 0: cold start); lam[n] out, iters[n] (may be NULL) = iterations taken. */
int sm_debug_host_force(const sm_potential_desc* desc, const double* xyz, int64_t n, double t, int precision, double* F, double* Phi);
int sm_debug_host_lambda(double a, double b, double c, const double* xyz, int64_t n, const float* guess, float* lam, int* iters);

/* Number of kernels this library has launched since load (bench.py's gpu_launches). */
int64_t sm_launch_count(void);
const char* sm_last_error(void);
int sm_version(void);

#ifdef __cplusplus
}
#endif
#endif
