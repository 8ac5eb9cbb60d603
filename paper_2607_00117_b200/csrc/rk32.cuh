// rk32.cuh -- the paper's own integrator (reading R23): adaptive
// Bogacki-Shampine RK3(2) in the bar's rotating frame with a fixed number of step attempts, every sample weighted by its
// accepted step size.  One thread per orbit, state and the four stage derivatives in registers, accept / reject as selects
// (no divergent control flow: "the absence of branching ensures that the orbit integration can be perfectly parallelised").
//   state y = (x_b, u), u = velocity in the rotating frame:  dx_b/dt = u,
//   du/dt = F(x_b) + (2 Om u_y + Om^2 x_b, -2 Om u_x + Om^2 y_b, 0)              (Coriolis + centrifugal, Om = Omega_p e_z)
//   k1 = f(y); k2 = f(y + h/2 k1); k3 = f(y + 3h/4 k2); y' = y + h (2/9 k1 + 1/3 k2 + 4/9 k3); k4 = f(y') (= next k1)
//   e = h (-5/72 k1 + 1/12 k2 + 1/9 k3 - 1/8 k4);  err = rms_i e_i / (atol_i + rtol max(|y_i|, |y'_i|));
//   accept iff err <= 1;  h <- h min(5, max(0.2, 0.9 err^(-1/3)));  rtol <= 0: fixed steps.
// rk32_rows_kernel builds the delta-t-weighted rows: cells are fp32 sums of w = dt / t_total instead of counts.
#pragma once
#include "kernels.cuh"

namespace smx {

struct Rk32Args {
    const PotDev* pots; int trial;  // first trial of the launch
    int n_trials;                  // trials in this launch (batched potentials): every per-orbit array below then holds n_trials x n_orb
                                   // orbits, trial-major (orbit index trial * n_orb + i); the projections are [n_trials][n_proj]
    long long ics_trial_stride;    // doubles between the ICs of consecutive trials (0: shared)
    int q_stride;                  // ints between the queues of consecutive trials (work / done below are trial 0's)
    long long state_trial_stride;  // doubles between the hand-over states of consecutive trials
    const double* tab;             // fp64 Ferrers anchor tables (global)
    const double* tab0;            // W000 tables (potential; Jacobi diagnostic only), may be null
    const double* ics;             // [n_orb][6] inertial at t = 0
    long long n_orb; int n_steps;
    double rtol, atol_x, atol_v, h0;
    double* samples;               // [n_steps][n_orb][6] or null
    double* dtw;                   // [n_steps][n_orb] or null
    double* t_end;                 // [n_orb] or null
    double* diag;                  // [n_orb][2] {max relative Jacobi-integral error over the accepted samples, non-finite flag} or null
    // library mode (stage != null): cells of every attempt's sample (and of its n_sym - 1 mirror copies) per histogram, and its weight
    const ProjDev<double>* proj; int n_proj;
    BinDev<double> bins;           // with the aperture map / cylindrical cells of the observable rows
    int n_sym;                     // 1, or 4 = the copies of PAPER.md:77-90 Table 1
    unsigned* stage;               // [n_proj + 1][stage_orb_stride][n_steps * n_sym]
    float* stage_v;                // Gauss-Hermite rows: v_los of the staged LOSVD samples [n_proj][stage_orb_stride][n_steps * n_sym], else null
    long long stage_orb_stride;
    float* stage_w;                // [n_orb][n_steps] accepted step size (0 = rejected attempt)
    // work queue: units = (segment of seg_len attempts) x (group of 32 orbits), one warp each (see integrate_kernel)
    int* work; int* done; double* state;
    int n_grp, n_seg; int seg_len;
};
constexpr int N_RKSTATE = 19;      // y[6] k1[6] h t lam ej0 drift bad | spare

// PHI: also return the potential at y (the Jacobi diagnostic takes it from the first-same-as-last evaluation, see rk32_kernel)
template <int POT, bool PHI = false>
__device__ __forceinline__ double rk32_rhs(const PotS<double>& P, const double* tab, const FerrersCtx<double, true>& FB, double om, double om2,
                                           const double* y, double* f, float& lam) {
    double ax, ay, az, phi = 0.0;
    // all components with the bar at rest along x (cos = 1, sin = 0: the rotation to bar axes is the identity)
    total_force<double, PHI, POT, true>(P, tab, FB, y[0], y[1], y[2], 1.0, 0.0, ax, ay, az, phi, lam);
    f[0] = y[3]; f[1] = y[4]; f[2] = y[5];
    f[3] = fma(om2, y[0], fma(2.0 * om, y[4], ax));
    f[4] = fma(om2, y[1], fma(-2.0 * om, y[3], ay));
    f[5] = az;
    return phi;
}

// Jacobi integral of a rotating-frame state: E_J = |u|^2/2 + Phi(x_b) - Omega^2 (x_b^2 + y_b^2)/2, which equals
// v^2/2 + Phi - Omega L_z with the inertial velocity.  Not inlined: one call per attempt, only when the diagnostic is asked for.
template <int POT>
__device__ __noinline__ double rk32_jacobi(const PotS<double>& P, const double* tab, const FerrersCtx<double, true>& FB, double om2, const double* y) {
    double ax, ay, az, phi = 0.0;
    float lam = -1.0f;
    total_force<double, true, POT, true>(P, tab, FB, y[0], y[1], y[2], 1.0, 0.0, ax, ay, az, phi, lam);
    return 0.5 * (y[3] * y[3] + y[4] * y[4] + y[5] * y[5]) + phi - 0.5 * om2 * (y[0] * y[0] + y[1] * y[1]);
}

// Cells of one sample (attempt k of orbit `orb`): density cell and one LOSVD cell per projection, times the n_sym copies of
// Table 1 (slots k n_sym + {0: (+,+), 1: (+,-z), 2: (-x-y,+), 3: (-,-)}; a projection is linear, so two give all four).
// Run-time variants (aperture map, cylindrical cells, Gauss-Hermite staging): once per attempt beside three force evaluations.
__device__ __forceinline__ void rk32_stage_sample(const Rk32Args& a, const ProjDev<double>* proj, long long orb, int k, double xb, double yb, double z,
                                                  double ub, double wb, double vz) {
    const int ns = a.n_sym;
    const long long nre = (long long)a.n_steps * ns, hs = a.stage_orb_stride * nre;
    unsigned* st = a.stage + orb * nre + (long long)k * ns;
    float* sv = a.stage_v ? a.stage_v + orb * nre + (long long)k * ns : nullptr;
    const DensCoord<double> dc = dens_coord<double, true>(a.bins, xb, yb);
    const int n_half = ns == 4 ? 2 : 1;
    for (int m = 0; m < n_half; ++m) {
        const double zm = m ? -z : z, vzm = m ? -vz : vz;
        st[a.n_proj * hs + m] = bin3<double>(a.bins, 3, dc.u0, dc.u1, zm);
        if (ns == 4) st[a.n_proj * hs + m + 2] = bin3<double>(a.bins, 3, dc.m0, dc.m1, zm);
        for (int p = 0; p < a.n_proj; ++p) {
            const ProjDev<double> R = proj[p];
            const double x1 = xb * R.ca - yb * R.sa, y1 = xb * R.sa + yb * R.ca;
            const double y2 = y1 * R.cb - zm * R.sb;
            const double X = x1 * R.cg - y2 * R.sg, Y = x1 * R.sg + y2 * R.cg;
            const double vlos = (ub * R.sa + wb * R.ca) * R.sb + vzm * R.cb;
            if (sv) {
                st[p * hs + m] = aperture_of<double>(a.bins, X, Y);
                sv[p * hs + m] = (float)vlos;
                if (ns == 4) { st[p * hs + 3 - m] = aperture_of<double>(a.bins, -X, -Y); sv[p * hs + 3 - m] = (float)(-vlos); }
            } else {
                st[p * hs + m] = bin3<double, true>(a.bins, 0, X, Y, vlos);
                if (ns == 4) st[p * hs + 3 - m] = bin3<double, true>(a.bins, 0, -X, -Y, -vlos);
            }
        }
    }
}

// POT: potential class (force.cuh) -- the specialised force bodies of the fixed-step integrator, Ferrers table in shared memory.
// Persistent: one CTA per SM, the attempts of every group of 32 orbits cut into segments that warps take from a queue
// (with a plain grid 20 000 orbits filled 125 of 148 SMs).  Later segments are handed out through a READY RING: the warp that
// finishes segment s of a group appends segment s+1 to the ring and warps take ring entries in order, so no warp ever holds a
// unit whose predecessor is still running.  With a fixed segment-major hand-out order the predecessor was always in the round just
// before and every warp lost the spread of that round's finishing times: 78 million polls per 34 ms launch, a quarter of the slot
// time, each poll (ld.acquire) flushing the SM's L1 (config-1 size: 25.6 -> 18.8 ms; profiles/r2g.md).
#ifndef SMX_RK32_MAXTHREADS
#define SMX_RK32_MAXTHREADS 256
#endif
#ifndef SMX_RK32_MAXREGS
#define SMX_RK32_MAXREGS 232   // leaves the SM room for a 64-thread zero_fill_kernel CTA (api_rk32.inc)
#endif
// FULL = false: plain rows only (one cell per histogram and attempt, no copies, apertures, cylindrical cells, v_los staging or
// Jacobi diagnostic) -- the first version's loop body, which the compiler schedules in 238 registers without spills; FULL = true
// carries the run-time row-form variants and the diagnostic (254 registers and a 200-byte stack frame: measured 1.5x slower
// per attempt at one warp per scheduler, profiles/r2g.md), so only the calls that need them pay for them.
// FEAT: 0 = plain rows (FULL = false), 1 = row-form variants, 2 = row-form variants + Jacobi diagnostic.  The diagnostic takes the
// potential from the fourth (first-same-as-last) force evaluation, which costs that evaluation ~10 % even when nobody reads it:
// hence its own instantiation (measured: 64-trial Gauss-Hermite batch 933 ms without, 1 041 ms with the potential computed).
template <int POT, int FEAT>
__global__ void __maxnreg__(SMX_RK32_MAXREGS) rk32_kernel(Rk32Args a) {
    constexpr bool FULL = FEAT != 0, DIAG = FEAT == 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PotS<double>* P = reinterpret_cast<PotS<double>*>(smem_raw);
    double* tab_s = reinterpret_cast<double*>(smem_raw + ((sizeof(PotS<double>) + 15) / 16) * 16);
    __shared__ int s_skip;
    const int lane = threadIdx.x & 31;
    const long long n_units = (long long)a.n_grp * a.n_seg;
    // Batched potentials: the 160 KB table of ONE trial fits the CTA's shared memory, so a CTA works on one trial at a time: it
    // starts on trial blockIdx mod n_trials, takes units of that trial's queue until it is exhausted and moves on to the next trial
    // (every CTA visits every trial, skipping those whose units have all been handed out), so no SM idles while any trial has work.
    for (int tp = 0; tp < a.n_trials; ++tp) {
    const int tr = a.n_trials > 1 ? (int)((blockIdx.x + tp) % a.n_trials) : 0;
    int* const q_work = a.work + (long long)tr * a.q_stride;
    int* const q_done = a.done + (long long)tr * a.q_stride;
    if (a.n_trials > 1) {
        __syncthreads();   // every warp has left the previous trial: its table may be overwritten
        if (threadIdx.x == 0) s_skip = ld_relaxed_gpu(q_work) >= n_units;
        __syncthreads();
        if (s_skip) continue;
    }
    const PotDev& G = a.pots[a.trial + tr];
    load_pot<double>(G, P, a.tab, a.tab0, tab_s, true, (int)threadIdx.x, (int)blockDim.x);
    __syncthreads();
    FerrersCtx<double, true> FB{};
    if (POT == POT_BARRED) FB = make_ferrers_ctx<double, true>(*P, tab_s, P->comp[P->i_fer]);
    const double om = G.omega_p, om2 = om * om;
    double c0, s0;
    sincos(G.phase0, &s0, &c0);
    const long long orb0 = (long long)tr * a.n_orb;          // this trial's first orbit in the per-orbit arrays
    const ProjDev<double>* const proj = a.proj + tr * a.n_proj;
    for (;;) {
        // hand-out position u; positions >= n_grp go through the ready ring (see integrate_kernel): a.done[0] = ring tail,
        // a.done[1 + i] = the i-th unit of a later segment that became ready (seg * n_grp + grp), -1 before
        int u = 0, unit = 0;
        if (lane == 0) {
            u = unit = atomicAdd(q_work, 1);
            if (u >= a.n_grp && u < n_units) {
                const int* e = q_done + 1 + (u - a.n_grp);
                while ((unit = ld_relaxed_gpu(e)) < 0) __nanosleep(64);
                __threadfence();
            }
        }
        u = __shfl_sync(0xFFFFFFFFu, u, 0);
        unit = __shfl_sync(0xFFFFFFFFu, unit, 0);
        if (u >= n_units) break;
        const int seg = unit / a.n_grp, grp = unit - seg * a.n_grp;
        const long long orb_raw = (long long)grp * 32 + lane;
        const bool live = orb_raw < a.n_orb;   // every lane stays alive (the Ferrers lambda iteration votes across the warp)
        const long long orb = orb0 + (live ? orb_raw : a.n_orb - 1);   // index in the per-orbit arrays
        double* sp = a.state + tr * a.state_trial_stride + (long long)grp * N_RKSTATE * 32 + lane;
        double y[6], k1[6], k2[6], k3[6], k4[6], yt[6], yn[6];
        float lam;
        double h, t, ej0 = 0.0, drift = 0.0, bad = 0.0;
        if (seg == 0) {
            const double* ic = a.ics + tr * a.ics_trial_stride + (orb - orb0) * 6;
            y[0] = c0 * ic[0] + s0 * ic[1]; y[1] = -s0 * ic[0] + c0 * ic[1]; y[2] = ic[2];
            y[3] = c0 * ic[3] + s0 * ic[4] + om * y[1]; y[4] = -s0 * ic[3] + c0 * ic[4] - om * y[0]; y[5] = ic[5];
            lam = -1.0f; h = a.h0; t = 0.0;
            rk32_rhs<POT>(*P, tab_s, FB, om, om2, y, k1, lam);
            if (DIAG && a.diag) ej0 = rk32_jacobi<POT>(*P, tab_s, FB, om2, y);
        } else {
#pragma unroll
            for (int j = 0; j < 6; ++j) { y[j] = __ldcg(sp + j * 32); k1[j] = __ldcg(sp + (6 + j) * 32); }
            h = __ldcg(sp + 12 * 32); t = __ldcg(sp + 13 * 32); lam = (float)__ldcg(sp + 14 * 32);
            if (DIAG) { ej0 = __ldcg(sp + 15 * 32); drift = __ldcg(sp + 16 * 32); bad = __ldcg(sp + 17 * 32); }
        }
        const int ka = seg * a.seg_len, kb = min(ka + a.seg_len, a.n_steps);
        for (int k = ka; k < kb; ++k) {
#pragma unroll
            for (int j = 0; j < 6; ++j) yt[j] = fma(h, 0.5 * k1[j], y[j]);
            rk32_rhs<POT>(*P, tab_s, FB, om, om2, yt, k2, lam);
#pragma unroll
            for (int j = 0; j < 6; ++j) yt[j] = fma(h, 0.75 * k2[j], y[j]);
            rk32_rhs<POT>(*P, tab_s, FB, om, om2, yt, k3, lam);
#pragma unroll
            for (int j = 0; j < 6; ++j) yn[j] = fma(h, (2.0 / 9.0) * k1[j] + (1.0 / 3.0) * k2[j] + (4.0 / 9.0) * k3[j], y[j]);
            // the fourth evaluation is next attempt's first (first-same-as-last) AND, in the FULL kernel, gives the potential at the new
            // state for the Jacobi diagnostic: a separate potential evaluation per attempt cost a fourth pass through the force body
            const double phi_n = rk32_rhs<POT, DIAG>(*P, tab_s, FB, om, om2, yn, k4, lam);
            bool accept = true;
            double h_next = h;
            if (a.rtol > 0.0) {
                double sum = 0.0;
#pragma unroll
                for (int j = 0; j < 6; ++j) {
                    const double e = h * ((-5.0 / 72.0) * k1[j] + (1.0 / 12.0) * k2[j] + (1.0 / 9.0) * k3[j] - (1.0 / 8.0) * k4[j]);
                    const double sc = (j < 3 ? a.atol_x : a.atol_v) + a.rtol * fmax(fabs(y[j]), fabs(yn[j]));
                    const double q = e * rcp_t(sc);       // sc > 0; reciprocal to ~1 ulp without the division's slow path
                    sum = fma(q, q, sum);
                }
                const double err = sqrt(sum * (1.0 / 6.0));
                accept = err <= 1.0;                              // NaN rejects
                double fac = err > 0.0 ? 0.9 * rcbrt(err) : (err == 0.0 ? 5.0 : 0.2);    // err^(-1/3); a NaN estimate (overflowed stage) shrinks the step
                if (!(fac >= 0.2)) fac = 0.2;
                if (fac > 5.0) fac = 5.0;
                h_next = h * fac;
            }
            const double w = accept ? h : 0.0;
#pragma unroll
            for (int j = 0; j < 6; ++j) { y[j] = accept ? yn[j] : y[j]; k1[j] = accept ? k4[j] : k1[j]; }
            t += w;
            h = h_next;
            if (DIAG && a.diag && accept) {   // y is yn here
                const double ej = 0.5 * (y[3] * y[3] + y[4] * y[4] + y[5] * y[5]) + phi_n - 0.5 * om2 * (y[0] * y[0] + y[1] * y[1]);
                if (isfinite(ej)) drift = fmax(drift, fabs(ej - ej0) / fabs(ej0)); else bad = 1.0;
            }
            // the sample: position on bar axes, inertial velocity on bar axes u + Omega x x_b (reading R1)
            const double vbx = fma(-om, y[1], y[3]), vby = fma(om, y[0], y[4]);
            if (live) {
                if (a.samples) {
                    double* o = a.samples + ((long long)k * a.n_orb + orb) * 6;
                    o[0] = y[0]; o[1] = y[1]; o[2] = y[2]; o[3] = vbx; o[4] = vby; o[5] = y[5];
                }
                if (a.dtw) a.dtw[(long long)k * a.n_orb + orb] = w;
                if (a.stage) {
                    if (FULL) {
                        rk32_stage_sample(a, proj, orb, k, y[0], y[1], y[2], vbx, vby, y[5]);
                    } else {
                        unsigned* st = a.stage + orb * (long long)a.n_steps + k;
                        const long long hs = a.stage_orb_stride * (long long)a.n_steps;
                        st[a.n_proj * hs] = bin3<double>(a.bins, 3, y[0], y[1], y[2]);
                        for (int p = 0; p < a.n_proj; ++p) {
                            const ProjDev<double> R = proj[p];
                            const double x1 = y[0] * R.ca - y[1] * R.sa, y1 = y[0] * R.sa + y[1] * R.ca;
                            const double y2 = y1 * R.cb - y[2] * R.sb;
                            const double X = x1 * R.cg - y2 * R.sg, Y = x1 * R.sg + y2 * R.cg;
                            const double vlos = (vbx * R.sa + vby * R.ca) * R.sb + y[5] * R.cb;
                            st[p * hs] = bin3<double>(a.bins, 0, X, Y, vlos);
                        }
                    }
                    a.stage_w[orb * (long long)a.n_steps + k] = (float)w;
                }
            }
        }
        if (seg + 1 < a.n_seg) {
#pragma unroll
            for (int j = 0; j < 6; ++j) { __stcg(sp + j * 32, y[j]); __stcg(sp + (6 + j) * 32, k1[j]); }
            __stcg(sp + 12 * 32, h); __stcg(sp + 13 * 32, t); __stcg(sp + 14 * 32, (double)lam);
            if (DIAG) { __stcg(sp + 15 * 32, ej0); __stcg(sp + 16 * 32, drift); __stcg(sp + 17 * 32, bad); }
            __syncwarp();
            if (lane == 0) {
                __threadfence();
                const int tpos = atomicAdd(q_done, 1);
                st_release_gpu(q_done + 1 + tpos, (seg + 1) * a.n_grp + grp);
            }
        } else if (live) {
            if (a.t_end) a.t_end[orb] = t;
            if (DIAG && a.diag) { a.diag[2 * orb] = drift; a.diag[2 * orb + 1] = bad; }
        }
    }
    }   // trials
}

// One CTA per (orbit, histogram): zero the dense fp32 row, then add w_k / t_total into the cell of every accepted sample
// (fp32 atomics on the row, which stays in L2: 192 KB for config 1's LOSVD block); the weight that falls outside the grid
// goes to wout.  Sums of ~n_steps positive fp32 terms in arbitrary order: relative error <= ~1e-6 per cell.
__global__ void __launch_bounds__(256) rk32_rows_kernel(const unsigned* stage, const float* stage_w, const double* t_end, long long n_orb,
                                                        int n_steps, int n_proj, long long nlos, long long nden,
                                                        float* losvd, float* dens, float* wout) {
    __shared__ float s_out[8];
    const long long orb = blockIdx.x;
    const int hst = blockIdx.y;
    const long long ncell = hst < n_proj ? nlos : nden;
    float* row = hst < n_proj ? losvd + ((long long)hst * n_orb + orb) * nlos : dens + orb * nden;
    for (long long i = threadIdx.x; i < ncell; i += blockDim.x) row[i] = 0.0f;
    __syncthreads();
    const double tt = t_end[orb];
    const float inv = tt > 0.0 ? (float)(1.0 / tt) : 0.0f;
    const unsigned* st = stage + ((long long)hst * n_orb + orb) * n_steps;
    const float* sw = stage_w + orb * (long long)n_steps;
    float out = 0.0f;
    for (int k = threadIdx.x; k < n_steps; k += blockDim.x) {
        const float w = sw[k] * inv;
        const unsigned c = st[k];
        if (w > 0.0f) {
            if (c != IDX_OUT) atomicAdd(row + c, w); else out += w;
        }
    }
    for (int o = 16; o > 0; o >>= 1) out += __shfl_down_sync(0xffffffffu, out, o);
    if ((threadIdx.x & 31) == 0) s_out[threadIdx.x >> 5] = out;
    __syncthreads();
    if (threadIdx.x == 0 && wout) {
        float s = 0.0f;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += s_out[i];
        wout[(long long)hst * n_orb + orb] = s;
    }
}

}  // namespace smx
