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
    const PotDev* pots; int trial;
    const double* tab;             // fp64 Ferrers anchor tables (global)
    const double* ics;             // [n_orb][6] inertial at t = 0
    long long n_orb; int n_steps;
    double rtol, atol_x, atol_v, h0;
    double* samples;               // [n_steps][n_orb][6] or null
    double* dtw;                   // [n_steps][n_orb] or null
    double* t_end;                 // [n_orb] or null
    // library mode (stage != null): cell of every attempt's sample per histogram, and its weight
    const ProjDev<double>* proj; int n_proj;
    BinDev<double> bins;
    unsigned* stage;               // [n_proj + 1][n_orb][n_steps]
    float* stage_w;                // [n_orb][n_steps] accepted step size (0 = rejected attempt)
};

template <int POT>
__device__ __forceinline__ void rk32_rhs(const PotS<double>& P, const double* tab, const FerrersCtx<double, true>& FB, double om, double om2,
                                         const double* y, double* f, float& lam) {
    double ax, ay, az, phi = 0.0;
    // all components with the bar at rest along x (cos = 1, sin = 0: the rotation to bar axes is the identity)
    total_force<double, false, POT, true>(P, tab, FB, y[0], y[1], y[2], 1.0, 0.0, ax, ay, az, phi, lam);
    f[0] = y[3]; f[1] = y[4]; f[2] = y[5];
    f[3] = fma(om2, y[0], fma(2.0 * om, y[4], ax));
    f[4] = fma(om2, y[1], fma(-2.0 * om, y[3], ay));
    f[5] = az;
}

// POT: potential class (force.cuh) -- the specialised force bodies of the fixed-step integrator, Ferrers table in shared memory
template <int POT>
__global__ void __launch_bounds__(256) rk32_kernel(Rk32Args a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PotS<double>* P = reinterpret_cast<PotS<double>*>(smem_raw);
    double* tab_s = reinterpret_cast<double*>(smem_raw + ((sizeof(PotS<double>) + 15) / 16) * 16);
    const PotDev& G = a.pots[a.trial];
    load_pot<double>(G, P, a.tab, nullptr, tab_s, true, (int)threadIdx.x, (int)blockDim.x);
    __syncthreads();
    FerrersCtx<double, true> FB{};
    if (POT == POT_BARRED) FB = make_ferrers_ctx<double, true>(*P, tab_s, P->comp[P->i_fer]);
    const long long orb_raw = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const bool live = orb_raw < a.n_orb;   // every lane stays alive (the Ferrers lambda iteration votes across the warp)
    const long long orb = live ? orb_raw : a.n_orb - 1;
    const double om = G.omega_p, om2 = om * om;
    double c0, s0;
    sincos(G.phase0, &s0, &c0);
    const double* ic = a.ics + orb * 6;
    double y[6], k1[6], k2[6], k3[6], k4[6], yt[6], yn[6];
    y[0] = c0 * ic[0] + s0 * ic[1]; y[1] = -s0 * ic[0] + c0 * ic[1]; y[2] = ic[2];
    y[3] = c0 * ic[3] + s0 * ic[4] + om * y[1]; y[4] = -s0 * ic[3] + c0 * ic[4] - om * y[0]; y[5] = ic[5];
    float lam = -1.0f;
    double h = a.h0, t = 0.0;
    rk32_rhs<POT>(*P, tab_s, FB, om, om2, y, k1, lam);
    const int n_hist = a.n_proj + 1;
    for (int k = 0; k < a.n_steps; ++k) {
#pragma unroll
        for (int j = 0; j < 6; ++j) yt[j] = fma(h, 0.5 * k1[j], y[j]);
        rk32_rhs<POT>(*P, tab_s, FB, om, om2, yt, k2, lam);
#pragma unroll
        for (int j = 0; j < 6; ++j) yt[j] = fma(h, 0.75 * k2[j], y[j]);
        rk32_rhs<POT>(*P, tab_s, FB, om, om2, yt, k3, lam);
#pragma unroll
        for (int j = 0; j < 6; ++j) yn[j] = fma(h, (2.0 / 9.0) * k1[j] + (1.0 / 3.0) * k2[j] + (4.0 / 9.0) * k3[j], y[j]);
        rk32_rhs<POT>(*P, tab_s, FB, om, om2, yn, k4, lam);
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
            double fac = err > 0.0 ? 0.9 * rcbrt(err) : 5.0;    // err^(-1/3)
            if (!(fac >= 0.2)) fac = 0.2;
            if (fac > 5.0) fac = 5.0;
            h_next = h * fac;
        }
        const double w = accept ? h : 0.0;
#pragma unroll
        for (int j = 0; j < 6; ++j) { y[j] = accept ? yn[j] : y[j]; k1[j] = accept ? k4[j] : k1[j]; }
        t += w;
        h = h_next;
        // the sample: position on bar axes, inertial velocity on bar axes u + Omega x x_b (reading R1)
        const double vbx = fma(-om, y[1], y[3]), vby = fma(om, y[0], y[4]);
        if (live) {
            if (a.samples) {
                double* o = a.samples + ((long long)k * a.n_orb + orb) * 6;
                o[0] = y[0]; o[1] = y[1]; o[2] = y[2]; o[3] = vbx; o[4] = vby; o[5] = y[5];
            }
            if (a.dtw) a.dtw[(long long)k * a.n_orb + orb] = w;
            if (a.stage) {
                unsigned* st = a.stage + orb * (long long)a.n_steps + k;
                const long long hs = a.n_orb * (long long)a.n_steps;
                st[a.n_proj * hs] = bin3<double>(a.bins, 3, y[0], y[1], y[2]);
                for (int p = 0; p < a.n_proj; ++p) {
                    const ProjDev<double> R = a.proj[p];
                    const double x1 = y[0] * R.ca - y[1] * R.sa, y1 = y[0] * R.sa + y[1] * R.ca;
                    const double y2 = y1 * R.cb - y[2] * R.sb;
                    const double X = x1 * R.cg - y2 * R.sg, Y = x1 * R.sg + y2 * R.cg;
                    const double vlos = (vbx * R.sa + vby * R.ca) * R.sb + y[5] * R.cb;
                    st[p * hs] = bin3<double>(a.bins, 0, X, Y, vlos);
                }
                a.stage_w[orb * (long long)a.n_steps + k] = (float)w;
            }
        }
    }
    (void)n_hist;
    if (live && a.t_end) a.t_end[orb] = t;
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

// The same rows through a shared-memory slab (the form of rowbuild_kernel, with fp32 weights in place of
// counts): persistent CTAs walk the rows orbit-fastest; for every slab of RK32_SLAB cells the CTA replays the orbit's staged
// (cell, weight) pairs into the slab with fp32 shared-memory atomics, then streams the slab to HBM with 16-byte stores and
// zeroes it behind itself, so every cell of the dense row is written exactly once and never read back.
constexpr int RK32_SLAB = 8192;   // cells = 32 KB: six CTAs of 256 threads per SM
__global__ void __launch_bounds__(256) rk32_rows_slab_kernel(const unsigned* stage, const float* stage_w, const double* t_end, long long n_orb,
                                                             int n_steps, int n_proj, long long nlos, long long nden,
                                                             float* losvd, float* dens, float* wout) {
    __shared__ __align__(16) float slab[RK32_SLAB];
    __shared__ float s_out[8];
    const int tid = threadIdx.x;
    for (int i = tid; i < RK32_SLAB; i += blockDim.x) slab[i] = 0.0f;
    __syncthreads();
    const long long n_rows = (long long)(n_proj + 1) * n_orb;
    for (long long row_id = blockIdx.x; row_id < n_rows; row_id += gridDim.x) {
        const long long orb = row_id % n_orb;
        const int hst = (int)(row_id / n_orb);
        const int ncell = (int)(hst < n_proj ? nlos : nden);
        float* row = hst < n_proj ? losvd + ((long long)hst * n_orb + orb) * nlos : dens + orb * nden;
        const double tt = t_end[orb];
        const float inv = tt > 0.0 ? (float)(1.0 / tt) : 0.0f;
        const unsigned* st = stage + ((long long)hst * n_orb + orb) * n_steps;
        const float* sw = stage_w + orb * (long long)n_steps;
        const bool vec_ok = ((ncell & 3) == 0) && ((((size_t)row) & 15) == 0);
        float out = 0.0f;
        for (int base = 0; base < ncell; base += RK32_SLAB) {
            const int n_here = min(RK32_SLAB, ncell - base);
            for (int k = tid; k < n_steps; k += blockDim.x) {
                const float w = __ldg(sw + k) * inv;
                const unsigned c = __ldg(st + k);
                const unsigned rel = c - (unsigned)base;           // wraps to a huge value below the slab
                if (w > 0.0f) {
                    if (c == IDX_OUT) { if (base == 0) out += w; }
                    else if (rel < (unsigned)n_here) atomicAdd(&slab[rel], w);
                }
            }
            __syncthreads();
            if (vec_ok) {
                float4* s4 = reinterpret_cast<float4*>(slab);
                float4* o4 = reinterpret_cast<float4*>(row + base);
                for (int i = tid; i < (n_here >> 2); i += blockDim.x) {
                    const float4 v = s4[i];
                    s4[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                    __stcs(o4 + i, v);
                }
            } else {
                for (int i = tid; i < n_here; i += blockDim.x) { row[base + i] = slab[i]; slab[i] = 0.0f; }
            }
            __syncthreads();
        }
        for (int o = 16; o > 0; o >>= 1) out += __shfl_down_sync(0xffffffffu, out, o);
        if ((tid & 31) == 0) s_out[tid >> 5] = out;
        __syncthreads();
        if (tid == 0 && wout) {
            float s = 0.0f;
            for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += s_out[i];
            wout[(long long)hst * n_orb + orb] = s;
        }
        __syncthreads();
    }
}

}  // namespace smx
