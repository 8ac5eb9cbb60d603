// kernels.cuh -- the CUDA kernels of the orbit-library path (sm_100a).
//
//   phase_table_kernel   (cos, sin)(Omega_p k dt + phase0), k = 0..n_steps, once per call: the bar
//                        phase is common to all orbits, so it is hoisted out of the orbit loop.
//   integrate_kernel     SURVEY.md 8(a) rows a-1..a-6: one thread per orbit, state in registers,
//                        KDK leapfrog, force from force.cuh/ferrers.cuh, record -> bar frame ->
//                        project -> bin index; writes one u32 cell index per histogram per sample
//                        to a staging buffer (or the trajectory for the test hook).
//   rowbuild_kernel      row a-7: one CTA per (orbit, histogram) row: replays the orbit's staged
//                        indices into a shared-memory slab with warp-aggregated shared atomics and
//                        flushes the dense fp32 row to HBM with 16-byte coalesced streaming stores.
//   eval_force_kernel    test hook.      fma_peak_kernel   roofline denominator.
#pragma once
#include <cuda_runtime.h>

#include "ferrers.cuh"

namespace smx {

constexpr int MAX_PROJ = 4;
constexpr unsigned IDX_OUT = 0xFFFFFFFFu;

template <typename T> struct Vec2;
template <> struct Vec2<double> { typedef double2 type; };
template <> struct Vec2<float> { typedef float2 type; };

template <typename T>
struct BinDev {
    T lo[6], inv[6];  // X, Y, v_los, then density x, y, z
    int n[6];
    const int* ap_map;  // [ny*nx] aperture of every image pixel (< 0: none), or null = no regrouping
    int n_ap;
    int dens_mode;      // 0 Cartesian (x_b, y_b, z_b); 1 cylindrical (R, phi in [0, 2 pi), z) cells of PAPER.md:106
};
template <typename T>
struct ProjDev { T ca, sa, cb, sb, cg, sg; };

template <typename T>
struct IntegrateArgs {
    const PotDev* pots;        // [n_trials_total]
    const T* tab;              // anchor tables, all trials
    const T* tab0;             // W000 tables (MODE_DIAG), may be null
    const typename Vec2<T>::type* cs;  // [n_trials][n_steps+2] bar phase (one spare entry)
    const double* ics;         // [n_trials or 1][n_orb][6]
    long long ics_trial_stride;  // 0 if shared
    const ProjDev<T>* proj;    // [n_trials][n_proj]
    BinDev<T> bins;
    int trial0, n_proj;
    long long n_orb, n_steps;
    int stride, n_rec;
    T dt;
    unsigned* stage;           // [n_trials][n_hist][stage_orb_stride][n_rec], offset to this launch's first orbit
    long long stage_orb_stride;  // orbits per histogram block of the staging buffer (>= n_orb)
    float* stage_v;            // Gauss-Hermite mode (OBS variants): v_los of every staged LOSVD sample, [n_trials][n_proj][stride][n_rec*n_sym]; else null
    double* traj;              // [n_rec][n_orb][6] (MODE_TRAJ)
    double* diag;              // [n_orb][2] or null
    // work queue (see integrate_kernel): units = (segment of seg_len loop iterations) x (trial) x (group of `team` orbits)
    int* work;                 // [0] next unit; zeroed before the launch
    int* done;                 // [1 + gid] = segments completed by (trial, group) gid, zeroed before the launch.  (SMX_QUEUE_RING: [0] = tail of
                               // the ready ring, [1 + i] = the i-th unit of a later segment that became ready, seg * n_groups + gid, -1 before.)
    T* state;                  // [n_trials * n_grp][N_STATE][team] orbit state between segments
    int n_trials, n_grp, n_seg;
    long long seg_len;         // loop iterations per segment, a multiple of stride
    int team_warp;             // 1: a unit belongs to ONE WARP (32 orbits), warps never wait for one another; 0: to the whole CTA
    int table_in_smem;         // 1: the Ferrers anchor table of the unit's trial is staged in shared memory (CTA teams, or a
                               // single-trial launch); 0: read from global memory through L1 (warp teams with several trials)
    int* ctas_done;            // counter of finished CTAs (zeroed before the launch)
    const int* perm;           // orbit order of this launch (see order_*_kernel), [n_trials or 1][n_orb] indices within the trial; null = as given
    int* pace;                 // device flag read by zero_fill_kernel: 1 while an integrator runs (pace the fill), cleared by the
                               // last CTA of the launch (the fill then runs flat out); may be null
};
constexpr int N_STATE = 12;    // x y z vx vy vz lam1 lam2 lam3 | ej0 drift bad (MODE_DIAG)

// SYM4: fourfold symmetrisation; OBS: aperture map and / or cylindrical density cells.  Compile-time variants, so that the
// plain path pays nothing for them (config 0 records every step: the run-time checks alone cost it 20 %).
enum { MODE_LIBRARY = 0, MODE_TRAJ = 1, MODE_NOREC = 2, MODE_DIAG = 3, MODE_LIBRARY_SYM4 = 4, MODE_LIBRARY_OBS = 5, MODE_LIBRARY_SYM4_OBS = 6 };

__global__ void phase_table_kernel(const PotDev* pots, int trial0, long long n_steps, double dt, double2* cs64, float2* cs32) {
    long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k > n_steps + 1) return;
    const PotDev& P = pots[trial0 + blockIdx.y];
    // t_k = k*dt and theta = Omega_p*t_k + phase0 with individually rounded fp64 operations
    double t = __dmul_rn((double)k, dt);
    double th = __dadd_rn(__dmul_rn(P.omega_p, t), P.phase0);
    double s, c;
    sincos(th, &s, &c);
    long long o = blockIdx.y * (n_steps + 2) + k;
    if (cs64) cs64[o] = make_double2(c, s);
    if (cs32) cs32[o] = make_float2((float)c, (float)s);
}

// ---------------------------------------------------------------- orbit order of a launch (round 2, notes M)
// The 32 orbits of a warp share the lambda iteration's vote (a second iteration is taken while ANY lane still moves) and the warp's
// instruction stream, so a warp costs what its most demanding orbit costs.  Orbits that visit the centre need the second iteration
// (lambda changes by a good fraction of c^2 + lambda per step there); spread at random over the warps they made 60 % of all warp-steps
// pay for it.  The launch therefore hands the orbits to the warps in order of their specific ENERGY (orbits of one energy reach the same
// radii; measured against the initial radius, L_z and the Jacobi integral as the key, profiles/r2m.md): a counting sort of the ICs
// over ORD_NB equal energy intervals between the smallest and the largest finite energy of the trial, four tiny kernels in front of the
// integrator.  The energy is that of a stand-in potential -- the spherical and axisymmetric components as they are, a triaxial bar as a
// Plummer sphere of its mass and half-length -- in fp32: only the ORDER matters.  Orbits are independent and a lane's result never
// depends on its neighbours, so every row stays bit for bit what it was (tested); the order inside an interval is left to the atomics.
// Measured (profiles/r2m.md): config 2 fp64 integrator 45.4 -> 43.0 ms, fp32 25.4 -> 23.9, config 1 9.6 -> 8.8.
constexpr int ORD_NB = 4096;
__device__ float order_energy(const PotDev& P, const double* ic) {
    const float x = (float)ic[0], y = (float)ic[1], z = (float)ic[2], vx = (float)ic[3], vy = (float)ic[4], vz = (float)ic[5];
    const float R2 = x * x + y * y, r2 = R2 + z * z;
    float phi = 0.0f;
    for (int i = 0; i < P.n_comp; ++i) {
        const CompDev& c = P.comp[i];
        const float gm = (float)c.c[0];
        if (c.kind == K_PLUMMER) phi -= gm * rsqrtf(r2 + (float)c.c[1]);
        else if (c.kind == K_MN) { const float s = (float)c.c[1] + sqrtf(z * z + (float)c.c[2]); phi -= gm * rsqrtf(R2 + s * s); }
        else if (c.kind == K_NFW) { const float r = sqrtf(r2); phi -= r > 0.0f ? gm * log1pf(r * (float)c.c[1]) / r : gm * (float)c.c[1]; }
        else if (c.kind == K_FERRERS) phi -= (16.0f / 105.0f) * gm * rsqrtf(r2 + (float)c.c[1]);                    // K = 105 GM / 16, c[1] = a^2
        else phi -= gm * rsqrtf(r2 + (float)(c.c[1] * c.c[1] + c.c[3] * c.c[3]));                                  // needle bars: GM, scale a, half-length L
    }
    return 0.5f * (vx * vx + vy * vy + vz * vz) + phi;
}
// floats as integers of the same order (for atomicMin / atomicMax)
__device__ __forceinline__ int order_f2i(float f) { const int i = __float_as_int(f); return i >= 0 ? i : i ^ 0x7FFFFFFF; }
__device__ __forceinline__ float order_i2f(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7FFFFFFF); }
__device__ __forceinline__ int order_bucket(float e, const int* mm) {
    const float lo = order_i2f(mm[0]), hi = order_i2f(mm[1]);
    if (!(hi > lo) || !isfinite(e)) return ORD_NB - 1;          // one energy only / an orbit without a finite energy: the last interval
    return min(max((int)((e - lo) * ((float)(ORD_NB - 1) / (hi - lo))), 0), ORD_NB - 1);
}
// All three: grid (ceil(n_orb / 256), n_sets); set s = the ICs of trial trial0 + s (pot_per_set) or the shared ICs in the launch's first
// trial potential; ics_set_stride in doubles.  mm [n_sets][2] = {min, max} finite energy (order_f2i), initialised to {large, small}.
__global__ void order_minmax_kernel(const PotDev* pots, int trial0, const double* ics, long long ics_set_stride, long long n_orb, int* mm) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    int lo = 0x7F7F7F7F, hi = (int)0x80808080;
    if (i < n_orb) {
        const float e = order_energy(pots[trial0 + blockIdx.y], ics + blockIdx.y * ics_set_stride + i * 6);
        if (isfinite(e)) lo = hi = order_f2i(e);
    }
    lo = __reduce_min_sync(0xFFFFFFFFu, lo);
    hi = __reduce_max_sync(0xFFFFFFFFu, hi);
    if ((threadIdx.x & 31) == 0) { atomicMin(&mm[2 * blockIdx.y], lo); atomicMax(&mm[2 * blockIdx.y + 1], hi); }
}
// counts [n_sets][ORD_NB] zeroed by the caller
__global__ void order_count_kernel(const PotDev* pots, int trial0, const double* ics, long long ics_set_stride, long long n_orb, const int* mm,
                                   int* counts) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n_orb) return;
    const float e = order_energy(pots[trial0 + blockIdx.y], ics + blockIdx.y * ics_set_stride + i * 6);
    atomicAdd(&counts[blockIdx.y * ORD_NB + order_bucket(e, mm + 2 * blockIdx.y)], 1);
}
// <<<n_sets, 1024>>>: counts -> exclusive prefix sums, in place (four consecutive intervals per thread)
__global__ void __launch_bounds__(1024) order_scan_kernel(int* counts) {
    static_assert(ORD_NB == 4096, "four intervals per thread of a 1024-thread CTA");
    __shared__ int s[1024];
    const int i = threadIdx.x;
    int4* c4 = reinterpret_cast<int4*>(counts + blockIdx.x * ORD_NB) + i;
    const int4 own = *c4;
    const int sum = own.x + own.y + own.z + own.w;
    s[i] = sum;
    __syncthreads();
    for (int d = 1; d < 1024; d <<= 1) {
        const int v = i >= d ? s[i - d] : 0;
        __syncthreads();
        s[i] += v;
        __syncthreads();
    }
    const int base = s[i] - sum;
    *c4 = make_int4(base, base + own.x, base + own.x + own.y, base + own.x + own.y + own.z);
}
__global__ void order_scatter_kernel(const PotDev* pots, int trial0, const double* ics, long long ics_set_stride, long long n_orb, const int* mm,
                                     int* offsets, int* perm) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n_orb) return;
    const float e = order_energy(pots[trial0 + blockIdx.y], ics + blockIdx.y * ics_set_stride + i * 6);
    const int pos = atomicAdd(&offsets[blockIdx.y * ORD_NB + order_bucket(e, mm + 2 * blockIdx.y)], 1);
    perm[blockIdx.y * n_orb + pos] = (int)i;
}

// copy one trial's PotDev into shared memory in the kernel's arithmetic type; executed by a team of `tsize` threads
// (a warp or the CTA), `tl` = the thread's index in the team; the caller synchronises the team afterwards
template <typename T>
__device__ void load_pot(const PotDev& g, PotS<T>* s, const T* tab_global, const T* tab0_global, T* tab_smem, bool stage_table,
                         int tl, int tsize) {
    if (tl == 0) {
        s->n_comp = g.n_comp; s->has_rot = g.has_rot; s->has_ferrers = g.has_ferrers;
        s->pot_class = g.pot_class; s->i_mn = g.i_mn; s->i_nfw = g.i_nfw; s->i_fer = g.i_fer; s->i_v4 = g.i_v4;
        s->ft_key0 = sizeof(T) == 8 ? g.ft_key0 : g.ft32_key0; s->ft_nint = sizeof(T) == 8 ? g.ft_nint : g.ft32_nint;
        s->tab0 = tab0_global ? tab0_global + g.ft_off0 : nullptr;
    }
    for (int i = tl; i < MAX_COMP * 6; i += tsize) s->comp[i / 6].c[i % 6] = (T)g.comp[i / 6].c[i % 6];
    for (int i = tl; i < MAX_COMP; i += tsize) { s->comp[i].kind = g.comp[i].kind; s->comp[i].rotating = g.comp[i].rotating; }
    for (int i = tl; i < FT_NFUNC * FT_NFAR; i += tsize) s->far[i / FT_NFAR][i % FT_NFAR] = (T)g.far[i / FT_NFAR][i % FT_NFAR];
    const long long off = sizeof(T) == 8 ? g.ft_off64 : g.ft_off32;
    const T* src = tab_global + off;
    if (g.has_ferrers && stage_table) {
        const int n = (sizeof(T) == 8 ? g.ft_nint : g.ft32_nint) * FT<T>::ROW;
        for (int i = tl; i < n; i += tsize) tab_smem[i] = src[i];
        if (tl == 0) s->tab = tab_smem;
    } else if (tl == 0) {
        s->tab = src;
    }
}

template <typename T, bool OBS = false>
__device__ __forceinline__ unsigned bin3(const BinDev<T>& b, int o, T u0, T u1, T u2) {
    T w0 = (u0 - b.lo[o]) * b.inv[o], w1 = (u1 - b.lo[o + 1]) * b.inv[o + 1], w2 = (u2 - b.lo[o + 2]) * b.inv[o + 2];
    bool ok = (w0 >= (T)0) && (w0 < (T)b.n[o]) && (w1 >= (T)0) && (w1 < (T)b.n[o + 1]) && (w2 >= (T)0) && (w2 < (T)b.n[o + 2]);
    int j0 = (int)w0, j1 = (int)w1, j2 = (int)w2;  // truncation == floor for w >= 0
    // LOSVD (o=0): (iy*nx+ix)*nv+iv with (u0,u1,u2)=(X,Y,v);  density (o=3): (iz*dy+iy)*dx+ix with (x,y,z)
    unsigned idx = (o == 0) ? (unsigned)((j1 * b.n[0] + j0) * b.n[2] + j2) : (unsigned)((j2 * b.n[4] + j1) * b.n[3] + j0);
    if (OBS && o == 0 && b.ap_map && ok) {  // regroup the pixel into its aperture: cell = ap*nv + iv
        const int ap = __ldg(b.ap_map + j1 * b.n[0] + j0);
        ok = ap >= 0 && ap < b.n_ap;
        idx = (unsigned)(ap * b.n[2] + j2);
    }
    return ok ? idx : IDX_OUT;
}

// aperture of an image position (Gauss-Hermite mode: the velocity axis is not binned)
template <typename T>
__device__ __forceinline__ unsigned aperture_of(const BinDev<T>& b, T X, T Y) {
    T w0 = (X - b.lo[0]) * b.inv[0], w1 = (Y - b.lo[1]) * b.inv[1];
    bool ok = (w0 >= (T)0) && (w0 < (T)b.n[0]) && (w1 >= (T)0) && (w1 < (T)b.n[1]);
    int ap = -1;
    if (ok) ap = __ldg(b.ap_map + (int)w1 * b.n[0] + (int)w0);
    return (ap >= 0 && ap < b.n_ap) ? (unsigned)ap : IDX_OUT;
}

// Density cell of a bar-frame position, and of its (x,y) -> (-x,-y) mirror copy.  Cylindrical cells need one
// sqrt and one atan2 per SAMPLE: the copies of the fourfold symmetrisation share R, and their azimuth is phi +- pi.
template <typename T>
struct DensCoord { T u0, u1, m0, m1; };  // (x, y) or (R, phi) of the sample; the same for the mirrored copy
template <typename T, bool OBS>
__device__ __forceinline__ DensCoord<T> dens_coord(const BinDev<T>& b, T xb, T yb) {
    DensCoord<T> c{xb, yb, -xb, -yb};
    if (OBS && b.dens_mode == 1) {
        const T pi = (T)3.141592653589793238463;
        T phi = atan2(yb, xb);
        if (phi < (T)0) phi += (T)2 * pi;
        c.u0 = c.m0 = sqrt(xb * xb + yb * yb);
        c.u1 = phi;
        c.m1 = phi < pi ? phi + pi : phi - pi;
    }
    return c;
}

// Opaque copies: the value stays in a register instead of being re-read from the constant bank (kernel parameters)
// inside the time loop, where an LDC/LDCU + its latency sat on the critical path of every step.
__device__ __forceinline__ double keep(double v) { double o; asm volatile("mov.f64 %0, %1;" : "=d"(o) : "d"(v)); return o; }
__device__ __forceinline__ float keep(float v) { float o; asm volatile("mov.f32 %0, %1;" : "=f"(o) : "f"(v)); return o; }
__device__ __forceinline__ int keep(int v) { int o; asm volatile("mov.s32 %0, %1;" : "=r"(o) : "r"(v)); return o; }

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// spin load that does not touch the SM's L1: ld.acquire in a polling loop compiles to LDG.STRONG + CCTL.IVALL, an invalidation of
// the whole L1 per poll (measured: 11 million of them per config-2 launch, 78 million in the adaptive integrator)
__device__ __forceinline__ int ld_relaxed_gpu(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

// Persistent kernel, one CTA per SM.  The time loop of every group of orbits is cut into segments and the
// (segment, trial, group) units are handed out through an atomic counter, segment-major, so that every SM stays busy
// until the whole launch ends whatever the ratio of groups to SMs.  A unit belongs to a TEAM: one warp (32 orbits;
// a.team_warp) or the whole CTA.  With warp teams no warp ever waits for another one: a CTA-wide barrier per segment made
// the sixteen warps of a CTA idle until its slowest warp arrived (the lambda iteration count differs from warp to warp):
// 7 % of all warp cycles in barrier stalls plus the drained tail of every segment (profiles/r2a).  The CTA is then only
// the container that shares the potential constants and the Ferrers table in shared memory.
// A unit of segment s > 0 waits until segment s-1 of its group has been released by whichever team ran it; that team
// is running already (units are handed out in order and every CTA of the grid is resident), so the wait cannot deadlock.
// (SMX_QUEUE_RING = 1, the A/B alternative and the adaptive integrator's scheme: later segments are handed out through a ready ring.)
// Between segments the orbit state goes through a small L2-resident scratch buffer (96 B per orbit and segment).
// The CTA has up to 512 threads at no more than 120 registers each: 61 440 of the SM's 65 536 registers, which leaves room for one
// small co-resident CTA of zero_fill_kernel (128 threads x 32 registers), so that the output rows are zeroed WHILE the
// integrator runs (cudaMemsetAsync and device-to-device copies are SM kernels of the driver's own and cannot start beside a
// CTA that owns the whole register file: measured serialised, profiles/r2b).
// Hand-out order of the later segments.  0 (default): fixed segment-major order, a unit waits for its predecessor's flag (polled with a
// relaxed load: an acquire load in the polling loop flushed the SM's L1 on every poll).  1: a READY RING -- the team that finishes
// segment s of a group appends segment s+1 to a ring and teams take ring entries in order, so nobody ever holds a unit that is not
// ready.  The ring removes the waiting (a quarter of the slot time of the adaptive integrator, whose kernel uses it: rk32.cuh) but
// measured 10 % SLOWER here (config 2 fp64 51.3 against 46.5 ms, fp32 29.1 against 25.6, config 1 12.7 against 11.7; ncu: 849
// against 797 cycles per warp-step and a longer tail; the cause was not isolated): at four warps per scheduler a waiting warp
// costs its scheduler little, so there was little to gain here in the first place.
#ifndef SMX_QUEUE_RING
#define SMX_QUEUE_RING 0
#endif
#ifndef SMX_INTEGRATE_MAXTHREADS
#define SMX_INTEGRATE_MAXTHREADS 512
#endif
// The fp32 kernel needs ~100 registers: capped at 104 it leaves room for a 256-thread fill, which it takes to finish the fill
// within the (shorter) fp32 integration: beside it a 128-thread fill reaches only 2.4 TB/s whatever its pacing.
#ifndef SMX_INTEGRATE_MAXREGS
#define SMX_INTEGRATE_MAXREGS 120
#endif
#ifndef SMX_INTEGRATE_MAXREGS_F32
#define SMX_INTEGRATE_MAXREGS_F32 104
#endif
// SMALL: the instantiation for launches of at most SMX_INTEGRATE_SMALLTHREADS threads per CTA (fewer than ~38 000 orbits: one or two
// warps per scheduler, bound by the latency of a single instruction stream).  There the cap only costs: uncapped the compiler takes
// 218 (fp64) / 186 (fp32) registers and config 1 runs in 9.8 instead of 11.7 ms (128 registers: 10.7, 168: 10.3); 232 x 256
// threads still leave the SM room for the zero fill.
#ifndef SMX_INTEGRATE_SMALLTHREADS
#define SMX_INTEGRATE_SMALLTHREADS 256
#endif
#ifndef SMX_INTEGRATE_MAXREGS_SMALL
#define SMX_INTEGRATE_MAXREGS_SMALL 232
#endif
template <typename T, int MODE, int POT, bool SMALL = false>
__global__ void __maxnreg__(SMALL ? SMX_INTEGRATE_MAXREGS_SMALL : (sizeof(T) == 8 ? SMX_INTEGRATE_MAXREGS : SMX_INTEGRATE_MAXREGS_F32)) integrate_kernel(IntegrateArgs<T> a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int s_unit, s_unit2;
    __shared__ int s_wunit[SMX_INTEGRATE_MAXTHREADS / 32];   // the unit every warp team is working on (kept out of the registers across the time loop)
    const int tid = threadIdx.x, lane = tid & 31;
    const bool team_warp = a.team_warp != 0;
    const int B = team_warp ? 32 : (int)blockDim.x;    // team size
    const int tl = team_warp ? lane : tid;             // index in the team
    // potential constants: one slot per CTA, or per warp when warps of one CTA work on different trials
    constexpr int SLOT = ((sizeof(PotS<T>) + 15) / 16) * 16;
    const int n_slots = (team_warp && !a.table_in_smem) ? (int)(blockDim.x >> 5) : 1;
    PotS<T>* P = reinterpret_cast<PotS<T>*>(smem_raw + (size_t)SLOT * (n_slots > 1 ? (tid >> 5) : 0));
    T* tab_s = reinterpret_cast<T*>(smem_raw + (size_t)SLOT * n_slots);
    const int n_groups = a.n_trials * a.n_grp;
    const long long n_units = (long long)n_groups * a.n_seg;
    const int n_hist = a.n_proj + 1;
    constexpr int NSYM = (MODE == MODE_LIBRARY_SYM4 || MODE == MODE_LIBRARY_SYM4_OBS) ? 4 : 1;
    constexpr bool OBS = MODE == MODE_LIBRARY_OBS || MODE == MODE_LIBRARY_SYM4_OBS;
    const int nre = a.n_rec * NSYM;     // staged indices per orbit and histogram
    const long long hist_stride = a.stage_orb_stride * nre;
    const T dt = keep(a.dt), hdt = keep((T)0.5 * a.dt);
    const int n_steps = keep((int)a.n_steps), stride = keep(a.stride);
    int cur_trial = -1;
    if (team_warp && a.table_in_smem) {   // single-trial launch: constants and table staged once, by the whole CTA
        load_pot<T>(a.pots[a.trial0], P, a.tab, a.tab0, tab_s, true, tid, (int)blockDim.x);
        cur_trial = 0;
        __syncthreads();
    }

    for (;;) {
        // Position u in the hand-out order = the unit itself (segment-major), or with SMX_QUEUE_RING the position whose unit is
        // read from the ready ring once u is past the first segments.
        int u, unit;
        if (team_warp) {
            u = unit = 0;
            if (lane == 0) {
                u = unit = atomicAdd(a.work, 1);
                if (SMX_QUEUE_RING && u >= n_groups && u < n_units) {
                    const int* e = a.done + 1 + (u - n_groups);
                    while ((unit = ld_relaxed_gpu(e)) < 0) __nanosleep(64);
                    __threadfence();   // acquire: the predecessor's state (written before its release) is visible
                }
            }
            u = __shfl_sync(0xFFFFFFFFu, u, 0);
            unit = __shfl_sync(0xFFFFFFFFu, unit, 0);
        } else {
            __syncthreads();  // the previous unit is finished by every thread (s_unit, the table and P may be rewritten)
            if (tid == 0) {
                int uu = atomicAdd(a.work, 1), vv = uu;
                if (SMX_QUEUE_RING && uu >= n_groups && uu < n_units) {
                    const int* e = a.done + 1 + (uu - n_groups);
                    while ((vv = ld_relaxed_gpu(e)) < 0) __nanosleep(64);
                    __threadfence();
                }
                s_unit = uu; s_unit2 = vv;
            }
            __syncthreads();
            u = s_unit; unit = s_unit2;
        }
        if (u >= n_units) {
            // no more work for this team.  The last CTA to get here tells a concurrent zero fill that the SMs are free
            // (by then at most one unit per slot is still running).
            if (a.pace && tid == 0 && atomicAdd(a.ctas_done, 1) == (int)gridDim.x - 1) *(volatile int*)a.pace = 0;
            break;
        }
        if (team_warp) { if (lane == 0) s_wunit[tid >> 5] = unit; __syncwarp(); }
        const int seg = unit / n_groups, gid = unit - seg * n_groups;
        if (!SMX_QUEUE_RING && seg > 0) {   // A/B: fixed segment-major hand-out order, wait for the predecessor's flag
            if (tl == 0) { while (ld_relaxed_gpu(a.done + 1 + gid) < seg) __nanosleep(128); __threadfence(); }
            if (team_warp) __syncwarp(); else __syncthreads();
        }
        const int trial = gid / a.n_grp, grp = gid - trial * a.n_grp;
        const PotDev& G = a.pots[a.trial0 + trial];
        if (trial != cur_trial) {
            load_pot<T>(G, P, a.tab, a.tab0, tab_s, a.table_in_smem != 0, tl, B);
            cur_trial = trial;
            if (team_warp) __syncwarp(); else __syncthreads();
        }
        // every lane stays alive to the end (the lambda iteration votes across the warp): lanes past the last orbit
        // integrate a copy of the last orbit and write nothing.
        const long long orb_raw = (long long)grp * B + tl;
        const bool live = orb_raw < a.n_orb;
        long long orb = live ? orb_raw : a.n_orb - 1;
        if (a.perm) orb = a.perm[(a.ics_trial_stride ? (long long)trial * a.n_orb : 0) + orb];   // the launch's orbit order (order_*_kernel)
        const int k0 = (int)(seg * a.seg_len);
        const int k1 = (int)((k0 + a.seg_len < a.n_steps + 1) ? k0 + a.seg_len : a.n_steps + 1);
        T* st = a.state + (long long)gid * N_STATE * B + tl;

        T x, y, z, vx, vy, vz;
        // Ferrers lambda of the last three steps (warm start by quadratic extrapolation), < 0 = none yet
        float lam1 = -1.0f, lam2 = -1.0f, lam3 = -1.0f;
        double ej0 = 0.0, drift = 0.0, bad = 0.0;
        if (seg == 0) {
            const double* ic = a.ics + trial * a.ics_trial_stride + orb * 6;
            x = (T)ic[0]; y = (T)ic[1]; z = (T)ic[2]; vx = (T)ic[3]; vy = (T)ic[4]; vz = (T)ic[5];
        } else {
            x = __ldcg(st); y = __ldcg(st + B); z = __ldcg(st + 2 * B);
            vx = __ldcg(st + 3 * B); vy = __ldcg(st + 4 * B); vz = __ldcg(st + 5 * B);
            lam1 = (float)__ldcg(st + 6 * B); lam2 = (float)__ldcg(st + 7 * B); lam3 = (float)__ldcg(st + 8 * B);
            if (MODE == MODE_DIAG) { ej0 = __ldcg(st + 9 * B); drift = __ldcg(st + 10 * B); bad = __ldcg(st + 11 * B); }
        }
        const typename Vec2<T>::type* cs = a.cs + (long long)trial * (a.n_steps + 2);
        // seg_len is a multiple of stride, so the first iteration of a later segment is a recording one;
        // iteration 0 records nothing and applies no closing kick (hk = 0)
        int until_rec = k0 == 0 ? stride + 1 : 1;
        int rec = k0 == 0 ? 0 : k0 / stride - 1;
        T hk = k0 == 0 ? (T)0 : hdt;
        unsigned* stage = a.stage + ((long long)trial * n_hist * a.stage_orb_stride + orb) * nre;
        float* stage_v = (OBS && a.stage_v) ? a.stage_v + ((long long)trial * a.n_proj * a.stage_orb_stride + orb) * nre : nullptr;
        const ProjDev<T>* proj = a.proj + trial * a.n_proj;
        FerrersCtx<T, true> FB{};
        if (POT == POT_BARRED) {
            FB = make_ferrers_ctx<T, true>(*P, P->tab, P->comp[P->i_fer]);
            if (seg == 0) {  // every orbit starts from a cold solve at its initial position; the time loop is warm-only
                const typename Vec2<T>::type c0 = a.cs[(long long)trial * (a.n_steps + 2)];
                const T xb = fma_t(c0.x, x, c0.y * y), yb = fma_t(c0.x, y, -c0.y * x);
                lam1 = lam2 = lam3 = ferrers_lambda32(FB.fa2, FB.fb2, FB.fc2, (float)(xb * xb), (float)(yb * yb), (float)(z * z), -1.0f);
            }
        }

        // Kick-drift-kick with ONE force evaluation site: iteration k evaluates a = F(x_k, t_k), which closes step k
        // (v += dt/2 a), is recorded, and opens step k+1 (v += dt/2 a; x += dt v).  The opening kick and drift after
        // the last iteration (k = n_steps) are computed and never used; the phase table has one spare entry for it.
        typename Vec2<T>::type c = cs[k0];
        for (int k = k0; k < k1; ++k) {
            const typename Vec2<T>::type c_next = cs[k + 1];  // prefetch: hides the L1/L2 latency
            T ax, ay, az, phi = (T)0;
            // extrapolated lambda; once lambda has been clamped to 0 (inside the bar) the guess stays >= 0
            float lam = (POT == POT_BARRED || lam3 >= 0.0f) ? fmaxf(0.0f, 3.0f * (lam1 - lam2) + lam3)
                      : (lam2 >= 0.0f ? fmaxf(0.0f, 2.0f * lam1 - lam2) : lam1);
            total_force<T, MODE == MODE_DIAG, POT, true, POT != POT_BARRED>(*P, P->tab, FB, x, y, z, c.x, c.y, ax, ay, az, phi, lam);
            lam3 = lam2; lam2 = lam1; lam1 = lam;
            vx = fma_t(hk, ax, vx); vy = fma_t(hk, ay, vy); vz = fma_t(hk, az, vz);
            hk = hdt;
            if (MODE == MODE_DIAG && k == 0) ej0 = 0.5 * (vx * vx + vy * vy + vz * vz) + phi - G.omega_p * (x * vy - y * vx);
            if (--until_rec == 0) {
                until_rec = stride;
                if (MODE == MODE_TRAJ) {
                    if (live) {
                        double* o = a.traj + ((long long)rec * a.n_orb + orb) * 6;
                        o[0] = x; o[1] = y; o[2] = z; o[3] = vx; o[4] = vy; o[5] = vz;
                    }
                } else if (MODE != MODE_NOREC) {
                    // sample -> bar frame (inertial velocity on bar axes)
                    const T xb = c.x * x + c.y * y, yb = c.x * y - c.y * x;
                    const T ub = c.x * vx + c.y * vy, wb = c.x * vy - c.y * vx;
                    // copies of PAPER.md:77-90 Table 1 (n_sym = 4): (x,y,z;v) (x,y,-z;vx,vy,-vz) (-x,-y,z;-vx,-vy,vz) (-x,-y,-z;-v).
                    // A projection is linear, so copy (-,-) is minus copy (+,+) and copy (-,+) minus copy (+,-): two
                    // projections per sample give all four (slots: 0 = (+,+), 1 = (+,-), 2 = (-,+), 3 = (-,-)).
                    constexpr int n_half = NSYM == 4 ? 2 : 1;
                    const DensCoord<T> dc = dens_coord<T, OBS>(a.bins, xb, yb);
#pragma unroll
                    for (int m = 0; m < n_half; ++m) {
                        const T sz = m ? (T)-1 : (T)1;
                        const T zm = sz * z, vzm = sz * vz;
                        const int slot = rec * NSYM + m;
                        if (live) {
                            stage[(long long)a.n_proj * hist_stride + slot] = bin3<T>(a.bins, 3, dc.u0, dc.u1, zm);
                            if (NSYM == 4) stage[(long long)a.n_proj * hist_stride + slot + 2] = bin3<T>(a.bins, 3, dc.m0, dc.m1, zm);
                        }
                        for (int p = 0; p < a.n_proj; ++p) {
                            const ProjDev<T> R = proj[p];
                            // R = Rz(gamma) Rx(beta) Rz(alpha), Eq.1
                            T x1 = xb * R.ca - yb * R.sa, y1 = xb * R.sa + yb * R.ca;
                            T y2 = y1 * R.cb - zm * R.sb;
                            T X = x1 * R.cg - y2 * R.sg, Y = x1 * R.sg + y2 * R.cg;
                            T vlos = (ub * R.sa + wb * R.ca) * R.sb + vzm * R.cb;
                            if (OBS && stage_v) {  // Gauss-Hermite mode: stage (aperture, v_los) instead of the LOSVD cell
                                if (live) {
                                    stage[(long long)p * hist_stride + slot] = aperture_of<T>(a.bins, X, Y);
                                    stage_v[(long long)p * hist_stride + slot] = (float)vlos;
                                    if (NSYM == 4) {
                                        stage[(long long)p * hist_stride + rec * 4 + (3 - m)] = aperture_of<T>(a.bins, -X, -Y);
                                        stage_v[(long long)p * hist_stride + rec * 4 + (3 - m)] = (float)(-vlos);
                                    }
                                }
                            } else if (live) {
                                stage[(long long)p * hist_stride + slot] = bin3<T, OBS>(a.bins, 0, X, Y, vlos);
                                // minus this projection is the copy with all signs flipped: slot 3 for m = 0, slot 2 for m = 1
                                if (NSYM == 4) stage[(long long)p * hist_stride + rec * 4 + (3 - m)] = bin3<T, OBS>(a.bins, 0, -X, -Y, -vlos);
                            }
                        }
                    }
                    if (MODE == MODE_DIAG) {
                        double ej = 0.5 * (vx * vx + vy * vy + vz * vz) + phi - G.omega_p * (x * vy - y * vx);
                        if (isfinite(ej)) drift = fmax(drift, fabs(ej - ej0) / fabs(ej0)); else bad = 1.0;
                    }
                }
                ++rec;
            }
            vx = fma_t(hdt, ax, vx); vy = fma_t(hdt, ay, vy); vz = fma_t(hdt, az, vz);
            x = fma_t(dt, vx, x); y = fma_t(dt, vy, y); z = fma_t(dt, vz, z);
            c = c_next;
        }
        // what follows the time loop is recomputed from the unit number parked in shared memory: nothing of it occupies a register
        // inside the loop (the kernel sits at its register cap: every value carried across the loop is a spill inside it)
        const int unit_b = team_warp ? *(volatile int*)&s_wunit[tid >> 5] : *(volatile int*)&s_unit2;
        const int seg_b = unit_b / n_groups, gid_b = unit_b - seg_b * n_groups;
        T* st_b = a.state + (long long)gid_b * N_STATE * B + tl;
        if (seg_b + 1 < a.n_seg) {
            T* st = st_b;
            __stcg(st, x); __stcg(st + B, y); __stcg(st + 2 * B, z);
            __stcg(st + 3 * B, vx); __stcg(st + 4 * B, vy); __stcg(st + 5 * B, vz);
            __stcg(st + 6 * B, (T)lam1); __stcg(st + 7 * B, (T)lam2); __stcg(st + 8 * B, (T)lam3);
            if (MODE == MODE_DIAG) { __stcg(st + 9 * B, (T)ej0); __stcg(st + 10 * B, (T)drift); __stcg(st + 11 * B, (T)bad); }
            if (team_warp) __syncwarp(); else __syncthreads();
            if (tl == 0) {   // release the state, then publish the group's next segment as ready
                __threadfence();
                if (SMX_QUEUE_RING) {
                    const int t = atomicAdd(a.done, 1);
                    st_release_gpu(a.done + 1 + t, unit_b + n_groups);
                } else {
                    st_release_gpu(a.done + 1 + gid_b, seg_b + 1);
                }
            }
        } else {
            if (MODE == MODE_NOREC && live) {  // keep the integration alive without the recording path
                stage[0] = __float_as_uint((float)(x + y + z + vx + vy + vz));
            }
            if (MODE == MODE_DIAG && a.diag && live) { a.diag[2 * orb] = drift; a.diag[2 * orb + 1] = bad; }
        }
    }
}

}  // namespace smx
