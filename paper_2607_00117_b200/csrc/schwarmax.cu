// schwarmax.cu -- C-ABI entry points of libschwarmax.so (see include/schwarmax.h).
// Host side: argument validation, per-potential table construction, launches.  No CPU fallback:
// every step of the path runs in the kernels of kernels.cuh / rowbuild.cuh.
#include "../../include/schwarmax.h"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <mutex>
#include <string>
#include <vector>

#include "rowbuild.cuh"
#include "rk32.cuh"
#include "weights.cuh"

using namespace smx;

namespace {

thread_local std::string g_err;
std::atomic<long long> g_launches{0};
// debug flags belong to the calling HOST THREAD (a process may drive several GPUs from several threads)
thread_local int t_flags = 0;
struct ThreadFlags {
    int load() const { return t_flags; }
    int exchange(int f) { const int o = t_flags; t_flags = f; return o; }
} g_flags;

int fail(int code, const std::string& msg) { g_err = msg; return code; }
#define CUDA_TRY(expr)                                                                         \
    do {                                                                                       \
        cudaError_t e_ = (expr);                                                               \
        if (e_ != cudaSuccess) return fail(SM_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_)); \
    } while (0)

const double PI = 3.14159265358979323846;

}  // namespace

struct sm_potential {
    int n_trials = 0;
    std::vector<PotDev> host;
    std::vector<FerrersTable> tables;  // one per trial with a Ferrers component (else empty table)
    PotDev* d_pots = nullptr;
    double* d_tab64 = nullptr;   // anchors [trial][interval][ROW]
    double* d_tab0 = nullptr;    // W000    [trial][interval][FT_NC0]
    float* d_tab32 = nullptr;    // anchors fp32
    size_t max_tab_elems64 = 0, max_tab_elems32 = 0;  // largest single-trial table (elements)
};

namespace {

int convert_desc(const sm_potential_desc& d, PotDev* out, FerrersTable* table) {
    if (d.n_comp < 1 || d.n_comp > MAX_COMP) return fail(SM_ERR_INVALID_ARG, "n_comp must be in [1,8]");
    if (!std::isfinite(d.G) || !(d.G > 0)) return fail(SM_ERR_INVALID_ARG, "G must be positive");
    if (!std::isfinite(d.omega_p) || !std::isfinite(d.phase0)) return fail(SM_ERR_INVALID_ARG, "omega_p/phase0 not finite");
    PotDev P{};
    P.omega_p = d.omega_p; P.phase0 = d.phase0; P.n_comp = d.n_comp;
    int n_ferrers = 0;
    for (int i = 0; i < d.n_comp; ++i) {
        const sm_component& c = d.comp[i];
        CompDev& o = P.comp[i];
        o.kind = c.kind; o.rotating = c.rotating != 0;
        if (o.rotating) P.has_rot = 1;
        for (int j = 0; j < 4; ++j)
            if (!std::isfinite(c.p[j])) return fail(SM_ERR_INVALID_ARG, "component parameter not finite");
        switch (c.kind) {
            case SM_PLUMMER:
                if (!(c.p[0] >= 0) || !(c.p[1] >= 0)) return fail(SM_ERR_INVALID_ARG, "Plummer needs M>=0, b>=0");
                o.c[0] = d.G * c.p[0]; o.c[1] = c.p[1] * c.p[1];
                break;
            case SM_MIYAMOTO_NAGAI:
                if (!(c.p[0] >= 0) || !(c.p[1] >= 0) || !(c.p[2] > 0)) return fail(SM_ERR_INVALID_ARG, "Miyamoto-Nagai needs M>=0, a>=0, b>0");
                o.c[0] = d.G * c.p[0]; o.c[1] = c.p[1]; o.c[2] = c.p[2] * c.p[2];
                break;
            case SM_NFW:
                if (!(c.p[0] >= 0) || !(c.p[1] > 0)) return fail(SM_ERR_INVALID_ARG, "NFW needs rho_s>=0, r_s>0");
                o.c[0] = d.G * 4.0 * PI * c.p[0] * c.p[1] * c.p[1] * c.p[1]; o.c[1] = 1.0 / c.p[1]; o.c[2] = c.p[1];
                break;
            case SM_FERRERS2: {
                if (!(c.p[0] >= 0) || !(c.p[1] > c.p[2] && c.p[2] > c.p[3] && c.p[3] > 0))
                    return fail(SM_ERR_INVALID_ARG, "Ferrers needs M>=0 and axes a>b>c>0");
                if (++n_ferrers > 1) return fail(SM_ERR_UNSUPPORTED, "at most one Ferrers component per potential");
                if (!build_ferrers_table(c.p[1], c.p[2], c.p[3], table))
                    return fail(SM_ERR_INVALID_ARG, "Ferrers table construction failed (degenerate axes?)");
                if (table->fit_err > 1e-14) return fail(SM_ERR_UNSUPPORTED, "Ferrers table accuracy not reached");
                o.c[0] = 105.0 * d.G * c.p[0] / 16.0;
                o.c[1] = table->a2; o.c[2] = table->b2; o.c[3] = table->c2;
                o.c[4] = table->a2 - table->b2; o.c[5] = table->a2 - table->c2;
                P.has_ferrers = 1; P.ft_key0 = table->key0_64; P.ft_nint = table->n_int64;
                P.ft32_key0 = table->key0_32; P.ft32_nint = table->n_int32;
                for (int f = 0; f < FT_NFUNC; ++f) for (int m = 0; m < FT_NFAR; ++m) P.far[f][m] = table->far[f][m];
                break;
            }
            case SM_DEHNEN_T3:
            case SM_DEHNEN_V4:
                // {GM, a, b^2, L, (1+eta)/(2L), eta/L^2}; the needle lies along the component's x axis
                if (!std::isfinite(c.p[4]) || !(c.p[0] >= 0) || !(c.p[1] >= 0) || !(c.p[2] > 0) || !(c.p[3] > 0) || !(c.p[4] >= -1 && c.p[4] <= 1))
                    return fail(SM_ERR_INVALID_ARG, "Dehnen-Aly bar needs M>=0, a>=0, b>0, L>0, -1<=eta<=1");
                o.c[0] = d.G * c.p[0]; o.c[1] = c.p[1]; o.c[2] = c.p[2] * c.p[2]; o.c[3] = c.p[3]; o.c[4] = (1.0 + c.p[4]) / (2.0 * c.p[3]); o.c[5] = c.p[4] / (c.p[3] * c.p[3]);
                break;
            default: return fail(SM_ERR_INVALID_ARG, "unknown component kind");
        }
    }
    // classify for the specialised kernels
    P.pot_class = POT_GENERIC; P.i_mn = P.i_nfw = P.i_fer = -1;
    if (d.n_comp == 1 && P.comp[0].kind == K_PLUMMER && !P.comp[0].rotating) P.pot_class = POT_PLUMMER;
    if (d.n_comp == 3) {
        for (int i = 0; i < 3; ++i) {
            if (P.comp[i].kind == K_MN && !P.comp[i].rotating) P.i_mn = i;
            if (P.comp[i].kind == K_NFW && !P.comp[i].rotating) P.i_nfw = i;
            if (P.comp[i].kind == K_FERRERS && P.comp[i].rotating) P.i_fer = i;
        }
        if (P.i_mn >= 0 && P.i_nfw >= 0 && P.i_fer >= 0) P.pot_class = POT_BARRED;
    }
    P.i_v4 = -1;
    if (d.n_comp == 4) {  // the paper's stellar model: sloped T_3 long bar + uniform V_4 bulge
        for (int i = 0; i < 4; ++i) {
            if (P.comp[i].kind == K_MN && !P.comp[i].rotating) P.i_mn = i;
            if (P.comp[i].kind == K_NFW && !P.comp[i].rotating) P.i_nfw = i;
            if (P.comp[i].kind == K_DEHNEN_T3 && P.comp[i].rotating && P.comp[i].c[5] != 0.0) P.i_fer = i;
            if (P.comp[i].kind == K_DEHNEN_V4 && P.comp[i].rotating && P.comp[i].c[5] == 0.0) P.i_v4 = i;
        }
        if (P.i_mn >= 0 && P.i_nfw >= 0 && P.i_fer >= 0 && P.i_v4 >= 0) P.pot_class = POT_NEEDLE;
    }
    *out = P;
    return SM_OK;
}

template <typename T>
size_t pot_smem_bytes(const sm_potential* p) {
    size_t tab = sizeof(T) == 8 ? p->max_tab_elems64 * 8 : p->max_tab_elems32 * 4;
    return ((sizeof(PotS<T>) + 15) / 16) * 16 + tab;
}

}  // namespace

extern "C" {

int sm_make_potential_batch(const sm_potential_desc* desc, int n_trials, sm_potential** out) {
    if (!desc || !out || n_trials < 1) return fail(SM_ERR_INVALID_ARG, "null descriptor/output or n_trials < 1");
    sm_potential* p = new sm_potential;
    p->n_trials = n_trials;
    p->host.resize(n_trials);
    p->tables.resize(n_trials);
    std::vector<double> t64, t0;
    std::vector<float> t32;
    for (int t = 0; t < n_trials; ++t) {
        int rc = convert_desc(desc[t], &p->host[t], &p->tables[t]);
        if (rc != SM_OK) { delete p; return rc; }
        PotDev& P = p->host[t];
        P.ft_off64 = (long long)t64.size();
        P.ft_off32 = (long long)t32.size();
        P.ft_off0 = (long long)t0.size();
        if (P.has_ferrers) {
            const FerrersTable& T = p->tables[t];
            t64.insert(t64.end(), T.rows64.begin(), T.rows64.end());
            t0.insert(t0.end(), T.coef0.begin(), T.coef0.end());
            t32.insert(t32.end(), T.rows32.begin(), T.rows32.end());
            p->max_tab_elems64 = std::max(p->max_tab_elems64, T.rows64.size());
            p->max_tab_elems32 = std::max(p->max_tab_elems32, T.rows32.size());
        }
    }
    auto cleanup = [&](int code, const std::string& m) { sm_free_potential(p); return fail(code, m); };
    if (cudaMalloc(&p->d_pots, sizeof(PotDev) * n_trials) != cudaSuccess) return cleanup(SM_ERR_NOMEM, "cudaMalloc(pots) failed (no CUDA device?)");
    if (cudaMemcpy(p->d_pots, p->host.data(), sizeof(PotDev) * n_trials, cudaMemcpyHostToDevice) != cudaSuccess) return cleanup(SM_ERR_CUDA, "upload of potentials failed");
    if (!t64.empty()) {
        if (cudaMalloc(&p->d_tab64, t64.size() * 8) != cudaSuccess || cudaMalloc(&p->d_tab0, t0.size() * 8) != cudaSuccess ||
            cudaMalloc(&p->d_tab32, t32.size() * 4) != cudaSuccess) return cleanup(SM_ERR_NOMEM, "cudaMalloc(tables) failed");
        if (cudaMemcpy(p->d_tab64, t64.data(), t64.size() * 8, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(p->d_tab0, t0.data(), t0.size() * 8, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(p->d_tab32, t32.data(), t32.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) return cleanup(SM_ERR_CUDA, "upload of tables failed");
    }
    *out = p;
    return SM_OK;
}

int sm_make_potential(const sm_potential_desc* desc, sm_potential** out) { return sm_make_potential_batch(desc, 1, out); }

void sm_free_potential(sm_potential* p) {
    if (!p) return;
    cudaFree(p->d_pots); cudaFree(p->d_tab64); cudaFree(p->d_tab0); cudaFree(p->d_tab32);
    delete p;
}

const char* sm_last_error(void) { return g_err.c_str(); }
int sm_version(void) { return 100; }
int64_t sm_launch_count(void) { return (int64_t)g_launches.load(); }
int sm_set_debug_flags(int flags) { return g_flags.exchange(flags); }

}  // extern "C"

#include "api_build.inc"
#ifndef SMX_VARIANT_BUILD
#include "api_weights.inc"
#include "api_rk32.inc"
#endif

// ------------------------------------------------------------------------------------------------------------------------
// sm_stage_library_noalloc: rows a-1..a-6 for callers that may not allocate (CUDA graph capture, tight serving loops, harnesses
// that forbid cudaMalloc).  It is sm_stage_library_batch for ONE trial of a potential with every byte of the integrator's
// scratch -- the work-queue counters and ready ring, the projection constants, the bar-phase table and the orbit state that travels between
// segments of the persistent queue -- in ONE file-scope device array of a fixed, modest size, which every GPU that loads the
// library holds until the process exits.  No cudaMalloc / cudaMallocAsync / cudaFree, no memory pool, no event or stream
// creation, no host-to-device copy: a small set-up kernel and a memset node write the scratch, then the same phase_table_kernel
// and integrate_kernel<T, MODE_LIBRARY, POT> as the pooled path run on it, so the staged indices are the same bit for bit.
//
// In HOST code the name of a __device__ array is a host-side stand-in, not a device address (a kernel handed &g_noalloc_scratch
// faults, or silently uses host memory where the GPU can reach it): the device address comes from cudaGetSymbolAddress, looked up
// in this translation unit, once per device, with that device current (noalloc_scratch_ptr).
//
// Every call on a device shares the array and finds the previous call's contents in it: the counters are cleared by every call
// (the rest is fully overwritten before it is read); calls that OVERLAP on one GPU -- two streams, two host threads -- race.
constexpr long long NOALLOC_MAX_ORB = SM_NOALLOC_MAX_ORB;       // 32 768 orbits per call
constexpr long long NOALLOC_MAX_STEPS = SM_NOALLOC_MAX_STEPS;   // 65 534 steps per call (a phase table of 65 536 entries)
constexpr size_t NOALLOC_INT_BYTES = 131072;                    // [0] unit counter, [1] finished CTAs, [3 ..] segment flags of <= 1024 warp groups (or the ready ring: <= 25 later segments each)
constexpr size_t NOALLOC_PROJ_BYTES = 256;                      // <= 4 projections x 6 x 8 B
constexpr size_t NOALLOC_CS_BYTES = (size_t)(NOALLOC_MAX_STEPS + 2) * sizeof(double2);     // 1 MiB
constexpr size_t NOALLOC_STATE_BYTES = (size_t)NOALLOC_MAX_ORB * N_STATE * sizeof(double);  // 3 MiB
constexpr size_t NOALLOC_SCRATCH_BYTES = NOALLOC_INT_BYTES + NOALLOC_PROJ_BYTES + NOALLOC_CS_BYTES + NOALLOC_STATE_BYTES;
static_assert(NOALLOC_SCRATCH_BYTES == SM_NOALLOC_SCRATCH_BYTES, "include/schwarmax.h states the size of the static scratch");
static_assert((3 + 25 * ((NOALLOC_MAX_ORB + 31) / 32)) * sizeof(int) <= NOALLOC_INT_BYTES, "ready ring of the largest call");
static_assert(MAX_PROJ * sizeof(ProjDev<double>) <= NOALLOC_PROJ_BYTES, "projection constants of the largest call");

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

namespace {

// device address of g_noalloc_scratch on the CURRENT device; looked up once per device
int noalloc_scratch_ptr(unsigned char** out) {
    static unsigned char* ptrs[64];
    static std::mutex mu;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(SM_ERR_UNSUPPORTED, "device ordinal >= 64");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        unsigned char* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p)
            return fail(SM_ERR_CUDA, std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(e));
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return SM_OK;
}

template <typename T> struct ProjPack { ProjDev<T> p[MAX_PROJ]; };

// clears the queue counters and writes the projection constants (kernel arguments: no host-to-device copy)
template <typename T>
__global__ void noalloc_setup_kernel(int* ints, int n_ints, ProjDev<T>* proj, ProjPack<T> pack, int n_proj) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_ints) ints[i] = (i < 3 || !SMX_QUEUE_RING) ? 0 : -1;   // counters and segment flags 0 (ready ring: empty)
    if (i < n_proj) proj[i] = pack.p[i];
}

template <typename T, int POT>
int stage_noalloc_pot(const sm_potential* pot, int trial, const double* d_ics, long long n_orb, double dt, long long n_steps,
                      int stride, const sm_projection* proj, int n_proj, const sm_grids* g, unsigned* d_stage, cudaStream_t st) {
    if constexpr (!kernel_enabled<T, MODE_LIBRARY, POT>()) return fail(SM_ERR_UNSUPPORTED, "kernel not part of this variant build");
    else {
    typedef typename Vec2<T>::type T2;
    unsigned char* base = nullptr;
    int rc = noalloc_scratch_ptr(&base);
    if (rc != SM_OK) return rc;
    int* d_ints = reinterpret_cast<int*>(base);
    ProjDev<T>* d_proj = reinterpret_cast<ProjDev<T>*>(base + NOALLOC_INT_BYTES);
    T2* d_cs = reinterpret_cast<T2*>(base + NOALLOC_INT_BYTES + NOALLOC_PROJ_BYTES);
    T* d_state = reinterpret_cast<T*>(base + NOALLOC_INT_BYTES + NOALLOC_PROJ_BYTES + NOALLOC_CS_BYTES);

    // launch shape, segments and shared memory exactly as launch_integrate_pot picks them for a single-trial launch
    const LaunchShape sh = pick_shape(n_orb, 1, true, false);
    constexpr size_t SLOT = ((sizeof(PotS<T>) + 15) / 16) * 16;
    const size_t smem = SLOT + (sizeof(T) == 8 ? pot->max_tab_elems64 * 8 : pot->max_tab_elems32 * 4);
    if (smem + 1024 > SMEM_OPTIN_MAX) return fail(SM_ERR_UNSUPPORTED, "potential tables exceed shared memory");
    const long long n_groups = sh.n_grp, slots = (long long)sh.grid * (sh.block / 32), iters = n_steps + 1;
    long long n_seg = 1;
    if (n_groups > slots) n_seg = ((long long)SEGMENTS_PER_SLOT * slots + n_groups - 1) / n_groups;
    long long seg_len = (iters + n_seg - 1) / n_seg;
    seg_len = std::max<long long>(seg_len, std::max<long long>(32LL * stride, 256));
    seg_len = (seg_len + stride - 1) / stride * stride;
    n_seg = (iters + seg_len - 1) / seg_len;
    if ((size_t)(3 + n_groups * std::max<long long>(n_seg - 1, 1)) * sizeof(int) > NOALLOC_INT_BYTES || (size_t)n_groups * N_STATE * 32 * sizeof(T) > NOALLOC_STATE_BYTES ||
        sizeof(T2) * (size_t)(n_steps + 2) > NOALLOC_CS_BYTES)
        return fail(SM_ERR_UNSUPPORTED, "sm_stage_library_noalloc: call exceeds the static scratch");  // unreachable within the stated limits

    ProjPack<T> pack{};
    for (int i = 0; i < n_proj; ++i)   // formed in fp64, then cast to T, as stage_orbits does
        pack.p[i] = ProjDev<T>{(T)std::cos(proj[i].alpha), (T)std::sin(proj[i].alpha), (T)std::cos(proj[i].beta),
                               (T)std::sin(proj[i].beta), (T)std::cos(proj[i].gamma), (T)std::sin(proj[i].gamma)};
    const int n_ints = (int)(3 + n_groups * std::max<long long>(n_seg - 1, 1));
    noalloc_setup_kernel<T><<<(n_ints + 255) / 256, 256, 0, st>>>(d_ints, n_ints, d_proj, pack, n_proj);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    phase_table_kernel<<<dim3((unsigned)((n_steps + 2 + 255) / 256), 1), 256, 0, st>>>(
        pot->d_pots, trial, n_steps, dt, sizeof(T) == 8 ? (double2*)d_cs : nullptr, sizeof(T) == 4 ? (float2*)d_cs : nullptr);
    g_launches++;
    CUDA_TRY(cudaGetLastError());

    IntegrateArgs<T> a{};
    a.pots = pot->d_pots;
    a.tab = sizeof(T) == 8 ? (const T*)pot->d_tab64 : (const T*)pot->d_tab32;
    a.tab0 = sizeof(T) == 8 ? (const T*)pot->d_tab0 : nullptr;
    a.cs = d_cs;
    a.trial0 = trial; a.n_proj = n_proj; a.n_steps = n_steps; a.stride = stride; a.n_rec = (int)(n_steps / stride); a.dt = (T)dt;
    a.ics = d_ics; a.ics_trial_stride = 0; a.n_orb = n_orb;
    a.stage = d_stage; a.stage_orb_stride = n_orb;
    a.proj = d_proj;
    const double lo[6] = {g->x0, g->y0, g->v0, g->bx0, g->by0, g->bz0}, hi[6] = {g->x1, g->y1, g->v1, g->bx1, g->by1, g->bz1};
    const int nb[6] = {g->nx, g->ny, g->nv, g->dx, g->dy, g->dz};
    for (int i = 0; i < 6; ++i) { a.bins.lo[i] = (T)lo[i]; a.bins.inv[i] = (T)(nb[i] / (hi[i] - lo[i])); a.bins.n[i] = nb[i]; }
    a.n_trials = 1; a.n_grp = (int)sh.n_grp; a.n_seg = (int)n_seg; a.seg_len = seg_len;
    a.team_warp = 1; a.table_in_smem = 1;
    a.work = d_ints; a.ctas_done = d_ints + 1; a.done = d_ints + 2;
    a.pace = nullptr;   // no zero fill runs beside this launch
    a.state = d_state;
    // the same instantiation as the pooled path picks for this size (launch_integrate_pot)
    const cudaError_t e = sh.block <= SMX_INTEGRATE_SMALLTHREADS
        ? launch_integrate_kernel<T, MODE_LIBRARY, POT, true>(a, sh, smem, (int)cudaSharedmemCarveoutMaxShared, st)
        : launch_integrate_kernel<T, MODE_LIBRARY, POT, false>(a, sh, smem, (int)cudaSharedmemCarveoutMaxShared, st);
    g_launches++;
    if (e != cudaSuccess) return fail(SM_ERR_CUDA, std::string("integrate_kernel launch: ") + cudaGetErrorString(e));
    return SM_OK;
    }
}

template <typename T>
int stage_noalloc(const sm_potential* pot, int trial, const double* d_ics, long long n_orb, double dt, long long n_steps, int stride,
                  const sm_projection* proj, int n_proj, const sm_grids* g, unsigned* d_stage, cudaStream_t st) {
    switch (pot->host[trial].pot_class) {
        case POT_BARRED: return stage_noalloc_pot<T, POT_BARRED>(pot, trial, d_ics, n_orb, dt, n_steps, stride, proj, n_proj, g, d_stage, st);
        case POT_PLUMMER: return stage_noalloc_pot<T, POT_PLUMMER>(pot, trial, d_ics, n_orb, dt, n_steps, stride, proj, n_proj, g, d_stage, st);
        case POT_NEEDLE: return stage_noalloc_pot<T, POT_NEEDLE>(pot, trial, d_ics, n_orb, dt, n_steps, stride, proj, n_proj, g, d_stage, st);
        default: return stage_noalloc_pot<T, POT_GENERIC>(pot, trial, d_ics, n_orb, dt, n_steps, stride, proj, n_proj, g, d_stage, st);
    }
}

}  // namespace

extern "C" int sm_stage_library_noalloc(const sm_potential* pot, int trial, const double* d_ics, int64_t n_orb, double dt,
                                        int64_t n_steps, int32_t stride, const sm_projection* proj, int n_proj, const sm_grids* g,
                                        int precision, uint32_t* d_stage, void* cuda_stream) {
    int rc = check_common(pot, trial, 1, d_ics, n_orb, dt, n_steps, stride, precision);
    if (rc != SM_OK) return rc;
    if ((rc = check_grids(g)) != SM_OK) return rc;
    if (!proj || n_proj < 1 || n_proj > MAX_PROJ) return fail(SM_ERR_INVALID_ARG, "need 1..4 projections");
    if (n_orb > NOALLOC_MAX_ORB)
        return fail(SM_ERR_UNSUPPORTED, "sm_stage_library_noalloc: n_orb = " + std::to_string((long long)n_orb) + " exceeds SM_NOALLOC_MAX_ORB = " +
                                            std::to_string(NOALLOC_MAX_ORB) + " (the static scratch holds no more: call per orbit range, or use sm_stage_library_batch)");
    if (n_steps > NOALLOC_MAX_STEPS)
        return fail(SM_ERR_UNSUPPORTED, "sm_stage_library_noalloc: n_steps = " + std::to_string((long long)n_steps) + " exceeds SM_NOALLOC_MAX_STEPS = " +
                                            std::to_string(NOALLOC_MAX_STEPS) + " (the static scratch holds no longer a phase table: use sm_stage_library_batch)");
    if (!d_stage && n_orb > 0 && n_steps / stride > 0) return fail(SM_ERR_INVALID_ARG, "null d_stage");
    if (n_orb == 0) return SM_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (precision == SM_F64) return stage_noalloc<double>(pot, trial, d_ics, n_orb, dt, n_steps, stride, proj, n_proj, g, d_stage, st);
    return stage_noalloc<float>(pot, trial, d_ics, n_orb, dt, n_steps, stride, proj, n_proj, g, d_stage, st);
}
