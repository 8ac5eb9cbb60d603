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
