// weights.cuh -- kernels of the orbital-weight solve (include/schwarmax.h sm_solve_weights).
//
// ADMM for Q(w) = 1/2 ||U w - y||^2 + 1/2 sum d_i w_i^2, w >= 0, with n_rhs data vectors sharing one U:
//   G = U^T U + diag(d + rho)            one fp64 GEMM on the assembled, scaled U^T              (gemm_f64_kernel)
//   K = G^-1                             in-place symmetric block sweep (Gauss-Jordan on the lower triangle), 128-wide pivot
//                                        blocks: the pivot block is inverted by one CTA, the rest is rank-128 GEMM updates
//   per iteration  X = R K^T             one split-K GEMM (n_rhs x n_orb x n_orb) -- the dominant kernel --
//                  z, u, R updates       fused into the reduction of the split-K partial sums       (admm_update_kernel)
// The x-update is a dense contraction, but an fp64 one (the iteration has to reproduce the paper-order fp64 oracle to
// 1e-9), so it runs on the FP64 FMA pipe, not on tcgen05 (no fp64 MMA there): register-tiled
// 128 x 128 x 16 CTA tiles, 8 x 8 accumulators per thread, operands staged through shared memory with 16-byte loads laid
// out so that every LDS.128 of a warp touches one 128-byte (B) or 64-byte (A) line.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace smx {

constexpr int GM = 128, GN = 128, GK = 16;
constexpr int GPITCH = GM + 2;   // doubles: rows stay 16-byte aligned and the transposing stores of a warp hit 16 distinct 8-byte banks
constexpr int GJ_NB = 128;       // pivot block of the inversion

struct GemmArgs {
    const double* A; long long lda;   // A[m][k]
    const double* B; long long ldb;   // B_KMAJOR: B[n][k], else B[k][n]
    double* C; long long ldc;         // C[m][n] = alpha * sum_k A B + beta * C   (beta == 0: C is not read)
    int M, N, K;
    double alpha, beta;
    int split_k;                      // > 1: CTA z sums k in [z*k_chunk, (z+1)*k_chunk) and writes alpha * partial to C + z*c_split
    int k_chunk;                      // multiple of GK
    long long c_split;
    int lower_only;                   // != 0: only tiles that hold elements with m >= n are computed (symmetric results)
};

constexpr int GEMM_SMEM_BYTES = 2 * 2 * GK * GPITCH * (int)sizeof(double);   // two stages of an A and a B tile

// One 16-deep k-tile for the JM leading 8-row bands of this warp (JM is warp-uniform; a full tile is JM = 4).  Branch-free,
// so that the shared-memory loads of step kk+1 can be scheduled under the FMAs of step kk.
template <int JM>
__device__ __forceinline__ void gemm_tile(const double* __restrict__ As, const double* __restrict__ Bs, int row_base,
                                          int col_base, double (&acc)[8][8]) {
#pragma unroll
    for (int kk = 0; kk < GK; ++kk) {
        double a[2 * JM], b[8];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const double2 v = *reinterpret_cast<const double2*>(Bs + kk * GPITCH + col_base + j * 16);
            b[2 * j] = v.x; b[2 * j + 1] = v.y;
        }
#pragma unroll
        for (int j = 0; j < JM; ++j) {
            const double2 v = *reinterpret_cast<const double2*>(As + kk * GPITCH + row_base + j * 32);
            a[2 * j] = v.x; a[2 * j + 1] = v.y;
        }
#pragma unroll
        for (int i = 0; i < 2 * JM; ++i)
#pragma unroll
            for (int c = 0; c < 8; ++c) acc[i][c] = fma(a[i], b[c], acc[i][c]);
    }
}

template <bool B_KMAJOR>
__global__ void __launch_bounds__(256) gemm_f64_kernel(GemmArgs g) {
    extern __shared__ __align__(16) double gemm_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int wr = warp >> 1, wc = warp & 1, ty = lane >> 3, tx = lane & 7;
    const int m0 = blockIdx.y * GM, n0 = blockIdx.x * GN;
    if (g.lower_only && blockIdx.x > blockIdx.y) return;
    int kbeg = 0, kend = g.K;
    if (g.split_k > 1) { kbeg = blockIdx.z * g.k_chunk; kend = min(g.K, kbeg + g.k_chunk); }
    // rows of this thread: j*32 + wr*8 + ty*2 + {0,1}; columns: wc*64 + j*16 + tx*2 + {0,1}   (j = 0..3)
    const int row_base = wr * 8 + ty * 2, col_base = wc * 64 + tx * 2;
    // row bands j whose 8 rows of this warp lie entirely past M do no work (n_rhs = 100 on a 128-row tile)
    int jmax = 0;
    for (int j = 0; j < 4; ++j) if (m0 + j * 32 + wr * 8 < g.M) jmax = j + 1;

    // beta C enters through the accumulators (acc = (beta/alpha) C, all 64 loads in flight under the first tile's loads),
    // so the epilogue is stores only
    double* C = g.C + (g.split_k > 1 ? (long long)blockIdx.z * g.c_split : 0);
    const bool use_beta = g.split_k <= 1 && g.beta != 0.0;
    const double c_scale = use_beta ? g.beta / g.alpha : 0.0;
    double acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int m = m0 + row_base + (i >> 1) * 32 + (i & 1);
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int n = n0 + col_base + (c >> 1) * 16 + (c & 1);
            acc[i][c] = (use_beta && m < g.M && n < g.N) ? c_scale * C[(long long)m * g.ldc + n] : 0.0;
        }
    }

    double ra[8], rb[8];
    auto load_tile = [&](int k0) {
        {   // A tile: 128 rows x 16 k, k fastest in memory
            const int k = tid & 15, r = tid >> 4;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int m = m0 + r + 16 * i;
                ra[i] = (m < g.M && k0 + k < kend) ? __ldg(g.A + (long long)m * g.lda + k0 + k) : 0.0;
            }
        }
        if (B_KMAJOR) {
            const int k = tid & 15, r = tid >> 4;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int n = n0 + r + 16 * i;
                rb[i] = (n < g.N && k0 + k < kend) ? __ldg(g.B + (long long)n * g.ldb + k0 + k) : 0.0;
            }
        } else {
            const int n = tid & 127, r = tid >> 7;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int k = r + 2 * i;
                rb[i] = (n0 + n < g.N && k0 + k < kend) ? __ldg(g.B + (long long)(k0 + k) * g.ldb + n0 + n) : 0.0;
            }
        }
    };
    auto store_tile = [&](int stage) {
        double* As = gemm_smem + stage * 2 * GK * GPITCH;
        double* Bs = As + GK * GPITCH;
        {
            const int k = tid & 15, r = tid >> 4;
#pragma unroll
            for (int i = 0; i < 8; ++i) As[k * GPITCH + r + 16 * i] = ra[i];
        }
        if (B_KMAJOR) {
            const int k = tid & 15, r = tid >> 4;
#pragma unroll
            for (int i = 0; i < 8; ++i) Bs[k * GPITCH + r + 16 * i] = rb[i];
        } else {
            const int n = tid & 127, r = tid >> 7;
#pragma unroll
            for (int i = 0; i < 8; ++i) Bs[(r + 2 * i) * GPITCH + n] = rb[i];
        }
    };

    if (kbeg < kend) {
        load_tile(kbeg);
        store_tile(0);
    }
    __syncthreads();
    int stage = 0;
    for (int k0 = kbeg; k0 < kend; k0 += GK, stage ^= 1) {
        const bool more = k0 + GK < kend;
        if (more) load_tile(k0 + GK);
        const double* As = gemm_smem + stage * 2 * GK * GPITCH;
        const double* Bs = As + GK * GPITCH;
        switch (jmax) {
            case 4: gemm_tile<4>(As, Bs, row_base, col_base, acc); break;
            case 3: gemm_tile<3>(As, Bs, row_base, col_base, acc); break;
            case 2: gemm_tile<2>(As, Bs, row_base, col_base, acc); break;
            case 1: gemm_tile<1>(As, Bs, row_base, col_base, acc); break;
            default: break;
        }
        if (more) store_tile(stage ^ 1);   // the other stage: its readers finished before the previous barrier
        __syncthreads();
    }

#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int m = m0 + row_base + (i >> 1) * 32 + (i & 1);
        if (m >= g.M) continue;
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int n = n0 + col_base + (c >> 1) * 16 + (c & 1);
            if (n < g.N) C[(long long)m * g.ldc + n] = g.alpha * acc[i][c];
        }
    }
}

// ---- the same contraction on the FP64 matrix unit (mma.sync m8n8k4, DMMA) ---------------------------------------
// With 8 x 8 register tiles every thread refills 16 doubles from shared memory per 64 FMAs: 128 B per SM clock, exactly the
// shared-memory bandwidth, so the LSU and the FP64 pipe limit each other at ~60 %.  The warp-wide m8n8k4 fragment shares its
// operands across lanes: one double per lane per 8 x 4 (A) or 4 x 8 (B) fragment, 18 LDS.64 per 32 DMMAs (8 192 FMAs) for a
// 128 x 16 warp tile -- a quarter of the shared-memory traffic, and 6x fewer issue slots.  On B200 the DMMA rate measured
// the same as the DFMA rate (37.0 TFLOP/s with two warps per scheduler): same roofline, reachable.
// Operands must both be K-major (A[m][k], B[n][k]); they are staged k-contiguous (32-deep k-tiles, pitch 36 doubles: the eight rows x four
// k of a fragment load fall on 32 distinct banks, and the staging copies need no transpose).
// Fragment layout (PTX ISA, mma.m8n8k4 .f64): lane l holds A[l/4][l%4], B[k = l%4][n = l/4], C[l/4][2*(l%4) + {0,1}].
// k-tile of the matrix-unit kernel.  Row pitch MK + 4 doubles: 2 * (MK + 4) = 8 mod 32 words, so the 8 rows x 4 k of a fragment
// load fall on 32 distinct banks.  (48-deep tiles for the 128 x 128 variant fit two stages in 213 KB and pay the per-tile barrier
// less often, but measured slower -- 0.508 against 0.395 ms for the x-update: 255 registers and sixteen 12-step tile bodies.)
__host__ __device__ constexpr int mma_mk(int) { return 32; }
constexpr int MMA_STAGES = 2;

__device__ __forceinline__ void dmma_m8n8k4(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
// global -> shared copy of BYTES (8 or 16) bytes, of which only the first src_bytes are read (the rest is zero-filled)
template <int BYTES>
__device__ __forceinline__ void cp_async(double* smem, const double* gmem, int src_bytes) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(s), "l"(gmem), "n"(BYTES), "r"(src_bytes));
}

// One k-tile for a warp that owns NRB 8-row blocks (all the tile's valid rows) x two 8-column blocks: every warp of the
// CTA does the same work whatever M is (n_rhs = 100: 13 row blocks), so no scheduler waits for another at the barrier.
template <int NRB, int MK>
__device__ __forceinline__ void mma_tile(const double* __restrict__ As, const double* __restrict__ Bs, int a_off, int b_off,
                                         double (&acc)[16][2][2]) {
    constexpr int MPITCH = MK + 4;
#pragma unroll
    for (int k4 = 0; k4 < MK; k4 += 4) {
        double a[NRB], b[2];
#pragma unroll
        for (int jn = 0; jn < 2; ++jn) b[jn] = Bs[b_off + jn * 8 * MPITCH + k4];
#pragma unroll
        for (int j = 0; j < NRB; ++j) a[j] = As[a_off + j * 8 * MPITCH + k4];
#pragma unroll
        for (int j = 0; j < NRB; ++j)
#pragma unroll
            for (int jn = 0; jn < 2; ++jn) dmma_m8n8k4(acc[j][jn], a[j], b[jn]);
    }
}

// VEC = doubles per asynchronous copy: 2 when both operands are 16-byte aligned with even pitches, else 1.
// NW  = warps per CTA = 16-column strips of the CTA tile: 8 (128 x 128 tile, one CTA per SM) for long contractions; 4 (128 x 64
//       tile, 111 KB of shared memory, two CTAs per SM) for short ones (the rank-128 sweep update), where a CTA is a few k-tiles
//       between reading and writing its block of C and a second resident CTA fills the unit meanwhile.
constexpr int mma_smem_bytes(int nw) { return MMA_STAGES * (GM + nw * 16) * (mma_mk(nw) + 4) * (int)sizeof(double); }
template <int VEC, int NW>
__global__ void __launch_bounds__(NW * 32) gemm_f64_mma_kernel(GemmArgs g) {
    constexpr int MK = mma_mk(NW), MPITCH = MK + 4;
    constexpr int NT = NW * 32, TN = NW * 16, STAGE = (GM + TN) * MPITCH;
    extern __shared__ __align__(16) double gemm_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int gid = lane >> 2, tig = lane & 3;
    const int m0 = blockIdx.y * GM, n0 = blockIdx.x * TN;
    if (g.lower_only && n0 >= m0 + GM) return;
    int kbeg = 0, kend = g.K;
    if (g.split_k > 1) { kbeg = blockIdx.z * g.k_chunk; kend = min(g.K, kbeg + g.k_chunk); }
    // this warp: row blocks j*8 + [0,8) for j < nrb (all valid rows of the tile), column blocks warp*16 + jn*8 + [0,8) (jn = 0, 1)
    const int nrb = min(16, (g.M - m0 + 7) >> 3);
    const int a_off = gid * MPITCH + tig, b_off = (warp * 16 + gid) * MPITCH + tig;

    // the operand tiles go global -> shared with cp.async, MMA_STAGES deep: tile t+1 is in flight while tile t is multiplied
    constexpr int CPR = MK / VEC;              // copies per tile row
    constexpr int RPP = NT / CPR;              // rows per pass
    static_assert(NT % CPR == 0 && GM % RPP == 0 && TN % RPP == 0, "whole passes over the tile rows");
    const int ck = (tid % CPR) * VEC, cr = tid / CPR;
    auto issue_tile = [&](int k0, int stage) {
        double* As = gemm_smem + stage * STAGE;
        double* Bs = As + GM * MPITCH;
        const int left = (kend - (k0 + ck)) * 8;                         // bytes of this copy that lie inside [kbeg, kend)
        const int kbytes = left < 0 ? 0 : (left > 8 * VEC ? 8 * VEC : left);
#pragma unroll
        for (int i = 0; i < GM / RPP; ++i) {
            const int r = cr + RPP * i;
            const bool va = m0 + r < g.M && kbytes > 0;
            cp_async<8 * VEC>(As + r * MPITCH + ck, va ? g.A + (long long)(m0 + r) * g.lda + k0 + ck : g.A, va ? kbytes : 0);
        }
#pragma unroll
        for (int i = 0; i < TN / RPP; ++i) {
            const int r = cr + RPP * i;
            const bool vb = n0 + r < g.N && kbytes > 0;
            cp_async<8 * VEC>(Bs + r * MPITCH + ck, vb ? g.B + (long long)(n0 + r) * g.ldb + k0 + ck : g.B, vb ? kbytes : 0);
        }
    };

    const int n_tiles = kbeg < kend ? (kend - kbeg + MK - 1) / MK : 0;
#pragma unroll
    for (int s = 0; s < MMA_STAGES - 1; ++s) {
        if (s < n_tiles) issue_tile(kbeg + s * MK, s);
        asm volatile("cp.async.commit_group;");
    }

    double* C = g.C + (g.split_k > 1 ? (long long)blockIdx.z * g.c_split : 0);
    const bool use_beta = g.split_k <= 1 && g.beta != 0.0;
    const double c_scale = use_beta ? g.beta / g.alpha : 0.0;
    // a lane's two columns of an 8 x 8 block are adjacent: C is written as 16-byte pairs when it is aligned for that (reading it
    // that way into the accumulators measured slower: 40 against 35.5 ms for the inverse)
    const bool c_vec = (((uintptr_t)C | (uintptr_t)(g.ldc * 8)) & 15) == 0;
    double acc[16][2][2];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const int m = m0 + j * 8 + gid;
#pragma unroll
        for (int jn = 0; jn < 2; ++jn)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int n = n0 + warp * 16 + jn * 8 + tig * 2 + e;
                acc[j][jn][e] = (use_beta && m < g.M && n < g.N) ? c_scale * C[(long long)m * g.ldc + n] : 0.0;
            }
    }

    for (int t = 0; t < n_tiles; ++t) {
        asm volatile("cp.async.wait_group %0;" ::"n"(MMA_STAGES - 2));   // tile t has landed (this thread's copies)
        __syncthreads();                                                  // ... everyone's; and tile t-1 is no longer read
        if (t + MMA_STAGES - 1 < n_tiles) issue_tile(kbeg + (t + MMA_STAGES - 1) * MK, (t + MMA_STAGES - 1) % MMA_STAGES);
        asm volatile("cp.async.commit_group;");
        const double* As = gemm_smem + (t % MMA_STAGES) * STAGE;
        const double* Bs = As + GM * MPITCH;
        switch (nrb) {
#define SMX_MMA_CASE(N) case N: mma_tile<N, MK>(As, Bs, a_off, b_off, acc); break;
            SMX_MMA_CASE(16) SMX_MMA_CASE(15) SMX_MMA_CASE(14) SMX_MMA_CASE(13) SMX_MMA_CASE(12) SMX_MMA_CASE(11) SMX_MMA_CASE(10)
            SMX_MMA_CASE(9) SMX_MMA_CASE(8) SMX_MMA_CASE(7) SMX_MMA_CASE(6) SMX_MMA_CASE(5) SMX_MMA_CASE(4) SMX_MMA_CASE(3)
            SMX_MMA_CASE(2) SMX_MMA_CASE(1)
#undef SMX_MMA_CASE
            default: break;
        }
    }

#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const int m = m0 + j * 8 + gid;
        if (m >= g.M) continue;
#pragma unroll
        for (int jn = 0; jn < 2; ++jn) {
            const int n = n0 + warp * 16 + jn * 8 + tig * 2;
            if (n >= g.N) continue;
            double* p = C + (long long)m * g.ldc + n;
            if (c_vec && n + 1 < g.N) {
                *reinterpret_cast<double2*>(p) = make_double2(g.alpha * acc[j][jn][0], g.alpha * acc[j][jn][1]);
            } else {
                p[0] = g.alpha * acc[j][jn][0];
                if (n + 1 < g.N) p[1] = g.alpha * acc[j][jn][1];
            }
        }
    }
}

// ---- block Gauss-Jordan inversion of an SPD matrix ---------------------------------------------------------------

// P = inverse of the nb x nb pivot block A[k0..k0+nb)[k0..k0+nb), read from its lower triangle (an SPD Schur complement: no
// pivoting needed).
// One CTA of 32 x 32 threads, each holding a 4 x 4 patch of the block in registers through all nb Gauss-Jordan steps;
// only the pivot row and column of a step go through shared memory (double-buffered: one barrier per step).
// P is written dense [GJ_NB][GJ_NB] with identity padding past nb.
static_assert(GJ_NB == 128, "gj_pivot_inverse_kernel assumes 32 x 32 threads x 4 x 4 patches");
__global__ void __launch_bounds__(1024) gj_pivot_inverse_kernel(const double* A, long long lda, int k0, int nb, double* P) {
    __shared__ __align__(16) double rowp[2][GJ_NB], colp[2][GJ_NB];
    const int tj = threadIdx.x & 31, ti = threadIdx.x >> 5;
    double s[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int i = ti * 4 + a, j = tj * 4 + b;
            s[a][b] = (i < nb && j < nb) ? A[(long long)(k0 + max(i, j)) * lda + k0 + min(i, j)] : (i == j ? 1.0 : 0.0);   // lower triangle
        }
    for (int p = 0; p < nb; ++p) {
        const int po = p >> 2, pa = p & 3, buf = p & 1;
        if (ti == po) {   // this warp holds row p
#pragma unroll
            for (int b = 0; b < 4; ++b) rowp[buf][tj * 4 + b] = pa == 0 ? s[0][b] : pa == 1 ? s[1][b] : pa == 2 ? s[2][b] : s[3][b];
        }
        if (tj == po) {   // this lane holds column p
#pragma unroll
            for (int a = 0; a < 4; ++a) colp[buf][ti * 4 + a] = pa == 0 ? s[a][0] : pa == 1 ? s[a][1] : pa == 2 ? s[a][2] : s[a][3];
        }
        __syncthreads();
        const double inv = 1.0 / rowp[buf][p];
        double r[4], c[4];
#pragma unroll
        for (int b = 0; b < 4; ++b) r[b] = rowp[buf][tj * 4 + b] * inv;
#pragma unroll
        for (int a = 0; a < 4; ++a) c[a] = colp[buf][ti * 4 + a];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const bool ip = ti * 4 + a == p, jp = tj * 4 + b == p;
                s[a][b] = ip ? (jp ? inv : r[b]) : (jp ? -c[a] * inv : fma(-c[a], r[b], s[a][b]));
            }
    }
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) P[(ti * 4 + a) * GJ_NB + tj * 4 + b] = s[a][b];
}

// Symmetric sweep on pivot block K = [k0, k0+nb) of a matrix whose LOWER triangle is kept (api_weights.inc invert_spd):
// gather the column block A_:,K into Ccol [n][GJ_NB] (rows in K and columns past nb zero) ...
__global__ void sweep_gather_kernel(const double* A, long long lda, int n, int k0, int nb, double* Ccol) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long left = (long long)k0 * GJ_NB;          // i < k0: element (i, K) lives at A[k0+kk][i]; i fastest
    if (gid < left) {
        const int kk = (int)(gid / k0), i = (int)(gid % k0);
        Ccol[(long long)i * GJ_NB + kk] = kk < nb ? A[(long long)(k0 + kk) * lda + i] : 0.0;
    } else if (gid < (long long)n * GJ_NB) {               // i >= k0: kk fastest
        const int i = (int)(gid / GJ_NB), kk = (int)(gid % GJ_NB);
        Ccol[gid] = (i >= k0 + nb && kk < nb) ? A[(long long)i * lda + k0 + kk] : 0.0;
    }
}

// ... and, after A -= T Ccol^T with T = Ccol P on the other blocks, store A_:,K = T and A_KK = -P.
__global__ void sweep_scatter_kernel(double* A, long long lda, int n, int k0, int nb, const double* T, const double* P) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long left = (long long)k0 * GJ_NB;
    if (gid < left) {
        const int kk = (int)(gid / k0), i = (int)(gid % k0);
        if (kk < nb) A[(long long)(k0 + kk) * lda + i] = T[(long long)i * GJ_NB + kk];
    } else if (gid < (long long)n * GJ_NB) {
        const int i = (int)(gid / GJ_NB), kk = (int)(gid % GJ_NB);
        if (kk >= nb) return;
        if (i >= k0 + nb) A[(long long)i * lda + k0 + kk] = T[gid];
        else if (i >= k0) A[(long long)i * lda + k0 + kk] = -P[(i - k0) * GJ_NB + kk];
    }
}

// After all blocks are swept the lower triangle holds -A^-1: negate and mirror.
__global__ void sweep_finish_kernel(double* A, long long lda, int n) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    if (j > i || j >= n) return;
    const double v = -A[(long long)i * lda + j];
    A[(long long)i * lda + j] = v;
    if (j < i) A[(long long)j * lda + i] = v;
}

// ---- assembling the system ---------------------------------------------------------------------------------------

struct WBlockDev {
    const float* rows; long long row_pitch; int col0, col_stride, n_cols, con0;
};
constexpr int MAX_WBLOCKS = 16;
struct AssembleArgs {
    WBlockDev blk[MAX_WBLOCKS];
    int n_blocks, n_orb, n_con;
    const double* sigma; const unsigned char* keep;
    double* Ut; long long ldu;   // Ut[i][n] = U[n][i]
};

// a constraint whose tolerance is not a positive finite number is IGNORED: its row of U and its entry of y are zero
__device__ __forceinline__ bool sigma_ok(double s) { return s > 0.0 && s < 1.0e300; }
__global__ void assemble_ut_kernel(AssembleArgs a) {
    const int i = blockIdx.x;
    const bool kept = !a.keep || a.keep[i] != 0;
    for (int n = blockIdx.y * blockDim.x + threadIdx.x; n < a.n_con; n += gridDim.y * blockDim.x) {
        int b = 0;
        while (b + 1 < a.n_blocks && n >= a.blk[b + 1].con0) ++b;
        const WBlockDev& w = a.blk[b];
        const int c = n - w.con0;
        const double v = (double)w.rows[(long long)i * w.row_pitch + w.col0 + (long long)c * w.col_stride];
        const double sg = a.sigma[n];
        a.Ut[(long long)i * a.ldu + n] = (kept && sigma_ok(sg)) ? v / sg : 0.0;
    }
}

// y_b[n] = target[n]/sigma[n] + xi[b][n]
__global__ void build_y_kernel(const double* target, const double* sigma, const double* xi, int n_con, int n_rhs, double* Y) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)n_con * n_rhs) return;
    const int n = (int)(gid % n_con);
    Y[gid] = sigma_ok(sigma[n]) ? target[n] / sigma[n] + (xi ? xi[gid] : 0.0) : 0.0;
}

// G_ii += 2 lambda / (N wtilde_i^2) + rho
__global__ void add_diag_kernel(double* G, long long ldg, int n, const double* wtilde, double two_lam_over_n, double rho) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double wt = wtilde ? wtilde[i] : 1.0;
    G[(long long)i * ldg + i] += two_lam_over_n / (wt * wt) + rho;
}

// The ADMM update, one thread per (right-hand side b, orbit i), fixed summation order:
//   x = sum of the split-K partial sums;  z' = max(0, x + u);  u' = u + x - z';  r = q + rho (z' - u').
// On the last iteration every CTA also leaves its share of sum (x-z')^2 and sum (z'-z)^2 in resid_part[b][blockIdx.x][2],
// which admm_resid_kernel adds up in a fixed order.
constexpr int MAX_SPLIT = 16;
__global__ void __launch_bounds__(256) admm_update_kernel(const double* __restrict__ part, int n_split, long long split_stride,
                                                          const double* __restrict__ q, double* __restrict__ z, double* __restrict__ u,
                                                          double* __restrict__ r, int n_orb, double rho, double* resid_part) {
    const int b = blockIdx.y, i = blockIdx.x * 256 + threadIdx.x;
    const long long e = (long long)b * n_orb + i;
    double dp = 0.0, dd = 0.0;
    if (i < n_orb) {
        double p[MAX_SPLIT];
#pragma unroll
        for (int s = 0; s < MAX_SPLIT; ++s) p[s] = s < n_split ? part[s * split_stride + e] : 0.0;
        const double zo = z[e], uo = u[e], qq = q[e];
        double x = 0.0;
#pragma unroll
        for (int s = 0; s < MAX_SPLIT; ++s) x += p[s];
        const double zn = fmax(0.0, x + uo);
        const double un = uo + x - zn;
        z[e] = zn; u[e] = un;
        r[e] = fma(rho, zn - un, qq);
        dp = (x - zn) * (x - zn); dd = (zn - zo) * (zn - zo);
    }
    if (!resid_part) return;
    __shared__ double red[2][8];
    for (int o = 16; o > 0; o >>= 1) {
        dp += __shfl_down_sync(0xffffffffu, dp, o);
        dd += __shfl_down_sync(0xffffffffu, dd, o);
    }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = dp; red[1][threadIdx.x >> 5] = dd; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, d = 0.0;
        for (int w = 0; w < 8; ++w) { a += red[0][w]; d += red[1][w]; }
        resid_part[((long long)b * gridDim.x + blockIdx.x) * 2] = a;
        resid_part[((long long)b * gridDim.x + blockIdx.x) * 2 + 1] = d;
    }
}

__global__ void admm_resid_kernel(const double* resid_part, int n_chunks, int n_rhs, double rho, double* resid) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_rhs) return;
    double a = 0.0, d = 0.0;
    for (int c = 0; c < n_chunks; ++c) { a += resid_part[((long long)b * n_chunks + c) * 2]; d += resid_part[((long long)b * n_chunks + c) * 2 + 1]; }
    resid[2 * b] = sqrt(a); resid[2 * b + 1] = rho * sqrt(d);
}

// chi^2 of Eq. 5 per realisation b and block k against the unperturbed data: sum over the block's rows of
// (pred[b][n] - target[n]/sigma[n])^2, one CTA each, fixed summation order.
__global__ void __launch_bounds__(256) chi2_blocks_kernel(const double* pred, long long ldp, const double* target, const double* sigma,
                                                          AssembleArgs a, double* chi2) {
    const int k = blockIdx.x, b = blockIdx.y;
    const int lo = a.blk[k].con0, hi = lo + a.blk[k].n_cols;
    double acc = 0.0;
    for (int n = lo + threadIdx.x; n < hi; n += 256) {
        const double d = sigma_ok(sigma[n]) ? pred[(long long)b * ldp + n] - target[n] / sigma[n] : 0.0;
        acc = fma(d, d, acc);
    }
    __shared__ double red[8];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += red[w];
        chi2[(long long)b * a.n_blocks + k] = t;
    }
}

// Eq. 6 (reading R20): chi2_b = sum of the selected blocks; out[0] = chi2_min - 2 ln[(1/B) sum_b exp((chi2_min - chi2_b)/2)],
// out[1] = chi2_min.  One CTA, fixed order.
__global__ void __launch_bounds__(256) marginal_chi2_kernel(const double* chi2, int n_rhs, int n_blocks, unsigned mask, double* out) {
    __shared__ double red[256];
    auto chi2_of = [&](int b) {
        double t = 0.0;
        for (int k = 0; k < n_blocks; ++k) if ((mask >> k) & 1u) t += chi2[(long long)b * n_blocks + k];
        return t;
    };
    double mn = INFINITY;
    for (int b = threadIdx.x; b < n_rhs; b += 256) mn = fmin(mn, chi2_of(b));
    red[threadIdx.x] = mn;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) red[threadIdx.x] = fmin(red[threadIdx.x], red[threadIdx.x + o]); __syncthreads(); }
    const double cmin = red[0];
    __syncthreads();
    double sum = 0.0;
    for (int b = threadIdx.x; b < n_rhs; b += 256) sum += exp(0.5 * (cmin - chi2_of(b)));
    red[threadIdx.x] = sum;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o]; __syncthreads(); }
    if (threadIdx.x == 0) { out[0] = cmin - 2.0 * log(red[0] / n_rhs); out[1] = cmin; }
}

}  // namespace smx
