// rowbuild.cuh -- SURVEY.md 8(a) row a-7: accumulate each orbit's histogram in shared memory with
// warp-aggregated atomics and flush it to HBM in coalesced, vectorised stores, once per orbit
// (north_star item 3).  Also the test-hook and microbenchmark kernels.
#pragma once
#include "kernels.cuh"

namespace smx {

struct RowArgs {
    const unsigned* stage;  // [n_trials][n_hist][stage_orb_stride][n_rec]
    long long stage_orb_stride, stage_orb0;  // pitch of a histogram block and first orbit to read
    float* losvd;           // [n_trials][n_proj][n_orb][nlos]
    float* dens;            // [n_trials][n_orb][nden]
    int* nout;              // [n_trials][n_hist][n_orb] or null
    long long n_orb;        // rows to build per histogram
    long long out_orb_stride;  // orbits in the caller's full output (row pitch between projections/trials)
    long long out_orb0;     // first orbit of this chunk in the output
    int n_trials, n_proj, n_rec;
    int nlos, nden;
    int slab;               // slab length in cells
    int h0;                 // first histogram to build (0; n_proj = the density grid only, Gauss-Hermite mode)
    int prezeroed;          // sparse kernel only: the rows are all-zero on entry (zero_fill_kernel beside the integrator),
                            // so the kernel writes nothing but the non-zero cells
    // compact form (sm_flush_rows_compact; sparse kernel, single batch per row): instead of dense rows, (cell, count) pairs
    unsigned* c_cell;       // [capacity] or null = dense output
    float* c_count;         // [capacity]
    long long* c_row_start; // [n_trials][n_hist][n_orb] first entry of the row
    int* c_row_nnz;         // [n_trials][n_hist][n_orb] entries of the row
    unsigned long long* c_total;   // [1] entries handed out so far (zeroed before the launch); may exceed capacity
    long long capacity;
};

// One CTA builds whole rows: row id -> (trial, hist, orbit).  The slab holds u32 counts; it is all-zero
// between rows (the flush loop writes zeros back as it reads), so the per-row cost is the replay of
// n_rec indices per slab plus the dense, HBM-bound flush.
template <bool GLOBAL_ATOMICS>
__global__ void __launch_bounds__(256) rowbuild_kernel(RowArgs a) {
    extern __shared__ __align__(16) unsigned slab[];
    __shared__ int s_nout;
    const int tid = threadIdx.x, lane = tid & 31;
    const int n_hist = a.n_proj + 1;
    const int n_hb = n_hist - a.h0;  // histograms built by this launch
    const long long n_rows = (long long)a.n_trials * n_hb * a.n_orb;
    if (!GLOBAL_ATOMICS) {
        for (int i = tid; i < a.slab; i += blockDim.x) slab[i] = 0u;
    }
    __syncthreads();
    for (long long row = blockIdx.x; row < n_rows; row += gridDim.x) {
        // rows are enumerated orbit-fastest within a histogram so that neighbouring CTAs write neighbouring rows
        const long long orb = row % a.n_orb;
        const int h = a.h0 + (int)((row / a.n_orb) % n_hb);
        const int trial = (int)(row / (a.n_orb * n_hb));
        const unsigned* idx = a.stage + (((long long)trial * n_hist + h) * a.stage_orb_stride + a.stage_orb0 + orb) * a.n_rec;
        const int len = h < a.n_proj ? a.nlos : a.nden;
        float* out = h < a.n_proj
            ? a.losvd + (((long long)trial * a.n_proj + h) * a.out_orb_stride + a.out_orb0 + orb) * a.nlos
            : a.dens + ((long long)trial * a.out_orb_stride + a.out_orb0 + orb) * a.nden;
        if (tid == 0) s_nout = 0;
        __syncthreads();
        if (GLOBAL_ATOMICS) {
            // A/B baseline: zero-fill the row, then one global atomic per sample
            for (int i = tid; i < len; i += blockDim.x) out[i] = 0.0f;
            __syncthreads();
            int cnt = 0;
            for (int r = tid; r < a.n_rec; r += blockDim.x) {
                unsigned d = idx[r];
                if (d == IDX_OUT) ++cnt; else atomicAdd(out + d, 1.0f);
            }
            if (cnt) atomicAdd(&s_nout, cnt);
        } else {
            const bool vec_ok = ((len & 3) == 0) && ((((size_t)out) & 15) == 0);
            for (int base = 0; base < len; base += a.slab) {
                const int n_here = min(a.slab, len - base);
                int cnt = 0;
                for (int r0 = 0; r0 < a.n_rec; r0 += blockDim.x) {
                    const int r = r0 + tid;
                    unsigned d = r < a.n_rec ? __ldg(idx + r) : IDX_OUT;
                    if (base == 0 && r < a.n_rec && d == IDX_OUT) ++cnt;
                    unsigned rel = d - (unsigned)base;               // wraps to a huge value below the slab
                    const bool in = rel < (unsigned)n_here && d != IDX_OUT;
                    // warp-aggregated shared atomic: lanes hitting the same cell elect a leader
                    unsigned key = in ? rel : IDX_OUT;
                    unsigned peers = __match_any_sync(0xFFFFFFFFu, key);
                    if (in && lane == (__ffs(peers) - 1)) atomicAdd(&slab[rel], (unsigned)__popc(peers));
                }
                if (base == 0 && cnt) atomicAdd(&s_nout, cnt);
                __syncthreads();
                // flush: u32 counts -> fp32, 16-byte streaming stores, zero the slab behind us
                if (vec_ok) {
                    uint4* s4 = reinterpret_cast<uint4*>(slab);
                    float4* o4 = reinterpret_cast<float4*>(out + base);
                    const int n4 = n_here >> 2;
                    for (int i = tid; i < n4; i += blockDim.x) {
                        uint4 v = s4[i];
                        s4[i] = make_uint4(0u, 0u, 0u, 0u);
                        __stcs(o4 + i, make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w));
                    }
                } else {
                    for (int i = tid; i < n_here; i += blockDim.x) {
                        unsigned v = slab[i];
                        slab[i] = 0u;
                        out[base + i] = (float)v;
                    }
                }
                __syncthreads();
            }
        }
        __syncthreads();
        if (tid == 0 && a.nout) a.nout[((long long)trial * n_hist + h) * a.out_orb_stride + a.out_orb0 + orb] = s_nout;
        __syncthreads();
    }
}

// Sparse variant of the same step: an orbit's row is ~98 % zeros (a few hundred distinct cells out of 48 000 ... 196 608),
// so the CTA (1) accumulates the orbit's samples in a shared-memory HASH histogram (open addressing at load <= 1/2; runs of
// consecutive samples in the same cell are merged within the warp and added by their first lane: warp-aggregated shared
// atomics), keeping a LIST of the slots it claims, (2) unless the caller has zeroed the rows (a.prezeroed: zero_fill_kernel beside
// the integrator), streams the zero row with 16-byte stores and (3) writes the few non-zero cells by walking the list (not the
// table: a row claims ~500 of 4 096 slots), emptying the claimed slots on the way.  One pass over the staged indices whatever the
// row length; rows with more samples than half the table (bundles) take further batches whose cells are added with global atomics.
// Shared memory: keys[n_slots] u32, cnts[n_slots] u32, list[n_slots / 2] u16.
__global__ void __launch_bounds__(256) rowbuild_sparse_kernel(RowArgs a, int log2_slots) {
    extern __shared__ __align__(16) unsigned hsm[];
    const int n_slots = 1 << log2_slots;
    unsigned* keys = hsm;               // IDX_OUT = empty
    unsigned* cnts = hsm + n_slots;
    unsigned short* list = reinterpret_cast<unsigned short*>(hsm + 2 * n_slots);
    __shared__ int s_nout[2], s_n[2];   // out-of-grid count of the row / claimed slots of the batch, double-buffered by parity
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x, lane = tid & 31;
    const int n_hist = a.n_proj + 1;
    const int batch = n_slots >> 1;     // samples per batch: the table never exceeds half load, so probing terminates
    int par = 0, rp = 0;
    const int n_hb = n_hist - a.h0;     // histograms built by this launch
    const long long n_rows = (long long)a.n_trials * n_hb * a.n_orb;
    for (int i = tid; i < n_slots; i += blockDim.x) { keys[i] = IDX_OUT; cnts[i] = 0u; }
    if (tid == 0) { s_nout[0] = s_nout[1] = 0; s_n[0] = s_n[1] = 0; }
    __syncthreads();
    for (long long row = blockIdx.x; row < n_rows; row += gridDim.x) {
        const long long orb = row % a.n_orb;
        const int h = a.h0 + (int)((row / a.n_orb) % n_hb);
        const int trial = (int)(row / (a.n_orb * n_hb));
        const unsigned* idx = a.stage + (((long long)trial * n_hist + h) * a.stage_orb_stride + a.stage_orb0 + orb) * a.n_rec;
        const int len = h < a.n_proj ? a.nlos : a.nden;
        float* out = h < a.n_proj
            ? a.losvd + (((long long)trial * a.n_proj + h) * a.out_orb_stride + a.out_orb0 + orb) * a.nlos
            : a.dens + ((long long)trial * a.out_orb_stride + a.out_orb0 + orb) * a.nden;
        int cnt_out = 0;
        const bool single = a.n_rec <= batch;
        for (int b0 = 0; b0 == 0 || b0 < a.n_rec; b0 += batch) {
            const int b1 = min(b0 + batch, a.n_rec);
            // (1) shared-memory hash histogram of this batch of samples
            // the staged indices come from HBM (written by the integrator long before): eight independent loads per thread are
            // in flight before the first one is used, instead of one latency per pass over the row
            for (int r0 = b0; r0 < b1; r0 += 8 * blockDim.x) {
                unsigned dd[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int r = r0 + j * blockDim.x + tid;
                    dd[j] = r < b1 ? __ldcs(idx + r) : IDX_OUT;
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int r = r0 + j * blockDim.x + tid;
                    if (r0 + j * (int)blockDim.x >= b1) break;    // uniform across the CTA
                    const unsigned d = dd[j];
                    if (r < b1 && d == IDX_OUT) ++cnt_out;
                    // lanes hold consecutive samples of the orbit: a run of equal cells (the orbit lingering in a cell) is added by its first
                    // lane in one atomic.  (Runs instead of __match_any_sync: MATCH.ANY takes time proportional to the number of distinct
                    // values in the warp -- 22 % of this kernel's stall samples -- and equal cells that are not adjacent are rare.)
                    const unsigned prev = __shfl_up_sync(0xFFFFFFFFu, d, 1);
                    const bool head = lane == 0 || d != prev;
                    const unsigned heads = __ballot_sync(0xFFFFFFFFu, head);
                    const unsigned above = (heads >> lane) >> 1;           // heads after this lane
                    const unsigned run = above ? (unsigned)__ffs(above) : 32u - (unsigned)lane;
                    if (d != IDX_OUT && head) {
                        unsigned slot = (d * 2654435761u) >> (32 - log2_slots);
                        for (;;) {
                            unsigned k = keys[slot];
                            if (k == IDX_OUT) {                      // empty: claim it (another warp may win the race)
                                k = atomicCAS(&keys[slot], IDX_OUT, d);
                                if (k == IDX_OUT) { k = d; list[atomicAdd(&s_n[par], 1)] = (unsigned short)slot; }
                            }
                            if (k == d) { atomicAdd(&cnts[slot], run); break; }
                            slot = (slot + 1) & (n_slots - 1);
                        }
                    }
                }
            }
            if (b1 >= a.n_rec && cnt_out) atomicAdd(&s_nout[rp], cnt_out);   // last batch: the row's out-of-grid count is complete
            __syncthreads();
            if (a.c_cell) {
                // compact form: the row's entries go to a run of the entry arrays handed out by one global atomic
                const int n_c = s_n[par];
                if (tid == 0) {
                    s_base = atomicAdd(a.c_total, (unsigned long long)n_c);
                    const long long ri = ((long long)trial * n_hist + h) * a.out_orb_stride + a.out_orb0 + orb;
                    a.c_row_start[ri] = (long long)s_base; a.c_row_nnz[ri] = n_c;
                    s_n[par ^ 1] = 0;
                    if (a.nout) a.nout[ri] = s_nout[rp];
                    s_nout[rp ^ 1] = 0;
                }
                __syncthreads();
                const unsigned long long base = s_base;
                for (int i = tid; i < n_c; i += blockDim.x) {
                    const int slot = list[i];
                    if ((long long)(base + i) < a.capacity) { a.c_cell[base + i] = keys[slot]; a.c_count[base + i] = (float)cnts[slot]; }
                    keys[slot] = IDX_OUT; cnts[slot] = 0u;
                }
                par ^= 1;
                __syncthreads();
                continue;
            }
            if (b0 == 0 && !a.prezeroed) {
                // (2) the zero row (default cache policy: the lines stay in L2 until step 3 has patched them)
                if (((len & 3) == 0) && ((((size_t)out) & 15) == 0)) {
                    float4* o4 = reinterpret_cast<float4*>(out);
                    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
                    const int n4 = len >> 2;
                    for (int i = tid; i < n4; i += blockDim.x) o4[i] = z4;
                } else {
                    for (int i = tid; i < len; i += blockDim.x) out[i] = 0.0f;
                }
                __syncthreads();  // the zeros are ordered before this CTA's later writes to the same row
            }
            // (3) the non-zero cells, by the list of claimed slots; the table is emptied for the next batch / row on the way
            const int n_claimed = s_n[par];
            if (tid == 0) {
                s_n[par ^ 1] = 0;             // the other counter was last read before the barrier that ended the previous batch
                if (b1 >= a.n_rec) {
                    if (a.nout) a.nout[((long long)trial * n_hist + h) * a.out_orb_stride + a.out_orb0 + orb] = s_nout[rp];
                    s_nout[rp ^ 1] = 0;       // the next row's counter (last read a whole row ago)
                }
            }
            for (int i = tid; i < n_claimed; i += blockDim.x) {
                const int slot = list[i];
                const unsigned k = keys[slot];
                if (single) out[k] = (float)cnts[slot]; else atomicAdd(out + k, (float)cnts[slot]);
                keys[slot] = IDX_OUT; cnts[slot] = 0u;
            }
            par ^= 1;
            __syncthreads();
        }
        rp ^= 1;
    }
}

// Weighted rows of the adaptive integrator (every sample weighs dt / t_total of its orbit).  The scheme of
// rowbuild_sparse_kernel with sums in place of counts: a shared-memory hash table per CTA accumulates the weights of a row in
// 64-bit FIXED POINT (2^-32; two 32-bit halves with carry: native shared atomics, order-independent, so rows are reproducible bit
// for bit), a list remembers the claimed slots, and the non-zero cells are written into the zero row (zeroed by zero_fill_kernel
// beside the integrator, a.prezeroed, or by this kernel).  A row = n_bundle consecutive orbits x n_steps attempts x n_sym copies
// (rejected attempts have weight 0 and are skipped).  The table is emptied into the row whenever it gets half full (bundles of
// dithered orbits visit more cells than it holds): from the second time on with atomic adds, one per cell and flush.
struct WRowArgs {
    const unsigned* stage;   // [n_hist][stage_orb_stride][n_steps * n_sym]
    const float* stage_w;    // [stage_orb_stride][n_steps]
    const double* t_end;     // [stage_orb_stride] total integrated time of every orbit of the chunk
    long long stage_orb_stride;
    float* losvd; float* dens; float* wout;   // rows [n_proj][out_stride][nlos], [out_stride][nden], [n_hist][out_stride] (may be null)
    long long n_rows, out_stride, out_row0;
    int n_proj, n_steps, n_sym, n_bundle, nlos, nden, h0, prezeroed;
    // batched potentials: n_trials (0 = 1) trials in one launch; trial t's staged orbits start t * t_orb orbits further on (in stage,
    // stage_w and t_end), its output rows t * out_stride rows per histogram block further on ([trial][n_proj][out_stride] ...)
    int n_trials; long long t_orb;
};
__global__ void __launch_bounds__(256) rowbuild_weighted_kernel(WRowArgs a, int log2_slots) {
    extern __shared__ __align__(16) unsigned hsm[];
    const int n_slots = 1 << log2_slots;
    unsigned* keys = hsm;
    unsigned* lo = hsm + n_slots;
    unsigned* hi = hsm + 2 * n_slots;
    unsigned short* list = reinterpret_cast<unsigned short*>(hsm + 3 * n_slots);
    __shared__ int s_n;
    __shared__ double s_red[8];
    const int tid = threadIdx.x, lane = tid & 31;
    const int n_hist = a.n_proj + 1, n_hb = n_hist - a.h0;
    const long long nre = (long long)a.n_steps * a.n_sym;
    const long long n_idx = nre * a.n_bundle;
    const int chunk = 4 * blockDim.x;   // samples between two looks at the table load (<= n_slots / 4)
    for (int i = tid; i < n_slots; i += blockDim.x) { keys[i] = IDX_OUT; lo[i] = 0u; hi[i] = 0u; }
    if (tid == 0) s_n = 0;
    __syncthreads();
    const int n_tr = a.n_trials > 0 ? a.n_trials : 1;
    const long long jobs_per_trial = a.n_rows * n_hb;
    for (long long job0 = blockIdx.x; job0 < jobs_per_trial * n_tr; job0 += gridDim.x) {
        const long long trial = job0 / jobs_per_trial, job = job0 - trial * jobs_per_trial;
        const long long r = job % a.n_rows;
        const int h = a.h0 + (int)(job / a.n_rows);
        const long long so = trial * a.t_orb + r * a.n_bundle;   // first staged orbit of the row
        const unsigned* idx = a.stage + ((long long)h * a.stage_orb_stride + so) * nre;
        const float* sw = a.stage_w + so * (long long)a.n_steps;
        const double* te = a.t_end + so;
        const int len = h < a.n_proj ? a.nlos : a.nden;
        float* out = h < a.n_proj ? a.losvd + (((long long)trial * a.n_proj + h) * a.out_stride + a.out_row0 + r) * a.nlos
                                  : a.dens + (trial * a.out_stride + a.out_row0 + r) * (long long)a.nden;
        if (!a.prezeroed) {
            for (int i = tid; i < len; i += blockDim.x) out[i] = 0.0f;
            __syncthreads();
        }
        double w_out = 0.0;
        bool flushed = false;
        for (long long c0 = 0; c0 < n_idx; c0 += chunk) {
            unsigned dd[4]; float ww[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const long long i = c0 + j * blockDim.x + tid;
                dd[j] = IDX_OUT; ww[j] = 0.0f;
                if (i < n_idx) {
                    const int member = (int)(i / nre);
                    const int k = (int)((i - member * nre) / a.n_sym);
                    const double tt = te[member];
                    ww[j] = tt > 0.0 ? __ldg(sw + (long long)member * a.n_steps + k) * (float)(1.0 / tt) : 0.0f;
                    dd[j] = __ldcs(idx + i);
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const unsigned d = dd[j];
                const float w = ww[j];
                if (!(w > 0.0f)) continue;
                if (d == IDX_OUT) { w_out += (double)w; continue; }
                const unsigned long long v = (unsigned long long)llrint((double)w * 4294967296.0);
                unsigned slot = (d * 2654435761u) >> (32 - log2_slots);
                for (;;) {
                    unsigned k = keys[slot];
                    if (k == IDX_OUT) {
                        k = atomicCAS(&keys[slot], IDX_OUT, d);
                        if (k == IDX_OUT) { k = d; list[atomicAdd(&s_n, 1)] = (unsigned short)slot; }
                    }
                    if (k == d) {
                        const unsigned vl = (unsigned)v;
                        unsigned vh = (unsigned)(v >> 32);
                        if (vl) vh += (atomicAdd(&lo[slot], vl) + vl) < vl;   // carry out of the low half
                        if (vh) atomicAdd(&hi[slot], vh);
                        break;
                    }
                    slot = (slot + 1) & (n_slots - 1);
                }
            }
            __syncthreads();
            // empty the table into the row when the next chunk could take it past half load, and at the end of the row
            const int n_c = s_n;
            const bool last = c0 + chunk >= n_idx;
            if (last || n_c + chunk > (n_slots >> 1)) {
                for (int i = tid; i < n_c; i += blockDim.x) {
                    const int slot = list[i];
                    const float val = (float)((double)(((unsigned long long)hi[slot] << 32) | lo[slot]) * (1.0 / 4294967296.0));
                    if (flushed) atomicAdd(out + keys[slot], val); else out[keys[slot]] = val;
                    keys[slot] = IDX_OUT; lo[slot] = 0u; hi[slot] = 0u;
                }
                flushed = true;
                __syncthreads();
                if (tid == 0) s_n = 0;
                __syncthreads();
            }
        }
        // the weight outside the grid: per-thread sums in a fixed sample order, reduced in a fixed order
        for (int o = 16; o > 0; o >>= 1) w_out += __shfl_down_sync(0xffffffffu, w_out, o);
        if (lane == 0) s_red[tid >> 5] = w_out;
        __syncthreads();
        if (tid == 0 && a.wout) {
            double t = 0.0;
            for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += s_red[i];
            a.wout[(trial * n_hist + h) * a.out_stride + a.out_row0 + r] = (float)t;
        }
        __syncthreads();
    }
}

// Gauss-Hermite rows (Eq.2): per (projection, row) the CTA accumulates, for every aperture, the sample count and
// sum_k alpha(w_k) H_m(w_k), m = 0..4, w = (v_los - v0[ap])/s[ap], from the staged (aperture, v_los) pairs.  Accumulation is in
// 64-bit fixed point (2^-32) with shared-memory integer atomics: exact for the counts and independent of the order of the
// additions, so the rows are reproducible bit for bit.  H_m: van der Marel & Franx (1993) normalisation (R17).
struct GhArgs {
    const unsigned* stage;   // apertures [n_proj+1][stage_orb_stride][n_idx] (the last block is the density grid, unused here)
    const float* stage_v;    // v_los    [n_proj][stage_orb_stride][n_idx]
    long long stage_orb_stride;
    const double* v0; const double* s;   // [n_ap]
    float* gh;               // [n_proj][out_stride][n_ap][6]
    int* nout;               // [n_proj+1][out_stride] or null
    long long n_rows, out_stride, out_row0;
    int n_proj, n_idx, n_ap;
    // weighted rows (adaptive integrator): weight of sample i of row r = stage_w[(r n_bundle + i / nre)][(i % nre) / n_sym] / t_end[...];
    // null = every sample counts 1 (fixed-step integrator)
    const float* stage_w; const double* t_end; float* wout;
    int n_steps, n_sym, n_bundle;
    // batched potentials: n_trials (0 = 1) trials in one launch.  Trial t's staged samples start t * t_stage elements further on in
    // stage, t * t_v in stage_v, its orbits t * t_orb orbits further on in stage_w / t_end (the fixed-step path stages
    // [trial][hist][row], the adaptive one [hist][trial][row]); its outputs are the t-th blocks of gh [trial][n_proj][out_stride][n_ap][6],
    // nout / wout [trial][n_hist][out_stride].
    int n_trials, n_hist; long long t_stage, t_v, t_orb;
};
__global__ void __launch_bounds__(256) rowbuild_gh_kernel(GhArgs a) {
    // [n_ap][6] 64-bit fixed-point sums kept as two 32-bit halves: a 64-bit shared atomicAdd compiles to a compare-and-swap
    // spin loop, whereas low half + carry into the high half are native 32-bit atomics and still exact and order-independent
    extern __shared__ __align__(16) unsigned acc_lo[];
    __shared__ int s_nout;
    __shared__ double s_red[8];
    const int tid = threadIdx.x;
    const int n_acc = a.n_ap * 6;
    unsigned* acc_hi = acc_lo + n_acc;
    const int n_tr = a.n_trials > 0 ? a.n_trials : 1;
    const long long n_jobs = (long long)a.n_proj * a.n_rows;
    for (long long job0 = blockIdx.x; job0 < n_jobs * n_tr; job0 += gridDim.x) {
        const long long trial = job0 / n_jobs, job = job0 - trial * n_jobs;
        const int p = (int)(job / a.n_rows);
        const long long r = job % a.n_rows;
        const long long orow = (trial * a.n_proj + p) * a.out_stride + a.out_row0 + r;      // output row of gh
        const long long crow = (trial * a.n_hist + p) * a.out_stride + a.out_row0 + r;      // its counter in nout / wout
        for (int i = tid; i < 2 * n_acc; i += blockDim.x) acc_lo[i] = 0u;
        if (tid == 0) s_nout = 0;
        __syncthreads();
        const unsigned* idx = a.stage + trial * a.t_stage + ((long long)p * a.stage_orb_stride + r) * a.n_idx;
        const float* vs = a.stage_v + trial * a.t_v + ((long long)p * a.stage_orb_stride + r) * a.n_idx;
        int cnt_out = 0;
        double w_out = 0.0;
        const long long nre = (long long)a.n_steps * a.n_sym;
        for (int k = tid; k < a.n_idx; k += blockDim.x) {
            const unsigned ap = __ldg(idx + k);
            float wt = 1.0f;
            if (a.stage_w) {
                const int member = (int)(k / nre);
                const long long orb = trial * a.t_orb + r * a.n_bundle + member;
                const double tt = a.t_end[orb];
                wt = tt > 0.0 ? __ldg(a.stage_w + orb * a.n_steps + (int)((k - member * nre) / a.n_sym)) * (float)(1.0 / tt) : 0.0f;
                if (!(wt > 0.0f)) continue;
            }
            if (ap == IDX_OUT) { ++cnt_out; w_out += (double)wt; continue; }
            const float w = (float)(((double)__ldg(vs + k) - a.v0[ap]) / a.s[ap]);
            const float w2 = w * w;
            const float al = expf(-0.5f * w2) * 0.3989422804014327f;
            float t[5];
            t[0] = al;
            t[1] = al * 1.4142135623730951f * w;
            t[2] = al * (2.0f * w2 - 1.0f) * 0.7071067811865476f;
            t[3] = al * w * (2.0f * w2 - 3.0f) * 0.5773502691896258f;            // (2 sqrt2 w^3 - 3 sqrt2 w)/sqrt6
            t[4] = al * (4.0f * w2 * w2 - 12.0f * w2 + 3.0f) * 0.2041241452319315f;  // /sqrt24
            const int base = (int)ap * 6;
            if (!a.stage_w) {
                atomicAdd(acc_hi + base, 1u);   // the count: 1 in units of 2^32
            } else {                            // the weight, in the same fixed point
                const unsigned long long v = (unsigned long long)llrint((double)wt * 4294967296.0);
                const unsigned lo = (unsigned)v;
                unsigned hi = (unsigned)(v >> 32);
                if (lo) hi += (atomicAdd(acc_lo + base, lo) + lo) < lo;
                if (hi) atomicAdd(acc_hi + base, hi);
            }
#pragma unroll
            for (int m = 0; m < 5; ++m) {
                const unsigned long long v = (unsigned long long)(long long)llrintf(t[m] * wt * 4294967296.0f);
                const unsigned lo = (unsigned)v;
                unsigned hi = (unsigned)(v >> 32);
                if (lo) hi += (atomicAdd(acc_lo + base + 1 + m, lo) + lo) < lo;   // carry out of the low half
                if (hi) atomicAdd(acc_hi + base + 1 + m, hi);
            }
        }
        if (cnt_out) atomicAdd(&s_nout, cnt_out);
        if (a.wout) {   // weighted rows: the weight outside the apertures, summed in a fixed order
            for (int o = 16; o > 0; o >>= 1) w_out += __shfl_down_sync(0xffffffffu, w_out, o);
            if ((tid & 31) == 0) s_red[tid >> 5] = w_out;
        }
        __syncthreads();
        if (a.wout && tid == 0) {
            double t = 0.0;
            for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += s_red[i];
            a.wout[crow] = (float)t;
        }
        float* out = a.gh + orow * n_acc;
        for (int i = tid; i < n_acc; i += blockDim.x)
            out[i] = (float)((double)(long long)(((unsigned long long)acc_hi[i] << 32) | acc_lo[i]) * (1.0 / 4294967296.0));
        if (tid == 0 && a.nout) a.nout[crow] = s_nout;
        __syncthreads();
    }
}

// Zero fill of the output rows with a footprint small enough (one CTA of <= 128 threads x <= 32 registers per SM, no shared
// memory) to run BESIDE the persistent integrator: the integrator is ALU-bound and leaves HBM idle, so the dense 98 %-zero part
// of the matrix is written while it runs and the row build afterwards only scatters the non-zero cells.  PACED: flat out, the
// fill keeps every SM's load/store queue full of stores that drain at the HBM rate, and the integrator's shared-memory table
// reads wait behind them (measured: +10 ms on a 44 ms integrator for a 12 ms fill); `n_st` 16-byte stores per thread, then
// `sleep_ns` of __nanosleep, keep the queue mostly empty.  sleep_ns = 0: flat out (nothing to hide behind).
__global__ void __launch_bounds__(256) zero_fill_kernel(uint4* p, unsigned long long n16, unsigned char* tail, int n_tail,
                                                        unsigned sleep_ns, int n_st, const int* pace) {
    const uint4 z = make_uint4(0u, 0u, 0u, 0u);
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned it = 0;
    // `pace` (may be null = always paced): non-zero while an integrator launch is running on this device, cleared by its last CTA;
    // looked at every 16 iterations, in both directions (an integrator may start while a fill is under way)
    bool paced = sleep_ns != 0 && (!pace || *(const volatile int*)pace != 0);
    while (i < n16) {
        for (int k = 0; k < n_st && i < n16; ++k, i += stride) p[i] = z;
        if (paced) __nanosleep(sleep_ns);
        if (sleep_ns && pace && (++it & 15u) == 0) paced = *(const volatile int*)pace != 0;
    }
    if (blockIdx.x == 0 && (int)threadIdx.x < n_tail) tail[threadIdx.x] = 0;
}

// The same fill through the SM's bulk-copy engine (TMA): ONE thread per SM issues cp.async.bulk shared -> global copies of a zeroed
// 16 KB shared-memory block, so the stores never enter the SM's load/store instruction queue, where the integrator's table reads
// wait behind them.  Alone on the GPU it writes 7.2 TB/s (the 128-thread store loop above: 6.7); beside the fp64 integrator ~3.3 TB/s
// (the engine reads shared memory, which the integrator's table rows keep 60 % busy) at a cost to the integrator of 0.3 ms in 45 (the
// paced store loop: 1.3 ms for 2.5 TB/s), and one warp of <= 32 registers needs a quarter of the store loop's room on the SM.
// It takes 16 KB + of shared memory beside the integrator's CTA: used where the integrator launches stage their table in shared
// memory (carve-out = all of it); launches that read their tables through L1 keep the store loop (profiles/r2l.md).
// CTA b writes blocks b, b + grid, ...; after every block the thread waits until the engine has READ the source (not until the
// write has landed), which is all the pipelining the engine needs, and sleeps `sleep_ns` while an integrator runs (see `pace` above).
constexpr unsigned FILL_TMA_SRC = 16384;
__global__ void __launch_bounds__(32) zero_fill_tma_kernel(unsigned char* p, unsigned long long n_bytes16, unsigned char* tail, int n_tail,
                                                           unsigned block_bytes, unsigned sleep_ns, const int* pace) {
    __shared__ __align__(128) unsigned char zsrc[FILL_TMA_SRC];
    for (unsigned i = threadIdx.x * 16; i < block_bytes; i += 32 * 16) *reinterpret_cast<uint4*>(zsrc + i) = make_uint4(0u, 0u, 0u, 0u);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the generic-proxy stores above are visible to the bulk-copy engine
    __syncwarp();
    if (blockIdx.x == 0 && (int)threadIdx.x < n_tail) tail[threadIdx.x] = 0;
    if (threadIdx.x != 0) return;
    const unsigned src = (unsigned)__cvta_generic_to_shared(zsrc);
    const unsigned long long n_blocks = (n_bytes16 + block_bytes - 1) / block_bytes;
    bool paced = sleep_ns != 0 && (!pace || *(const volatile int*)pace != 0);
    unsigned it = 0;
    for (unsigned long long b = blockIdx.x; b < n_blocks; b += gridDim.x) {
        const unsigned long long off = b * block_bytes;
        const unsigned long long left = n_bytes16 - off;
        const unsigned sz = left < block_bytes ? (unsigned)left : block_bytes;
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" :: "l"(p + off), "r"(src), "r"(sz) : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        if (paced) __nanosleep(sleep_ns);
        if (sleep_ns && pace && (++it & 15u) == 0) paced = *(const volatile int*)pace != 0;
    }
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // every block has been written before the kernel ends
}

// ---------------------------------------------------------------- test hook: force / potential at points
template <typename T>
__global__ void eval_force_kernel(const PotDev* pots, int trial, const T* tab, const double* tab0, const double* tab64,
                                  const double* xyz, long long n, double c, double s, double* F, double* Phi) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PotS<T>* P = reinterpret_cast<PotS<T>*>(smem_raw);
    PotS<double>* P64 = reinterpret_cast<PotS<double>*>(smem_raw + ((sizeof(PotS<T>) + 15) / 16) * 16);
    load_pot<T>(pots[trial], P, tab, nullptr, nullptr, false, (int)threadIdx.x, (int)blockDim.x);
    if (Phi) load_pot<double>(pots[trial], P64, tab64, tab0, nullptr, false, (int)threadIdx.x, (int)blockDim.x);
    __syncthreads();
    const long long i_raw = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const bool live = i_raw < n;  // all lanes stay alive: the lambda iteration votes across the warp
    const long long i = live ? i_raw : n - 1;
    T fx, fy, fz, ph;
    float lam = -1.0f;
    total_force<T, false, POT_GENERIC>(*P, P->tab, (T)xyz[3 * i], (T)xyz[3 * i + 1], (T)xyz[3 * i + 2], (T)c, (T)s, fx, fy, fz, ph, lam);
    if (live) { F[3 * i] = fx; F[3 * i + 1] = fy; F[3 * i + 2] = fz; }
    if (Phi) {
        double gx, gy, gz, p64;
        lam = -1.0f;
        total_force<double, true, POT_GENERIC>(*P64, P64->tab, xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], c, s, gx, gy, gz, p64, lam);
        if (live) Phi[i] = p64;
    }
}

// ---------------------------------------------------------------- roofline denominator: plain FMA throughput
template <typename T>
__global__ void __launch_bounds__(256) fma_peak_kernel(T* out, int iters, T seed) {
    T a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const T m = (T)0.999999, b = (T)1e-6;
#pragma unroll 8
    for (int i = 0; i < iters; ++i) {   // unrolled so that the loop counter and branch are 1 in 66 instructions, not 1 in 5
        a0 = fma_t(a0, m, b); a1 = fma_t(a1, m, b); a2 = fma_t(a2, m, b); a3 = fma_t(a3, m, b);
        a4 = fma_t(a4, m, b); a5 = fma_t(a5, m, b); a6 = fma_t(a6, m, b); a7 = fma_t(a7, m, b);
    }
    out[blockIdx.x * (long long)blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

}  // namespace smx
