// stage1.cu -- isochrone weighting and sampler tables (DESIGN.md R-C2,R-C3).
// Everything that decides a star count is fp64 with explicit round-to-nearest intrinsics
// (__dmul_rn etc. are never contracted into FMAs), so the tables are bit-identical on any
// IEEE machine.
#include "pcmd_internal.cuh"

#define TWO_M64 5.42101086242752217e-20
#define TWO32 4294967296.0

// e^-t, t >= 0, from basic operations only (R-C3): degree-6 Taylor polynomial of e^-r at
// r = t 2^-16 in Horner form, then sixteen squarings.
__device__ double expneg_basic(double t) {
    if (t > 64.0) return 0.0;
    const double c[7] = {0.0, 1.0, 1.0 / 2.0, 1.0 / 3.0, 1.0 / 4.0, 1.0 / 5.0, 1.0 / 6.0};
    double r = __dmul_rn(t, 1.0 / 65536.0);
    double p = 1.0;
#pragma unroll
    for (int k = 6; k >= 1; --k) p = __dsub_rn(1.0, __dmul_rn(__dmul_rn(r, c[k]), p));
#pragma unroll
    for (int i = 0; i < 16; ++i) p = __dmul_rn(p, p);
    return p;
}

// grid = (blocks over points, n_models).  Thread 0 of every block computes the MDF weights in the
// stated order (Z values; block 0 stores them); all threads then compute lambda_j and the fluxes.
__global__ void __launch_bounds__(256) k_weights(const DevModel *__restrict__ mdl, const double *__restrict__ sfh,
                          const double *__restrict__ feh_grid, const int32_t *__restrict__ age_idx,
                          const int32_t *__restrict__ feh_idx, const double *__restrict__ imf_w,
                          const double *__restrict__ absmag, int A, int Z, int J, int Jpad, int B,
                          double mdf_cut, double zp0, double zp1, double zp2, double zp3,
                          double *__restrict__ mdfw_out, double *__restrict__ lambda_out,
                          PointRec *__restrict__ rec_out, int32_t *status) {
    extern __shared__ double w[];  // [Z]
    const int m = blockIdx.y;
    const DevModel M = mdl[m];
    if (threadIdx.x == 0) {
        double e_min = INFINITY;
        for (int z = 0; z < Z; ++z) {
            double d = __dsub_rn(feh_grid[z], M.feh_mean);
            w[z] = __ddiv_rn(__dmul_rn(d, d), __dmul_rn(__dmul_rn(2.0, M.feh_sigma), M.feh_sigma));
            if (w[z] < e_min) e_min = w[z];
        }
        double G = 0.0;
        for (int z = 0; z < Z; ++z) { w[z] = expneg_basic(__dsub_rn(w[z], e_min)); G = __dadd_rn(G, w[z]); }
        double G2 = 0.0;
        for (int z = 0; z < Z; ++z) {
            w[z] = __ddiv_rn(w[z], G);
            if (w[z] < mdf_cut) w[z] = 0.0;
            G2 = __dadd_rn(G2, w[z]);
        }
        for (int z = 0; z < Z; ++z) {
            w[z] = __ddiv_rn(w[z], G2);
            if (blockIdx.x == 0) mdfw_out[(size_t)m * Z + z] = w[z];
        }
    }
    __syncthreads();
    const double zp[4] = {zp0, zp1, zp2, zp3};
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Jpad) return;
    PointRec r;
    r.T0 = 0xFFFFFFFFu; r.off = 0; r.len = 0; r.k0 = 0;
    r.f[0] = r.f[1] = r.f[2] = r.f[3] = 0.f;
    if (j < J) {
        double lam = __dmul_rn(__dmul_rn(sfh[(size_t)m * A + age_idx[j]], w[feh_idx[j]]), imf_w[j]);
        lambda_out[(size_t)m * J + j] = lam;
        if (!(lam >= 0.0) || lam > PCMD_LAMBDA_MAX) atomicMin(status, PCMD_ERANGE);
        for (int b = 0; b < B; ++b)  // fluxes according to the distance
            r.f[b] = (float)exp10(-0.4 * (absmag[(size_t)j * B + b] + M.dmod - zp[b]));
    }
    rec_out[(size_t)m * Jpad + j] = r;
}

// Range [k_lo, k_hi] of the relative pmf q[k] >= 2^-64 (R-C2 step 1), one thread per point.
__global__ void k_table_range(const double *__restrict__ lambda, int J, int n_models,
                              uint32_t *__restrict__ rawcnt, uint32_t *__restrict__ klo_out) {
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= J * n_models) return;
    int m = idx / J, j = idx - m * J;
    double lam = lambda[idx];
    uint32_t n = 0, klo = 0;
    if (lam > 0.0 && lam <= PCMD_LAMBDA_MAX) {
        long long mode = (long long)floor(lam), k_hi = mode, k_lo = mode;
        double v = 1.0;
        for (long long k = mode + 1;; ++k) {
            v = __dmul_rn(v, __ddiv_rn(lam, (double)k));
            if (v < TWO_M64) break;
            k_hi = k;
        }
        v = 1.0;
        for (long long k = mode - 1; k >= 0; --k) {
            v = __dmul_rn(v, __ddiv_rn((double)(k + 1), lam));
            if (v < TWO_M64) break;
            k_lo = k;
        }
        n = (uint32_t)(k_hi - k_lo + 1);
        klo = (uint32_t)k_lo;
    }
    rawcnt[(size_t)m * (J + 1) + j] = n;
    klo_out[idx] = klo;
}

// In-place exclusive scan of cnt[m][0..J] (entry J receives the total), one block per model.
__global__ void k_scan(uint32_t *__restrict__ cnt, int J, int64_t cap, int32_t *status) {
    __shared__ uint32_t warp_sum[32];
    __shared__ uint32_t carry;
    uint32_t *c = cnt + (size_t)blockIdx.x * (J + 1);
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int base = 0; base < J; base += blockDim.x) {
        int j = base + threadIdx.x;
        uint32_t v = (j < J) ? c[j] : 0, x = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
        if (lane == 31) warp_sum[wid] = x;
        __syncthreads();
        if (wid == 0) {
            uint32_t s = (lane < nw) ? warp_sum[lane] : 0;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, s, d); if (lane >= d) s += y; }
            warp_sum[lane] = s;
        }
        __syncthreads();
        uint32_t before = carry + (wid ? warp_sum[wid - 1] : 0) + (x - v);
        if (j < J) c[j] = before;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = before + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        c[J] = carry;
        if ((int64_t)carry > cap) atomicMin(status, PCMD_ENOMEM);
    }
}

// R-C2 steps 1-3 for one point per thread: q[k] by the two recurrences into scratch, S summed
// in increasing k, thresholds T[k] = (uint64)((c/S) 2^32 + 0.5) written over q.  Also counts
// the stored thresholds (0 < T < 2^32) and k0 = first k with T > 0.
__global__ void k_table_fill(const double *__restrict__ lambda, int J, int n_models,
                             const uint32_t *__restrict__ rawoff, const uint32_t *__restrict__ klo_in,
                             double *__restrict__ qbuf, int64_t cap, uint32_t *__restrict__ stcnt,
                             PointRec *__restrict__ rec, int Jpad) {
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= J * n_models) return;
    int m = idx / J, j = idx - m * J;
    const uint32_t *ro = rawoff + (size_t)m * (J + 1);
    uint32_t off = ro[j], n = ro[j + 1] - off, stored = 0, k0 = 0;
    if (n > 0 && (int64_t)ro[J] <= cap) {
        double lam = lambda[idx];
        double *q = qbuf + (size_t)m * cap + off;
        long long k_lo = klo_in[idx], mode = (long long)floor(lam), k_hi = k_lo + n - 1;
        q[mode - k_lo] = 1.0;
        double v = 1.0;
        for (long long k = mode + 1; k <= k_hi; ++k) { v = __dmul_rn(v, __ddiv_rn(lam, (double)k)); q[k - k_lo] = v; }
        v = 1.0;
        for (long long k = mode - 1; k >= k_lo; --k) { v = __dmul_rn(v, __ddiv_rn((double)(k + 1), lam)); q[k - k_lo] = v; }
        double S = 0.0;
        for (uint32_t i = 0; i < n; ++i) S = __dadd_rn(S, q[i]);
        double c = 0.0;
        uint32_t zeros = 0;
        for (uint32_t i = 0; i < n; ++i) {
            c = __dadd_rn(c, q[i]);
            unsigned long long t = __double2ull_rz(__dadd_rn(__dmul_rn(__ddiv_rn(c, S), TWO32), 0.5));
            q[i] = __longlong_as_double((long long)t);  // q[i] is no longer needed
            if (t == 0ull) zeros++;
            else if (t < 4294967296ull) stored++;
        }
        k0 = (uint32_t)k_lo + zeros;
    }
    stcnt[(size_t)m * (J + 1) + j] = stored;
    rec[(size_t)m * Jpad + j].k0 = k0;
    rec[(size_t)m * Jpad + j].len = stored;
}

// Compacts the stored thresholds (minus 1) into the model's table and completes the records.
__global__ void k_table_compact(int J, int n_models, const uint32_t *__restrict__ rawoff,
                                const double *__restrict__ qbuf, int64_t cap,
                                const uint32_t *__restrict__ stoff, uint32_t *__restrict__ tab,
                                PointRec *__restrict__ rec, int Jpad) {
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= J * n_models) return;
    int m = idx / J, j = idx - m * J;
    const uint32_t *ro = rawoff + (size_t)m * (J + 1);
    const uint32_t *so = stoff + (size_t)m * (J + 1);
    if ((int64_t)ro[J] > cap) return;
    uint32_t off = ro[j], n = ro[j + 1] - off, dst = so[j];
    const double *T = qbuf + (size_t)m * cap + off;
    uint32_t *out = tab + (size_t)m * cap;
    uint32_t w = dst;
    for (uint32_t i = 0; i < n; ++i) {
        unsigned long long t = (unsigned long long)__double_as_longlong(T[i]);
        if (t != 0ull && t < 4294967296ull) out[w++] = (uint32_t)(t - 1ull);
    }
    PointRec *r = rec + (size_t)m * Jpad + j;
    r->off = dst;
    r->T0 = (w > dst) ? out[dst] : 0xFFFFFFFFu;
}


// ---------------------------------------------------------------------------------------------
// Stage-2 work layout: classify the groups of four points, sort them by class, cut segments, and
// lay out the padded search tables of the D classes.  One block per model.
// Class of a point:  L1/L2/L4: k0 = 0 and the probability of more than L stars is below 2^-10
// (its (L+1)-th threshold is above 2^32 (1 - 2^-10)): L inline compares decide the draw;
// S3/S4: k0 = 0 and more than 7 / 15 stars have probability below 2^-10: the first 2^D - 1 thresholds are
// searched branch-free in shared memory, the overflow path finishes the rest;
// D5/D7/D9: table of at most 2^D - 1 thresholds, searched branch-free in shared memory;
// class 0: longer tables, bisection in global memory.  A group takes the most expensive class
// of its four points.
#ifndef S2_OVF_LOG2
#define S2_OVF_LOG2 10
#endif
#define S2_OVF_THR (0xFFFFFFFFu - (1u << (32 - S2_OVF_LOG2)))   /* 2^32 (1 - 2^-10) - 1 */

#ifndef S2_RARE_LOG2
#define S2_RARE_LOG2 8
#endif
#define S2_RARE_THR (0xFFFFFFFFu - (1u << (32 - S2_RARE_LOG2)))   /* P(any star) < 2^-8 per draw */

__device__ __forceinline__ int point_class(const PointRec &r, const uint32_t *__restrict__ tab) {
    if (r.len == 0 && r.k0 == 0) return S2_CLS_NONE;      // never a star
    if (r.k0 == 0) {
        if (r.T0 >= S2_RARE_THR && (r.len <= 1 || tab[r.off + 1] >= S2_OVF_THR)) return S2_CLS_L0;
        if (r.len <= 1 || tab[r.off + 1] >= S2_OVF_THR) return S2_CLS_L1;
        if (r.len <= 2 || tab[r.off + 2] >= S2_OVF_THR) return S2_CLS_L2;
        if (r.len <= 4 || tab[r.off + 4] >= S2_OVF_THR) return S2_CLS_L4;
        if (r.len <= 7 || tab[r.off + 7] >= S2_OVF_THR) return S2_CLS_S3;
        if (r.len <= 15 || tab[r.off + 15] >= S2_OVF_THR) return S2_CLS_S4;
    }
    if (r.len <= 31) return S2_CLS_D5;
    if (r.len <= 63) return S2_CLS_D6;
    if (r.len <= 127) return S2_CLS_D7;
    if (r.len <= 255) return S2_CLS_D8;
    if (r.len <= 511) return S2_CLS_D9;
    return 0;
}

// Stable counting sort of the groups by class (positions only), chunk layout, arena layout.
// One block per model.
//
// Cost model of stage 2 (cost units ~ SM cycles per warp and group, measured per class loop with
// ncu, profiles/): the static partition of the chunk sequence among the persistent CTAs is by cost.
__constant__ uint32_t c_s2_group_cost[S2_NCLASS] = {S2_COST_G, S2_COST_D9, S2_COST_D8, S2_COST_D7, S2_COST_D6, S2_COST_D5, S2_COST_S4, S2_COST_S3,
                                                    S2_COST_L4, S2_COST_L2, S2_COST_L1, S2_COST_L0};
__global__ void __launch_bounds__(1024) k_group_sort(const uint8_t *__restrict__ cls_all, int Jpad,
                                                     int64_t arena_cap, int n_seg, uint32_t *__restrict__ pos_all,
                                                     ModelPlan *__restrict__ plan_all) {
    pdl_enter<PDL_EARLY_SORT>();
    __shared__ uint32_t wcnt[32][S2_NCLASS];
    __shared__ uint32_t count[S2_NCLASS + 1], carry[S2_NCLASS], cls_start[S2_NCLASS + 1];
    const int m = blockIdx.x, n_groups = Jpad >> 2;
    const uint8_t *gcls = cls_all + (size_t)m * n_groups;
    uint32_t *gpos = pos_all + (size_t)m * n_groups;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if (threadIdx.x <= S2_NCLASS) count[threadIdx.x] = 0;
    __syncthreads();
    for (int g = threadIdx.x; g < n_groups; g += blockDim.x) atomicAdd(&count[gcls[g]], 1u);
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0;
        for (int c = 0; c < S2_NCLASS; ++c) { cls_start[c] = run; carry[c] = 0; run += count[c]; }
        cls_start[S2_NCLASS] = run;
    }
    __syncthreads();
    for (int base = 0; base < n_groups; base += blockDim.x) {
        const int g = base + threadIdx.x;
        const int cls = (g < n_groups) ? (int)gcls[g] : S2_CLS_NONE;
        uint32_t rank = 0;
#pragma unroll
        for (int k = 0; k < S2_NCLASS; ++k) {
            const uint32_t bal = __ballot_sync(0xffffffffu, cls == k);
            if (cls == k) rank = __popc(bal & ((1u << lane) - 1u));
            if (lane == 0) wcnt[wid][k] = __popc(bal);
        }
        __syncthreads();
        if (threadIdx.x < S2_NCLASS) {
            const int k = threadIdx.x;
            uint32_t run = carry[k];
            for (int w = 0; w < nw; ++w) { const uint32_t t = wcnt[w][k]; wcnt[w][k] = run; run += t; }
            carry[k] = run;
        }
        __syncthreads();
        if (g < n_groups) gpos[g] = (cls < S2_NCLASS) ? cls_start[cls] + wcnt[wid][cls] + rank : 0xFFFFFFFFu;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        ModelPlan t;
        // padded search tables: D9 first, then D7, D5; a class that does not fit the arena is
        // demoted to bisection in global memory (run_cls = 0)
        const int64_t stride[8] = {0, 4 << 9, 4 << 8, 4 << 7, 4 << 6, 4 << 5, 4 << 4, 4 << 3};      // words of padded tables per group
        int first_d = S2_CLS_D9;
        for (;;) {
            int64_t need = 0;
            for (int c = first_d; c <= S2_CLS_S3; ++c) need += stride[c] * (int64_t)count[c];
            if (need <= arena_cap || first_d > S2_CLS_S3) break;
            first_d++;
        }
        // A small model (c1: 64 groups) cut into full-size chunks has fewer chunks than the n_seg segments stage 2
        // wants per tile (a segment is at least one chunk), and its few work units then run their groups one after
        // the other: chunks are shrunk to about 1/n_seg of the model's cost.  Models of the larger configurations
        // (cost / n_seg above a full chunk) keep their chunk sizes.
        uint32_t group_cost_total = 0;        // 32-bit like the plan's cost_total
        for (int c = 0; c < S2_NCLASS; ++c) {
            const bool demoted_c = c >= S2_CLS_D9 && c <= S2_CLS_S3 && !(c >= first_d && c <= S2_CLS_S3);
            group_cost_total += count[c] * c_s2_group_cost[demoted_c ? 0 : c];
        }
        const uint32_t chunk_cost_target = group_cost_total / (uint32_t)max(n_seg, 1);
        int64_t off = 0;
        int32_t chunks = 0;
        uint32_t cost = 0, cmax = 0;
        for (int c = 0; c < S2_NCLASS; ++c) {
            t.cls_start[c] = (int32_t)cls_start[c];
            t.arena_off[c] = 0;
            const bool in_arena = c >= first_d && c <= S2_CLS_S3;
            if (in_arena) { t.arena_off[c] = off; off += stride[c] * (int64_t)count[c]; }
            const bool demoted = c >= S2_CLS_D9 && c <= S2_CLS_S3 && !in_arena;
            t.run_cls[c] = demoted ? 0 : c;
            int cg = in_arena ? min((int)(S2_TABW / stride[c]), S2_CHUNK) : S2_CHUNK;     // groups per chunk
            if (chunk_cost_target < (uint32_t)cg * c_s2_group_cost[t.run_cls[c]])
                cg = (int)max(chunk_cost_target / c_s2_group_cost[t.run_cls[c]], 1u);
            t.chunk_groups[c] = cg;
            t.chunk_cost[c] = (uint32_t)cg * c_s2_group_cost[t.run_cls[c]] + S2_COST_CHUNK;
            const int n = (int)count[c], nch = (n + cg - 1) / cg;
            t.chunk_start[c] = chunks;
            t.cost_start[c] = cost;
            chunks += nch;
            cost += (uint32_t)nch * t.chunk_cost[c];     // the last (ragged) chunk is charged as a full one
            if (nch > 0 && t.chunk_cost[c] > cmax) cmax = t.chunk_cost[c];
        }
        t.cls_start[S2_NCLASS] = (int32_t)cls_start[S2_NCLASS];
        t.chunk_start[S2_NCLASS] = chunks;
        t.cost_start[S2_NCLASS] = cost;
        t.n_chunks = chunks; t.first_d = first_d; t.cost_total = cost; t.cost_max = cmax;
        plan_all[m] = t;
    }
}

// Stage 1 for one point per thread, fused (the main path; the separate kernels above still build the few
// tables of the Poisson sky and of the aggregated sampler): MDF weights (thread 0 of the block, R-C3 order),
// lambda_j, per-star fluxes, the R-C2 table (range pass, raw entries into a scratch region taken from a
// per-model bump allocator, thresholds, compaction into a second bump-allocated region), the point record
// and the class of the point's group.  Table regions are handed out in completion order, so their PLACE
// varies from run to run; their contents, and everything stage 2 computes from them, do not.
__global__ void __launch_bounds__(128) k_points(const DevModel *__restrict__ mdl, const double *__restrict__ sfh,
                         const double *__restrict__ feh_grid, const int32_t *__restrict__ age_idx,
                         const int32_t *__restrict__ feh_idx, const double *__restrict__ imf_w,
                         const double *__restrict__ absmag, int A, int Z, int J, int Jpad, int B,
                         double mdf_cut, double zp0, double zp1, double zp2, double zp3,
                         double *__restrict__ mdfw_out, double *__restrict__ lambda_out,
                         double *__restrict__ qbuf, int64_t cap, uint32_t *__restrict__ tab_all,
                         uint32_t *__restrict__ alloc, PointRec *__restrict__ rec_out,
                         uint8_t *__restrict__ gcls_out, int32_t *status) {
    pdl_enter<PDL_EARLY_POINTS>();
    extern __shared__ double w[];  // [Z]
    const int m = blockIdx.y;
    const DevModel M = mdl[m];
    if (threadIdx.x == 0) {
        double e_min = INFINITY;
        for (int z = 0; z < Z; ++z) {
            double d = __dsub_rn(feh_grid[z], M.feh_mean);
            w[z] = __ddiv_rn(__dmul_rn(d, d), __dmul_rn(__dmul_rn(2.0, M.feh_sigma), M.feh_sigma));
            if (w[z] < e_min) e_min = w[z];
        }
        double G = 0.0;
        for (int z = 0; z < Z; ++z) { w[z] = expneg_basic(__dsub_rn(w[z], e_min)); G = __dadd_rn(G, w[z]); }
        double G2 = 0.0;
        for (int z = 0; z < Z; ++z) {
            w[z] = __ddiv_rn(w[z], G);
            if (w[z] < mdf_cut) w[z] = 0.0;
            G2 = __dadd_rn(G2, w[z]);
        }
        for (int z = 0; z < Z; ++z) {
            w[z] = __ddiv_rn(w[z], G2);
            if (blockIdx.x == 0) mdfw_out[(size_t)m * Z + z] = w[z];
        }
    }
    __syncthreads();
    const double zp[4] = {zp0, zp1, zp2, zp3};
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    PointRec r;
    r.T0 = 0xFFFFFFFFu; r.off = 0; r.len = 0; r.k0 = 0;
    r.f[0] = r.f[1] = r.f[2] = r.f[3] = 0.f;
    int pcls = S2_CLS_NONE;
    if (j < J) {
        const double lam = __dmul_rn(__dmul_rn(sfh[(size_t)m * A + age_idx[j]], w[feh_idx[j]]), imf_w[j]);
        lambda_out[(size_t)m * J + j] = lam;
        if (!(lam >= 0.0) || lam > PCMD_LAMBDA_MAX) atomicMin(status, PCMD_ERANGE);
        for (int b = 0; b < B; ++b)  // fluxes according to the distance
            r.f[b] = (float)exp10(-0.4 * (absmag[(size_t)j * B + b] + M.dmod - zp[b]));
        if (lam > 0.0 && lam <= PCMD_LAMBDA_MAX) {
            // R-C2 step 1: range of the relative pmf >= 2^-64
            const long long mode = (long long)floor(lam);
            long long k_hi = mode, k_lo = mode;
            double v = 1.0;
            for (long long k = mode + 1;; ++k) {
                v = __dmul_rn(v, __ddiv_rn(lam, (double)k));
                if (v < TWO_M64) break;
                k_hi = k;
            }
            v = 1.0;
            for (long long k = mode - 1; k >= 0; --k) {
                v = __dmul_rn(v, __ddiv_rn((double)(k + 1), lam));
                if (v < TWO_M64) break;
                k_lo = k;
            }
            const uint32_t n = (uint32_t)(k_hi - k_lo + 1);
            const uint32_t off = atomicAdd(&alloc[2 * m], n);
            if ((int64_t)off + n > cap) atomicMin(status, PCMD_ENOMEM);
            else {
                double *q = qbuf + (size_t)m * cap + off;
                q[mode - k_lo] = 1.0;
                v = 1.0;
                for (long long k = mode + 1; k <= k_hi; ++k) { v = __dmul_rn(v, __ddiv_rn(lam, (double)k)); q[k - k_lo] = v; }
                v = 1.0;
                for (long long k = mode - 1; k >= k_lo; --k) { v = __dmul_rn(v, __ddiv_rn((double)(k + 1), lam)); q[k - k_lo] = v; }
                double S = 0.0;
                for (uint32_t i = 0; i < n; ++i) S = __dadd_rn(S, q[i]);
                double cs = 0.0;
                uint32_t zeros = 0, stored = 0;
                for (uint32_t i = 0; i < n; ++i) {      // R-C2 step 3; q[i] is no longer needed once its threshold is known
                    cs = __dadd_rn(cs, q[i]);
                    const unsigned long long t = __double2ull_rz(__dadd_rn(__dmul_rn(__ddiv_rn(cs, S), TWO32), 0.5));
                    q[i] = __longlong_as_double((long long)t);
                    if (t == 0ull) zeros++;
                    else if (t < 4294967296ull) stored++;
                }
                const uint32_t dst = atomicAdd(&alloc[2 * m + 1], stored);    // stored <= n: the compact region cannot overflow if the raw one did not
                uint32_t *out = tab_all + (size_t)m * cap;
                uint32_t wr = dst;
                PCMD_CHK((int64_t)dst + stored <= cap && mode >= k_lo && mode <= k_hi);
                for (uint32_t i = 0; i < n; ++i) {
                    const unsigned long long t = (unsigned long long)__double_as_longlong(q[i]);
                    if (t != 0ull && t < 4294967296ull) out[wr++] = (uint32_t)(t - 1ull);
                }
                PCMD_CHK(wr == dst + stored);
                r.k0 = (uint32_t)k_lo + zeros; r.len = stored; r.off = dst;
                r.T0 = stored ? out[dst] : 0xFFFFFFFFu;
                pcls = point_class(r, out);
            }
        }
    }
    if (j < Jpad) rec_out[(size_t)m * Jpad + j] = r;
    // class of the group of four points = its most expensive point (threads 4g .. 4g+3 are neighbouring lanes)
    pcls = min(pcls, __shfl_xor_sync(0xffffffffu, pcls, 1));
    pcls = min(pcls, __shfl_xor_sync(0xffffffffu, pcls, 2));
    if (j < Jpad && (j & 3) == 0) gcls_out[(size_t)m * (Jpad >> 2) + (j >> 2)] = (uint8_t)pcls;
}

// Group records at their sorted places and the padded search tables of the D classes: one warp
// per group.  Lane w < 4 writes point w's part of the record; all lanes write the padded tables
// (2^D words per point: the stored thresholds minus 1, then 0xFFFFFFFF).
__global__ void __launch_bounds__(256) k_group_emit(const PointRec *__restrict__ rec_all,
                                                    const uint32_t *__restrict__ tab_all, int64_t cap, int Jpad,
                                                    const uint8_t *__restrict__ cls_all,
                                                    const uint32_t *__restrict__ pos_all,
                                                    const ModelPlan *__restrict__ plan_all, GroupRec *__restrict__ grp_all,
                                                    uint32_t *__restrict__ arena_all, int64_t arena_cap) {
    pdl_enter<PDL_EARLY_EMIT>();
    const int m = blockIdx.y, n_groups = Jpad >> 2, lane = threadIdx.x & 31;
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (g >= n_groups) return;
    const int cls = (int)cls_all[(size_t)m * n_groups + g];
    if (cls >= S2_NCLASS) return;
    const uint32_t pos = pos_all[(size_t)m * n_groups + g];
    const PointRec *rec = rec_all + (size_t)m * Jpad;
    const uint32_t *tab = tab_all + (size_t)m * cap;
    GroupRec *o = grp_all + (size_t)m * n_groups + pos;
    if (lane < 4) {
        const int w = lane;
        const PointRec r = rec[4 * g + w];
        uint32_t tmin = r.T0;                       // smallest first threshold of the four points
        tmin = min(tmin, __shfl_xor_sync(0xFu, tmin, 1));
        tmin = min(tmin, __shfl_xor_sync(0xFu, tmin, 2));
        if (w == 0) { o->g_orig = (uint32_t)g; o->cls = (uint32_t)cls; o->tmin = tmin; o->pad1 = 0; }
#pragma unroll
        for (int i = 0; i < 5; ++i) o->T[i][w] = ((uint32_t)i < r.len) ? tab[r.off + i] : 0xFFFFFFFFu;
        if (cls <= S2_CLS_S3) {
            // the search classes keep the first count here: k0 (bisection class), or, for a class whose padded
            // tables are staged in shared memory, the float k0 - (word offset of the point's table in its
            // chunk's stage buffer): stage 2 then gets the count from the ADDRESS of the found entry
            const ModelPlan *pl = plan_all + m;
            if (cls >= pl->first_d) {
                const int D = s2_class_depth(cls);
                const int g_local = ((int)pos - pl->cls_start[cls]) % pl->chunk_groups[cls];
                o->T[4][w] = __float_as_uint((float)((int)r.k0 - ((g_local * 4 + w) << D)));
                if (cls >= S2_CLS_S4) o->T[3][w] = ((1u << D) - 1u < r.len) ? tab[r.off + (1u << D) - 1u] : 0xFFFFFFFFu;
            } else o->T[4][w] = r.k0;
        }
#pragma unroll
        for (int b = 0; b < 4; ++b) o->f[w][b] = r.f[b];
    }
    const ModelPlan *t = plan_all + m;
    if (cls >= t->first_d && cls <= S2_CLS_S3) {
        const int D = s2_class_depth(cls);
        uint32_t *dst = arena_all + (size_t)m * arena_cap + t->arena_off[cls] +
                        (int64_t)((int)pos - t->cls_start[cls]) * (4 << D);
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const uint32_t off = rec[4 * g + w].off, len = min(rec[4 * g + w].len, (1u << D) - 1u);   // S3/S4: the first 2^D - 1 only
            for (int i = lane; i < (1 << D); i += 32) dst[(w << D) + i] = ((uint32_t)i < len) ? tab[off + i] : 0xFFFFFFFFu;
        }
    }
}

int pcmd_build_tables(pcmd_ctx *c, const double *d_lambda, int J, int n_models, uint32_t *rawcnt,
                      uint32_t *klo, double *q, int64_t cap, uint32_t *stcnt, uint32_t *tab,
                      PointRec *rec, int Jpad, cudaStream_t s) {
    int total = J * n_models, tb = 128, gb = (total + tb - 1) / tb;
    k_table_range<<<gb, tb, 0, s>>>(d_lambda, J, n_models, rawcnt, klo);
    PCMD_LAUNCHED(c);
    k_scan<<<n_models, 1024, 0, s>>>(rawcnt, J, cap, c->d_status);
    PCMD_LAUNCHED(c);
    k_table_fill<<<gb, tb, 0, s>>>(d_lambda, J, n_models, rawcnt, klo, q, cap, stcnt, rec, Jpad);
    PCMD_LAUNCHED(c);
    k_scan<<<n_models, 1024, 0, s>>>(stcnt, J, cap, c->d_status);
    PCMD_LAUNCHED(c);
    k_table_compact<<<gb, tb, 0, s>>>(J, n_models, rawcnt, q, cap, stcnt, tab, rec, Jpad);
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}

int pcmd_launch_stage1(pcmd_ctx *c, int n_models, cudaStream_t s) {
    const int n_groups = c->Jpad >> 2;
    if (c->sampler_mode == 1) {      // aggregated sampler: lambda and fluxes only, then its own tables (agg.cu)
        k_weights<<<dim3((c->Jpad + 255) / 256, n_models), 256, c->Z * sizeof(double), s>>>(
            c->d_model, c->d_sfh, c->d_feh_grid, c->d_age_idx, c->d_feh_idx, c->d_imf_w, c->d_absmag, c->A,
            c->Z, c->J, c->Jpad, c->B, c->mdf_cut, c->zp[0], c->zp[1], c->zp[2], c->zp[3], c->d_mdfw,
            c->d_lambda, c->d_rec, c->d_status);
        PCMD_LAUNCHED(c);
        return pcmd_launch_agg_tables(c, n_models, s);
    }
    PCMD_CUDA(c, cudaMemsetAsync(c->d_alloc, 0, (size_t)n_models * 2 * sizeof(uint32_t), s));
    pcmd_launch_pdl(k_points, dim3((c->Jpad + 127) / 128, n_models), dim3(128), c->Z * sizeof(double), s, 
        c->d_model, c->d_sfh, c->d_feh_grid, c->d_age_idx, c->d_feh_idx, c->d_imf_w, c->d_absmag, c->A, c->Z, c->J,
        c->Jpad, c->B, c->mdf_cut, c->zp[0], c->zp[1], c->zp[2], c->zp[3], c->d_mdfw, c->d_lambda, c->d_q,
        c->cap_raw, c->d_tab, c->d_alloc, c->d_rec, c->d_gcls, c->d_status);
    PCMD_LAUNCHED(c);
    pcmd_launch_pdl(k_group_sort, dim3(n_models), dim3(1024), 0, s, c->d_gcls, c->Jpad, c->arena_cap, c->n_seg, c->d_gpos, c->d_plan);
    PCMD_LAUNCHED(c);
    pcmd_launch_pdl(k_group_emit, dim3((n_groups + 7) / 8, n_models), dim3(256), 0, s, c->d_rec, c->d_tab, c->cap_raw, c->Jpad, c->d_gcls,
                                                                    c->d_gpos, c->d_plan, c->d_grp, c->d_arena,
                                                                    c->arena_cap);
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}

// One sampler table per band for Poisson(sky_b) (R-Q11), built once at pcmd_create with the
// same kernels (J = B "points", one "model").
int pcmd_build_sky_tables(pcmd_ctx *c) {
    const int B = c->B;
    double maxsky = 0.0;
    for (int b = 0; b < B; ++b) maxsky = c->sky[b] > maxsky ? c->sky[b] : maxsky;
    int64_t cap = (int64_t)B * (int64_t)(20.0 * sqrt(maxsky) + 96.0);
    double *d_lam = nullptr, *d_q = nullptr;
    uint32_t *d_raw = nullptr, *d_klo = nullptr, *d_st = nullptr;
    PointRec *d_rec = nullptr;
    PCMD_CUDA(c, cudaMalloc(&d_lam, B * sizeof(double)));
    PCMD_CUDA(c, cudaMalloc(&d_q, cap * sizeof(double)));
    PCMD_CUDA(c, cudaMalloc(&d_raw, (B + 1) * sizeof(uint32_t)));
    PCMD_CUDA(c, cudaMalloc(&d_st, (B + 1) * sizeof(uint32_t)));
    PCMD_CUDA(c, cudaMalloc(&d_klo, B * sizeof(uint32_t)));
    PCMD_CUDA(c, cudaMalloc(&d_rec, 4 * sizeof(PointRec)));
    PCMD_CUDA(c, cudaMalloc(&c->d_sky_tab, cap * sizeof(uint32_t)));
    PCMD_CUDA(c, cudaMemset(d_rec, 0, 4 * sizeof(PointRec)));
    PCMD_CUDA(c, cudaMemcpy(d_lam, c->sky, B * sizeof(double), cudaMemcpyHostToDevice));
    int rc = pcmd_build_tables(c, d_lam, B, 1, d_raw, d_klo, d_q, cap, d_st, c->d_sky_tab, d_rec, 4, 0);
    if (rc) return rc;
    PointRec h[4];
    PCMD_CUDA(c, cudaMemcpy(h, d_rec, 4 * sizeof(PointRec), cudaMemcpyDeviceToHost));
    c->sky_cap = (uint32_t)cap;
    for (int b = 0; b < B; ++b) c->sky_rec[b] = h[b];   // (off, len, k0) of each band's table
    cudaFree(d_lam); cudaFree(d_q); cudaFree(d_raw); cudaFree(d_st); cudaFree(d_klo); cudaFree(d_rec);
    return PCMD_OK;
}
