// agg.cu -- the aggregated sampler (sampler_mode = 1; PAPER.md:75 footnote 3: the sum of the Poisson star
// counts of a pixel is itself Poisson with mean N_pix; DESIGN.md R-A1): one Poisson draw of the pixel's number
// of stars, then every star placed on an isochrone point with probability lambda_j / N_pix by inversion of an
// integer cumulative weight table.  O(N_pix) random numbers per pixel instead of O(J): the cheaper path when
// N_pix << J (BASELINE c2 / c4).  A different random stream from the per-point sampler (stream 4 of R-C1), with
// its own oracle function; everything that decides a star is integer or explicitly rounded fp64.
#include "pcmd_internal.cuh"

#define AGG_SHIFT 28                 // guide cell = r >> 28 (r < W ~ 2^40: 4096 cells, + 2 for W slightly above 2^40)
#define AGG_CELLS 4098
#define AGG_THREADS 512

// One block per model.  Lambda = sum_j lambda_j in increasing j (thread 0: the order is part of the definition),
// w_j = (uint64)((lambda_j / Lambda) 2^40 + 0.5), C = exclusive prefix sums (integers: any order), guide cells.
__global__ void __launch_bounds__(1024) k_agg_tables(const double *__restrict__ lambda_all, int J,
                                                     double *__restrict__ lam_tot, uint64_t *__restrict__ C_all,
                                                     uint32_t *__restrict__ G_all) {
    __shared__ double s_tot;
    __shared__ unsigned long long warp_sum[32];
    __shared__ unsigned long long carry;
    const int m = blockIdx.x;
    const double *lam = lambda_all + (size_t)m * J;
    uint64_t *C = C_all + (size_t)m * (J + 1);
    // the sum is sequential by definition; thread 0 walks chunks staged in shared memory (coalesced loads by the block)
    __shared__ double s_chunk[2048];
    double t = 0.0;
    for (int base = 0; base < J; base += 2048) {
        const int n = min(2048, J - base);
        for (int i = threadIdx.x; i < n; i += blockDim.x) s_chunk[i] = lam[base + i];
        __syncthreads();
        if (threadIdx.x == 0) {
            int i = 0;
            for (; i + 8 <= n; i += 8) {
                double v[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = s_chunk[i + k];
#pragma unroll
                for (int k = 0; k < 8; ++k) t = __dadd_rn(t, v[k]);
            }
            for (; i < n; ++i) t = __dadd_rn(t, s_chunk[i]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { s_tot = t; lam_tot[m] = t; carry = 0ull; }
    __syncthreads();
    const double tot = s_tot;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int base = 0; base < J; base += blockDim.x) {
        const int j = base + threadIdx.x;
        unsigned long long v = 0ull;
        if (j < J && tot > 0.0)
            v = __double2ull_rz(__dadd_rn(__dmul_rn(__ddiv_rn(lam[j], tot), 1099511627776.0), 0.5));
        unsigned long long x = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { unsigned long long y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
        if (lane == 31) warp_sum[wid] = x;
        __syncthreads();
        if (wid == 0) {
            unsigned long long sw = (lane < nw) ? warp_sum[lane] : 0ull;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { unsigned long long y = __shfl_up_sync(0xffffffffu, sw, d); if (lane >= d) sw += y; }
            warp_sum[lane] = sw;
        }
        __syncthreads();
        const unsigned long long before = carry + (wid ? warp_sum[wid - 1] : 0ull) + (x - v);
        if (j < J) C[j] = before;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = before + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) C[J] = carry;
    __syncthreads();
    // guide: G[c] = the largest j <= J-1 with C_j <= c 2^28
    uint32_t *G = G_all + (size_t)m * AGG_CELLS;
    for (int cidx = threadIdx.x; cidx < AGG_CELLS; cidx += blockDim.x) {
        const unsigned long long v = (unsigned long long)cidx << AGG_SHIFT;
        int lo = 0, hi = J - 1;                    // C_0 = 0 <= v
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (C[mid] <= v) lo = mid; else hi = mid - 1;
        }
        G[cidx] = (uint32_t)lo;
    }
}

struct AggArgs {
    const double *lam_tot;     // [n_tab]
    const uint64_t *C;         // [n_tab][J+1]
    const uint32_t *G;         // [n_tab][AGG_CELLS]
    const PointRec *rec;       // [n_tab][Jpad]: per-star fluxes
    const PointRec *trec;      // [n_tab]: (off, len, k0) of the Poisson(Lambda) table
    const uint32_t *ttab;      // [n_tab][tcap]
    const uint64_t *mult;      // [Jpad]
    int64_t tcap, P;
    int J, Jpad, B, mts;
    uint32_t key0, key1, model0;
    float *part;               // [n_models][1][B][P]
    uint64_t *hash; uint32_t *total;
};

// One thread per pixel.  The cumulative table and the guide sit in shared memory when they fit.
template <bool SMEM, bool COUNTS>
__global__ void __launch_bounds__(AGG_THREADS) k_stage2_agg(const AggArgs a) {
    extern __shared__ __align__(16) unsigned char agg_smem[];
    const int m = blockIdx.y, mt = m * a.mts, J = a.J;
    const uint64_t *C = a.C + (size_t)mt * (J + 1);
    const uint32_t *G = a.G + (size_t)mt * AGG_CELLS;
    if (SMEM) {
        uint64_t *sC = reinterpret_cast<uint64_t *>(agg_smem);
        uint32_t *sG = reinterpret_cast<uint32_t *>(sC + (J + 1));
        for (int t = threadIdx.x; t <= J; t += AGG_THREADS) sC[t] = C[t];
        for (int t = threadIdx.x; t < AGG_CELLS; t += AGG_THREADS) sG[t] = G[t];
        __syncthreads();
        C = sC; G = sG;
    }
    const int64_t p64 = (int64_t)blockIdx.x * AGG_THREADS + threadIdx.x;
    if (p64 >= a.P) return;
    const uint32_t p = (uint32_t)p64, mctr = a.model0 + (uint32_t)m;
    const uint64_t W = C[J];
    const PointRec *rec = a.rec + (size_t)mt * a.Jpad;
    uint32_t w[4];
    uint32_t N = 0;
    if (a.lam_tot[mt] > 0.0 && W > 0) {
        const PointRec tr = a.trec[mt];
        philox4x32_10(a.key0, a.key1, p, 0u, mctr, 4u, w);
        N = tr.k0 + count_below(a.ttab + (size_t)mt * a.tcap + tr.off, tr.len, w[0]);
    }
    double F[4] = {0.0, 0.0, 0.0, 0.0};
    uint64_t h = 0;
    // two stars per Philox call, their two searches interleaved (independent chains)
    for (uint32_t s = 0; s < N; s += 2) {
        philox4x32_10(a.key0, a.key1, p, 1u + (s >> 1), mctr, 4u, w);
        const uint64_t r0 = __umul64hi(((uint64_t)w[0] << 32) | w[1], W), r1 = __umul64hi(((uint64_t)w[2] << 32) | w[3], W);
        int lo0 = (int)G[(uint32_t)(r0 >> AGG_SHIFT)], hi0 = (int)G[(uint32_t)(r0 >> AGG_SHIFT) + 1];
        int lo1 = (int)G[(uint32_t)(r1 >> AGG_SHIFT)], hi1 = (int)G[(uint32_t)(r1 >> AGG_SHIFT) + 1];
        PCMD_CHK((r0 >> AGG_SHIFT) + 1 < AGG_CELLS && (r1 >> AGG_SHIFT) + 1 < AGG_CELLS && r0 < W && r1 < W);
        PCMD_CHK(lo0 >= 0 && lo0 <= hi0 && hi0 < a.J && lo1 >= 0 && lo1 <= hi1 && hi1 < a.J);
        while (lo0 < hi0 || lo1 < hi1) {            // the j with C_j <= r < C_{j+1}
            const int m0 = (lo0 + hi0 + 1) >> 1, m1 = (lo1 + hi1 + 1) >> 1;
            const uint64_t c0 = C[m0], c1 = C[m1];
            if (lo0 < hi0) { if (c0 <= r0) lo0 = m0; else hi0 = m0 - 1; }
            if (lo1 < hi1) { if (c1 <= r1) lo1 = m1; else hi1 = m1 - 1; }
        }
        const bool two = s + 1 < N;
        PCMD_CHK(C[lo0] <= r0 && r0 < C[lo0 + 1] && C[lo1] <= r1 && r1 < C[lo1 + 1]);
        const float4 f0 = *reinterpret_cast<const float4 *>(rec[lo0].f);
        const float4 f1 = two ? *reinterpret_cast<const float4 *>(rec[lo1].f) : make_float4(0.f, 0.f, 0.f, 0.f);
        F[0] += (double)f0.x; F[1] += (double)f0.y; F[2] += (double)f0.z; F[3] += (double)f0.w;
        F[0] += (double)f1.x; F[1] += (double)f1.y; F[2] += (double)f1.z; F[3] += (double)f1.w;
        if (COUNTS) { h += a.mult[lo0]; if (two) h += a.mult[lo1]; }
    }
    for (int b = 0; b < a.B; ++b) a.part[((size_t)m * a.B + b) * a.P + p] = (float)F[b];
    if (COUNTS) { a.total[(size_t)m * a.P + p] = N; a.hash[(size_t)m * a.P + p] = h; }
}

int pcmd_launch_agg_tables(pcmd_ctx *c, int n_models, cudaStream_t s) {
    k_agg_tables<<<n_models, 1024, 0, s>>>(c->d_lambda, c->J, c->d_agg_lam, c->d_agg_C, c->d_agg_G);
    PCMD_LAUNCHED(c);
    // the R-C2 table of Lambda: the same kernels as the per-point tables, with one "point" per model
    return pcmd_build_tables(c, c->d_agg_lam, 1, n_models, c->d_agg_rawcnt, c->d_agg_klo, c->d_agg_q, c->agg_tcap,
                             c->d_agg_stcnt, c->d_agg_tab, c->d_agg_rec, 1, s);
}

int pcmd_launch_stage2_agg(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, uint64_t *d_hash,
                           uint32_t *d_total, cudaStream_t s) {
    AggArgs a;
    a.lam_tot = c->d_agg_lam; a.C = c->d_agg_C; a.G = c->d_agg_G; a.rec = c->d_rec; a.trec = c->d_agg_rec;
    a.ttab = c->d_agg_tab; a.mult = c->d_mult; a.tcap = c->agg_tcap; a.P = c->P; a.J = c->J; a.Jpad = c->Jpad;
    a.B = c->B; a.mts = c->tab_stride;
    a.key0 = (uint32_t)(seed & 0xFFFFFFFFull); a.key1 = (uint32_t)(seed >> 32); a.model0 = model0;
    a.part = c->d_part; a.hash = d_hash; a.total = d_total;
    const size_t smem = (size_t)(c->J + 1) * sizeof(uint64_t) + AGG_CELLS * sizeof(uint32_t);
    const bool in_smem = smem <= 200 * 1024;
    if (in_smem && smem > 48 * 1024 && smem > c->smem_agg) {
        PCMD_CUDA(c, cudaFuncSetAttribute(k_stage2_agg<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        PCMD_CUDA(c, cudaFuncSetAttribute(k_stage2_agg<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        c->smem_agg = smem;
    }
    const dim3 grid((unsigned)((c->P + AGG_THREADS - 1) / AGG_THREADS), n_models);
    if (in_smem) {
        if (d_hash) k_stage2_agg<true, true><<<grid, AGG_THREADS, smem, s>>>(a);
        else k_stage2_agg<true, false><<<grid, AGG_THREADS, smem, s>>>(a);
    } else {
        if (d_hash) k_stage2_agg<false, true><<<grid, AGG_THREADS, 0, s>>>(a);
        else k_stage2_agg<false, false><<<grid, AGG_THREADS, 0, s>>>(a);
    }
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}
