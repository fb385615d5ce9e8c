// stage2.cu -- Poisson star count for every (pixel, isochrone point) pair, summed into pixel
// fluxes, then the reduction of the partial fluxes with the dust screen
// applied on the way out.
//
// Work layout: lanes of a warp are consecutive pixels, every thread owns
// S2_PX pixels, and the warp walks class-sorted groups of four isochrone points (one Philox call
// = the four draws of one pixel, R-C1), so every table read is a warp-uniform shared-memory
// broadcast and every loop is specialised for its class.  A work unit is (model, 512-pixel
// tile, segment of one class); persistent CTAs pull units from an atomic counter, stage the
// segment's group records through shared memory with bulk async copies (TMA, double buffered)
// and write one partial flux per (segment, band, pixel); k_reduce_dust adds the partials in
// segment order.
#include "pcmd_internal.cuh"

#ifndef S2_THREADS
#define S2_THREADS 256
#endif
#ifndef S2_PX
#define S2_PX 2
#endif
#ifndef S2_MINB
#define S2_MINB 1
#endif
#ifndef S2_UNITS_PER_SLOT
#define S2_UNITS_PER_SLOT 16
#endif
#define S2_TILE (S2_THREADS * S2_PX)
#ifndef S2_CHUNK
#define S2_CHUNK 48          // groups per staged chunk (48 * 160 B = 7.5 KB; with the 16 KB table stage: 48 KB static)
#endif
#define S2_FLUSH 16          // groups between flushes of the fp32 partial sums into fp64
#define S2_TABW 4096         // words of staged search tables per buffer (16 KB): 32 / 8 / 2 groups of D5 / D7 / D9

struct S2Args {
    const GroupRec *grp;     // [n_models][n_groups] class-sorted
    const SegTable *seg;     // [n_models]
    const PointRec *rec;     // [n_models][Jpad]  (generic class and overflow fix-up: k0, len, off)
    const uint32_t *tab;     // [n_models][cap]
    const uint64_t *mult;    // [Jpad]
    const uint32_t *arena;   // [n_models][arena_cap] padded search tables of the D classes
    int64_t cap, arena_cap;
    int Jpad, n_groups, B, n_models, n_tiles, seg_cap, mts;   // mts: table stride per realisation (1, or 0 in repeat mode)
    int64_t P;
    uint32_t key0, key1, model0;
    float *part;             // [n_models][seg_cap][B][P]
    uint64_t *hash;          // optional [n_models][P], zeroed before the launch
    uint32_t *total;         // optional [n_models][P], zeroed before the launch
    int32_t *counter;        // work-unit counter, zeroed before the launch
};

// ---- bulk async copy (TMA) + mbarrier ---------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---- per-thread state ---------------------------------------------------------------------------
template <int NB, bool COUNTS>
struct S2State {
    float F[S2_PX][NB];      // fp32 partial sums since the last flush
    double D[S2_PX][NB];     // fp64 running sums (R: flux accuracy)
    uint32_t tot[S2_PX];
    uint64_t hsh[S2_PX];
    __device__ __forceinline__ void reset() {
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
#pragma unroll
            for (int b = 0; b < NB; ++b) { F[i][b] = 0.f; D[i][b] = 0.0; }
            tot[i] = 0; hsh[i] = 0;
        }
    }
    __device__ __forceinline__ void flush() {
#pragma unroll
        for (int i = 0; i < S2_PX; ++i)
#pragma unroll
            for (int b = 0; b < NB; ++b) { D[i][b] += (double)F[i][b]; F[i][b] = 0.f; }
    }
};

// Adds n stars of (group g_orig, word w) to pixel slot i: flux by FMA, exact counts in the parity build.
template <int NB, bool COUNTS>
__device__ __forceinline__ void add_stars(S2State<NB, COUNTS> &st, int i, uint32_t n, const float4 f,
                                          uint32_t j, const uint64_t *__restrict__ mult) {
    const float nf = (float)n;
    st.F[i][0] = fmaf(nf, f.x, st.F[i][0]);
    if (NB > 1) st.F[i][1] = fmaf(nf, f.y, st.F[i][1]);
    if (NB > 2) st.F[i][2] = fmaf(nf, f.z, st.F[i][2]);
    if (NB > 3) st.F[i][3] = fmaf(nf, f.w, st.F[i][3]);
    if (COUNTS) { st.tot[i] += n; st.hsh[i] += (uint64_t)n * mult[j]; }
}

// Stars beyond the L inline thresholds (probability < 2^-10 per draw): the rest of the table.
template <int NB, bool COUNTS, int L>
__device__ __forceinline__ void overflow_fixup(S2State<NB, COUNTS> &st, const GroupRec *__restrict__ g,
                                            const uint32_t (&u)[S2_PX][4], const PointRec *__restrict__ rec,
                                            const uint32_t *__restrict__ tab, const uint64_t *__restrict__ mult) {
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t Tov = g->T[L][w];
        const uint32_t j = g->g_orig * 4u + (uint32_t)w;
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
            if (u[i][w] > Tov) {
                const PointRec r = rec[j];
                const uint32_t extra = 1u + count_below(tab + r.off + L + 1, r.len - (L + 1), u[i][w]);
                add_stars<NB, COUNTS>(st, i, extra, *reinterpret_cast<const float4 *>(g->f[w]), j, mult);
            }
        }
    }
}

// One group of class L in {1, 2}: a star is added per exceeded threshold with a predicated FADD.
template <int NB, bool COUNTS, int L>
__device__ __forceinline__ void group_short(S2State<NB, COUNTS> &st, const GroupRec *__restrict__ g,
                                            const uint32_t (&u)[S2_PX][4], const PointRec *__restrict__ rec,
                                            const uint32_t *__restrict__ tab, const uint64_t *__restrict__ mult) {
    const uint4 T0 = *reinterpret_cast<const uint4 *>(g->T[0]);
    const uint4 T1 = *reinterpret_cast<const uint4 *>(g->T[1]);
    const uint4 T2 = *reinterpret_cast<const uint4 *>(g->T[2]);   // used by L == 2 only
    const uint32_t t0[4] = {T0.x, T0.y, T0.z, T0.w}, t1[4] = {T1.x, T1.y, T1.z, T1.w},
                   t2[4] = {T2.x, T2.y, T2.z, T2.w};
    bool ovf = false;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const float4 f = *reinterpret_cast<const float4 *>(g->f[w]);
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
            const uint32_t x = u[i][w];
            const bool p0 = x > t0[w], p1 = x > t1[w];
            if (p0) {
                st.F[i][0] += f.x;
                if (NB > 1) st.F[i][1] += f.y;
                if (NB > 2) st.F[i][2] += f.z;
                if (NB > 3) st.F[i][3] += f.w;
            }
            if (L == 1) ovf |= p1;
            else {
                if (p1) {
                    st.F[i][0] += f.x;
                    if (NB > 1) st.F[i][1] += f.y;
                    if (NB > 2) st.F[i][2] += f.z;
                    if (NB > 3) st.F[i][3] += f.w;
                }
                ovf |= x > t2[w];
            }
            if (COUNTS) {
                const uint32_t n = (uint32_t)p0 + ((L == 2) ? (uint32_t)p1 : 0u);
                st.tot[i] += n; st.hsh[i] += (uint64_t)n * mult[g->g_orig * 4u + w];
            }
        }
    }
    if (__any_sync(0xffffffffu, ovf)) overflow_fixup<NB, COUNTS, L>(st, g, u, rec, tab, mult);
}

// Class L0: a star anywhere in the group is rare (< 2^-8 per draw): one compare of the largest of
// the thread's draws against the smallest first threshold, a vote, and class L1's path if any lane hit.
template <int NB, bool COUNTS>
__device__ __forceinline__ void group_rare(S2State<NB, COUNTS> &st, const GroupRec *__restrict__ g,
                                           const uint32_t (&u)[S2_PX][4], const PointRec *__restrict__ rec,
                                           const uint32_t *__restrict__ tab, const uint64_t *__restrict__ mult) {
    uint32_t mx = 0;
#pragma unroll
    for (int i = 0; i < S2_PX; ++i)
#pragma unroll
        for (int w = 0; w < 4; ++w) mx = max(mx, u[i][w]);
    if (__any_sync(0xffffffffu, mx > g->tmin)) group_short<NB, COUNTS, 1>(st, g, u, rec, tab, mult);
}

// Class L = 4: count the exceeded thresholds, one FMA per band.
template <int NB, bool COUNTS>
__device__ __forceinline__ void group_four(S2State<NB, COUNTS> &st, const GroupRec *__restrict__ g,
                                           const uint32_t (&u)[S2_PX][4], const PointRec *__restrict__ rec,
                                           const uint32_t *__restrict__ tab, const uint64_t *__restrict__ mult) {
    bool ovf = false;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const float4 f = *reinterpret_cast<const float4 *>(g->f[w]);
        const uint32_t a0 = g->T[0][w], a1 = g->T[1][w], a2 = g->T[2][w], a3 = g->T[3][w], a4 = g->T[4][w];
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
            const uint32_t x = u[i][w];
            const uint32_t n = (uint32_t)(x > a0) + (uint32_t)(x > a1) + (uint32_t)(x > a2) + (uint32_t)(x > a3);
            ovf |= x > a4;
            add_stars<NB, COUNTS>(st, i, n, f, g->g_orig * 4u + w, mult);
        }
    }
    if (__any_sync(0xffffffffu, ovf)) overflow_fixup<NB, COUNTS, 4>(st, g, u, rec, tab, mult);
}

// Generic class: n = k0 + #{stored thresholds below u} by bisection of the point's table.
template <int NB, bool COUNTS>
__device__ __forceinline__ void group_generic(S2State<NB, COUNTS> &st, const GroupRec *__restrict__ g,
                                              const uint32_t (&u)[S2_PX][4], const PointRec *__restrict__ rec,
                                              const uint32_t *__restrict__ tab, const uint64_t *__restrict__ mult) {
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t j = g->g_orig * 4u + (uint32_t)w;
        const float4 f = *reinterpret_cast<const float4 *>(g->f[w]);
        const uint32_t t0 = g->T[0][w];
        const uint4 r = *reinterpret_cast<const uint4 *>(&rec[j]);   // T0, off, len, k0
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
            uint32_t n = r.w;
            if (u[i][w] > t0) n += 1u + count_below(tab + r.y + 1, r.z - 1, u[i][w]);
            add_stars<NB, COUNTS>(st, i, n, f, j, mult);
        }
    }
}

// Classes D5/D7/D9: branch-free lower bound in the point's padded table (2^D words, staged in shared
// memory): pos = #{stored thresholds below u}; every probe of a warp hits one table.
// xbuf: the staged table buffer; xoff: byte offset of this group's four tables inside it.
template <int NB, bool COUNTS, int D>
__device__ __forceinline__ void group_search(S2State<NB, COUNTS> &st, const GroupRec *__restrict__ g,
                                             const uint32_t (&u)[S2_PX][4], const uint32_t *__restrict__ xbuf,
                                             uint32_t xoff, const uint64_t *__restrict__ mult) {
    const char *X = reinterpret_cast<const char *>(xbuf);
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const float4 f = *reinterpret_cast<const float4 *>(g->f[w]);
        const uint32_t lo = xoff + ((uint32_t)w << (D + 2)), hi = lo + (2u << D);   // byte offsets of X[0], X[2^(D-1)]
        const uint32_t kb = g->T[4][w] - (lo >> 2);                                 // k0 - lo/4 (mod 2^32)
        const uint32_t t0 = *reinterpret_cast<const uint32_t *>(X + hi - 4u);       // first probe: warp-uniform
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
            const uint32_t x = u[i][w];
            uint32_t off = (x > t0) ? hi : lo;                                      // byte offset of X[pos]
#pragma unroll
            for (int sft = D - 2; sft >= 0; --sft) {
                const uint32_t t = *reinterpret_cast<const uint32_t *>(X + off + ((4u << sft) - 4u));
                asm("{\n.reg .pred p;\nsetp.gt.u32 p, %1, %2;\n@p add.u32 %0, %0, %3;\n}"
                    : "+r"(off) : "r"(x), "r"(t), "r"(4u << sft));
            }
            add_stars<NB, COUNTS>(st, i, (off >> 2) + kb, f, g->g_orig * 4u + w, mult);
        }
    }
}

// ---- the persistent kernel ----------------------------------------------------------------------
template <int NB, bool COUNTS>
__global__ void __launch_bounds__(S2_THREADS, S2_MINB) k_stage2(const S2Args a) {
    __shared__ __align__(128) GroupRec sbuf[2][S2_CHUNK];
    __shared__ __align__(128) uint32_t stab[2][S2_TABW];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_unit;
    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1); mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    uint32_t phase0 = 0, phase1 = 0;                 // parity of the next completion of each barrier
    const int n_units = a.n_models * a.n_tiles * a.seg_cap;
    S2State<NB, COUNTS> st;
    for (;;) {
        if (threadIdx.x == 0) s_unit = atomicAdd(a.counter, 1);
        __syncthreads();
        const int unit = s_unit;
        __syncthreads();
        if (unit >= n_units) break;
        // segment-minor order: consecutive units are different segments (classes) of one tile, so the
        // CTAs resident on an SM mix multiply-bound (L) and compare-bound (D) classes
        const int sg = unit % a.seg_cap;
        const int rem = unit / a.seg_cap;
        const int m = rem / a.n_tiles, tile = rem - m * a.n_tiles;
        const int mt = m * a.mts;                        // whose tables realisation m reads
        const SegTable *seg = a.seg + mt;
        if (sg >= seg->n_seg) continue;
        const int g_lo = seg->g_lo[sg], g_hi = seg->g_hi[sg], cls = seg->cls[sg];
        const GroupRec *grp = a.grp + (size_t)mt * a.n_groups;
        const PointRec *rec = a.rec + (size_t)mt * a.Jpad;
        const uint32_t *tab = a.tab + (size_t)mt * a.cap;
        const uint32_t mctr = a.model0 + (uint32_t)m;
        uint32_t pix[S2_PX];
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) pix[i] = (uint32_t)tile * S2_TILE + (uint32_t)i * S2_THREADS + threadIdx.x;
        PhiloxPix ph[S2_PX];          // the group-independent part of the Philox rounds, per pixel
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) ph[i] = philox_pix_setup(a.key0, a.key1, pix[i], mctr);
        st.reset();
        const int D = cls == S2_CLS_D9 ? 9 : (cls == S2_CLS_D7 ? 7 : (cls == S2_CLS_D5 ? 5 : 0));
        const int csz = D ? (S2_TABW >> (D + 2)) : S2_CHUNK;       // groups per chunk
        const uint32_t *xsrc = a.arena + (size_t)mt * a.arena_cap + seg->arena_off[cls];
        const int cls0 = seg->cls_start[cls];
        const int n_chunks = (g_hi - g_lo + csz - 1) / csz;
        auto stage = [&](int c, int buf) {      // thread 0: bulk copies (TMA) of chunk c into buffer buf
            const int g0 = g_lo + c * csz;
            const uint32_t ng = (uint32_t)min(csz, g_hi - g0);
            const uint32_t rbytes = ng * (uint32_t)sizeof(GroupRec), tbytes = D ? (ng << (D + 4)) : 0u;
            mbar_expect_tx(&bar[buf], rbytes + tbytes);
            bulk_g2s(sbuf[buf], grp + g0, rbytes, &bar[buf]);
            if (D) bulk_g2s(stab[buf], xsrc + ((size_t)(g0 - cls0) << (D + 2)), tbytes, &bar[buf]);
        };
        if (threadIdx.x == 0 && n_chunks > 0) stage(0, 0);
        for (int c = 0; c < n_chunks; ++c) {
            const int cur = c & 1;
            if (threadIdx.x == 0 && c + 1 < n_chunks) stage(c + 1, cur ^ 1);   // prefetch
            if (cur == 0) { mbar_wait(&bar[0], phase0); phase0 ^= 1; }
            else { mbar_wait(&bar[1], phase1); phase1 ^= 1; }
            const int ng = min(csz, g_hi - (g_lo + c * csz));
            const uint32_t *xt = stab[cur];
            const GroupRec *sb = sbuf[cur];
#define S2_LOOP(BODY)                                                                          \
            for (int g = 0; g < ng; ++g) {                                                     \
                const GroupRec *gr = sb + g;                                                   \
                uint32_t u[S2_PX][4];                                                          \
                const PhiloxGrp pq = philox_grp_setup(a.key0, mctr, gr->g_orig);               \
                _Pragma("unroll") for (int i = 0; i < S2_PX; ++i)                              \
                    philox_stage2(a.key0, a.key1, ph[i], pq, u[i]);                            \
                BODY;                                                                          \
                if ((g & (S2_FLUSH - 1)) == S2_FLUSH - 1) st.flush();                          \
            }
            if (cls == S2_CLS_L0) { S2_LOOP((group_rare<NB, COUNTS>(st, gr, u, rec, tab, a.mult))) }
            else if (cls == S2_CLS_L1) { S2_LOOP((group_short<NB, COUNTS, 1>(st, gr, u, rec, tab, a.mult))) }
            else if (cls == S2_CLS_L2) { S2_LOOP((group_short<NB, COUNTS, 2>(st, gr, u, rec, tab, a.mult))) }
            else if (cls == S2_CLS_L4) { S2_LOOP((group_four<NB, COUNTS>(st, gr, u, rec, tab, a.mult))) }
            else if (cls == S2_CLS_D5) { S2_LOOP((group_search<NB, COUNTS, 5>(st, gr, u, xt, (uint32_t)g << 9, a.mult))) }
            else if (cls == S2_CLS_D7) { S2_LOOP((group_search<NB, COUNTS, 7>(st, gr, u, xt, (uint32_t)g << 11, a.mult))) }
            else if (cls == S2_CLS_D9) { S2_LOOP((group_search<NB, COUNTS, 9>(st, gr, u, xt, (uint32_t)g << 13, a.mult))) }
            else { S2_LOOP((group_generic<NB, COUNTS>(st, gr, u, rec, tab, a.mult))) }
#undef S2_LOOP
            st.flush();
            __syncthreads();   // every warp is done with the buffers of chunk c before they are refilled
        }
        // partial flux of this (segment, tile); exact integer counts by atomics (parity build)
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
            if ((int64_t)pix[i] >= a.P) continue;
#pragma unroll
            for (int b = 0; b < NB; ++b)
                if (b < a.B)
                    a.part[(((size_t)m * a.seg_cap + sg) * a.B + b) * a.P + pix[i]] = (float)st.D[i][b];
            if (COUNTS) {
                atomicAdd(&a.total[(size_t)m * a.P + pix[i]], st.tot[i]);
                atomicAdd((unsigned long long *)&a.hash[(size_t)m * a.P + pix[i]], (unsigned long long)st.hsh[i]);
            }
        }
    }
}

// ---- partial sums -> raw flux -> dust (stage 3; R-Q7, R-Q8) --------------------
struct RdArgs {
    const float *part; const SegTable *seg; const DevModel *mdl;
    float *flux_raw, *flux_dust;
    int B, seg_cap, dust_mode, n_models, mts;
    int64_t P;
    uint32_t key0, key1, model0;
    double dust_frac, coef[4];
};

__global__ void __launch_bounds__(256) k_reduce_dust(const RdArgs a) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= a.P * a.n_models) return;
    const int m = (int)(idx / a.P);
    const uint32_t p = (uint32_t)(idx - (int64_t)m * a.P);
    const int n_seg = a.seg[m * a.mts].n_seg;
    float A = 0.f; bool behind = true;
    if (a.dust_mode != 0) {       // fp32: the factor needs 1e-5 relative, expf / exp10f give 1e-7
        const DevModel M = a.mdl[m * a.mts];
        uint32_t w[4];
        philox4x32_10(a.key0, a.key1, p, 0u, a.model0 + (uint32_t)m, 1u, w);
        A = (float)M.dust_med * expf((float)M.dust_sigma * normal_f32(w[0], w[1]));
        if (a.dust_mode == 2) behind = ((double)w[2] < a.dust_frac * 4294967296.0);
    }
    const float Fd = (float)a.dust_frac;
    for (int b = 0; b < a.B; ++b) {
        double s = 0.0;
        for (int sg = 0; sg < n_seg; ++sg)
            s += (double)a.part[(((size_t)m * a.seg_cap + sg) * a.B + b) * a.P + p];
        const float F = (float)s;
        const size_t o = ((size_t)m * a.B + b) * a.P + p;
        if (a.flux_raw) a.flux_raw[o] = F;
        float fac = 1.f;
        if (a.dust_mode == 1) fac = (1.f - Fd) + Fd * exp10f(-0.4f * (float)a.coef[b] * A);
        else if (a.dust_mode == 2) fac = behind ? exp10f(-0.4f * (float)a.coef[b] * A) : 1.f;
        a.flux_dust[o] = F * fac;
    }
}

// ---- host side ------------------------------------------------------------------------------------
// Number of cost-equal segments a model's groups are cut into: enough work units (model x tile x
// segment) to fill every resident CTA slot ~16 times, so the tail of the persistent loop is short.
int pcmd_stage2_seg_budget(const pcmd_ctx *c, int n_models) {
    const int64_t tiles = (c->P + S2_TILE - 1) / S2_TILE;
    const int64_t slots = (int64_t)c->sm_count * 4;
    int64_t b = (S2_UNITS_PER_SLOT * slots + n_models * tiles - 1) / (n_models * tiles);
    if (b < 1) b = 1;
    if (b > S2_SEG_MAX - S2_NCLASS) b = S2_SEG_MAX - S2_NCLASS;
    return (int)b;
}

template <int NB>
static cudaError_t launch_s2(const S2Args &a, bool counts, int grid, cudaStream_t s) {
    if (counts) k_stage2<NB, true><<<grid, S2_THREADS, 0, s>>>(a);
    else k_stage2<NB, false><<<grid, S2_THREADS, 0, s>>>(a);
    return cudaGetLastError();
}

int pcmd_launch_stage2(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, float *d_flux_raw,
                       uint64_t *d_hash, uint32_t *d_total, cudaStream_t s) {
    S2Args a;
    a.grp = c->d_grp; a.seg = c->d_seg; a.rec = c->d_rec; a.tab = c->d_tab; a.mult = c->d_mult;
    a.arena = c->d_arena; a.arena_cap = c->arena_cap;
    a.cap = c->cap_raw; a.Jpad = c->Jpad; a.n_groups = c->Jpad >> 2; a.B = c->B; a.n_models = n_models;
    a.n_tiles = (int)((c->P + S2_TILE - 1) / S2_TILE); a.seg_cap = c->seg_cap; a.P = c->P; a.mts = c->tab_stride;
    a.key0 = (uint32_t)(seed & 0xFFFFFFFFull); a.key1 = (uint32_t)(seed >> 32); a.model0 = model0;
    a.part = c->d_part; a.hash = d_hash; a.total = d_total; a.counter = c->d_status + 1;
    if (d_hash) {
        PCMD_CUDA(c, cudaMemsetAsync(d_hash, 0, (size_t)n_models * c->P * sizeof(uint64_t), s));
        PCMD_CUDA(c, cudaMemsetAsync(d_total, 0, (size_t)n_models * c->P * sizeof(uint32_t), s));
    }
    const int64_t n_units = (int64_t)n_models * a.n_tiles * a.seg_cap;
    const int per_sm = d_hash ? 2 : c->s2_ctas_per_sm;
    const int grid = (int)(n_units < (int64_t)c->sm_count * per_sm ? n_units : (int64_t)c->sm_count * per_sm);
    cudaError_t e;
    const bool counts = d_hash != nullptr;
    if (c->B <= 2) e = launch_s2<2>(a, counts, grid, s);
    else if (c->B == 3) e = launch_s2<3>(a, counts, grid, s);
    else e = launch_s2<4>(a, counts, grid, s);
    c->launches++;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return PCMD_ECUDA; }

    RdArgs r;
    r.part = c->d_part; r.seg = c->d_seg; r.mdl = c->d_model; r.flux_raw = d_flux_raw; r.flux_dust = c->d_fdust;
    r.mts = c->tab_stride; r.B = c->B; r.seg_cap = c->seg_cap; r.dust_mode = c->dust_mode; r.n_models = n_models; r.P = c->P;
    r.key0 = a.key0; r.key1 = a.key1; r.model0 = model0; r.dust_frac = c->dust_frac;
    for (int b = 0; b < 4; ++b) r.coef[b] = c->dust_coef[b];
    const int64_t n = c->P * n_models;
    k_reduce_dust<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(r);
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}

// Resident CTAs per SM of the production kernels (occupancy query, once per ctx).
int pcmd_stage2_occupancy(pcmd_ctx *c) {
    int n2 = 0, n3 = 0, n4 = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n2, k_stage2<2, false>, S2_THREADS, 0);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n3, k_stage2<3, false>, S2_THREADS, 0);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n4, k_stage2<4, false>, S2_THREADS, 0);
    const int n = c->B <= 2 ? n2 : (c->B == 3 ? n3 : n4);
    c->s2_ctas_per_sm = n > 0 ? n : 1;
    return PCMD_OK;
}
