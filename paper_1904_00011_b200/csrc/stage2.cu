// stage2.cu -- Poisson star count for every (pixel, isochrone point) pair, summed into pixel
// fluxes, then the reduction of the partial fluxes with the dust screen
// applied on the way out.
//
// Work layout: lanes of a warp are consecutive pixels, every thread owns
// S2_PX pixels, and the warp walks class-sorted groups of four isochrone points (one Philox call
// = the four draws of one pixel, R-C1), so every table read is a warp-uniform shared-memory
// broadcast and every loop is specialised for its class.  A work unit = (model, 512-pixel tile, segment of the
// model's chunk list); persistent CTAs take units from an atomic counter, one ahead, and stream the chunks
// (<= 48 groups of one class) of successive units through a ring of shared-memory stages filled by bulk async
// copies (TMA) with full/empty mbarriers -- no CTA-wide barrier inside the stream -- and write one partial
// flux per (unit, band, pixel); k_reduce_dust adds the segments of a tile in a fixed order.
#include "pcmd_internal.cuh"

#ifndef S2_THREADS
#define S2_THREADS 256
#endif
#ifndef S2_PX
#define S2_PX 2
#endif
#ifndef S2_MINB
#define S2_MINB 2
#endif
#ifndef S2_NST
#define S2_NST 3             // stages of the chunk ring
#endif
#define S2_WARPS (S2_THREADS / 32)
#define S2_TILE (S2_THREADS * S2_PX)
#define S2_FLUSH 16          // groups between flushes of the fp32 partial sums into fp64
#ifndef S2_UNITS_PER_SLOT
#define S2_UNITS_PER_SLOT 24
#endif
#define S2_SEG_MAX 32

struct S2Args {
    const GroupRec *grp;     // [n_models][n_groups] class-sorted
    const ModelPlan *plan;   // [n_models]
    const PointRec *rec;     // [n_models][Jpad]  (generic class and overflow fix-up: k0, len, off)
    const uint32_t *tab;     // [n_models][cap]
    const uint64_t *mult;    // [Jpad]
    const uint32_t *arena;   // [n_models][arena_cap] padded search tables of the D classes
    int64_t cap, arena_cap;
    int Jpad, n_groups, B, n_models, n_tiles, n_seg, mts;   // mts: table stride per realisation (1, or 0 in repeat mode)
    int64_t P;
    uint32_t key0, key1, model0;
    float *part;             // [n_models][n_seg][B][P]
    int32_t *counter;        // work-unit counter, zeroed before the launch
    uint64_t *hash;          // optional [n_models][P], zeroed before the launch
    uint32_t *total;         // optional [n_models][P], zeroed before the launch
};

// ---- bulk async copy (TMA) + mbarrier: the plain forms are in pcmd_internal.cuh ------------------
// lane-predicated forms for the warp-uniform producer
__device__ __forceinline__ void mbar_expect_tx_if(bool lead, uint64_t *bar, uint32_t bytes) {
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n}"
                 ::"r"(smem_u32(bar)), "r"(bytes), "r"((int)lead) : "memory");
}
__device__ __forceinline__ void mbar_arrive_if(bool lead, uint64_t *bar) {
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %1, 0;\n@q mbarrier.arrive.shared::cta.b64 _, [%0];\n}"
                 ::"r"(smem_u32(bar)), "r"((int)lead) : "memory");
}
__device__ __forceinline__ void bulk_g2s_if(bool lead, void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %4, 0;\n"
                 "@q cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n}"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "r"((int)lead) : "memory");
}
// Stores of the producer thread into shared memory.  They go through inline PTX on purpose: a plain C++
// store to shared memory inside the chunk loop makes the compiler give up warp-uniformity of everything
// read back from shared memory there (descriptors, loop bounds, table addresses), and with it the
// uniform datapath (uniform registers for the Philox round keys, uniform branches) in all the loops.
// The producer code is executed by all lanes of warp 0 with identical values (warp-uniform control flow, for
// the same reason); `lead` (lane 0) predicates the side effects.
__device__ __forceinline__ void sts32(bool lead, void *p, int32_t v) {
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q st.shared.b32 [%0], %1;\n}" ::"r"(smem_u32(p)), "r"(v), "r"((int)lead) : "memory");
}
__device__ __forceinline__ void sts128(bool lead, void *p, int4 v) {
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %5, 0;\n@q st.shared.v4.b32 [%0], {%1, %2, %3, %4};\n}"
                 ::"r"(smem_u32(p)), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "r"((int)lead) : "memory");
}
// volatile load that the compiler may not move other memory accesses across (spin on a flag another warp sets)
__device__ __forceinline__ uint32_t lds_acquire_u32(const void *p) {
    uint32_t v;
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
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

// Adds nf (an exact small integer held as a float) stars of (group g_orig, word w) to pixel slot i:
// flux by FMA, exact integer counts in the parity build.
template <int NB, bool COUNTS>
__device__ __forceinline__ void add_stars(S2State<NB, COUNTS> &st, int i, float nf, const float4 f,
                                          uint32_t j, const uint64_t *__restrict__ mult) {
    st.F[i][0] = fmaf(nf, f.x, st.F[i][0]);
    if (NB > 1) st.F[i][1] = fmaf(nf, f.y, st.F[i][1]);
    if (NB > 2) st.F[i][2] = fmaf(nf, f.z, st.F[i][2]);
    if (NB > 3) st.F[i][3] = fmaf(nf, f.w, st.F[i][3]);
    if (COUNTS) { const uint32_t n = (uint32_t)nf; st.tot[i] += n; st.hsh[i] += (uint64_t)n * mult[j]; }
}

// nf += 1 if x > t: one integer compare (ALU pipe) and one predicated FADD (FMA pipe); no int->float
// conversion and no integer add.
__device__ __forceinline__ void count_if_above(float &nf, uint32_t x, uint32_t t) {
    asm("{\n.reg .pred p;\nsetp.gt.u32 p, %1, %2;\n@p add.f32 %0, %0, 0f3F800000;\n}" : "+f"(nf) : "r"(x), "r"(t));
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
                PCMD_CHK(r.len >= (uint32_t)L + 1u);      // the overflow threshold is entry L of the table
                const uint32_t extra = 1u + count_below(tab + r.off + L + 1, r.len - (L + 1), u[i][w]);
                add_stars<NB, COUNTS>(st, i, (float)extra, *reinterpret_cast<const float4 *>(g->f[w]), j, mult);
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

// Class L = 4: count the exceeded thresholds in a float (compare + predicated FADD each), one FMA per band.
template <int NB, bool COUNTS>
__device__ __forceinline__ void group_four(S2State<NB, COUNTS> &st, const GroupRec *__restrict__ g,
                                           const uint32_t (&u)[S2_PX][4], const PointRec *__restrict__ rec,
                                           const uint32_t *__restrict__ tab, const uint64_t *__restrict__ mult) {
    const uint4 A0 = *reinterpret_cast<const uint4 *>(g->T[0]), A1 = *reinterpret_cast<const uint4 *>(g->T[1]),
                A2 = *reinterpret_cast<const uint4 *>(g->T[2]), A3 = *reinterpret_cast<const uint4 *>(g->T[3]),
                A4 = *reinterpret_cast<const uint4 *>(g->T[4]);
    const uint32_t a0[4] = {A0.x, A0.y, A0.z, A0.w}, a1[4] = {A1.x, A1.y, A1.z, A1.w}, a2[4] = {A2.x, A2.y, A2.z, A2.w},
                   a3[4] = {A3.x, A3.y, A3.z, A3.w}, a4[4] = {A4.x, A4.y, A4.z, A4.w};
    bool ovf = false;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const float4 f = *reinterpret_cast<const float4 *>(g->f[w]);
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
            const uint32_t x = u[i][w];
            float nf = 0.f;
            count_if_above(nf, x, a0[w]);
            count_if_above(nf, x, a1[w]);
            count_if_above(nf, x, a2[w]);
            count_if_above(nf, x, a3[w]);
            ovf |= x > a4[w];
            add_stars<NB, COUNTS>(st, i, nf, f, g->g_orig * 4u + w, mult);
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
            add_stars<NB, COUNTS>(st, i, (float)n, f, j, mult);
        }
    }
}

// Classes D5/D7/D9: branch-free lower bound in the point's padded table (2^D words, staged in shared
// memory): pos = #{stored thresholds below u}; every probe of a warp hits one table.  The shared-memory
// byte ADDRESS of X[pos] is carried as the bit pattern of a (denormal) float: adding two such floats
// adds their bit patterns exactly, so a level is LDS [bits + imm], ISETP (ALU pipe) and a predicated
// FADD (FMA pipe), and the count comes out of the final address with an FMUL and an FMA -- no integer
// add, no int->float conversion.  xs: byte address of this group's four tables; cx = -(stage buffer
// address) / 4 as a float; the record holds k0 - (word offset of the table in the stage buffer).
template <int NB, bool COUNTS, int D, bool OVF>
__device__ __forceinline__ void group_search(S2State<NB, COUNTS> &st, const GroupRec *__restrict__ g,
                                             const uint32_t (&u)[S2_PX][4], uint32_t xs, float cx,
                                             const PointRec *__restrict__ rec, const uint32_t *__restrict__ tab,
                                             const uint64_t *__restrict__ mult) {
    const float4 K = *reinterpret_cast<const float4 *>(g->T[4]);
    const uint4 TO = *reinterpret_cast<const uint4 *>(g->T[3]);     // classes S3/S4: the overflow thresholds
    const uint32_t tov[4] = {TO.x, TO.y, TO.z, TO.w};
    bool ovf = false;
    const float kq[4] = {K.x + cx, K.y + cx, K.z + cx, K.w + cx};                  // k0 - (address of X[0]) / 4
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const float4 f = *reinterpret_cast<const float4 *>(g->f[w]);
        const uint32_t base = xs + ((uint32_t)w << (D + 2));                        // byte address of X[0]
        const float lo = __uint_as_float(base), hi = __uint_as_float(base + (2u << D));
        const uint32_t t0 = lds_u32(base + (2u << D) - 4u);                         // first probe: warp-uniform
#pragma unroll
        for (int i = 0; i < S2_PX; ++i) {
            const uint32_t x = u[i][w];
            if (OVF) ovf |= x > tov[w];
            float off = (x > t0) ? hi : lo;                                         // bits = byte address of X[pos]
#pragma unroll
            for (int sft = D - 2; sft >= 0; --sft) {
                const uint32_t t = lds_u32(__float_as_uint(off) + ((4u << sft) - 4u));
                asm("{\n.reg .pred p;\nsetp.gt.u32 p, %1, %2;\n@p add.f32 %0, %0, %3;\n}"
                    : "+f"(off) : "r"(x), "r"(t), "f"(__uint_as_float(4u << sft)));
            }
            // off = (address of X[pos]) 2^-149 -> address / 4 + kq = k0 + pos, in two exact steps (2^147 is not a float)
            const float nf = fmaf(off * 8.507059173023462e37f, 2097152.0f, kq[w]);
            PCMD_CHK(__float_as_uint(off) - base <= (4u << D) - 4u && ((__float_as_uint(off) - base) & 3u) == 0u);
            PCMD_CHK(nf >= 0.f && nf < 4194304.f && nf == floorf(nf));
            add_stars<NB, COUNTS>(st, i, nf, f, g->g_orig * 4u + w, mult);
        }
    }
    // S3/S4: more stars than the 2^D - 1 searched thresholds (probability < 2^-10 per draw): the rest of the table
    if (OVF && __any_sync(0xffffffffu, ovf)) {
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const uint32_t j = g->g_orig * 4u + (uint32_t)w;
#pragma unroll
            for (int i = 0; i < S2_PX; ++i) {
                if (u[i][w] > tov[w]) {
                    const PointRec r = rec[j];
                    PCMD_CHK(r.len >= (1u << D));            // the overflow threshold is entry 2^D - 1
                    const uint32_t extra = 1u + count_below(tab + r.off + (1u << D), r.len - (1u << D), u[i][w]);
                    add_stars<NB, COUNTS>(st, i, (float)extra, *reinterpret_cast<const float4 *>(g->f[w]), j, mult);
                }
            }
        }
    }
}

// ---- work units and the chunk stream ----------------------------------------------------------------
// A work unit = (model, 512-pixel tile, segment): the segment is a contiguous range of the model's chunk
// list, one of n_seg pieces of (nearly) equal estimated cost.  Units are fixed, so the partial flux of a
// unit does not depend on which CTA ran it (deterministic results); CTAs take units from an atomic
// counter (the two CTAs of an SM do not progress at the same rate, a static split leaves one of them idle
// at the end), one unit ahead, and the chunks of successive units form ONE continuous stream through the
// shared-memory ring, so a unit boundary costs no pipeline bubble.
struct __align__(16) ChunkDesc { int32_t m, tile, cls, ng, flags, slot, pad0, pad1; };
#define S2_F_FIRST 1      // first chunk of a unit: set up the pixels, reset the sums
#define S2_F_LAST 2       // last chunk of a unit: write the partial flux
#define S2_F_END 8        // last chunk of this CTA

struct S2Shared {
    uint64_t full[S2_NST], empty[S2_NST];
    ChunkDesc desc[S2_NST];
    ModelPlan plan;                      // the plan of model plan_m (the producer's current model)
    int32_t m_, tile, seg, chunk;        // current unit (model, tile, segment); next chunk to issue
    int32_t chunk_end, cls, live, issued;// end of the unit's chunk range; class of `chunk`; more to issue; chunks issued so far
    int32_t plan_m, unit_first, unit_next, ticket;  // model of `plan`; the next chunk issued starts a unit; the unit fetched
                                          // one step ahead; producer turns completed
};

// First chunk of plan p whose cost start is >= q; n_chunks if there is none.
__device__ __forceinline__ int s2_first_chunk_at(const ModelPlan &p, uint32_t q) {
    for (int c = 0; c < S2_NCLASS; ++c) {
        const int nch = p.chunk_start[c + 1] - p.chunk_start[c];
        if (nch == 0) continue;
        const uint32_t cs = p.cost_start[c], cc = p.chunk_cost[c];
        if (q <= cs + (uint32_t)(nch - 1) * cc) return p.chunk_start[c] + (q <= cs ? 0 : (int)((q - cs + cc - 1) / cc));
    }
    return p.n_chunks;
}

// Segments a model's chunk list is cut into: at most n_seg, and few enough that every segment is at least one
// chunk long (then none is empty).  Used by the kernel and by k_reduce_dust alike.
__device__ __forceinline__ int s2_model_segments(const ModelPlan &p, int n_seg) {
    if (p.n_chunks == 0) return 0;
    const uint32_t k = p.cost_total / p.cost_max;
    return (int)min((uint32_t)n_seg, max(k, 1u));
}

// Producer warp: make sh.unit_next (or the first valid unit the counter hands out after it) the current unit
// and fetch the one after it.
__device__ __forceinline__ void s2_advance(const S2Args &a, S2Shared &sh, bool lead) {
    const int n_units = a.n_models * a.n_tiles * a.n_seg;
    for (;;) {
        const int u = sh.unit_next;
        if (u >= n_units) { sts32(lead, &sh.live, 0); __syncwarp(); return; }
        int nx = 0;
        if (lead) nx = atomicAdd(a.counter, 1);
        __syncwarp();
        sts32(lead, &sh.unit_next, (int)gridDim.x + __shfl_sync(0xffffffffu, nx, 0));
        __syncwarp();
        const int seg = u % a.n_seg, r = u / a.n_seg;
        const int m = r / a.n_tiles, tile = r - m * a.n_tiles;
        if (m != sh.plan_m) {
            const int4 *src = reinterpret_cast<const int4 *>(a.plan + (size_t)m * a.mts);
            int4 *dst = reinterpret_cast<int4 *>(&sh.plan);
#pragma unroll
            for (int i = 0; i < (int)(sizeof(ModelPlan) / 16); ++i) sts128(lead, dst + i, src[i]);
            sts32(lead, &sh.plan_m, m);
            __syncwarp();
        }
        const ModelPlan &p = sh.plan;
        const int ns = s2_model_segments(p, a.n_seg);
        if (seg >= ns) continue;                         // this model has fewer segments
        const uint32_t C = p.cost_total;
        const int lo = s2_first_chunk_at(p, (uint32_t)((uint64_t)C * seg / ns));
        const int hi = seg + 1 == ns ? p.n_chunks : s2_first_chunk_at(p, (uint32_t)((uint64_t)C * (seg + 1) / ns));
        int cls = 0;
        while (lo >= p.chunk_start[cls + 1]) cls++;
        PCMD_CHK(m >= 0 && m < a.n_models && tile >= 0 && tile < a.n_tiles && lo >= 0 && lo < hi && hi <= p.n_chunks &&
                 cls < S2_NCLASS);
        sts128(lead, &sh.m_, make_int4(m, tile, seg, lo));
        sts128(lead, &sh.chunk_end, make_int4(hi, cls, 1, sh.issued));
        __syncwarp();
        return;
    }
}

// Thread 0: issue the current unit's next chunk into stage s (descriptor + bulk copies) and step to the next
// chunk of the stream.
__device__ __forceinline__ void s2_issue(const S2Args &a, S2Shared &sh, GroupRec *sbuf, uint32_t *stab, int s, bool lead) {
    const ModelPlan &p = sh.plan;
    const int m = sh.m_, mt = m * a.mts, cls = sh.cls, chunk = sh.chunk;
    const int li = chunk - p.chunk_start[cls], cg = p.chunk_groups[cls];
    const int g0 = p.cls_start[cls] + li * cg;
    const int ng = min(cg, p.cls_start[cls + 1] - g0);
    const int run = p.run_cls[cls];
    const int D = s2_class_depth(run);
    const uint32_t rbytes = (uint32_t)ng * (uint32_t)sizeof(GroupRec), tbytes = D ? ((uint32_t)ng << (D + 4)) : 0u;
    const GroupRec *rsrc = a.grp + (size_t)mt * a.n_groups + g0;
    const uint32_t *tsrc = a.arena + (size_t)mt * a.arena_cap + p.arena_off[cls] + ((size_t)(g0 - p.cls_start[cls]) << (D + 2));
    PCMD_CHK(cls >= 0 && cls < S2_NCLASS && li >= 0 && ng >= 1 && ng <= S2_CHUNK && g0 >= 0 && g0 + ng <= a.n_groups);
    PCMD_CHK(tbytes <= (uint32_t)S2_TABW * 4u && (rbytes & 15u) == 0u && s >= 0 && s < S2_NST);
    PCMD_CHK(!D || (size_t)p.arena_off[cls] + ((size_t)(g0 - p.cls_start[cls] + ng) << (D + 2)) <= (size_t)a.arena_cap);
    ChunkDesc d;
    d.m = m; d.tile = sh.tile; d.cls = run; d.ng = ng; d.slot = sh.seg; d.pad0 = d.pad1 = 0;
    // step: next chunk of the unit, or the next unit (which may replace sh.plan: everything above is in locals)
    const bool unit_first = sh.unit_first != 0;
    const bool unit_last = chunk + 1 == sh.chunk_end;
    const int issued = sh.issued;
    __syncwarp();
    sts32(lead, &sh.issued, issued + 1);
    __syncwarp();
    if (unit_last) { s2_advance(a, sh, lead); sts32(lead, &sh.unit_first, 1); }
    else {
        int c2 = cls;
        while (chunk + 1 >= p.chunk_start[c2 + 1]) c2++;
        sts32(lead, &sh.chunk, chunk + 1); sts32(lead, &sh.cls, c2); sts32(lead, &sh.unit_first, 0);
    }
    __syncwarp();
    d.flags = (unit_first ? S2_F_FIRST : 0) | (unit_last ? S2_F_LAST : 0) | ((unit_last && !sh.live) ? S2_F_END : 0);
    sts128(lead, &sh.desc[s], make_int4(d.m, d.tile, d.cls, d.ng));
    sts128(lead, &sh.desc[s].flags, make_int4(d.flags, d.slot, 0, 0));
    mbar_expect_tx_if(lead, &sh.full[s], rbytes + tbytes);
    bulk_g2s_if(lead, sbuf + (size_t)s * S2_CHUNK, rsrc, rbytes, &sh.full[s]);
    if (D) bulk_g2s_if(lead, stab + (size_t)s * S2_TABW, tsrc, tbytes, &sh.full[s]);
}

// ---- the persistent kernel ----------------------------------------------------------------------
template <int NB, bool COUNTS>
__global__ void __launch_bounds__(S2_THREADS, S2_MINB) k_stage2(const S2Args a) {
    pdl_enter<PDL_EARLY_STAGE2>();
    extern __shared__ __align__(128) unsigned char s2_smem[];
    GroupRec *sbuf = reinterpret_cast<GroupRec *>(s2_smem);                                     // [S2_NST][S2_CHUNK]
    uint32_t *stab = reinterpret_cast<uint32_t *>(s2_smem + (size_t)S2_NST * S2_CHUNK * sizeof(GroupRec));   // [S2_NST][S2_TABW]
    S2Shared &sh = *reinterpret_cast<S2Shared *>(s2_smem + (size_t)S2_NST * (S2_CHUNK * sizeof(GroupRec) + S2_TABW * 4));
    const int lane = threadIdx.x & 31;
    const bool lead = lane == 0;
    const bool producer = __all_sync(0xffffffffu, threadIdx.x < 32);     // warp 0, as a warp-uniform predicate
    const int wid = __reduce_max_sync(0xffffffffu, threadIdx.x >> 5);    // warp index, warp-uniform
    if (producer) {
        sts32(lead, &sh.plan_m, -1); sts32(lead, &sh.issued, 0); sts32(lead, &sh.live, 0); sts32(lead, &sh.unit_first, 1);
        sts32(lead, &sh.unit_next, blockIdx.x);      // the first unit is static; the counter hands out the rest
        sts32(lead, &sh.ticket, 0);
        if (lead) {
            for (int s = 0; s < S2_NST; ++s) { mbar_init(&sh.full[s], 1); mbar_init(&sh.empty[s], S2_WARPS); }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncwarp();
        s2_advance(a, sh, lead);
        for (int s = 0; s < S2_NST && sh.live; ++s) s2_issue(a, sh, sbuf, stab, s, lead);
        if (sh.issued == 0) {            // nothing for this CTA (tiny job): an empty last chunk ends the stream
            sts128(lead, &sh.desc[0], make_int4(0, 0, S2_CLS_L1, 0));
            sts128(lead, &sh.desc[0].flags, make_int4(S2_F_END, 0, 0, 0));
            mbar_arrive_if(lead, &sh.full[0]);
        }
    }
    __syncthreads();
    S2State<NB, COUNTS> st;
    uint32_t pix[S2_PX];
    PhiloxPix ph[S2_PX];                 // the group-independent part of the Philox rounds, per pixel
    uint32_t mctr = 0;
    // stage and phase parity of chunk q and of chunk q-1 (kept as counters: no division in the loop)
    int s = 0, sp = 0;
    uint32_t par = 0, parp = 0;
    for (int q = 0;; ++q) {
        mbar_wait(&sh.full[s], par);
        const ChunkDesc d = sh.desc[s];
        const int mt = d.m * a.mts;
        PCMD_CHK(d.m >= 0 && d.m < a.n_models && d.tile >= 0 && d.tile < a.n_tiles && d.slot >= 0 && d.slot < a.n_seg &&
                 d.ng >= 0 && d.ng <= S2_CHUNK && d.cls >= 0 && d.cls <= S2_NCLASS);
        if (d.flags & S2_F_FIRST) {
            mctr = a.model0 + (uint32_t)d.m;
#pragma unroll
            for (int i = 0; i < S2_PX; ++i) {
                pix[i] = (uint32_t)d.tile * S2_TILE + (uint32_t)i * S2_THREADS + threadIdx.x;
                ph[i] = philox_pix_setup(a.key0, a.key1, pix[i], mctr);
            }
            st.reset();
        }
        const PointRec *rec = a.rec + (size_t)mt * a.Jpad;
        const uint32_t *tab = a.tab + (size_t)mt * a.cap;
        const GroupRec *sb = sbuf + (size_t)s * S2_CHUNK;
        const uint32_t xs = smem_u32(stab + (size_t)s * S2_TABW);
        const float cx = -(float)(xs >> 2);
        const int ng = d.ng;
#ifndef S2_UNROLL
#define S2_UNROLL 1
#endif
#define S2_PRAGMA_(x) _Pragma(#x)
#define S2_PRAGMA_UNROLL(n) S2_PRAGMA_(unroll n)
#define S2_LOOP(BODY)                                                                          \
        for (int g0 = 0; g0 < ng; g0 += S2_FLUSH) {     /* fp32 sums of at most S2_FLUSH groups, then into fp64 */ \
            const int g1 = min(ng, g0 + S2_FLUSH);                                             \
            S2_PRAGMA_UNROLL(S2_UNROLL)                                                        \
            for (int g = g0; g < g1; ++g) {                                                    \
                const GroupRec *gr = sb + g;                                                   \
                uint32_t u[S2_PX][4];                                                          \
                const PhiloxGrp pq = philox_grp_setup(a.key0, mctr, gr->g_orig);               \
                _Pragma("unroll") for (int i = 0; i < S2_PX; ++i)                              \
                    philox_stage2(a.key0, a.key1, ph[i], pq, u[i]);                            \
                BODY;                                                                          \
            }                                                                                  \
            st.flush();                                                                        \
        }
        if (d.cls == S2_CLS_L0) { S2_LOOP((group_rare<NB, COUNTS>(st, gr, u, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_L1) { S2_LOOP((group_short<NB, COUNTS, 1>(st, gr, u, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_L2) { S2_LOOP((group_short<NB, COUNTS, 2>(st, gr, u, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_L4) { S2_LOOP((group_four<NB, COUNTS>(st, gr, u, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_S3) { S2_LOOP((group_search<NB, COUNTS, 3, true>(st, gr, u, xs + ((uint32_t)g << 7), cx, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_S4) { S2_LOOP((group_search<NB, COUNTS, 4, true>(st, gr, u, xs + ((uint32_t)g << 8), cx, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_D5) { S2_LOOP((group_search<NB, COUNTS, 5, false>(st, gr, u, xs + ((uint32_t)g << 9), cx, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_D6) { S2_LOOP((group_search<NB, COUNTS, 6, false>(st, gr, u, xs + ((uint32_t)g << 10), cx, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_D7) { S2_LOOP((group_search<NB, COUNTS, 7, false>(st, gr, u, xs + ((uint32_t)g << 11), cx, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_D8) { S2_LOOP((group_search<NB, COUNTS, 8, false>(st, gr, u, xs + ((uint32_t)g << 12), cx, rec, tab, a.mult))) }
        else if (d.cls == S2_CLS_D9) { S2_LOOP((group_search<NB, COUNTS, 9, false>(st, gr, u, xs + ((uint32_t)g << 13), cx, rec, tab, a.mult))) }
        else { S2_LOOP((group_generic<NB, COUNTS>(st, gr, u, rec, tab, a.mult))) }
#undef S2_LOOP
        // the stage is free once every warp has arrived; warp 0 refills the PREVIOUS chunk's stage, which
        // every warp has normally left long ago, so nobody waits for the slowest warp
        __syncwarp();
        if (lane == 0) mbar_arrive(&sh.empty[s]);
        if (d.flags & S2_F_LAST) {
            // partial flux of this unit; exact integer counts by atomics (parity build)
#pragma unroll
            for (int i = 0; i < S2_PX; ++i) {
                if ((int64_t)pix[i] >= a.P) continue;
#pragma unroll
                for (int b = 0; b < NB; ++b)
                    if (b < a.B)
                        a.part[(((size_t)d.m * a.n_seg + d.slot) * a.B + b) * a.P + pix[i]] = (float)st.D[i][b];
                if (COUNTS) {
                    atomicAdd(&a.total[(size_t)d.m * a.P + pix[i]], st.tot[i]);
                    atomicAdd((unsigned long long *)&a.hash[(size_t)d.m * a.P + pix[i]], (unsigned long long)st.hsh[i]);
                }
            }
        }
        if (d.flags & S2_F_END) {
            break;
        }
        // Producer turn q (after chunk q >= 1): chunk q-1's stage, which every warp has normally left long ago,
        // takes chunk q-1+S2_NST.  The turns rotate over the warps (no warp is slowed more than the others, nobody
        // waits for a producer warp) and run in order (ticket).
        if (q >= 1 && ((q - 1) & (S2_WARPS - 1)) == wid) {
            while (lds_acquire_u32(&sh.ticket) != (uint32_t)(q - 1)) { }
            __threadfence_block();
            if (lds_acquire_u32(&sh.live)) {
                mbar_wait(&sh.empty[sp], parp);
                s2_issue(a, sh, sbuf, stab, sp, lead);
            }
            __threadfence_block();
            sts32(lead, &sh.ticket, q);
        }
        sp = s; parp = par;
        if (++s == S2_NST) { s = 0; par ^= 1u; }
    }
}

// ---- partial sums -> raw flux -> dust (stage 3; R-Q7, R-Q8) --------------------
struct RdArgs {
    const float *part; const ModelPlan *plan; const DevModel *mdl;
    float *flux_raw, *flux_dust;
    int B, n_seg, dust_mode, n_models, mts, n_frag;   // n_frag >= 0: partial fluxes per pixel (else from the plan)
    int64_t P;
    uint32_t key0, key1, model0;
    double dust_frac, coef[4];
};

__global__ void __launch_bounds__(256) k_reduce_dust(const RdArgs a) {
    pdl_enter<PDL_EARLY_REDUCE>();
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= a.P * a.n_models) return;
    const int m = (int)(idx / a.P);
    const uint32_t p = (uint32_t)(idx - (int64_t)m * a.P);
    const int n_frag = a.n_frag >= 0 ? a.n_frag : s2_model_segments(a.plan[(size_t)m * a.mts], a.n_seg);   // partial fluxes written per pixel
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
        for (int sl = 0; sl < n_frag; ++sl)     // the segments in their fixed order (deterministic)
            s += (double)a.part[(((size_t)m * a.n_seg + sl) * a.B + b) * a.P + p];
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
static size_t s2_smem_bytes() {
    return (size_t)S2_NST * (S2_CHUNK * sizeof(GroupRec) + S2_TABW * sizeof(uint32_t)) + sizeof(S2Shared);
}

int pcmd_stage2_tiles(const pcmd_ctx *c) { return (int)((c->P + S2_TILE - 1) / S2_TILE); }

// Segments per (model, tile): enough work units (model x tile x segment) to give every resident CTA slot ~24
// of them, so that the tail of the dynamic schedule is short; one partial flux image per segment.
int pcmd_stage2_segments(const pcmd_ctx *c, int n_models) {
    const int64_t G = (int64_t)c->sm_count * c->s2_ctas_per_sm;
    const int64_t tiles = (int64_t)pcmd_stage2_tiles(c) * n_models;
    int64_t n = (S2_UNITS_PER_SLOT * G + tiles - 1) / tiles;
    if (n < 1) n = 1;
    if (n > S2_SEG_MAX) n = S2_SEG_MAX;
    return (int)n;
}

template <int NB>
static cudaError_t launch_s2(const S2Args &a, bool counts, int grid, cudaStream_t s) {
    if (counts) pcmd_launch_pdl((k_stage2<NB, true>), grid, dim3(S2_THREADS), s2_smem_bytes(), s, a);
    else pcmd_launch_pdl((k_stage2<NB, false>), grid, dim3(S2_THREADS), s2_smem_bytes(), s, a);
    return cudaGetLastError();
}

int pcmd_launch_stage2(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, float *d_flux_raw,
                       uint64_t *d_hash, uint32_t *d_total, cudaStream_t s) {
    S2Args a;
    a.grp = c->d_grp; a.plan = c->d_plan; a.rec = c->d_rec; a.tab = c->d_tab; a.mult = c->d_mult;
    a.arena = c->d_arena; a.arena_cap = c->arena_cap;
    a.cap = c->cap_raw; a.Jpad = c->Jpad; a.n_groups = c->Jpad >> 2; a.B = c->B; a.n_models = n_models;
    a.n_tiles = pcmd_stage2_tiles(c); a.n_seg = c->n_seg; a.P = c->P; a.mts = c->tab_stride;
    a.key0 = (uint32_t)(seed & 0xFFFFFFFFull); a.key1 = (uint32_t)(seed >> 32); a.model0 = model0;
    a.part = c->d_part; a.hash = d_hash; a.total = d_total; a.counter = c->d_status + 1;   // zeroed by the caller
    if (d_hash) {
        PCMD_CUDA(c, cudaMemsetAsync(d_hash, 0, (size_t)n_models * c->P * sizeof(uint64_t), s));
        PCMD_CUDA(c, cudaMemsetAsync(d_total, 0, (size_t)n_models * c->P * sizeof(uint32_t), s));
    }
    if (c->sampler_mode == 1) {      // aggregated sampler (agg.cu): one partial flux per pixel
        int rc = pcmd_launch_stage2_agg(c, n_models, seed, model0, d_hash, d_total, s);
        if (rc) return rc;
    } else {
    const int64_t n_units = (int64_t)n_models * a.n_tiles * a.n_seg;
    const int64_t slots = (int64_t)c->sm_count * (d_hash ? 1 : c->s2_ctas_per_sm);
    const int grid = (int)(n_units < slots ? n_units : slots);
    cudaError_t e;
    const bool counts = d_hash != nullptr;
    if (c->B <= 2) e = launch_s2<2>(a, counts, grid, s);
    else if (c->B == 3) e = launch_s2<3>(a, counts, grid, s);
    else e = launch_s2<4>(a, counts, grid, s);
    c->launches++;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return PCMD_ECUDA; }
    }

    RdArgs r;
    r.n_frag = c->sampler_mode == 1 ? 1 : -1;
    r.part = c->d_part; r.plan = c->d_plan; r.mdl = c->d_model; r.flux_raw = d_flux_raw; r.flux_dust = c->d_fdust;
    r.mts = c->tab_stride; r.B = c->B; r.n_seg = c->n_seg; r.dust_mode = c->dust_mode;
    r.n_models = n_models; r.P = c->P;
    r.key0 = a.key0; r.key1 = a.key1; r.model0 = model0; r.dust_frac = c->dust_frac;
    for (int b = 0; b < 4; ++b) r.coef[b] = c->dust_coef[b];
    const int64_t n = c->P * n_models;
    pcmd_launch_pdl(k_reduce_dust, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, s, r);
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}

// Resident CTAs per SM of the production kernels (occupancy query, once per ctx), and the opt-in to
// more than 48 KB of dynamic shared memory for every instantiation.
int pcmd_stage2_occupancy(pcmd_ctx *c) {
    const int smem = (int)s2_smem_bytes();
    PCMD_CUDA(c, cudaFuncSetAttribute(k_stage2<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    PCMD_CUDA(c, cudaFuncSetAttribute(k_stage2<3, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    PCMD_CUDA(c, cudaFuncSetAttribute(k_stage2<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    PCMD_CUDA(c, cudaFuncSetAttribute(k_stage2<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    PCMD_CUDA(c, cudaFuncSetAttribute(k_stage2<3, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    PCMD_CUDA(c, cudaFuncSetAttribute(k_stage2<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int n2 = 0, n3 = 0, n4 = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n2, k_stage2<2, false>, S2_THREADS, smem);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n3, k_stage2<3, false>, S2_THREADS, smem);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n4, k_stage2<4, false>, S2_THREADS, smem);
    const int n = c->B <= 2 ? n2 : (c->B == 3 ? n3 : n4);
    c->s2_ctas_per_sm = n > 0 ? n : 1;
    return PCMD_OK;
}
