// pcmd_internal.cuh -- shared declarations of the CUDA path (never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/pcmd.h"

// Self-check build (PCMD_NVCC_EXTRA=-DPCMD_SELFCHECK, profiles/r2_sanitizers.md): device-side assertions on the
// staged addresses, table ranges, work-unit indices and shared-memory indices of every kernel; a failed
// assertion ends the launch with cudaErrorAssert (the call returns PCMD_ECUDA) and prints file:line.
// The product build compiles them away.
#ifdef PCMD_SELFCHECK
#undef NDEBUG
#include <assert.h>
#define PCMD_CHK(c) assert(c)
#else
#define PCMD_CHK(c) ((void)0)
#endif

#define PCMD_LAMBDA_MAX 4194304.0 /* 2^22, R-C2 */

// Per isochrone point record consumed by stage 2 (32 bytes, one group of 4 points = 128 B).
struct __align__(16) PointRec {
    uint32_t T0;    // first stored threshold minus 1 (draw > T0 <=> n > k0); 0xFFFFFFFF if none
    uint32_t off;   // offset of the stored thresholds (minus 1 each) in the model's table
    uint32_t len;   // number of stored thresholds
    uint32_t k0;    // first count whose T > 0
    float f[4];     // flux of one star in each band (electrons), unused bands 0
};

// Stage-2 work layout.  Groups of four consecutive isochrone points (one
// Philox call, R-C1) are classified by how many sampler thresholds decide almost every draw and
// sorted by class; a class is cut into chunks (the unit of shared-memory staging); a model's chunk list
// is cut by estimated cost into n_seg segments, and a work unit = (model, 512-pixel tile, segment).
// Persistent CTAs take units from an atomic counter (units are fixed, so results do not depend on which
// CTA ran them) and stream their chunks through a shared-memory ring.
#define S2_NCLASS 12       // classes, most expensive first:
#define S2_CLS_D9 1        //   0 bisection in global memory (tables longer than 511)
#define S2_CLS_D8 2        //   1-5 branch-free search of a padded table of 2^D words in shared memory
#define S2_CLS_D7 3
#define S2_CLS_D6 4
#define S2_CLS_D5 5
#define S2_CLS_S4 6        //   6-7 the same search over the first 2^D - 1 thresholds only (k0 = 0 and more stars than that
#define S2_CLS_S3 7        //       have probability < 2^-10: the overflow path finishes them)
#define S2_CLS_L4 8        //   8-10 L inline thresholds decide the draw (more stars: probability < 2^-10)
#define S2_CLS_L2 9
#define S2_CLS_L1 10
#define S2_CLS_L0 11       //   11 rare: P(any star) < 2^-8 per draw: one max-compare per group, then class L1's path
#define S2_CLS_NONE 12     //   no point of the group can have a star: dropped
#ifndef S2_CHUNK
#define S2_CHUNK 48         // group records per staged chunk (48 * 160 B = 7.5 KB)
#endif
#ifndef S2_TABW
#define S2_TABW 6144        // words of staged search tables per chunk (24 KB): 48 / 24 / 12 / 6 / 3 groups of D5 / D6 / D7 / D8 / D9
#endif
// cost model of the segment cut: ~SM cycles per warp and group of each class loop (profiles/), and per chunk
#define S2_COST_G 1500u
#define S2_COST_D9 420u
#define S2_COST_D8 390u
#define S2_COST_D7 340u
#define S2_COST_D6 295u
#define S2_COST_D5 250u
#define S2_COST_S4 225u
#define S2_COST_S3 205u
#define S2_COST_L4 190u
#define S2_COST_L2 160u
#define S2_COST_L1 155u
#define S2_COST_L0 150u
#define S2_COST_CHUNK 100u
// log2 of the padded table size of a search class
__host__ __device__ __forceinline__ int s2_class_depth(int cls) {
    return cls == S2_CLS_D9 ? 9 : cls == S2_CLS_D8 ? 8 : cls == S2_CLS_D7 ? 7 : cls == S2_CLS_D6 ? 6 : cls == S2_CLS_D5 ? 5
           : cls == S2_CLS_S4 ? 4 : cls == S2_CLS_S3 ? 3 : 0;
}
struct __align__(16) GroupRec {      // 160 bytes
    uint32_t g_orig, cls, tmin, pad1; // original group index (Philox counter word 1), class, min over w of T[0][w]
    uint32_t T[5][4];                 // T[i][w]: (i+1)-th stored threshold minus 1 of point w; 0xFFFFFFFF if none.
                                      // Search classes: T[4][w] = float bits of k0 - (table offset in the stage buffer);
                                      // S3/S4: T[3][w] = the overflow threshold (the 2^D-th stored threshold minus 1)
    float f[4][4];                    // f[w][b]: flux of one star of point w in band b
};
// Per model: the class-sorted group list cut into chunks.  Chunk i of class c (chunk_start[c] <= i <
// chunk_start[c+1]) holds groups cls_start[c] + (i - chunk_start[c]) * chunk_groups[c] ... (at most
// chunk_groups[c] of them) and starts at cost position cost_start[c] + (i - chunk_start[c]) * chunk_cost[c].
struct __align__(16) ModelPlan {
    int32_t n_chunks, first_d;                    // first D class whose padded tables are in the arena
    uint32_t cost_total, cost_max;                // cost of one pixel tile of this model; largest chunk cost
    int32_t cls_start[S2_NCLASS + 1];             // sorted-group range of each class
    int32_t chunk_start[S2_NCLASS + 1];           // chunk range of each class
    uint32_t cost_start[S2_NCLASS + 1];           // cost position of each class's first chunk
    int32_t chunk_groups[S2_NCLASS];              // groups per full chunk
    uint32_t chunk_cost[S2_NCLASS];               // cost of a full chunk
    int32_t run_cls[S2_NCLASS];                   // the loop that runs a class (0 for a D class demoted to bisection)
    int64_t arena_off[S2_NCLASS];                 // word offset of a class's padded tables in the model's arena
};

struct DevHess {
    int32_t band_plus, band_minus, band_y, nx, ny;
    float x_lo, y_lo, inv_dx, inv_dy;
    int64_t bin_off;  // offset of this diagram inside a model's Hess block
};

struct DevModel {          // per-model scalars staged from pcmd_params
    double feh_mean, feh_sigma, dmod, dust_med, dust_sigma;
};

struct pcmd_ctx {
    // ---- configuration (host copies)
    int32_t psf_grid;      // G >= 1 cells per side, PSF table [B][G*G][K][K]
    int32_t N, B, A, Z, J, Jpad, K, psf_sep, shot_noise, poisson_sky, n_hess, dust_mode;
    int64_t P, hess_bins;
    double like_floor, dust_frac, mdf_cut;
    double zp[PCMD_MAX_BANDS], dust_coef[PCMD_MAX_BANDS], sky[PCMD_MAX_BANDS], read_sigma[PCMD_MAX_BANDS];
    pcmd_hess_spec hess[PCMD_MAX_HESS];
    double *h_imf_w;       // [J] host copy, used only to size scratch
    double imf_sqrt_sum, imf_w_max;   // sum_j sqrt(imf_w_j), max_j imf_w_j (scratch sizing)
    // ---- device constants
    int32_t *d_age_idx, *d_feh_idx;
    double *d_imf_w, *d_absmag, *d_feh_grid;
    float *d_psf;          // [B][K][K] (a separable PSF expanded)
    float *d_psf_sep;      // [B][2][K] row and column factors of a separable PSF, else NULL
    float *h_psf_sep;      // host copy of the same (kernel parameters of k_conv2)
    uint64_t *d_mult;      // [Jpad] splitmix64(j)|1
    double *d_lfact;       // ln(d!) table of the Poisson lnL
    DevHess *d_hess_spec;  // [n_hess]
    uint32_t *d_sky_tab;   // [B][sky_cap] stored thresholds minus 1 of Poisson(sky_b)
    PointRec sky_rec[PCMD_MAX_BANDS]; uint32_t sky_cap;
    // ---- per-call scratch, sized for cap_models
    int32_t cap_models;
    int64_t cap_raw;       // entries of raw table scratch per model
    double *d_sfh;         // [cap_models][A]
    DevModel *d_model;     // [cap_models]
    double *h_stage;       // pinned staging for sfh + DevModel: two halves used alternately
    size_t h_stage_bytes;  // bytes of one half
    int stage_flip;
    double *d_mdfw;        // [cap_models][Z]
    double *d_lambda;      // [cap_models][J]
    uint32_t *d_alloc;     // [cap_models][2] bump allocators of the raw and the compact table regions (k_points)
    double *d_q;           // [cap_models][cap_raw] pmf ratios, then thresholds (as uint64)
    uint32_t *d_tab;       // [cap_models][cap_raw] stored thresholds minus 1
    PointRec *d_rec;       // [cap_models][Jpad]
    float *d_fdust; int64_t fdust_elems;   // [realisations][B][P] dusty flux
    int32_t tab_stride;    // 1: realisation m reads model m's tables; 0: all read model 0's (repeat mode)
    GroupRec *d_grp;       // [cap_models][Jpad/4] class-sorted group records
    ModelPlan *d_plan;     // [cap_models]
    uint8_t *d_gcls;       // [cap_models][Jpad/4] class of each group (original order)
    uint32_t *d_gpos;      // [cap_models][Jpad/4] sorted position of each group
    uint32_t *d_arena; int64_t arena_cap;  // [cap_models][arena_cap] padded search tables of the D classes
    float *d_part;  int64_t part_elems;  // stage-2 partial fluxes [realisations][n_seg][B][P]
    int32_t n_seg, s2_ctas_per_sm;
    // aggregated sampler (sampler_mode = 1, agg.cu): total lambda, cumulative integer weights, guide cells and the
    // R-C2 table of the total, per model
    int32_t sampler_mode;
    double *d_agg_lam; uint64_t *d_agg_C; uint32_t *d_agg_G;
    uint32_t *d_agg_rawcnt, *d_agg_klo, *d_agg_stcnt, *d_agg_tab; double *d_agg_q; PointRec *d_agg_rec;
    int64_t agg_tcap; int32_t agg_models; size_t smem_agg;
    int32_t *d_status;     // device status word
    // hess / loglike scratch
    pcmd_hess_stats *d_hpart; int64_t hpart_cap; // per-block partial stats
    // evaluate_host scratch
    float *d_mag; uint32_t *d_hessbuf; pcmd_hess_stats *d_statbuf; double *d_lnl;
    uint32_t *d_hess_data; pcmd_hess_stats *d_data_stats;
    int32_t eval_cap;
    void *h_pin; size_t h_pin_bytes;
    // taps / options / bookkeeping
    float *tap_dust, *tap_conv;
    size_t smem_conv, smem_conv_sep, smem_hess;   // opted-in dynamic shared memory of this ctx's device
    int32_t last_models;
    int last_cuda;
    int64_t launches;
    int sm_count;
    cudaEvent_t stage_ev[2]; int stage_ev_valid;
    // per-stage timing (pcmd_profile): events recorded on the caller's stream around each stage
    cudaEvent_t prof_ev[8]; int prof_on, prof_made; uint32_t prof_seen;
};

#define PCMD_PROF(ctx, i, s)                                              \
    do {                                                                  \
        if ((ctx)->prof_on) {                                             \
            PCMD_CUDA(ctx, cudaEventRecord((ctx)->prof_ev[i], s));        \
            (ctx)->prof_seen |= 1u << (i);                                \
        }                                                                 \
    } while (0)

// Programmatic dependent launch (PDL) -------------------------------------------------------
// The kernels of one evaluation form a chain on the caller's stream, and on small jobs (c1: 64 x 64 pixels) the
// launch latency between them is a large part of the step.  Every kernel of the chain starts with pdl_enter<EARLY>():
// griddepcontrol.wait (returns once the previous kernel of the stream has completed and its writes are visible;
// a no-op for a kernel launched without the attribute) followed by griddepcontrol.launch_dependents (lets the
// NEXT kernel, if it was launched with the attribute, be set up and made resident while this one runs; it then
// sits in its own wait).  Completion is transitive along the chain because every kernel waits before it does
// anything else.  pcmd_launch_pdl launches with cudaLaunchAttributeProgrammaticStreamSerialization; only
// kernels that begin with pdl_enter() may be launched through it.  PCMD_NO_PDL=1 in the environment switches
// the attribute off (plain stream order).
// EARLY = false leaves the trigger to the kernel's exit: the warps of an early-resident dependent poll in their wait
// and take issue slots from the kernel that is still running, which costs more than the hidden launch latency when
// that kernel is a handful of latency-bound threads (k_points: a serial fp64 recurrence per thread; measured 3 us of
// stage 1 in every configuration).  Per-kernel switches (PDL_EARLY_*) below.
template <bool EARLY>
__device__ __forceinline__ void pdl_enter() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (EARLY) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
#ifndef PDL_EARLY_POINTS
#define PDL_EARLY_POINTS 0
#endif
#ifndef PDL_EARLY_SORT
#define PDL_EARLY_SORT 1
#endif
#ifndef PDL_EARLY_EMIT
#define PDL_EARLY_EMIT 1
#endif
#ifndef PDL_EARLY_STAGE2
#define PDL_EARLY_STAGE2 0        // k_reduce_dust blocks that fill in next to the last running k_stage2 blocks poll beside them (c1: -1.5 us)
#endif
#ifndef PDL_EARLY_REDUCE
#define PDL_EARLY_REDUCE 1
#endif
#ifndef PDL_EARLY_CONV
#define PDL_EARLY_CONV 1
#endif
#ifndef PDL_EARLY_HESS
#define PDL_EARLY_HESS 1
#endif
#ifndef PDL_EARLY_LIKE
#define PDL_EARLY_LIKE 1
#endif
int pcmd_pdl_enabled();     // api.cu
template <typename... KA, typename... A>
static inline cudaError_t pcmd_launch_pdl(void (*kern)(KA...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                          A &&...args) {
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cfg.attrs = at; cfg.numAttrs = pcmd_pdl_enabled() ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<A &&>(args)...);
}

// error helpers ---------------------------------------------------------------------------
#define PCMD_CUDA(ctx, call)                                              \
    do {                                                                  \
        cudaError_t e__ = (call);                                         \
        if (e__ != cudaSuccess) {                                         \
            if (ctx) (ctx)->last_cuda = (int)e__;                         \
            return (e__ == cudaErrorMemoryAllocation) ? PCMD_ENOMEM : PCMD_ECUDA; \
        }                                                                 \
    } while (0)
#define PCMD_LAUNCHED(ctx)                                                \
    do {                                                                  \
        (ctx)->launches++;                                                \
        cudaError_t e__ = cudaGetLastError();                             \
        if (e__ != cudaSuccess) { (ctx)->last_cuda = (int)e__; return PCMD_ECUDA; } \
    } while (0)

// Philox4x32-10 (R-C1), device side ----------------------------------------------------------
#define PHILOX_M0 0xD2511F53u
#define PHILOX_M1 0xCD9E8D57u
#define PHILOX_W0 0x9E3779B9u
#define PHILOX_W1 0xBB67AE85u

__device__ __forceinline__ void philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1,
                                              uint32_t c2, uint32_t c3, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0 = __umulhi(PHILOX_M0, c0), l0 = PHILOX_M0 * c0;
        uint32_t h1 = __umulhi(PHILOX_M1, c2), l1 = PHILOX_M1 * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += PHILOX_W0; k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The same generator for the stage-2 counter (pixel, group, model, 0), with everything that does
// not depend on the group taken out of the group loop.  Round 1 multiplies only the pixel and the
// model; of round 2, M1*c2 is pixel-only and M0*c0 depends on the group alone (one product serves
// every pixel of the thread); of round 3, M0*c0 is pixel-only.  7 full rounds remain per call.
struct PhiloxPix {          // per (pixel, model, key): 4 registers
    uint32_t X;             // lo(M0 pix) ^ (k1 + W1)          -> c2 after round 2 = hi(M0 c0') ^ X
    uint32_t Y;             // lo(M1 c2') ^ (k0 + 2 W0)        -> c0 after round 3 = hi(M1 c2'') ^ Y
    uint32_t Z;             // hi(M0 c0'') ^ (k1 + 2 W1)       -> c2 after round 3 = Z ^ lo(M0 c0')
    uint32_t L3;            // lo(M0 c0'')                     -> c3 after round 3
};
struct PhiloxGrp { uint32_t qh, ql; };   // hi, lo of M0 * c0' (c0' = hi(M1 model) ^ group ^ k0)

__device__ __forceinline__ PhiloxPix philox_pix_setup(uint32_t k0, uint32_t k1, uint32_t pix, uint32_t model) {
    PhiloxPix h;
    const uint32_t hi0 = __umulhi(PHILOX_M0, pix), lo0 = PHILOX_M0 * pix;     // round 1, c0 = pix
    const uint32_t lo1 = PHILOX_M1 * model;                                   // round 1, c2 = model
    const uint32_t c2p = hi0 ^ k1;                                            // c2' (c3 = stream 0)
    const uint32_t k0b = k0 + PHILOX_W0, k1b = k1 + PHILOX_W1;                // round-2 keys
    const uint32_t h2 = __umulhi(PHILOX_M1, c2p), l2 = PHILOX_M1 * c2p;       // round 2, pixel-only product
    const uint32_t c0pp = h2 ^ lo1 ^ k0b;                                     // c0'' (c1' = lo1)
    const uint32_t k0c = k0b + PHILOX_W0, k1c = k1b + PHILOX_W1;              // round-3 keys
    h.X = lo0 ^ k1b;
    h.Y = l2 ^ k0c;
    h.Z = __umulhi(PHILOX_M0, c0pp) ^ k1c;
    h.L3 = PHILOX_M0 * c0pp;
    return h;
}
__device__ __forceinline__ PhiloxGrp philox_grp_setup(uint32_t k0, uint32_t model, uint32_t group) {
    const uint32_t c0p = __umulhi(PHILOX_M1, model) ^ group ^ k0;             // c0' (c1 = group)
    PhiloxGrp q;
    q.qh = __umulhi(PHILOX_M0, c0p); q.ql = PHILOX_M0 * c0p;
    return q;
}
__device__ __forceinline__ void philox_stage2(uint32_t k0, uint32_t k1, const PhiloxPix &h, const PhiloxGrp &q,
                                              uint32_t out[4]) {
    // state after round 3
    const uint32_t c2pp = q.qh ^ h.X;                                         // c2''
    const uint32_t hm = __umulhi(PHILOX_M1, c2pp), lm = PHILOX_M1 * c2pp;     // round 3, the one real product
    uint32_t c0 = hm ^ h.Y, c1 = lm, c2 = h.Z ^ q.ql, c3 = h.L3;
    k0 += 3u * PHILOX_W0; k1 += 3u * PHILOX_W1;
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        uint32_t h0 = __umulhi(PHILOX_M0, c0), l0 = PHILOX_M0 * c0;
        uint32_t h1 = __umulhi(PHILOX_M1, c2), l1 = PHILOX_M1 * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += PHILOX_W0; k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Box-Muller normal from two words (R-C4), fp64: it is O(P) work, not O(P J).
__device__ __forceinline__ double normal_from_words(uint32_t w0, uint32_t w1) {
    double u1 = ((double)w0 + 0.5) * (1.0 / 4294967296.0);
    double u2 = ((double)w1 + 0.5) * (1.0 / 4294967296.0);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925 * u2);
}

// The same normal in fp32 (stages 3 and 5).  Special-function-unit approximations: ln with an
// absolute error of ~1e-7 on -ln u (relative 1e-6 near u = 1), cos with ~2e-6; the normal is good to
// ~2e-6, which moves a magnitude by < 1e-7 when the noise is a few per cent of the counts
// (DESIGN.md "Tolerances").
__device__ __forceinline__ float normal_f32(uint32_t w0, uint32_t w1) {
    const float u1 = fminf(((float)w0 + 0.5f) * 2.3283064365386963e-10f, 0.99999994f);
    const float u2 = ((float)w1 + 0.5f) * 2.3283064365386963e-10f;
    const float L = -1.3862943611198906f * __log2f(u1);          // -2 ln u1 = -2 ln2 log2 u1
    return L * rsqrtf(L) * __cosf(6.2831853071795865f * u2 - 3.1415926535897932f) * -1.0f;   // cos(x) = -cos(x - pi)
}

// log2 of a positive normal float with an absolute error of ~2.4e-7: exponent exactly, mantissa by
// the special-function unit (whose absolute error bound holds on [0.5, 2]).
__device__ __forceinline__ float log2_pos(float x) {
    const int e = (int)((__float_as_uint(x) >> 23) & 0xFFu) - 127;
    const float mant = __uint_as_float((__float_as_uint(x) & 0x007FFFFFu) | 0x3F800000u);
    return (float)e + __log2f(mant);
}

// #{i < len : u > T[i]} for non-decreasing T (thresholds stored minus 1)
__device__ __forceinline__ uint32_t count_below(const uint32_t *__restrict__ T, uint32_t len, uint32_t u) {
    uint32_t lo = 0, hi = len;
    while (lo < hi) {
        uint32_t mid = (lo + hi) >> 1;
        if (u > T[mid]) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// bulk async copy (TMA, UBLKCP in SASS) + mbarrier helpers shared by stage 2 and the convolution ------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE_%=;\n"
        "bra WAIT_LOOP_%=;\n"
        "WAIT_DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// launchers implemented in the stage files ---------------------------------------------------
int pcmd_launch_stage1(pcmd_ctx *c, int n_models, cudaStream_t s);
int pcmd_build_sky_tables(pcmd_ctx *c);
int pcmd_build_tables(pcmd_ctx *c, const double *d_lambda, int J, int n_models, uint32_t *rawcnt, uint32_t *klo,
                      double *q, int64_t cap, uint32_t *stcnt, uint32_t *tab, PointRec *rec, int Jpad, cudaStream_t s);
int pcmd_launch_agg_tables(pcmd_ctx *c, int n_models, cudaStream_t s);
int pcmd_launch_stage2_agg(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, uint64_t *d_hash,
                           uint32_t *d_total, cudaStream_t s);
int pcmd_build_lfact(pcmd_ctx *c);
int pcmd_launch_stage2(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, float *d_flux_raw,
                       uint64_t *d_hash, uint32_t *d_total, cudaStream_t s);
int pcmd_stage2_segments(const pcmd_ctx *c, int n_models);
int pcmd_stage2_tiles(const pcmd_ctx *c);
int pcmd_stage2_occupancy(pcmd_ctx *c);
int pcmd_conv_setup(pcmd_ctx *c);
int pcmd_launch_conv_noise(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, float *d_mag,
                           cudaStream_t s);
int pcmd_launch_hess(pcmd_ctx *c, const float *d_mag, int n_models, uint32_t *d_hess,
                     pcmd_hess_stats *d_stats, cudaStream_t s);
int pcmd_launch_loglike(pcmd_ctx *c, const uint32_t *d_hm, const pcmd_hess_stats *d_sm, int n_models,
                        const uint32_t *d_hd, const pcmd_hess_stats *d_sd, int mode, double *d_out,
                        cudaStream_t s);
