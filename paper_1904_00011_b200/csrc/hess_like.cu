// hess_like.cu -- stage 6: Hess diagram = 2-D histogram of (colour, magnitude) (PAPER.md:57,130,
// 218; R-Q13) with a block-private shared-memory histogram, and stage 7: Poisson log-likelihood
// (north_star; R-Q15) and the paper's Eq. 2-4 (R-Q14).
#include "pcmd_internal.cuh"

#ifndef HS_THREADS
#define HS_THREADS 512
#endif
#ifndef HS_MINB
#define HS_MINB 2        // blocks per SM of the 512-thread instance (64-register cap; without it the compiler takes 96 registers: one block per SM)
#endif
#define HS_PIX_PER_BLOCK 4096

// Binning arithmetic, fp32, no contraction:
// x = fl(mp - mm); t = fl(fl(x - x_lo) * inv_dx); ix = floor(t); half-open.
// NT threads per block: HS_THREADS, or 1024 when the histogram leaves room for one block per SM only
template <bool SMEM, int NT>
__global__ void __launch_bounds__(NT, (NT == HS_THREADS ? HS_MINB : 1)) k_hess(const float *__restrict__ mag, int B, int64_t P,
                                                     const DevHess *__restrict__ specs, int n_hess, int64_t ppb,
                                                     int64_t bins_total, uint32_t *__restrict__ hess,
                                                     pcmd_hess_stats *__restrict__ part,
                                                     pcmd_hess_stats *__restrict__ stats_out) {
    pdl_enter<PDL_EARLY_HESS>();
    extern __shared__ uint32_t sh[];
    const int h = blockIdx.y, m = blockIdx.z;
    const DevHess S = specs[h];
    const int nbins = S.nx * S.ny;
    uint32_t *gh = hess + (size_t)m * bins_total + S.bin_off;
    if (SMEM) {
        for (int t = threadIdx.x; t < nbins + 2; t += NT) sh[t] = 0;      // + the spare counters sh[nbins], sh[nbins + 1]
        __syncthreads();
    }
    const float *mp = mag + ((size_t)m * B + S.band_plus) * P;
    const float *mm = mag + ((size_t)m * B + S.band_minus) * P;
    const float *my = mag + ((size_t)m * B + S.band_y) * P;
    uint32_t n_in = 0, n_out = 0, n_bad = 0;
    double sx = 0.0, sy = 0.0;
    const int64_t p0 = (int64_t)blockIdx.x * ppb;
    const int64_t p1 = min(P, p0 + ppb);
    auto one = [&](float a, float b, float y) {
        const float x = __fsub_rn(a, b);
        // floor and conversion in one instruction (saturating, so a far-out value stays out); 0 <= ix < nx as one
        // unsigned compare: the same decision as floorf + float range test
        const int ix = __float2int_rd(__fmul_rn(__fsub_rn(x, S.x_lo), S.inv_dx));
        const int iy = __float2int_rd(__fmul_rn(__fsub_rn(y, S.y_lo), S.inv_dy));
        if (SMEM) {
            // branch-free (a warp's pixels rarely agree, and a branch per pixel costs its compare, its reconvergence
            // pair and the tail of the block around it): a pixel outside the window goes to the spare counter
            // sh[nbins], a NaN pixel to sh[nbins + 1] (the conversion gives 0 for NaN, so NaN is tested apart: both
            // scaled coordinates in one two-operand test -- NaN propagates from a, b and y into them), and both add
            // 0.0 to the sums; n_out, n_bad and n_in come out of the two counters and the block's pixel count (below)
            const float tx = __fmul_rn(__fsub_rn(x, S.x_lo), S.inv_dx), ty = __fmul_rn(__fsub_rn(y, S.y_lo), S.inv_dy);
            int bad;
            asm("{\n.reg .pred p;\nsetp.nan.f32 p, %1, %2;\nselp.s32 %0, 1, 0, p;\n}" : "=r"(bad) : "f"(tx), "f"(ty));
            const bool in = !bad && (unsigned)ix < (unsigned)S.nx && (unsigned)iy < (unsigned)S.ny;
            const int bin = in ? iy * S.nx + ix : nbins + bad;
            PCMD_CHK(bin >= 0 && bin <= nbins + 1);
            atomicAdd(&sh[bin], 1u);
            // the select is taken on the fp32 bit pattern, before the conversion (one select, not two on the halves of a double)
            sx += (double)__uint_as_float(in ? __float_as_uint(x) : 0u);
            sy += (double)__uint_as_float(in ? __float_as_uint(y) : 0u);
        } else {
            if (isnan(a) || isnan(b) || isnan(y)) { n_bad++; return; }
            if ((unsigned)ix >= (unsigned)S.nx || (unsigned)iy >= (unsigned)S.ny) { n_out++; return; }
            const int bin = iy * S.nx + ix;
            PCMD_CHK(bin >= 0 && bin < nbins);
            atomicAdd(&gh[bin], 1u);
            n_in++; sx += (double)x; sy += (double)y;
        }
    };
    if (((P | p0) & 3) == 0 && (reinterpret_cast<uintptr_t>(mag) & 15) == 0) {      // 16-byte loads: every band of every image starts 16-byte aligned
        const float4 *vp = reinterpret_cast<const float4 *>(mp), *vm = reinterpret_cast<const float4 *>(mm),
                     *vy = reinterpret_cast<const float4 *>(my);
        const int64_t q1 = (p1 + 3) >> 2;
        PCMD_CHK((p1 & 3) == 0);
        const bool y_is_minus = (my == mm), y_is_plus = (my == mp);    // the usual case: y is one of the colour's bands
        auto four = [&](int64_t q, const float4 &A, const float4 &Bv, const float4 &Y) {
            // P, p0 and ppb are multiples of 4 here: every quad of the block's range is a full one
            one(A.x, Bv.x, Y.x);
            one(A.y, Bv.y, Y.y);
            one(A.z, Bv.z, Y.z);
            one(A.w, Bv.w, Y.w);
        };
        int64_t q = (p0 >> 2) + threadIdx.x;
        for (; q + NT < q1; q += 2 * NT) {             // two 16-byte loads per band in flight
            const float4 A0 = vp[q], B0 = vm[q], A1 = vp[q + NT], B1 = vm[q + NT];
            const float4 Y0 = y_is_minus ? B0 : (y_is_plus ? A0 : vy[q]);
            const float4 Y1 = y_is_minus ? B1 : (y_is_plus ? A1 : vy[q + NT]);
            four(q, A0, B0, Y0);
            four(q + NT, A1, B1, Y1);
        }
        for (; q < q1; q += NT) {
            const float4 A = vp[q], Bv = vm[q];
            const float4 Y = y_is_minus ? Bv : (y_is_plus ? A : vy[q]);
            four(q, A, Bv, Y);
        }
    } else {
        for (int64_t p = p0 + threadIdx.x; p < p1; p += NT) one(mp[p], mm[p], my[p]);
    }
    // block reduction of the stats in a fixed order (deterministic)
    __shared__ double r_sx[NT / 32], r_sy[NT / 32];
    __shared__ uint32_t r_n[3][NT / 32];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_in += __shfl_down_sync(0xffffffffu, n_in, d);
        n_out += __shfl_down_sync(0xffffffffu, n_out, d);
        n_bad += __shfl_down_sync(0xffffffffu, n_bad, d);
        sx += __shfl_down_sync(0xffffffffu, sx, d);
        sy += __shfl_down_sync(0xffffffffu, sy, d);
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { r_n[0][wid] = n_in; r_n[1][wid] = n_out; r_n[2][wid] = n_bad; r_sx[wid] = sx; r_sy[wid] = sy; }
    __syncthreads();
    if (threadIdx.x == 0) {
        pcmd_hess_stats st = {0, 0, 0, 0, 0.0, 0.0};
        for (int w = 0; w < NT / 32; ++w) {
            st.n_in += r_n[0][w]; st.n_out += r_n[1][w]; st.n_bad += r_n[2][w];
            st.sum_x += r_sx[w]; st.sum_y += r_sy[w];
        }
        if (SMEM) { st.n_out = sh[nbins]; st.n_bad = sh[nbins + 1]; st.n_in = (uint32_t)(p1 - p0) - st.n_out - st.n_bad; }
        if (gridDim.x == 1 && stats_out) stats_out[(size_t)m * n_hess + h] = st;   // the only block: final stats
        else part[((size_t)m * n_hess + h) * gridDim.x + blockIdx.x] = st;
    }
    if (SMEM) {
        if (gridDim.x == 1) {       // the only block of this diagram: plain stores, no memset needed
            for (int t = threadIdx.x; t < nbins; t += NT) gh[t] = sh[t];
        } else {
            for (int t = threadIdx.x; t < nbins; t += NT) {
                uint32_t v = sh[t];
                if (v) atomicAdd(&gh[t], v);
            }
        }
    }
}

__global__ void k_hess_stats(const pcmd_hess_stats *__restrict__ part, int nblk,
                             pcmd_hess_stats *__restrict__ out) {
    pdl_enter<PDL_EARLY_HESS>();
    // one warp per (model, hess): lane l adds partials l, l+32, ... in order, then a shuffle tree
    // (a fixed order: deterministic sums)
    const pcmd_hess_stats *p = part + (size_t)blockIdx.x * nblk;
    uint32_t n_in = 0, n_out = 0, n_bad = 0;
    double sx = 0.0, sy = 0.0;
    for (int b = threadIdx.x; b < nblk; b += 32) {
        n_in += p[b].n_in; n_out += p[b].n_out; n_bad += p[b].n_bad;
        sx += p[b].sum_x; sy += p[b].sum_y;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_in += __shfl_down_sync(0xffffffffu, n_in, d);
        n_out += __shfl_down_sync(0xffffffffu, n_out, d);
        n_bad += __shfl_down_sync(0xffffffffu, n_bad, d);
        sx += __shfl_down_sync(0xffffffffu, sx, d);
        sy += __shfl_down_sync(0xffffffffu, sy, d);
    }
    if (threadIdx.x == 0) {
        pcmd_hess_stats st = {n_in, n_out, n_bad, 0, sx, sy};
        out[blockIdx.x] = st;
    }
}

// Memset (when several blocks share a diagram), k_hess and k_hess_stats for a given geometry; `parts` is the scratch
// for the per-block partial statistics (the ctx's, or the fixed array of pcmd_hess_noalloc).
static int hess_run(pcmd_ctx *c, const float *d_mag, int n_models, int nblk, int64_t ppb, uint32_t *d_hess,
                    pcmd_hess_stats *parts, pcmd_hess_stats *d_stats, cudaStream_t s) {
    int maxbins = 0;
    for (int h = 0; h < c->n_hess; ++h) maxbins = max(maxbins, c->hess[h].nx * c->hess[h].ny);
    const size_t smem = ((size_t)maxbins + 2) * sizeof(uint32_t);      // + the two spare counters
    if (!(nblk == 1 && smem <= 200 * 1024))    // a single block per diagram stores its histogram itself
        PCMD_CUDA(c, cudaMemsetAsync(d_hess, 0, (size_t)n_models * c->hess_bins * sizeof(uint32_t), s));
    dim3 grid(nblk, c->n_hess, n_models);
    if (smem <= 200 * 1024) {
        // a histogram that leaves room for one block per SM only (c5: 200 x 200 bins = 160 KB) takes 1024 threads:
        // the same number of warps per SM as two 512-thread blocks
        const bool wide = smem > 100 * 1024;
        if (smem > 48 * 1024 && smem > c->smem_hess) {      // an attribute of the functions, not an allocation
            PCMD_CUDA(c, cudaFuncSetAttribute(k_hess<true, HS_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            PCMD_CUDA(c, cudaFuncSetAttribute(k_hess<true, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            c->smem_hess = smem;
        }
        if (wide)
            PCMD_CUDA(c, pcmd_launch_pdl((k_hess<true, 1024>), grid, dim3(1024), smem, s, d_mag, c->B, c->P, c->d_hess_spec,
                                         c->n_hess, ppb, c->hess_bins, d_hess, parts, d_stats));
        else
            PCMD_CUDA(c, pcmd_launch_pdl((k_hess<true, HS_THREADS>), grid, dim3(HS_THREADS), smem, s, d_mag, c->B, c->P,
                                         c->d_hess_spec, c->n_hess, ppb, c->hess_bins, d_hess, parts, d_stats));
    } else {
        PCMD_CUDA(c, pcmd_launch_pdl((k_hess<false, HS_THREADS>), grid, dim3(HS_THREADS), 0, s, d_mag, c->B, c->P,
                                     c->d_hess_spec, c->n_hess, ppb, c->hess_bins, d_hess, parts, d_stats));
    }
    PCMD_LAUNCHED(c);
    if (d_stats && nblk > 1) {
        PCMD_CUDA(c, pcmd_launch_pdl(k_hess_stats, dim3(n_models * c->n_hess), dim3(32), 0, s, parts, nblk, d_stats));
        PCMD_LAUNCHED(c);
    }
    return PCMD_OK;
}

int pcmd_launch_hess(pcmd_ctx *c, const float *d_mag, int n_models, uint32_t *d_hess,
                     pcmd_hess_stats *d_stats, cudaStream_t s) {
    // Pixels per block: at least HS_PIX_PER_BLOCK (a block zeroes and flushes a whole private histogram, so long
    // pixel runs amortise that); a batch that fills the GPU by itself takes one block per diagram, which also
    // saves the memset, the global atomics and the stats kernel (measured: splitting diagrams to fill the last
    // wave of CTAs costs more than it gains).
    int64_t want_blocks = ((int64_t)c->sm_count * 8) / ((int64_t)n_models * c->n_hess);
    if (want_blocks < 1) want_blocks = 1;
    int64_t ppb = (c->P + want_blocks - 1) / want_blocks;
    if (ppb < HS_PIX_PER_BLOCK) ppb = HS_PIX_PER_BLOCK;
    ppb = (ppb + 1023) & ~(int64_t)1023;
    const int nblk = (int)((c->P + ppb - 1) / ppb);
    const int64_t need = (int64_t)n_models * c->n_hess * nblk;
    if (need > c->hpart_cap) {
        if (c->d_hpart) cudaFree(c->d_hpart);
        c->d_hpart = nullptr; c->hpart_cap = 0;
        PCMD_CUDA(c, cudaMalloc(&c->d_hpart, need * sizeof(pcmd_hess_stats)));
        c->hpart_cap = need;
    }
    return hess_run(c, d_mag, n_models, nblk, ppb, d_hess, c->d_hpart, d_stats, s);
}

// ---------------------------------------------------------------------------------------------
// Stage 7.  One block per model; every reduction is a fixed-order tree (deterministic).
#define LL_THREADS 1024
#define LL_LFACT 4096        // ln(d!) = lgamma(d + 1) tabulated for d < LL_LFACT (computed on the device at pcmd_create)

__global__ void k_lfact(double *__restrict__ t) {
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d < LL_LFACT) t[d] = lgamma((double)d + 1.0);
}

int pcmd_build_lfact(pcmd_ctx *c) {
    PCMD_CUDA(c, cudaMalloc(&c->d_lfact, LL_LFACT * sizeof(double)));
    k_lfact<<<LL_LFACT / 256, 256>>>(c->d_lfact);
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}

__device__ double block_sum(double v, double *scratch) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_down_sync(0xffffffffu, v, d);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) scratch[wid] = v;
    __syncthreads();
    double t = 0.0;
    for (int w = 0; w < LL_THREADS / 32; ++w) t += scratch[w];
    return t;  // same value in every thread
}

__global__ void __launch_bounds__(LL_THREADS) k_loglike(const uint32_t *__restrict__ hm_all,
                                                        const pcmd_hess_stats *__restrict__ sm_all,
                                                        const uint32_t *__restrict__ hd_all,
                                                        const pcmd_hess_stats *__restrict__ sd_all,
                                                        const DevHess *__restrict__ specs, int n_hess,
                                                        int64_t bins_total, int mode, double m_floor,
                                                        const double *__restrict__ lfact,
                                                        double *__restrict__ out) {
    pdl_enter<PDL_EARLY_LIKE>();
    __shared__ double scratch[LL_THREADS / 32];
    const int m = blockIdx.x;
    double total = 0.0;
    for (int h = 0; h < n_hess; ++h) {
        const DevHess S = specs[h];
        const int nb = S.nx * S.ny;
        const uint32_t *hm = hm_all + (size_t)m * bins_total + S.bin_off;
        const uint32_t *hd = hd_all + S.bin_off;
        double nd = 0.0, nm = 0.0;
        for (int i = threadIdx.x; i < nb; i += LL_THREADS) { nd += (double)hd[i]; nm += (double)hm[i]; }
        const double Nd = block_sum(nd, scratch), Nm = block_sum(nm, scratch);
        if (!(Nm > 0.0) || !(Nd > 0.0)) { total = -INFINITY; continue; }
        double L = 0.0;
        if (mode == PCMD_LIKE_POISSON) {
            const double sc = Nd / Nm;
            for (int i = threadIdx.x; i < nb; i += LL_THREADS) {
                const uint32_t d = hd[i], mo = hm[i];
                if (d == 0 && mo == 0) continue;
                const double mu = sc * fmax((double)mo, m_floor);
                L += (double)d * log(mu) - mu - (d < LL_LFACT ? lfact[d] : lgamma((double)d + 1.0));
            }
            L = block_sum(L, scratch);
        } else {
            for (int i = threadIdx.x; i < nb; i += LL_THREADS) {
                const double d = (double)hd[i], mo = (double)hm[i];
                const double diff = d / Nd - mo / Nm;
                double var;
                if (mode == PCMD_LIKE_GAUSS_LITERAL) { double sg = fmax(sqrt(d * d + mo * mo), 2.0); var = sg * sg; }
                else {
                    double ed = fmax(sqrt(d), 1.0) / Nd, em = fmax(sqrt(mo), 1.0) / Nm;
                    var = ed * ed + em * em;
                }
                L += -(diff * diff) / (2.0 * var);
            }
            L = block_sum(L, scratch);
            const pcmd_hess_stats a = sm_all[(size_t)m * n_hess + h], b = sd_all[h];
            const double Cd = b.sum_x / (double)b.n_in, Cm = a.sum_x / (double)a.n_in;
            const double Md = b.sum_y / (double)b.n_in, Mm = a.sum_y / (double)a.n_in;
            L += -((Cd - Cm) * (Cd - Cm)) / (2.0 * 0.05 * 0.05) - ((Md - Mm) * (Md - Mm)) / (2.0 * 0.05 * 0.05);
        }
        total += L;
    }
    if (threadIdx.x == 0) out[m] = total;
}

int pcmd_launch_loglike(pcmd_ctx *c, const uint32_t *d_hm, const pcmd_hess_stats *d_sm, int n_models,
                        const uint32_t *d_hd, const pcmd_hess_stats *d_sd, int mode, double *d_out,
                        cudaStream_t s) {
    pcmd_launch_pdl(k_loglike, dim3(n_models), dim3(LL_THREADS), 0, s, d_hm, d_sm, d_hd, d_sd, c->d_hess_spec, c->n_hess,
                                              c->hess_bins, mode, c->like_floor, c->d_lfact, d_out);
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}

// ---------------------------------------------------------------------------------------------
// pcmd_hess_noalloc (include/pcmd.h): stage 6 without any allocation.  The per-block partial statistics of
// k_hess go to a fixed array in this module's device image (one per device that loads the library, held
// until exit) instead of ctx->d_hpart.  Same kernels, same launch geometry as pcmd_launch_hess: results
// are bit-identical.  Nothing in the array has to start at zero (k_hess writes every slot k_hess_stats
// reads); it is shared by every call on the device, so calls that overlap on the GPU race on it.
static __device__ __align__(256) pcmd_hess_stats g_hess_parts[PCMD_HESS_NOALLOC_MAX_PARTS];

#define HS_MAX_DEVICES 64
// In host code `g_hess_parts` is only a handle for the runtime's symbol table, not a device address: the
// address is looked up per device (with that device current) and cached here.
static pcmd_hess_stats *g_hess_parts_addr[HS_MAX_DEVICES];

static cudaError_t hess_noalloc_addr(pcmd_hess_stats **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= HS_MAX_DEVICES) return cudaErrorInvalidDevice;
    pcmd_hess_stats *p = __atomic_load_n(&g_hess_parts_addr[dev], __ATOMIC_ACQUIRE);
    if (!p) {
        e = cudaGetSymbolAddress((void **)&p, g_hess_parts);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        __atomic_store_n(&g_hess_parts_addr[dev], p, __ATOMIC_RELEASE);   // every thread looks up the same address
    }
    *out = p;
    return cudaSuccess;
}

extern "C" int pcmd_hess_noalloc_setup(void) {
    pcmd_hess_stats *p = nullptr;
    return hess_noalloc_addr(&p) == cudaSuccess ? PCMD_OK : PCMD_ECUDA;
}

// blocks per diagram and pixels per block: the rule of pcmd_launch_hess
static int hess_geometry(const pcmd_ctx *c, int n_models, int64_t *ppb_out) {
    int64_t want_blocks = ((int64_t)c->sm_count * 8) / ((int64_t)n_models * c->n_hess);
    if (want_blocks < 1) want_blocks = 1;
    int64_t ppb = (c->P + want_blocks - 1) / want_blocks;
    if (ppb < HS_PIX_PER_BLOCK) ppb = HS_PIX_PER_BLOCK;
    ppb = (ppb + 1023) & ~(int64_t)1023;
    if (ppb_out) *ppb_out = ppb;
    return (int)((c->P + ppb - 1) / ppb);
}

extern "C" int64_t pcmd_hess_noalloc_parts(const pcmd_ctx *c, int32_t n_models) {
    if (!c || n_models < 1 || c->n_hess < 1) return 0;
    return (int64_t)n_models * c->n_hess * hess_geometry(c, n_models, nullptr);
}

extern "C" int pcmd_hess_noalloc(pcmd_ctx *c, const float *d_mag, int32_t n_models, uint32_t *d_hess,
                                 pcmd_hess_stats *d_stats, void *cuda_stream) {
    if (!c || !d_mag || !d_hess || n_models < 1 || c->n_hess < 1) return PCMD_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int64_t ppb = 0;
    const int nblk = hess_geometry(c, n_models, &ppb);
    if ((int64_t)n_models * c->n_hess * nblk > PCMD_HESS_NOALLOC_MAX_PARTS) return PCMD_ELIMIT;
    pcmd_hess_stats *parts = nullptr;
    PCMD_CUDA(c, hess_noalloc_addr(&parts));
    PCMD_PROF(c, 4, s);
    const int rc = hess_run(c, d_mag, n_models, nblk, ppb, d_hess, parts, d_stats, s);
    if (rc) return rc;
    PCMD_PROF(c, 5, s);
    return PCMD_OK;
}
