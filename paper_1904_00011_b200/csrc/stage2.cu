// stage2.cu -- Poisson star count for every (pixel, isochrone point) pair, summed into pixel
// fluxes, with the dust screen applied in the epilogue.
//
// Mapping: lanes of a warp are consecutive pixels and every thread owns PX pixels; the warp walks
// the isochrone points in groups of four (one Philox call = the four draws of one pixel, R-C1),
// so every table read is warp-uniform.  Records are staged through shared memory.
#include "pcmd_internal.cuh"

struct S2Args {
    const PointRec *rec;     // [n_models][Jpad]
    const uint32_t *tab;     // [n_models][cap]
    const uint64_t *mult;    // [Jpad]
    const DevModel *mdl;     // [n_models]
    int64_t cap;
    int Jpad, N, B, dust_mode;
    int64_t P;
    uint32_t key0, key1, model0;
    double dust_frac;
    double coef[4];
    float *flux_raw;         // optional [n_models][B][P]
    float *flux_dust;        // [n_models][B][P]
    uint64_t *hash;          // optional [n_models][P]
    uint32_t *total;         // optional [n_models][P]
};

#define S2_THREADS 256
#define S2_CHUNK 64          // groups per staged chunk (64 * 128 B = 8 KB)

template <int PX, bool COUNTS>
__global__ void __launch_bounds__(S2_THREADS) k_stage2_generic(const S2Args a) {
    __shared__ PointRec srec[S2_CHUNK * 4];
    const int m = blockIdx.y;
    const PointRec *rec = a.rec + (size_t)m * a.Jpad;
    const uint32_t *tab = a.tab + (size_t)m * a.cap;
    const int64_t tile0 = (int64_t)blockIdx.x * (S2_THREADS * PX);
    uint32_t pix[PX];
    float F[PX][4];
    uint32_t tot[PX];
    uint64_t hsh[PX];
#pragma unroll
    for (int i = 0; i < PX; ++i) {
        pix[i] = (uint32_t)(tile0 + (int64_t)i * S2_THREADS + threadIdx.x);
        F[i][0] = F[i][1] = F[i][2] = F[i][3] = 0.f;
        tot[i] = 0; hsh[i] = 0;
    }
    const uint32_t mctr = a.model0 + (uint32_t)m;
    const int n_groups = a.Jpad >> 2;
    for (int g0 = 0; g0 < n_groups; g0 += S2_CHUNK) {
        const int ng = min(S2_CHUNK, n_groups - g0);
        __syncthreads();
        {   // stage ng*4 records: 2 x 16 B per record
            const uint4 *src = reinterpret_cast<const uint4 *>(rec + (size_t)g0 * 4);
            uint4 *dst = reinterpret_cast<uint4 *>(srec);
            for (int t = threadIdx.x; t < ng * 8; t += S2_THREADS) dst[t] = src[t];
        }
        __syncthreads();
        for (int g = 0; g < ng; ++g) {
            uint32_t u[PX][4];
#pragma unroll
            for (int i = 0; i < PX; ++i)
                philox4x32_10(a.key0, a.key1, pix[i], (uint32_t)(g0 + g), mctr, 0u, u[i]);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                const PointRec r = srec[g * 4 + w];
#pragma unroll
                for (int i = 0; i < PX; ++i) {
                    uint32_t n = r.k0;
                    if (u[i][w] > r.T0) n += count_below(tab + r.off, r.len, u[i][w]);
                    if (n) {
                        float nf = (float)n;
                        F[i][0] = fmaf(nf, r.f[0], F[i][0]);
                        F[i][1] = fmaf(nf, r.f[1], F[i][1]);
                        F[i][2] = fmaf(nf, r.f[2], F[i][2]);
                        F[i][3] = fmaf(nf, r.f[3], F[i][3]);
                        if (COUNTS) { tot[i] += n; hsh[i] += (uint64_t)n * a.mult[(g0 + g) * 4 + w]; }
                    }
                }
            }
        }
    }
    // epilogue: raw flux, counts, dust (stage 3)
    const DevModel M = a.mdl[m];
#pragma unroll
    for (int i = 0; i < PX; ++i) {
        if ((int64_t)pix[i] >= a.P) continue;
        if (COUNTS) { a.total[(size_t)m * a.P + pix[i]] = tot[i]; a.hash[(size_t)m * a.P + pix[i]] = hsh[i]; }
        double A = 0.0; bool behind = true;
        if (a.dust_mode != 0) {
            uint32_t w[4];
            philox4x32_10(a.key0, a.key1, pix[i], 0u, mctr, 1u, w);
            A = M.dust_med * exp(M.dust_sigma * normal_from_words(w[0], w[1]));
            if (a.dust_mode == 2) behind = ((double)w[2] < a.dust_frac * 4294967296.0);
        }
        for (int b = 0; b < a.B; ++b) {
            size_t o = ((size_t)m * a.B + b) * a.P + pix[i];
            if (a.flux_raw) a.flux_raw[o] = F[i][b];
            double fac = 1.0;
            if (a.dust_mode == 1) fac = (1.0 - a.dust_frac) + a.dust_frac * pow(10.0, -0.4 * a.coef[b] * A);
            else if (a.dust_mode == 2) fac = behind ? pow(10.0, -0.4 * a.coef[b] * A) : 1.0;
            a.flux_dust[o] = (float)((double)F[i][b] * fac);
        }
    }
}

int pcmd_launch_stage2(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, float *d_flux_raw,
                       uint64_t *d_hash, uint32_t *d_total, cudaStream_t s) {
    S2Args a;
    a.rec = c->d_rec; a.tab = c->d_tab; a.mult = c->d_mult; a.mdl = c->d_model;
    a.cap = c->cap_raw; a.Jpad = c->Jpad; a.N = c->N; a.B = c->B; a.dust_mode = c->dust_mode; a.P = c->P;
    a.key0 = (uint32_t)(seed & 0xFFFFFFFFull); a.key1 = (uint32_t)(seed >> 32); a.model0 = model0;
    a.dust_frac = c->dust_frac;
    for (int b = 0; b < 4; ++b) a.coef[b] = c->dust_coef[b];
    a.flux_raw = d_flux_raw; a.flux_dust = c->d_fdust;
    a.hash = d_hash; a.total = d_total;
    const int PX = 4;
    dim3 grid((unsigned)((c->P + S2_THREADS * PX - 1) / (S2_THREADS * PX)), (unsigned)n_models);
    if (d_hash) k_stage2_generic<PX, true><<<grid, S2_THREADS, 0, s>>>(a);
    else k_stage2_generic<PX, false><<<grid, S2_THREADS, 0, s>>>(a);
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}
