// conv_noise.cu -- stage 4: per-band PSF convolution with circular boundary (
// R-Q9), and stage 5 fused into its epilogue: sky, shot/read noise, magnitudes (PAPER.md:83,
// 127-128,178; R-Q11).  Shared-memory tiled direct 2-D convolution (works for any PSF).
#include "pcmd_internal.cuh"

#define CV_TX 32
#define CV_TY 32
#define CV_ROWS 8   // blockDim.y; each thread computes CV_TY / CV_ROWS outputs

// v mod N for v in [-N, 2N) by one conditional add/subtract; the general case (image smaller than
// the PSF halo) falls back to the division.
__device__ __forceinline__ int wrap_index(int v, int N) {
    if (v < 0) v += N;
    if (v >= N) v -= N;
    if ((unsigned)v >= (unsigned)N) { v %= N; if (v < 0) v += N; }
    return v;
}

struct CvArgs {
    const float *F;      // [n_models][B][P] dusty flux
    const float *psf;    // [B][K][K]
    const float *psf_sep; // [B][2][K] row factor, column factor (separable PSFs only)
    float *mag;          // [n_models][B][P]
    float *tap_conv;     // optional
    const uint32_t *sky_tab;
    PointRec sky_rec[4];
    int N, B, K, G;      // G: PSF grid cells per side (1: one PSF per band)
    int64_t P;
    int shot_noise, poisson_sky;
    uint32_t key0, key1, model0;
    double zp[4], sky[4], read_sigma[4];
};

__device__ __forceinline__ void noise_mag_epilogue(const CvArgs &a, const float (&acc)[CV_TY / CV_ROWS], int x0, int y0,
                                                   int lx, int m, int b, int mb);

__global__ void __launch_bounds__(CV_TX * CV_ROWS) k_conv_noise(const CvArgs a) {
    extern __shared__ float sm[];
    const int K = a.K, r = (K - 1) / 2, N = a.N;
    const int TW = CV_TX + K - 1, TH = CV_TY + K - 1;
    float *tile = sm;              // [TH][TW]
    float *spsf = sm + TH * TW;    // [K][K]
    const int mb = blockIdx.z, m = mb / a.B, b = mb - m * a.B;
    const float *F = a.F + (size_t)mb * a.P;
    const int x0 = blockIdx.x * CV_TX, y0 = blockIdx.y * CV_TY;
    const int tid = threadIdx.y * CV_TX + threadIdx.x, nt = CV_TX * CV_ROWS;
    for (int i = threadIdx.y; i < TH; i += CV_ROWS) {      // halo tile with circular wrap (R-Q9)
        const float *row = F + (size_t)wrap_index(y0 - r + i, N) * N;
        for (int j = threadIdx.x; j < TW; j += CV_TX) tile[i * TW + j] = row[wrap_index(x0 - r + j, N)];
    }
    const int lx = threadIdx.x;
    float acc[CV_TY / CV_ROWS];
#pragma unroll
    for (int q = 0; q < CV_TY / CV_ROWS; ++q) acc[q] = 0.f;
    // Sub-pixel PSF grid (R-Q19): G x G cells of `cell` pixels, an output pixel uses its
    // cell's PSF.  The tile is convolved once per cell it touches (G = 1: once).
    const int G = a.G, cell = (N + G - 1) / G;
    const int gy0 = min(G - 1, y0 / cell), gy1 = min(G - 1, min(N - 1, y0 + CV_TY - 1) / cell);
    const int gx0 = min(G - 1, x0 / cell), gx1 = min(G - 1, min(N - 1, x0 + CV_TX - 1) / cell);
    const int my_gx = min(G - 1, (x0 + lx) / cell);
    for (int gy = gy0; gy <= gy1; ++gy)
        for (int gx = gx0; gx <= gx1; ++gx) {
            __syncthreads();           // the previous cell's PSF (and, first time, the tile stores) are done
            for (int t = tid; t < K * K; t += nt) spsf[t] = a.psf[(((size_t)b * G + gy) * G + gx) * K * K + t];
            __syncthreads();
            if (my_gx != gx) continue;
            bool mine[CV_TY / CV_ROWS];
            bool any = false;
#pragma unroll
            for (int q = 0; q < CV_TY / CV_ROWS; ++q) {
                mine[q] = min(G - 1, (y0 + (int)threadIdx.y + q * CV_ROWS) / cell) == gy;
                any |= mine[q];
            }
            if (!any) continue;
            float part[CV_TY / CV_ROWS];
#pragma unroll
            for (int q = 0; q < CV_TY / CV_ROWS; ++q) part[q] = 0.f;
            for (int ka = 0; ka < K; ++ka)
                for (int kb = 0; kb < K; ++kb) {
                    const float w = spsf[ka * K + kb];
#pragma unroll
                    for (int q = 0; q < CV_TY / CV_ROWS; ++q) {
                        const int ly = threadIdx.y + q * CV_ROWS;
                        part[q] = fmaf(w, tile[(ly + 2 * r - ka) * TW + (lx + 2 * r - kb)], part[q]);
                    }
                }
#pragma unroll
            for (int q = 0; q < CV_TY / CV_ROWS; ++q) if (mine[q]) acc[q] = part[q];
        }
    noise_mag_epilogue(a, acc, x0, y0, lx, m, b, mb);
}

// Separable PSF (column factor (x) row factor, R-Q10): row pass over the halo tile into shared
// memory, then the column pass: 2K FMAs per output instead of K^2.  Same tile, halo and epilogue.
template <int KT>
__global__ void __launch_bounds__(CV_TX * CV_ROWS) k_conv_noise_sep(const CvArgs a) {
    extern __shared__ float sm[];
    const int K = KT ? KT : a.K, r = (K - 1) / 2, N = a.N;
    const int TW = CV_TX + K - 1, TH = CV_TY + K - 1;
    float *tile = sm;                  // [TH][TW]
    float *hrow = sm + TH * TW;        // [TH][CV_TX] row-convolved
    float *fac = hrow + TH * CV_TX;    // [2][K]: row factor, column factor
    const int mb = blockIdx.z, m = mb / a.B, b = mb - m * a.B;
    const float *F = a.F + (size_t)mb * a.P;
    const int x0 = blockIdx.x * CV_TX, y0 = blockIdx.y * CV_TY;
    const int tid = threadIdx.y * CV_TX + threadIdx.x, nt = CV_TX * CV_ROWS;
    for (int t = tid; t < 2 * K; t += nt) fac[t] = a.psf_sep[(size_t)b * 2 * K + t];
    for (int i = threadIdx.y; i < TH; i += CV_ROWS) {      // halo tile with circular wrap (R-Q9)
        const float *row = F + (size_t)wrap_index(y0 - r + i, N) * N;
        for (int j = threadIdx.x; j < TW; j += CV_TX) tile[i * TW + j] = row[wrap_index(x0 - r + j, N)];
    }
    __syncthreads();
    const int lx = threadIdx.x;
    for (int i = threadIdx.y; i < TH; i += CV_ROWS) {
        float h = 0.f;
#pragma unroll
        for (int kb = 0; kb < K; ++kb) h = fmaf(fac[kb], tile[i * TW + (lx + 2 * r - kb)], h);
        hrow[i * CV_TX + lx] = h;
    }
    __syncthreads();
    float acc[CV_TY / CV_ROWS];
#pragma unroll
    for (int q = 0; q < CV_TY / CV_ROWS; ++q) acc[q] = 0.f;
#pragma unroll
    for (int ka = 0; ka < K; ++ka) {
        const float w = fac[K + ka];
#pragma unroll
        for (int q = 0; q < CV_TY / CV_ROWS; ++q) {
            const int ly = threadIdx.y + q * CV_ROWS;
            acc[q] = fmaf(w, hrow[(ly + 2 * r - ka) * CV_TX + lx], acc[q]);
        }
    }
    noise_mag_epilogue(a, acc, x0, y0, lx, m, b, mb);
}

// Stage 5 for the CV_TY / CV_ROWS outputs of one thread (R-Q11): sky, noise, magnitude.
__device__ __forceinline__ void noise_mag_epilogue(const CvArgs &a, const float (&acc)[CV_TY / CV_ROWS], int x0, int y0,
                                                   int lx, int m, int b, int mb) {
    const int N = a.N;
    const int x = x0 + lx;
    if (x >= N) return;
    const uint32_t mctr = a.model0 + (uint32_t)m;
    const double sky = a.sky[b], rs = a.read_sigma[b], zp = a.zp[b];
    const float skyf = (float)sky, rs2 = (float)(rs * rs);
    const bool psky = a.poisson_sky && sky > 0.0;
    const bool need_g = a.shot_noise || rs > 0.0;
#pragma unroll
    for (int q = 0; q < CV_TY / CV_ROWS; ++q) {
        const int y = y0 + threadIdx.y + q * CV_ROWS;
        if (y >= N) continue;
        const uint32_t p = (uint32_t)y * (uint32_t)N + (uint32_t)x;
        const size_t o = (size_t)mb * a.P + p;
        if (a.tap_conv) a.tap_conv[o] = acc[q];
        // fp32 arithmetic (the noise term is a few per cent of the counts, so a
        // 1e-7 error of the normal moves the magnitude by < 1e-8); only zp - 2.5 log10 is finished in fp64
        const float Gi = acc[q];
        uint32_t w[4];
        float g = 0.f;
        if (need_g) {
            philox4x32_10(a.key0, a.key1, p, (uint32_t)b, mctr, 2u, w);
            g = normal_f32(w[0], w[1]);
        }
        float arg;      // C' - sky
        if (psky) {
            philox4x32_10(a.key0, a.key1, p, (uint32_t)b, mctr, 3u, w);
            const PointRec sr = a.sky_rec[b];
            const float Kc = (float)(sr.k0 + count_below(a.sky_tab + sr.off, sr.len, w[0]));
            const float var = (a.shot_noise ? fmaxf(Gi, 0.f) : 0.f) + rs2;
            arg = Gi + (Kc - skyf) + sqrtf(var) * g;
        } else {
            const float var = (a.shot_noise ? fmaxf(Gi + skyf, 0.f) : 0.f) + rs2;
            arg = Gi + sqrtf(var) * g;
        }
        a.mag[o] = (arg > 0.f) ? (float)fma((double)log2_pos(arg), -0.75257498915995298, zp) : __int_as_float(0x7fc00000);
    }
}

int pcmd_launch_conv_noise(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, float *d_mag,
                           cudaStream_t s) {
    CvArgs a;
    a.F = c->d_fdust; a.psf = c->d_psf; a.psf_sep = c->d_psf_sep; a.mag = d_mag; a.tap_conv = c->tap_conv;
    a.sky_tab = c->d_sky_tab;
    for (int b = 0; b < 4; ++b) {
        a.sky_rec[b] = c->sky_rec[b];
        a.zp[b] = c->zp[b]; a.sky[b] = c->sky[b]; a.read_sigma[b] = c->read_sigma[b];
    }
    a.N = c->N; a.B = c->B; a.K = c->K; a.G = c->psf_grid; a.P = c->P;
    a.shot_noise = c->shot_noise; a.poisson_sky = c->poisson_sky;
    a.key0 = (uint32_t)(seed & 0xFFFFFFFFull); a.key1 = (uint32_t)(seed >> 32); a.model0 = model0;
    const int K = c->K;
    dim3 grid((c->N + CV_TX - 1) / CV_TX, (c->N + CV_TY - 1) / CV_TY, n_models * c->B);
    if (c->psf_sep) {
        size_t smem = ((size_t)(CV_TX + K - 1) * (CV_TY + K - 1) + (size_t)(CV_TY + K - 1) * CV_TX + 2 * (size_t)K) * sizeof(float);
        const dim3 blk(CV_TX, CV_ROWS);
        if (K == 5) k_conv_noise_sep<5><<<grid, blk, smem, s>>>(a);
        else if (K == 7) k_conv_noise_sep<7><<<grid, blk, smem, s>>>(a);
        else if (K == 15) k_conv_noise_sep<15><<<grid, blk, smem, s>>>(a);
        else if (K == 21) k_conv_noise_sep<21><<<grid, blk, smem, s>>>(a);
        else {
            if (smem > 48 * 1024 && smem > c->smem_conv_sep) {
                PCMD_CUDA(c, cudaFuncSetAttribute(k_conv_noise_sep<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                c->smem_conv_sep = smem;
            }
            k_conv_noise_sep<0><<<grid, blk, smem, s>>>(a);
        }
    } else {
        size_t smem = ((size_t)(CV_TX + K - 1) * (CV_TY + K - 1) + (size_t)K * K) * sizeof(float);
        if (smem > 48 * 1024 && smem > c->smem_conv) {
            PCMD_CUDA(c, cudaFuncSetAttribute(k_conv_noise, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            c->smem_conv = smem;
        }
        k_conv_noise<<<grid, dim3(CV_TX, CV_ROWS), smem, s>>>(a);
    }
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}
