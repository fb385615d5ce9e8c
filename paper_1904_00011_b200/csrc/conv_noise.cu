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
    pdl_enter<PDL_EARLY_CONV>();
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
    pdl_enter<PDL_EARLY_CONV>();
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


// ---------------------------------------------------------------------------------------------
// Separable PSF, register-blocked.  One launch per band, so the 2K PSF factors
// are kernel parameters with static indices: every FMA of the two passes takes its weight from the
// constant bank (no register, no shared-memory read).  A CTA makes a 64 x 64 output tile:
//   load   the halo tile (rows y0-r .. y0+63+r, columns rounded out to multiples of four) with 16-byte
//          loads, circular wrap applied per 16-byte segment (R-Q9);
//   rows   each thread makes 4 consecutive outputs of one halo-tile row from a sliding window of K+3
//          inputs held in registers (16-byte shared-memory loads), 16-byte store of the row result;
//   cols   each thread makes a 4 (x) x 4 (y) block of outputs from K+3 16-byte loads of row results;
//   out    stage 5 (noise, magnitude) on the 16 outputs in registers, 16-byte stores.
// K(4+K+3)/4... per output: 2K FMAs, ~2.4 shared-memory loads and ~0.3 stores (K = 15).
#define C2_TW 64
#define C2_TH 64
#define C2_THREADS 256
#define C2_KMAX 21
#ifndef C2_MINB_CLEAN
#define C2_MINB_CLEAN 6       // CTAs per SM of the noise-free instances (register cap 40, no spills; 5 -> 6: K = 7 +3 %, K = 15 flat)
#endif

struct Cv2Args {
    const float *F;      // [n_models][B][P] dusty flux
    float *mag;          // [n_models][B][P]
    float *tap_conv;     // optional
    const uint32_t *sky_tab;
    PointRec sky_rec;    // this band's Poisson-sky table
    int N, B, band;
    int64_t P;
    int shot_noise, poisson_sky;
    uint32_t key0, key1, model0;
    double zp, sky, read_sigma;
    float fr[C2_KMAX], fc[C2_KMAX];    // row factor, column factor of this band
    float2 rp[C2_KMAX];                // rp[t] = (fr[t], fr[t-1]): coefficient pair of an aligned input pair in the row pass
    float2 cp[C2_KMAX];                // cp[k] = (fc[k], fc[k]): coefficient pair of an output pair in the column pass
};

// packed FP32 pairs (FFMA2 on sm_100a: two FMAs per instruction, half the issue slots of the two passes)
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {      // a * b + c, lane-wise
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 as_pair(const float2 &p) { return *reinterpret_cast<const f32x2 *>(&p); }

__device__ __forceinline__ int wrap_any(int v, int N) {
    v %= N;
    return v < 0 ? v + N : v;
}

// zp - 2.5 log10(arg) for arg > 0, NaN for arg <= 0: one lg2.approx on the special-function unit (it handles the
// exponent itself: no exponent / mantissa split, no denormal pre-scaling of __log2f), finished in fp32 with zp and
// -2.5 log10(2) as float pairs: two fp32 FMAs instead of float->double, fp64 FMA, double->float (the conversion unit is
// a scarce pipe here).  The split of -2.5 log10(2) is chosen with a NEGATIVE high part and a POSITIVE low part, so that
// arg = 0 (lg2 = -inf) gives (+inf) + (-inf) = NaN and arg < 0 (lg2 = NaN) gives NaN with no compare and no select.
// Measured against the oracle's stage 5: max 1.7e-6 mag (fp64 finish: 1.6e-6).  A flux below FLT_MIN (1.2e-38: fainter
// than zp + 94.8 mag) is flushed to zero by the .ftz form and gives NaN (DESIGN.md R-Q20).
__device__ __forceinline__ float mag_of(float arg, double zp) {
    const float zph = (float)zp, zpl = (float)(zp - (double)zph);
    float l2;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l2) : "f"(arg));
    return fmaf(l2, -0.75257503986358642578125f, zph) + fmaf(l2, 5.0703633e-8f, zpl);
}
__device__ __forceinline__ float sqrt_approx(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));     // relative error ~1e-7: moves a magnitude by < 1e-8
    return r;
}
// #{i < 2^D : u > T[i]} in a table padded with 0xFFFFFFFF to 2^D entries (branch-free)
__device__ __forceinline__ uint32_t count_below_padded(const uint32_t *__restrict__ T, int D, uint32_t u) {
    uint32_t pos = 0;
    for (int sft = D - 1; sft >= 0; --sft) {
        const uint32_t probe = pos + (1u << sft);
        if (u > T[probe - 1]) pos = probe;
    }
    return pos;
}

// stage 5 for one pixel (R-Q11); `stab`: this band's sky table padded to 2^sky_d entries (shared memory), or the
// compact table in global memory (sky_d < 0)
__device__ __forceinline__ float noise_mag_one(const Cv2Args &a, float Gi, uint32_t p, uint32_t mctr, float skyf, float rs2,
                                               bool psky, bool need_g, const uint32_t *__restrict__ stab, int sky_d) {
    uint32_t w[4];
    float g = 0.f;
    if (need_g) {
        philox4x32_10(a.key0, a.key1, p, (uint32_t)a.band, mctr, 2u, w);
        g = normal_f32(w[0], w[1]);
    }
    float arg;      // C' - sky
    if (psky) {
        philox4x32_10(a.key0, a.key1, p, (uint32_t)a.band, mctr, 3u, w);
        const uint32_t n = sky_d >= 0 ? count_below_padded(stab, sky_d, w[0]) : count_below(stab, a.sky_rec.len, w[0]);
        const float Kc = (float)(a.sky_rec.k0 + n);
        const float var = (a.shot_noise ? fmaxf(Gi, 0.f) : 0.f) + rs2;
        arg = Gi + (Kc - skyf) + sqrt_approx(var) * g;
    } else {
        const float var = (a.shot_noise ? fmaxf(Gi + skyf, 0.f) : 0.f) + rs2;
        arg = Gi + sqrt_approx(var) * g;
    }
    return mag_of(arg, a.zp);
}

// NOISE = false: no shot / read noise and no Poisson sky (stage 5 is the magnitude only): a leaner instance
template <int K, bool VEC, bool NOISE>
__global__ void __launch_bounds__(C2_THREADS, (NOISE ? 4 : C2_MINB_CLEAN)) k_conv2(const Cv2Args a) {
    pdl_enter<PDL_EARLY_CONV>();
    constexpr int R = (K - 1) / 2, RA = (R + 3) & ~3, OFF = RA - R;
    constexpr int SW = C2_TW + 2 * RA;            // halo-tile row stride (floats), a multiple of 4
    constexpr int SH = C2_TH + K - 1;             // halo-tile rows
    constexpr int NV = (OFF + K + 3 + 3) / 4;     // 16-byte loads of one row-pass window
    constexpr int SKY_CAP = 1024;                 // Poisson-sky thresholds kept in shared memory
    static_assert((C2_TW / 4 - 1 + NV) * 4 <= SW, "row-pass window leaves the halo row");
    static_assert(C2_TH - 4 + K + 2 < SH, "column-pass window leaves the halo tile");
    extern __shared__ __align__(16) float sm[];
    float *tile = sm;                             // [SH + 1][SW]: row SH is a spare row nobody writes (row pass, idle lanes)
    float *hrow = sm;                             // row results overwrite the first 64 columns of their own tile row (stride SW)
    uint32_t *ssky = reinterpret_cast<uint32_t *>(sm + (SH + 1) * SW);        // [SKY_CAP], noisy instances only
    const int N = a.N, m = blockIdx.z, mb = m * a.B + a.band, tid = threadIdx.x;
    const float *F = a.F + (size_t)mb * a.P;
    const int x0 = blockIdx.x * C2_TW, y0 = blockIdx.y * C2_TH;
    const bool psky = NOISE && a.poisson_sky && a.sky > 0.0;
    int sky_d = -1;                                // log2 of the padded sky table in shared memory; -1: table stays in global memory
    if (psky && a.sky_rec.len < SKY_CAP) {
        sky_d = 32 - __clz(a.sky_rec.len);         // 2^sky_d > len: at least one 0xFFFFFFFF pad entry
        for (int t = tid; t < (1 << sky_d); t += C2_THREADS)
            ssky[t] = t < (int)a.sky_rec.len ? a.sky_tab[a.sky_rec.off + t] : 0xFFFFFFFFu;
    }
    // ---- load: rows y0-R .., columns x0-RA ..; rows past the last needed output row are skipped
    const int rows_used = min(SH, N - y0 + K - 1);          // halo rows that feed an output row < N
    // one conditional add / subtract wraps an index when the image is at least as large as the halo tile
    const bool big = N >= SW && N >= SH;
    if (VEC) {
        constexpr int NQ = SW / 4;                 // 16-byte segments per halo row (18 ... 22)
        // N % 4 == 0: a segment never straddles the edge.  Flat index over (row, segment): every lane copies.
        if (big) {      // a thread keeps its 16-byte column segment and walks down the rows: only the wrapped source row changes
            constexpr int RPI = C2_THREADS / NQ;                  // rows per sweep of the CTA (11 ... 14)
            if (tid < RPI * NQ) {
                const int r0 = tid / NQ, q = tid - r0 * NQ;
                int gx = x0 - RA + 4 * q, gy = y0 - R + r0;
                gx += gx < 0 ? N : 0; gx -= gx >= N ? N : 0;
                gy += gy < 0 ? N : 0; gy -= gy >= N ? N : 0;
                // byte offset of the wrapped source row, stepped by RPI rows (one conditional subtract wraps it):
                // 32-bit arithmetic and one 64-bit add per copy; the column's base address is pinned in a register
                // pair (the compiler otherwise recomputes the whole 64-bit chain under every copy's predicate)
                unsigned long long src = reinterpret_cast<unsigned long long>(F + gx);
                asm volatile("" : "+l"(src));
                const uint32_t NN = (uint32_t)N * (uint32_t)N * 4u, step = (uint32_t)(RPI * N) * 4u;
                uint32_t off = (uint32_t)gy * (uint32_t)N * 4u;
                uint32_t dst = (uint32_t)__cvta_generic_to_shared(reinterpret_cast<float4 *>(tile) + tid);
                const int rem = rows_used - r0;
#pragma unroll
                for (int it = 0; it < (SH + RPI - 1) / RPI; ++it) {
                    PCMD_CHK(it * RPI >= rem || (gx >= 0 && gx + 3 < N && off < NN && off % (4u * (uint32_t)N) == 0u && tid + it * RPI * NQ < SH * NQ));
                    if (it * RPI < rem)
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src + off) : "memory");
                    off += step; off -= off >= NN ? NN : 0u;
                    dst += RPI * NQ * 16;
                }
            }
        } else {
            for (int t = tid; t < rows_used * NQ; t += C2_THREADS) {
                const int i = t / NQ, q = t - i * NQ;
                const int gy = wrap_any(y0 - R + i, N), gx = wrap_any(x0 - RA + 4 * q, N);
                PCMD_CHK(gx >= 0 && gx + 3 < N && gy >= 0 && gy < N && t < SH * NQ);
                const uint32_t dst = (uint32_t)__cvta_generic_to_shared(reinterpret_cast<float4 *>(tile) + t);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(F + (size_t)gy * N + gx) : "memory");
            }
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
    } else {
        for (int t = tid; t < rows_used * SW; t += C2_THREADS) {
            const int i = t / SW, j = t - i * SW;
            tile[i * SW + j] = F[(size_t)wrap_any(y0 - R + i, N) * N + wrap_any(x0 - RA + j, N)];
        }
    }
    __syncthreads();
    // ---- row pass: h[i][x] = sum_k fr[k] F[i][x - (k - R)]
    constexpr int ROW_IT = (SH * (C2_TW / 4) + C2_THREADS - 1) / C2_THREADS;
#pragma unroll
    for (int it = 0; it < ROW_IT; ++it) {
        const int t = tid + it * C2_THREADS;
        const int i = t / (C2_TW / 4), sgm = t - i * (C2_TW / 4);
        const bool live = i < rows_used;        // a warp holds two rows: both halves reach the __syncwarp below
        float v[NV * 4];
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            // idle lanes read the spare row (values unused): an unconditional load, no zero-filling of the window
            const float4 f4 = reinterpret_cast<const float4 *>(tile + (live ? i : SH) * SW)[sgm + q];
            v[4 * q] = f4.x; v[4 * q + 1] = f4.y; v[4 * q + 2] = f4.z; v[4 * q + 3] = f4.w;
        }
        // h[c] = sum_i fr[b - i] v[i], i = OFF + c ... OFF + c + K - 1, b = OFF + c + K - 1: aligned input pairs
        // (v[2m], v[2m+1]) take the coefficient pair rp[b - 2m] in one FFMA2, the odd end(s) a plain FMA
        float h[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            constexpr int dummy = 0; (void)dummy;
            const int lo = OFF + c, hi = OFF + c + K - 1;
            f32x2 acc2 = pack2(0.f, 0.f);
            float single = 0.f;
#pragma unroll
            for (int i = lo; i <= hi; ++i) {
                if ((i & 1) == 0 && i + 1 <= hi) acc2 = fma2(pack2(v[i], v[i + 1]), as_pair(a.rp[hi - i]), acc2);
                else if ((i & 1) == 1 && i == lo) single = fmaf(a.fr[hi - i], v[i], single);
                else if ((i & 1) == 0 && i == hi) single = fmaf(a.fr[0], v[i], single);
            }
            float p0, p1;
            unpack2(acc2, p0, p1);
            h[c] = (p0 + p1) + single;
        }
        // in place: the 16 tasks of a row sit in one warp; every lane has its window in registers before any lane stores
        __syncwarp();
        if (live) reinterpret_cast<float4 *>(hrow + i * SW)[sgm] = make_float4(h[0], h[1], h[2], h[3]);
    }
    __syncthreads();
    // ---- column pass: G[y][x] = sum_k fc[k] h[y - (k - R)][x], 4 x 4 outputs per thread
    const int xg = tid & 15, yb = tid >> 4;
    float acc[4][4];
    {
        f32x2 a01[4], a23[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) { a01[j] = pack2(0.f, 0.f); a23[j] = pack2(0.f, 0.f); }
        if (y0 + 4 * yb < N) {
#pragma unroll
            for (int n = 0; n < K + 3; ++n) {
                const float4 hv = reinterpret_cast<const float4 *>(hrow + (4 * yb + n) * SW)[xg];
                const f32x2 h01 = pack2(hv.x, hv.y), h23 = pack2(hv.z, hv.w);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int k = j + (K - 1) - n;
                    if (k >= 0 && k < K) {
                        a01[j] = fma2(h01, as_pair(a.cp[k]), a01[j]);
                        a23[j] = fma2(h23, as_pair(a.cp[k]), a23[j]);
                    }
                }
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) { unpack2(a01[j], acc[j][0], acc[j][1]); unpack2(a23[j], acc[j][2], acc[j][3]); }
    }
    // ---- stage 5 on the 16 outputs
    const uint32_t mctr = a.model0 + (uint32_t)m;
    const float skyf = (float)a.sky, rs2 = (float)(a.read_sigma * a.read_sigma);
    const bool need_g = NOISE && (a.shot_noise || a.read_sigma > 0.0);
    const uint32_t *stab = sky_d >= 0 ? ssky : a.sky_tab + a.sky_rec.off;
    const int x = x0 + 4 * xg, yt = y0 + 4 * yb;
    if (x >= N || yt >= N) return;
    const uint32_t p0 = (uint32_t)yt * (uint32_t)N + (uint32_t)x;
    float *mag = a.mag + (size_t)mb * a.P + p0;
    if (VEC && yt + 3 < N) {                        // the whole 4 x 4 block is inside the image, 16-byte stores
        PCMD_CHK((int64_t)p0 + 3 * (int64_t)N + 3 < a.P);
        if (a.tap_conv) {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                *reinterpret_cast<float4 *>(a.tap_conv + (size_t)mb * a.P + p0 + (size_t)j * N) = make_float4(acc[j][0], acc[j][1], acc[j][2], acc[j][3]);
        }
        if (!NOISE) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float mg[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) mg[c] = mag_of(acc[j][c], a.zp);
                *reinterpret_cast<float4 *>(mag + (size_t)j * N) = make_float4(mg[0], mg[1], mg[2], mg[3]);
            }
        } else {
#pragma unroll 1
            for (int j = 0; j < 4; ++j) {       // one row of four pixels at a time: sixteen interleaved Philox calls would spill
                float mg[4];
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    mg[c] = noise_mag_one(a, acc[j][c], p0 + (uint32_t)(j * N + c), mctr, skyf, rs2, psky, need_g, stab, sky_d);
                *reinterpret_cast<float4 *>(mag + (size_t)j * N) = make_float4(mg[0], mg[1], mg[2], mg[3]);
            }
        }
        return;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (yt + j >= N) continue;
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if (x + c < N) {
                const size_t o = (size_t)j * N + c;
                if (a.tap_conv) a.tap_conv[(size_t)mb * a.P + p0 + o] = acc[j][c];
                mag[o] = noise_mag_one(a, acc[j][c], p0 + (uint32_t)o, mctr, skyf, rs2, psky, need_g, stab, sky_d);
            }
    }
}

template <int K>
static size_t conv2_smem(bool noise) {
    constexpr int R = (K - 1) / 2, RA = (R + 3) & ~3;
    return ((size_t)(C2_TH + K - 1 + 1) * (C2_TW + 2 * RA) + (noise ? 1024 : 0)) * sizeof(float);   // + the spare row
}

template <int K>
static cudaError_t conv2_launch(const Cv2Args &a, int n_models, cudaStream_t s) {
    const dim3 grid((a.N + C2_TW - 1) / C2_TW, (a.N + C2_TH - 1) / C2_TH, n_models);
    const bool vec = (a.N & 3) == 0 && ((reinterpret_cast<uintptr_t>(a.F) | reinterpret_cast<uintptr_t>(a.mag) |
                                         reinterpret_cast<uintptr_t>(a.tap_conv)) & 15) == 0;
    const bool noise = a.shot_noise || a.read_sigma > 0.0 || (a.poisson_sky && a.sky > 0.0);
    if (vec && noise) pcmd_launch_pdl((k_conv2<K, true, true>), grid, dim3(C2_THREADS), conv2_smem<K>(true), s, a);
    else if (vec) pcmd_launch_pdl((k_conv2<K, true, false>), grid, dim3(C2_THREADS), conv2_smem<K>(false), s, a);
    else if (noise) pcmd_launch_pdl((k_conv2<K, false, true>), grid, dim3(C2_THREADS), conv2_smem<K>(true), s, a);
    else pcmd_launch_pdl((k_conv2<K, false, false>), grid, dim3(C2_THREADS), conv2_smem<K>(false), s, a);
    return cudaGetLastError();
}

int pcmd_conv_setup(pcmd_ctx *) { return PCMD_OK; }     // k_conv2 needs at most 33 KB of dynamic shared memory: no opt-in

static int launch_conv2(pcmd_ctx *c, int n_models, uint64_t seed, uint32_t model0, float *d_mag, const float *h_fac,
                        cudaStream_t s) {
    for (int b = 0; b < c->B; ++b) {
        Cv2Args a;
        a.F = c->d_fdust; a.mag = d_mag; a.tap_conv = c->tap_conv; a.sky_tab = c->d_sky_tab; a.sky_rec = c->sky_rec[b];
        a.N = c->N; a.B = c->B; a.band = b; a.P = c->P; a.shot_noise = c->shot_noise; a.poisson_sky = c->poisson_sky;
        a.key0 = (uint32_t)(seed & 0xFFFFFFFFull); a.key1 = (uint32_t)(seed >> 32); a.model0 = model0;
        a.zp = c->zp[b]; a.sky = c->sky[b]; a.read_sigma = c->read_sigma[b];
        for (int k = 0; k < C2_KMAX; ++k) {
            a.fr[k] = k < c->K ? h_fac[((size_t)b * 2) * c->K + k] : 0.f;
            a.fc[k] = k < c->K ? h_fac[((size_t)b * 2 + 1) * c->K + k] : 0.f;
        }
        for (int k = 0; k < C2_KMAX; ++k) {
            a.rp[k] = make_float2(a.fr[k], k > 0 ? a.fr[k - 1] : 0.f);
            a.cp[k] = make_float2(a.fc[k], a.fc[k]);
        }
        cudaError_t e;
        switch (c->K) {
            case 5: e = conv2_launch<5>(a, n_models, s); break;
            case 7: e = conv2_launch<7>(a, n_models, s); break;
            case 15: e = conv2_launch<15>(a, n_models, s); break;
            default: e = conv2_launch<21>(a, n_models, s); break;
        }
        c->launches++;
        if (e != cudaSuccess) { c->last_cuda = (int)e; return PCMD_ECUDA; }
    }
    return PCMD_OK;
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
    // k_conv2 (64 x 64 tiles, one launch per band) when a launch fills the GPU; small jobs take the 32 x 32-tile kernel
    // below in one launch over all bands (4x the CTAs: latency-bound there, not bandwidth-bound)
    const int64_t ctas2 = (int64_t)((c->N + C2_TW - 1) / C2_TW) * ((c->N + C2_TH - 1) / C2_TH) * n_models;
    if (c->psf_sep && c->h_psf_sep && (K == 5 || K == 7 || K == 15 || K == 21) && ctas2 >= 2 * (int64_t)c->sm_count)
        return launch_conv2(c, n_models, seed, model0, d_mag, c->h_psf_sep, s);
    if (c->psf_sep) {
        size_t smem = ((size_t)(CV_TX + K - 1) * (CV_TY + K - 1) + (size_t)(CV_TY + K - 1) * CV_TX + 2 * (size_t)K) * sizeof(float);
        const dim3 blk(CV_TX, CV_ROWS);
        if (K == 5) pcmd_launch_pdl((k_conv_noise_sep<5>), grid, blk, smem, s, a);
        else if (K == 7) pcmd_launch_pdl((k_conv_noise_sep<7>), grid, blk, smem, s, a);
        else if (K == 15) pcmd_launch_pdl((k_conv_noise_sep<15>), grid, blk, smem, s, a);
        else if (K == 21) pcmd_launch_pdl((k_conv_noise_sep<21>), grid, blk, smem, s, a);
        else {
            if (smem > 48 * 1024 && smem > c->smem_conv_sep) {
                PCMD_CUDA(c, cudaFuncSetAttribute(k_conv_noise_sep<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                c->smem_conv_sep = smem;
            }
            pcmd_launch_pdl((k_conv_noise_sep<0>), grid, blk, smem, s, a);
        }
    } else {
        size_t smem = ((size_t)(CV_TX + K - 1) * (CV_TY + K - 1) + (size_t)K * K) * sizeof(float);
        if (smem > 48 * 1024 && smem > c->smem_conv) {
            PCMD_CUDA(c, cudaFuncSetAttribute(k_conv_noise, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            c->smem_conv = smem;
        }
        pcmd_launch_pdl(k_conv_noise, grid, dim3(CV_TX, CV_ROWS), smem, s, a);
    }
    PCMD_LAUNCHED(c);
    return PCMD_OK;
}
