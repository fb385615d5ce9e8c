/*
 * pcmd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see pcmd_oracle.h).
 *
 * fp64, single translation unit, no blocking / fusion / reordering beyond what
 * the cited passages and DESIGN.md readings state.  Build:
 *   gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC -o liboracle_pcmd.so pcmd_oracle.c -lm
 * (-ffp-contract=off: the bit-exact parts -- lambda and the sampler tables -- must
 * not be contracted into FMAs.)  OpenMP only distributes independent pixels.
 */
#include "pcmd_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TWO32 4294967296.0
#define TWO_M64 5.42101086242752217e-20 /* 2^-64 */
#define ORC_LAMBDA_MAX 4194304.0        /* 2^22 */

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------
 * Random stream.  Paper silent (PAPER.md:194 says only "random Poisson calls");
 * DESIGN.md R-C1: Philox4x32-10 (Salmon et al. 2011), key = (seed_lo, seed_hi),
 * counter = (pixel, group, model, stream).
 * ---------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; /* Weyl key schedule, bumped after each round */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void stream_words(uint64_t seed, uint32_t pixel, uint32_t group, uint32_t model,
                         uint32_t stream, uint32_t out[4]) {
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { pixel, group, model, stream };
    orc_philox4x32_10(key, ctr, out);
}

/* order-independent exact checksum multiplier (DESIGN.md R-C4) */
uint64_t orc_splitmix64(uint64_t j) {
    uint64_t z = j + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

/* ------------------------------------------------------------------------
 * Poisson sampler: inverse CDF on a 32-bit fixed-point table (DESIGN.md R-C2).
 * ---------------------------------------------------------------------- */
int64_t orc_poisson_table(double lambda, uint64_t *T_out, int64_t cap, int64_t *k_lo_out,
                          int64_t *k_hi_out) {
    if (!(lambda >= 0.0) || lambda > ORC_LAMBDA_MAX) return -1;
    if (lambda == 0.0) { /* n = 0 always */
        if (cap < 1) return -1 - 1;
        T_out[0] = (uint64_t)TWO32; *k_lo_out = 0; *k_hi_out = 0;
        return 1;
    }
    int64_t m = (int64_t)floor(lambda);
    /* step 1: relative pmf q[k] = pmf(k)/pmf(m) by the two recurrences; first count */
    int64_t k_hi = m, k_lo = m;
    {
        double v = 1.0;
        for (int64_t k = m + 1;; ++k) {
            v = v * (lambda / (double)k);
            if (v < TWO_M64) break;
            k_hi = k;
        }
        v = 1.0;
        for (int64_t k = m - 1; k >= 0; --k) {
            v = v * ((double)(k + 1) / lambda);
            if (v < TWO_M64) break;
            k_lo = k;
        }
    }
    int64_t n = k_hi - k_lo + 1;
    if (n > cap) return -n - 1;
    double *q = (double *)malloc((size_t)n * sizeof(double));
    if (!q) return -1;
    q[m - k_lo] = 1.0;
    for (int64_t k = m + 1; k <= k_hi; ++k) q[k - k_lo] = q[k - 1 - k_lo] * (lambda / (double)k);
    for (int64_t k = m - 1; k >= k_lo; --k) q[k - k_lo] = q[k + 1 - k_lo] * ((double)(k + 1) / lambda);
    /* step 2: S = sum in increasing k */
    double S = 0.0;
    for (int64_t i = 0; i < n; ++i) S += q[i];
    /* step 3: T[k] = (uint64)((c/S) 2^32 + 0.5) */
    double c = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        c += q[i];
        T_out[i] = (uint64_t)((c / S) * TWO32 + 0.5);
    }
    free(q);
    *k_lo_out = k_lo; *k_hi_out = k_hi;
    return n;
}

uint32_t orc_poisson_draw_linear(const uint64_t *T, int64_t k_lo, int64_t k_hi, uint32_t u) {
    /* T[k] = 0 for k < k_lo, so the scan can start at k_lo */
    for (int64_t k = k_lo; k <= k_hi; ++k)
        if ((uint64_t)u < T[k - k_lo]) return (uint32_t)k;
    return (uint32_t)k_hi; /* unreachable: T[k_hi] = 2^32 > u */
}

uint32_t orc_poisson_draw(const uint64_t *T, int64_t k_lo, int64_t k_hi, uint32_t u) {
    /* first index i with T[i] > u (T is non-decreasing) */
    int64_t lo = 0, hi = k_hi - k_lo; /* answer in [lo, hi] since T[hi] = 2^32 > u */
    while (lo < hi) {
        int64_t mid = lo + (hi - lo) / 2;
        if (T[mid] > (uint64_t)u) hi = mid; else lo = mid + 1;
    }
    return (uint32_t)(k_lo + lo);
}

/* ------------------------------------------------------------------------
 * Stage 1: isochrone weighting ("assigning each point a weight ...
 * normalizing the weights to equal N_pix"; PAPER.md:134-139 Gaussian MDF on the
 * grid, weights < 1 % removed).  Arithmetic order: DESIGN.md R-C3.
 * ---------------------------------------------------------------------- */
double orc_expneg(double t) {
    /* e^-t for t >= 0 from basic operations only: degree-6 Taylor polynomial of
     * e^-r at r = t 2^-16 in Horner form, then sixteen squarings. */
    static const double c[7] = { 0.0, 1.0, 1.0 / 2.0, 1.0 / 3.0, 1.0 / 4.0, 1.0 / 5.0, 1.0 / 6.0 };
    if (t > 64.0) return 0.0;
    double r = t * (1.0 / 65536.0);
    double p = 1.0;
    for (int k = 6; k >= 1; --k) p = 1.0 - (r * c[k]) * p;
    for (int i = 0; i < 16; ++i) p = p * p;
    return p;
}

int orc_stage1(const orc_config *c, const orc_params *p, double *mdfw, double *lambda, double *flux) {
    const int Z = c->n_feh, J = c->n_points, B = c->n_bands;
    if (!(p->feh_sigma > 0.0)) return -1;
    double *w = (double *)malloc((size_t)Z * sizeof(double));
    double e_min = INFINITY;
    for (int z = 0; z < Z; ++z) {
        double d = c->feh_grid[z] - p->feh_mean;
        w[z] = (d * d) / ((2.0 * p->feh_sigma) * p->feh_sigma);
        if (w[z] < e_min) e_min = w[z];
    }
    double G = 0.0;
    for (int z = 0; z < Z; ++z) { w[z] = orc_expneg(w[z] - e_min); G += w[z]; }
    double G2 = 0.0;
    for (int z = 0; z < Z; ++z) {
        w[z] = w[z] / G;
        if (w[z] < c->mdf_cut) w[z] = 0.0;
        G2 += w[z];
    }
    for (int z = 0; z < Z; ++z) { w[z] = w[z] / G2; if (mdfw) mdfw[z] = w[z]; }
    for (int j = 0; j < J; ++j) {
        if (lambda)
            lambda[j] = (p->sfh[c->age_idx[j]] * w[c->feh_idx[j]]) * c->imf_w[j];
        if (flux)  /* PAPER.md:81 "converted to fluxes according to the distance" */
            for (int b = 0; b < B; ++b)
                flux[(size_t)j * B + b] = pow(10.0, -0.4 * (c->absmag[(size_t)j * B + b] + p->dmod - c->zp[b]));
    }
    free(w);
    return 0;
}

/* ------------------------------------------------------------------------
 * Stage 2: Poisson star count for every (pixel, isochrone point) pair, summed
 * into pixel fluxes ("For every pixel ... we randomly draw the number
 * of stars in each bin according to a Poisson distribution with the given
 * weights"; "summed into their respective pixels").
 * ---------------------------------------------------------------------- */
typedef struct { uint64_t *T; int64_t *off, *k_lo, *k_hi; } orc_tables;

static int build_tables(int J, const double *lambda, orc_tables *t) {
    t->off = (int64_t *)malloc((size_t)(J + 1) * sizeof(int64_t));
    t->k_lo = (int64_t *)malloc((size_t)J * sizeof(int64_t));
    t->k_hi = (int64_t *)malloc((size_t)J * sizeof(int64_t));
    t->T = NULL;
    int64_t cap = 0, used = 0;
    for (int j = 0; j < J; ++j) {
        t->off[j] = used;
        for (;;) {
            int64_t n = orc_poisson_table(lambda[j], t->T ? t->T + used : NULL, cap - used,
                                          &t->k_lo[j], &t->k_hi[j]);
            if (n >= 0) { used += n; break; }
            if (n == -1) return -1;
            int64_t need = used + (-n - 1);
            cap = need * 2 + 1024;
            t->T = (uint64_t *)realloc(t->T, (size_t)cap * sizeof(uint64_t));
            if (!t->T) return -1;
        }
    }
    t->off[J] = used;
    return 0;
}
static void free_tables(orc_tables *t) { free(t->T); free(t->off); free(t->k_lo); free(t->k_hi); }

int orc_stage2(const orc_config *c, const double *lambda, const double *flux,
               uint64_t seed, uint32_t model, const uint32_t *pix, int64_t n_pix,
               double *F_raw, uint32_t *total, uint64_t *hash, uint32_t *counts) {
    const int J = c->n_points, B = c->n_bands;
    orc_tables t;
    if (build_tables(J, lambda, &t)) { return -1; }
    uint64_t *mult = (uint64_t *)malloc((size_t)J * sizeof(uint64_t));
    for (int j = 0; j < J; ++j) mult[j] = orc_splitmix64((uint64_t)j) | 1ull;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n_pix; ++i) {
        uint32_t p = pix ? pix[i] : (uint32_t)i;
        double F[16];
        for (int b = 0; b < B; ++b) F[b] = 0.0;
        uint32_t tot = 0; uint64_t h = 0; uint32_t w[4] = {0, 0, 0, 0};
        for (int j = 0; j < J; ++j) {
            if ((j & 3) == 0) stream_words(seed, p, (uint32_t)(j >> 2), model, 0u, w);
            uint32_t n = 0;
            if (lambda[j] > 0.0)
                n = orc_poisson_draw(t.T + t.off[j], t.k_lo[j], t.k_hi[j], w[j & 3]);
            if (counts) counts[(size_t)i * J + j] = n;
            if (n) {
                for (int b = 0; b < B; ++b) F[b] += (double)n * flux[(size_t)j * B + b];
                tot += n; h += (uint64_t)n * mult[j];
            }
        }
        if (F_raw) for (int b = 0; b < B; ++b) F_raw[(size_t)b * n_pix + i] = F[b];
        if (total) total[i] = tot;
        if (hash) hash[i] = h;
    }
    free(mult); free_tables(&t);
    return 0;
}

/* ------------------------------------------------------------------------
 * Aggregated sampler (PAPER.md:75 footnote 3; DESIGN.md R-A1): the number of stars of a pixel is one
 * Poisson draw with mean Lambda = sum_j lambda_j, and, given that number, every star is of point j with
 * probability lambda_j / Lambda (the counts of independent Poisson variables conditioned on their sum are
 * multinomial).  In integers, so that any implementation draws the same stars:
 *   Lambda = sum_j lambda_j added in increasing j;   w_j = (uint64)((lambda_j / Lambda) 2^40 + 0.5);
 *   C_j = sum_{i<j} w_i,  W = C_J;
 *   N_p: word 0 of Philox counter (pixel, 0, model, 4) through the R-C2 table of Lambda;
 *   star s < N_p: counter (pixel, 1 + (s >> 1), model, 4), U = word[2(s&1)] 2^32 + word[2(s&1)+1],
 *   r = floor(U W / 2^64), the star is of the point j with C_j <= r < C_{j+1}.
 * Returns 0, -1 (Lambda out of range).  weights_out (optional): w_j. */
int orc_stage2_agg(const orc_config *c, const double *lambda, const double *flux,
                   uint64_t seed, uint32_t model, const uint32_t *pix, int64_t n_pix,
                   double *F_raw, uint32_t *total, uint64_t *hash, uint32_t *counts, uint64_t *weights_out) {
    const int J = c->n_points, B = c->n_bands;
    double Lambda = 0.0;
    for (int j = 0; j < J; ++j) Lambda += lambda[j];
    uint64_t *C = (uint64_t *)malloc((size_t)(J + 1) * sizeof(uint64_t));
    C[0] = 0;
    for (int j = 0; j < J; ++j) {
        uint64_t w = 0;
        if (Lambda > 0.0) w = (uint64_t)((lambda[j] / Lambda) * 1099511627776.0 + 0.5);
        if (weights_out) weights_out[j] = w;
        C[j + 1] = C[j] + w;
    }
    const uint64_t W = C[J];
    uint64_t *T = NULL; int64_t tcap = 0, k_lo = 0, k_hi = 0, n;
    while ((n = orc_poisson_table(Lambda, T, tcap, &k_lo, &k_hi)) < -1) {
        tcap = (-n - 1) * 2; T = (uint64_t *)realloc(T, (size_t)tcap * sizeof(uint64_t));
    }
    if (n == -1) { free(T); free(C); return -1; }
    uint64_t *mult = (uint64_t *)malloc((size_t)J * sizeof(uint64_t));
    for (int j = 0; j < J; ++j) mult[j] = orc_splitmix64((uint64_t)j) | 1ull;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n_pix; ++i) {
        uint32_t p = pix ? pix[i] : (uint32_t)i;
        double F[16];
        for (int b = 0; b < B; ++b) F[b] = 0.0;
        uint64_t h = 0; uint32_t w[4];
        if (counts) for (int j = 0; j < J; ++j) counts[(size_t)i * J + j] = 0;
        stream_words(seed, p, 0u, model, 4u, w);
        const uint32_t N = (Lambda > 0.0 && W > 0) ? orc_poisson_draw(T, k_lo, k_hi, w[0]) : 0;
        for (uint32_t s = 0; s < N; ++s) {
            if ((s & 1) == 0) stream_words(seed, p, 1u + (s >> 1), model, 4u, w);
            const uint64_t U = ((uint64_t)w[2 * (s & 1)] << 32) | (uint64_t)w[2 * (s & 1) + 1];
            const uint64_t r = (uint64_t)(((unsigned __int128)U * (unsigned __int128)W) >> 64);
            int lo = 0, hi = J;                      /* the j with C[j] <= r < C[j+1]: C[lo] <= r < C[hi] throughout */
            while (hi - lo > 1) {
                int mid = (lo + hi) / 2;
                if (C[mid] <= r) lo = mid; else hi = mid;
            }
            for (int b = 0; b < B; ++b) F[b] += flux[(size_t)lo * B + b];
            h += mult[lo];
            if (counts) counts[(size_t)i * J + lo] += 1;
        }
        if (F_raw) for (int b = 0; b < B; ++b) F_raw[(size_t)b * n_pix + i] = F[b];
        if (total) total[i] = N;
        if (hash) hash[i] = h;
    }
    free(mult); free(T); free(C);
    return 0;
}

int orc_stage2_brute(const orc_config *c, const double *lambda, const double *flux,
                     uint64_t seed, uint32_t model, double *F_raw, uint32_t *total) {
    /* materialise every star: a growing list of (pixel, point) records, one per star,
     * each count found by the linear-scan definition; then add the stars one by one */
    const int J = c->n_points, B = c->n_bands;
    const int64_t P = (int64_t)c->n_im * c->n_im;
    uint32_t *star_pix = NULL, *star_pt = NULL; int64_t n_star = 0, cap = 0;
    uint64_t *T = NULL; int64_t tcap = 0;
    for (int j = 0; j < J; ++j) {
        int64_t k_lo, k_hi, n;
        while ((n = orc_poisson_table(lambda[j], T, tcap, &k_lo, &k_hi)) < -1) {
            tcap = (-n - 1) * 2; T = (uint64_t *)realloc(T, (size_t)tcap * sizeof(uint64_t));
        }
        if (n == -1) { free(T); free(star_pix); free(star_pt); return -1; }
        for (int64_t p = 0; p < P; ++p) {
            uint32_t w[4];
            stream_words(seed, (uint32_t)p, (uint32_t)(j >> 2), model, 0u, w);
            uint32_t cnt = (lambda[j] > 0.0) ? orc_poisson_draw_linear(T, k_lo, k_hi, w[j & 3]) : 0;
            for (uint32_t s = 0; s < cnt; ++s) {
                if (n_star == cap) {
                    cap = cap ? cap * 2 : 1024;
                    star_pix = (uint32_t *)realloc(star_pix, (size_t)cap * 4);
                    star_pt = (uint32_t *)realloc(star_pt, (size_t)cap * 4);
                }
                star_pix[n_star] = (uint32_t)p; star_pt[n_star] = (uint32_t)j; ++n_star;
            }
        }
    }
    for (int64_t i = 0; i < P * B; ++i) F_raw[i] = 0.0;
    for (int64_t p = 0; p < P; ++p) total[p] = 0;
    for (int64_t s = 0; s < n_star; ++s) {
        for (int b = 0; b < B; ++b) F_raw[(size_t)b * P + star_pix[s]] += flux[(size_t)star_pt[s] * B + b];
        total[star_pix[s]] += 1;
    }
    free(T); free(star_pix); free(star_pt);
    return 0;
}

/* ------------------------------------------------------------------------
 * Box-Muller normal from two 32-bit words (DESIGN.md R-C4):
 * u_i = (w_i + 1/2) 2^-32, z = sqrt(-2 ln u_1) cos(2 pi u_2).
 * ---------------------------------------------------------------------- */
double orc_normal(uint32_t w0, uint32_t w1) {
    double u1 = ((double)w0 + 0.5) * (1.0 / TWO32);
    double u2 = ((double)w1 + 0.5) * (1.0 / TWO32);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925 * u2);
}

/* ------------------------------------------------------------------------
 * Stage 3: dust screen (E1 constant, E2/E3 log-normal per pixel,
 * F_dust = fraction reddened).  Readings R-Q7, R-Q8 in DESIGN.md.
 * ---------------------------------------------------------------------- */
int orc_stage3(const orc_config *c, const orc_params *p, uint64_t seed, uint32_t model,
               const double *F_raw, double *A_pix, double *F_dust) {
    const int B = c->n_bands;
    const int64_t P = (int64_t)c->n_im * c->n_im;
#pragma omp parallel for
    for (int64_t i = 0; i < P; ++i) {
        double A = 0.0; int behind = 1;
        if (c->dust_mode != 0) {
            uint32_t w[4];
            stream_words(seed, (uint32_t)i, 0u, model, 1u, w);
            double z = orc_normal(w[0], w[1]);
            A = p->dust_med * exp(p->dust_sigma * z);
            if (c->dust_mode == 2) behind = ((double)w[2] < c->dust_frac * TWO32);
        }
        if (A_pix) A_pix[i] = A;
        for (int b = 0; b < B; ++b) {
            double fac = 1.0;
            if (c->dust_mode == 1)
                fac = (1.0 - c->dust_frac) + c->dust_frac * pow(10.0, -0.4 * c->dust_coef[b] * A);
            else if (c->dust_mode == 2)
                fac = behind ? pow(10.0, -0.4 * c->dust_coef[b] * A) : 1.0;
            F_dust[(size_t)b * P + i] = F_raw[(size_t)b * P + i] * fac;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * Stage 4: PSF convolution per band ("The raw images are convolved with
 * models for the point-spread function (PSF) in each filter"), circular boundary
 * (DESIGN.md R-Q9):  G[y][x] = sum_{dy,dx} PSF[dy+r][dx+r] F[(y-dy) mod N][(x-dx) mod N].
 * ---------------------------------------------------------------------- */
int orc_stage4(const orc_config *c, const double *F_in, double *G) {
    const int B = c->n_bands, N = c->n_im, K = c->psf_k, r = (K - 1) / 2;
    const int64_t P = (int64_t)N * N;
    /* PAPER.md:180 "we subdivide each image into a 4 x 4 grid and apply to each a different PSF
     * convolution, shifted by fractions of a pixel" (DESIGN.md R-Q19): cells of ceil(N/G) pixels; the
     * output pixel (y, x) uses the PSF of its cell; the sum runs over the whole (circular) image. */
    const int Gd = c->psf_grid > 1 ? c->psf_grid : 1;
    const int cell = (N + Gd - 1) / Gd;
    for (int b = 0; b < B; ++b) {
        const double *F = F_in + (size_t)b * P;
#pragma omp parallel for
        for (int y = 0; y < N; ++y)
            for (int x = 0; x < N; ++x) {
                int gy = y / cell, gx = x / cell;
                if (gy > Gd - 1) gy = Gd - 1;
                if (gx > Gd - 1) gx = Gd - 1;
                const double *psf = c->psf + ((size_t)b * Gd * Gd + (size_t)gy * Gd + gx) * K * K;
                double s = 0.0;
                for (int dy = -r; dy <= r; ++dy)
                    for (int dx = -r; dx <= r; ++dx) {
                        int yy = ((y - dy) % N + N) % N, xx = ((x - dx) % N + N) % N;
                        s += psf[(dy + r) * K + (dx + r)] * F[(size_t)yy * N + xx];
                    }
                G[(size_t)b * P + (size_t)y * N + x] = s;
            }
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * Stage 5: sky + noise + magnitudes ("Sky flux can be added at this
 * stage.  Poisson shot noise is added, assuming the data are in electrons, such
 * that noise = sqrt(counts).  The resulting pCMD is computed by converting the
 * pixel counts to magnitudes").  Readings R-Q11 in DESIGN.md.
 * ---------------------------------------------------------------------- */
int orc_stage5(const orc_config *c, uint64_t seed, uint32_t model, const double *G, double *mag) {
    const int B = c->n_bands;
    const int64_t P = (int64_t)c->n_im * c->n_im;
    for (int b = 0; b < B; ++b) {
        const double sky = c->sky[b], rs = c->read_sigma[b];
        const int psky = (c->poisson_sky && sky > 0.0);
        uint64_t *T = NULL; int64_t k_lo = 0, k_hi = 0;
        if (psky) { /* one table per band, shared by all pixels */
            int64_t n, cap = 0;
            while ((n = orc_poisson_table(sky, T, cap, &k_lo, &k_hi)) < -1) {
                cap = -n - 1; T = (uint64_t *)realloc(T, (size_t)cap * sizeof(uint64_t));
            }
            if (n == -1) { free(T); return -1; }
        }
#pragma omp parallel for
        for (int64_t i = 0; i < P; ++i) {
            uint32_t w[4];
            double g = 0.0;
            const int need_g = (c->shot_noise || rs > 0.0);
            if (need_g) {
                stream_words(seed, (uint32_t)i, (uint32_t)b, model, 2u, w);
                g = orc_normal(w[0], w[1]);
            }
            double Gi = G[(size_t)b * P + i], Cp;
            if (psky) {
                stream_words(seed, (uint32_t)i, (uint32_t)b, model, 3u, w);
                double Kc = (double)orc_poisson_draw(T, k_lo, k_hi, w[0]);
                double var = (c->shot_noise ? fmax(Gi, 0.0) : 0.0) + rs * rs;
                Cp = Gi + Kc + sqrt(var) * g;
            } else {
                double C = Gi + sky;
                double var = (c->shot_noise ? fmax(C, 0.0) : 0.0) + rs * rs;
                Cp = C + sqrt(var) * g;
            }
            double arg = Cp - sky;
            mag[(size_t)b * P + i] = (arg > 0.0) ? c->zp[b] - 2.5 * log10(arg) : NAN;
        }
        free(T);
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * Stage 6: Hess diagram = 2-D histogram of (colour, magnitude),
 * half-open bins, out-of-window and NaN pixels dropped and counted (R-Q13).
 * ---------------------------------------------------------------------- */
static int near_edge(double v, double lo, double d, int n, double tol) {
    double t = (v - lo) / d;
    double k = floor(t + 0.5); /* nearest edge index */
    if (k < 0.0 || k > (double)n) return 0;
    return fabs(v - (lo + k * d)) <= tol;
}

int orc_hess(const orc_hess_spec *h, int64_t n_pix, int32_t n_bands, const double *mag,
             uint32_t *hess, orc_hess_stats *st, double edge_tol,
             uint32_t *n_edge_out, uint32_t *edge_list, int64_t edge_cap) {
    (void)n_bands;
    const double dx = (h->x_hi - h->x_lo) / h->nx, dy = (h->y_hi - h->y_lo) / h->ny;
    memset(hess, 0, (size_t)h->nx * h->ny * sizeof(uint32_t));
    orc_hess_stats s = {0, 0, 0, 0.0, 0.0};
    uint32_t n_edge = 0;
    for (int64_t i = 0; i < n_pix; ++i) {
        double mp = mag[(size_t)h->band_plus * n_pix + i], mm = mag[(size_t)h->band_minus * n_pix + i];
        double my = mag[(size_t)h->band_y * n_pix + i];
        if (isnan(mp) || isnan(mm) || isnan(my)) { s.n_bad++; continue; }
        double x = mp - mm, y = my;
        if (near_edge(x, h->x_lo, dx, h->nx, edge_tol) || near_edge(y, h->y_lo, dy, h->ny, edge_tol)) {
            if (edge_list && n_edge < edge_cap) edge_list[n_edge] = (uint32_t)i;
            n_edge++;
        }
        double fx = floor((x - h->x_lo) / dx), fy = floor((y - h->y_lo) / dy);
        if (fx < 0.0 || fx >= (double)h->nx || fy < 0.0 || fy >= (double)h->ny) { s.n_out++; continue; }
        hess[(size_t)fy * h->nx + (size_t)fx] += 1;
        s.n_in++; s.sum_x += x; s.sum_y += y;
    }
    if (st) *st = s;
    if (n_edge_out) *n_edge_out = n_edge;
    return 0;
}

int orc_hess_f32(const orc_hess_spec *h, int64_t n_pix, int32_t n_bands, const float *mag,
                 uint32_t *hess, orc_hess_stats *st) {
    (void)n_bands;
    /* kernel-precision decision:
     * x = fl32(mp - mm); t = fl32(fl32(x - fl32(x_lo)) * fl32(nx / (x_hi - x_lo))); ix = floor(t) */
    const float x_lo = (float)h->x_lo, y_lo = (float)h->y_lo;
    const float inv_dx = (float)((double)h->nx / (h->x_hi - h->x_lo));
    const float inv_dy = (float)((double)h->ny / (h->y_hi - h->y_lo));
    memset(hess, 0, (size_t)h->nx * h->ny * sizeof(uint32_t));
    orc_hess_stats s = {0, 0, 0, 0.0, 0.0};
    for (int64_t i = 0; i < n_pix; ++i) {
        float mp = mag[(size_t)h->band_plus * n_pix + i], mm = mag[(size_t)h->band_minus * n_pix + i];
        float my = mag[(size_t)h->band_y * n_pix + i];
        if (isnan(mp) || isnan(mm) || isnan(my)) { s.n_bad++; continue; }
        volatile float x = mp - mm;
        volatile float tx0 = x - x_lo, ty0 = my - y_lo;
        volatile float tx = tx0 * inv_dx, ty = ty0 * inv_dy;
        float fx = floorf(tx), fy = floorf(ty);
        if (!(fx >= 0.0f) || !(fx < (float)h->nx) || !(fy >= 0.0f) || !(fy < (float)h->ny)) { s.n_out++; continue; }
        hess[(size_t)fy * h->nx + (size_t)fx] += 1;
        s.n_in++; s.sum_x += (double)x; s.sum_y += (double)my;
    }
    if (st) *st = s;
    return 0;
}

/* Per-pixel form of the two functions above, for the parity tests: bin[i] = iy*nx + ix of pixel i
 * (the very statements of orc_hess / orc_hess_f32), -1 outside the window, -2 for a NaN magnitude;
 * near[i] (optional): bit 0 = x within tol_x of a bin edge, bit 1 = y within tol_y of one
 * (north_star: "Hess bins may differ only for pixels lying within 1e-5 mag of a bin edge"; a colour
 * is the difference of two magnitudes, so tol_x = 2 tol_y, DESIGN.md R-Q17).
 * Pinned by tests/test_oracle_stages.py: the histogram of bin[] is orc_hess's, near != 0 is its edge list. */
int orc_hess_pixels(const orc_hess_spec *h, int64_t n_pix, int32_t n_bands, const double *mag,
                    double tol_x, double tol_y, int32_t *bin, uint8_t *near) {
    (void)n_bands;
    const double dx = (h->x_hi - h->x_lo) / h->nx, dy = (h->y_hi - h->y_lo) / h->ny;
    for (int64_t i = 0; i < n_pix; ++i) {
        double mp = mag[(size_t)h->band_plus * n_pix + i], mm = mag[(size_t)h->band_minus * n_pix + i];
        double my = mag[(size_t)h->band_y * n_pix + i];
        if (near) near[i] = 0;
        if (isnan(mp) || isnan(mm) || isnan(my)) { bin[i] = -2; continue; }
        double x = mp - mm, y = my;
        if (near) near[i] = (uint8_t)((near_edge(x, h->x_lo, dx, h->nx, tol_x) ? 1 : 0) |
                                      (near_edge(y, h->y_lo, dy, h->ny, tol_y) ? 2 : 0));
        double fx = floor((x - h->x_lo) / dx), fy = floor((y - h->y_lo) / dy);
        if (fx < 0.0 || fx >= (double)h->nx || fy < 0.0 || fy >= (double)h->ny) { bin[i] = -1; continue; }
        bin[i] = (int32_t)((size_t)fy * h->nx + (size_t)fx);
    }
    return 0;
}

int orc_hess_pixels_f32(const orc_hess_spec *h, int64_t n_pix, int32_t n_bands, const float *mag, int32_t *bin) {
    (void)n_bands;
    const float x_lo = (float)h->x_lo, y_lo = (float)h->y_lo;
    const float inv_dx = (float)((double)h->nx / (h->x_hi - h->x_lo));
    const float inv_dy = (float)((double)h->ny / (h->y_hi - h->y_lo));
    for (int64_t i = 0; i < n_pix; ++i) {
        float mp = mag[(size_t)h->band_plus * n_pix + i], mm = mag[(size_t)h->band_minus * n_pix + i];
        float my = mag[(size_t)h->band_y * n_pix + i];
        if (isnan(mp) || isnan(mm) || isnan(my)) { bin[i] = -2; continue; }
        volatile float x = mp - mm;
        volatile float tx0 = x - x_lo, ty0 = my - y_lo;
        volatile float tx = tx0 * inv_dx, ty = ty0 * inv_dy;
        float fx = floorf(tx), fy = floorf(ty);
        if (!(fx >= 0.0f) || !(fx < (float)h->nx) || !(fy >= 0.0f) || !(fy < (float)h->ny)) { bin[i] = -1; continue; }
        bin[i] = (int32_t)((size_t)fy * h->nx + (size_t)fx);
    }
    return 0;
}

/* ------------------------------------------------------------------------
 * Stage 7.  Poisson lnL of the data Hess given the model Hess scaled to the data's
 * pixel count, with a floor on empty model bins (north_star; PAPER.md:226 explains
 * why a bare Poisson model fails on empty model bins; DESIGN.md R-Q15):
 *   s = N_d/N_m;  mu_i = s max(m_i, m_floor);
 *   lnL = sum over bins with d_i>0 or m_i>0 of  d_i ln mu_i - mu_i - lgamma(d_i+1).
 * ---------------------------------------------------------------------- */
double orc_loglike_poisson(const uint32_t *hm, const uint32_t *hd, int64_t n_bins, double m_floor) {
    double Nd = 0.0, Nm = 0.0;
    for (int64_t i = 0; i < n_bins; ++i) { Nd += (double)hd[i]; Nm += (double)hm[i]; }
    if (!(Nm > 0.0) || !(Nd > 0.0)) return -INFINITY;
    double s = Nd / Nm, L = 0.0;
    for (int64_t i = 0; i < n_bins; ++i) {
        if (hd[i] == 0 && hm[i] == 0) continue;
        double mu = s * fmax((double)hm[i], m_floor);
        L += (double)hd[i] * log(mu) - mu - lgamma((double)hd[i] + 1.0);
    }
    return L;
}

/* Eq. 2-4.  Reading R-Q14: e_d = max(sqrt d,1)/N_d,
 * e_m = max(sqrt m,1)/N_m, sigma^2 = e_d^2 + e_m^2.  literal=1: sigma_i =
 * max(sqrt(d^2+m^2), 2) exactly as printed in Eq. 3.  Eq. 4 uses the mean colour
 * and magnitude of in-window pixels. */
double orc_loglike_gauss(const uint32_t *hm, const orc_hess_stats *sm,
                         const uint32_t *hd, const orc_hess_stats *sd,
                         int64_t n_bins, int literal) {
    double Nd = 0.0, Nm = 0.0;
    for (int64_t i = 0; i < n_bins; ++i) { Nd += (double)hd[i]; Nm += (double)hm[i]; }
    if (!(Nm > 0.0) || !(Nd > 0.0)) return -INFINITY;
    double L = 0.0;
    for (int64_t i = 0; i < n_bins; ++i) {
        double d = (double)hd[i], m = (double)hm[i];
        double diff = d / Nd - m / Nm, var;
        if (literal) { double sg = fmax(sqrt(d * d + m * m), 2.0); var = sg * sg; }
        else {
            double ed = fmax(sqrt(d), 1.0) / Nd, em = fmax(sqrt(m), 1.0) / Nm;
            var = ed * ed + em * em;
        }
        L += -(diff * diff) / (2.0 * var);
    }
    double Cd = sd->sum_x / (double)sd->n_in, Cm = sm->sum_x / (double)sm->n_in;
    double Md = sd->sum_y / (double)sd->n_in, Mm = sm->sum_y / (double)sm->n_in;
    L += -((Cd - Cm) * (Cd - Cm)) / (2.0 * 0.05 * 0.05) - ((Md - Mm) * (Md - Mm)) / (2.0 * 0.05 * 0.05);
    return L;
}
