/*
 * pcmd_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle of the pCMD Monte Carlo forward model of
 * Cook, Conroy, van Dokkum & Speagle (arXiv:1904.00011; PAPER.md), stages 1-7
 * of SURVEY.md section 8(a).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library.
 * It shares no code, header, table or constant generator with the CUDA path
 * under paper_1904_00011_b200/ (that path has its own include/pcmd.h).
 *
 * Every function cites the passage it follows.  Where the paper is silent the
 * reading is the one listed in DESIGN.md ("Readings of the paper").
 *
 * Parity pins: tests/test_oracle_*.py (-m "not gpu").  End-to-end absolute
 * values are "parity unpinned" (the paper prints no worked numerical example);
 * every stage is pinned separately, see DESIGN.md section "Oracle pins".
 */
#ifndef PCMD_ORACLE_H
#define PCMD_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Hyper-parameters fixed for a fit (Table 2) plus the
 * isochrone table.  All arrays are caller-owned host memory. */
typedef struct {
    int32_t n_im, n_bands, n_age, n_feh, n_points;   /* N, B, A, Z, J */
    const int32_t *age_idx;      /* [J] age index a(j) of isochrone point j      */
    const int32_t *feh_idx;      /* [J] [Fe/H] grid index z(j)                   */
    const double  *imf_w;        /* [J] IMF weight, sum = 1 within each isochrone */
    const double  *absmag;       /* [J][B] absolute magnitudes                   */
    const double  *feh_grid;     /* [Z]                                          */
    const double  *zp;           /* [B] magnitude giving 1 electron              */
    const double  *dust_coef;    /* [B] A_b per unit of the dust parameter       */
    const double  *psf;          /* [B][K][K], centre at (r,r), r=(K-1)/2        */
    int32_t        psf_k;
    const double  *sky;          /* [B] electrons                                */
    const double  *read_sigma;   /* [B] electrons                                */
    int32_t        shot_noise;   /* 0/1                                          */
    int32_t        poisson_sky;  /* 0/1                                          */
    double         dust_frac;    /* F_dust                        */
    int32_t        dust_mode;    /* 0 none, 1 star fraction, 2 pixel mixture     */
    double         mdf_cut;      /* 0.01                          */
    int32_t        psf_grid;     /* G: 0/1 one PSF per band; G > 1: psf is [B][G*G][K][K], the image is
                                    divided into a G x G grid of cells and an output pixel uses the PSF
                                    of its cell (DESIGN.md R-Q19)  */
} orc_config;

/* One model = the paper's free parameters (Table 1). */
typedef struct {
    const double *sfh;           /* [A] stars per pixel per age (linear)         */
    double feh_mean, feh_sigma;  /* M2/M3                     */
    double dmod;                 /* D2                        */
    double dust_med, dust_sigma; /* E1-E3                     */
} orc_params;

typedef struct {
    int32_t band_plus, band_minus, band_y;  /* x = mag[plus]-mag[minus], y = mag[y] */
    double  x_lo, x_hi, y_lo, y_hi;
    int32_t nx, ny;
} orc_hess_spec;

typedef struct {
    uint32_t n_in, n_out, n_bad;
    double   sum_x, sum_y;       /* over in-window pixels */
} orc_hess_stats;

/* ---- random stream (DESIGN.md R-C1) ------------------------------------ */
void     orc_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]);
uint64_t orc_splitmix64(uint64_t j);

/* ---- Poisson sampler (DESIGN.md R-C2) ---------------------------------- */
/* Builds T[k], k = k_lo..k_hi (as uint64, T[k_hi] == 2^32) into T_out[0..k_hi-k_lo].
 * Returns the number of entries written, or -(needed) if cap is too small,
 * or -1 if lambda is negative, NaN or > 2^22.  lambda == 0: 1 entry, k_lo=k_hi=0. */
int64_t  orc_poisson_table(double lambda, uint64_t *T_out, int64_t cap, int64_t *k_lo, int64_t *k_hi);
/* n = min{k >= 0 : u < T[k]}, linear scan (the definition). */
uint32_t orc_poisson_draw_linear(const uint64_t *T, int64_t k_lo, int64_t k_hi, uint32_t u);
/* same n by bisection (used inside stage 2 for speed; pinned equal to linear). */
uint32_t orc_poisson_draw(const uint64_t *T, int64_t k_lo, int64_t k_hi, uint32_t u);

/* ---- stage 1 (DESIGN.md R-C3) ------------------- */
double orc_expneg(double t);
/* mdfw[Z], lambda[J], flux[J][B] (fp64 electrons per star).  Returns 0 / -1. */
int orc_stage1(const orc_config *c, const orc_params *p, double *mdfw, double *lambda, double *flux);

/* ---- stage 2 ---------------------------------------- */
/* Pixels pix[0..n_pix) (NULL: 0..n_pix-1).  F_raw[b*n_pix + i], total[i], hash[i];
 * counts (optional) [i*J + j]. */
int orc_stage2(const orc_config *c, const double *lambda, const double *flux,
               uint64_t seed, uint32_t model, const uint32_t *pix, int64_t n_pix,
               double *F_raw, uint32_t *total, uint64_t *hash, uint32_t *counts);
/* Aggregated sampler (PAPER.md:75 footnote 3; DESIGN.md R-A1): one Poisson draw of the pixel's number of
 * stars (mean sum_j lambda_j), then each star placed on a point with probability lambda_j / sum, by
 * inversion of an integer cumulative table.  Same outputs as orc_stage2; weights_out (optional) [J]. */
int orc_stage2_agg(const orc_config *c, const double *lambda, const double *flux,
                   uint64_t seed, uint32_t model, const uint32_t *pix, int64_t n_pix,
                   double *F_raw, uint32_t *total, uint64_t *hash, uint32_t *counts, uint64_t *weights_out);
/* Brute force: materialises every star of every pixel one at a time (a list of
 * (pixel, point) records built from the same draws), then sums star by star. */
int orc_stage2_brute(const orc_config *c, const double *lambda, const double *flux,
                     uint64_t seed, uint32_t model, double *F_raw, uint32_t *total);

/* ---- stage 3 dust --------------------------------- */
int orc_stage3(const orc_config *c, const orc_params *p, uint64_t seed, uint32_t model,
               const double *F_raw, double *A_pix, double *F_dust);
/* ---- stage 4 PSF, circular boundary ------------------- */
int orc_stage4(const orc_config *c, const double *F_in, double *G);
/* ---- stage 5 noise + magnitudes ---------------- */
int orc_stage5(const orc_config *c, uint64_t seed, uint32_t model, const double *G, double *mag);
/* one standard normal from two Philox words (Box-Muller, DESIGN.md R-C4) */
double orc_normal(uint32_t w0, uint32_t w1);

/* ---- stage 6 Hess ---------------------------------- */
/* fp64 binning of fp64 magnitudes; n_edge = pixels within edge_tol mag of a bin edge
 * (either axis); edge_list (optional, cap entries) receives their pixel indices. */
int orc_hess(const orc_hess_spec *h, int64_t n_pix, int32_t n_bands, const double *mag,
             uint32_t *hess, orc_hess_stats *st, double edge_tol,
             uint32_t *n_edge, uint32_t *edge_list, int64_t edge_cap);
/* The same decision taken in the kernel's precision (fp32 mags, fp32 arithmetic in the
 * order DESIGN.md "Hess binning arithmetic" states).  Bit-exact target for the GPU Hess. */
int orc_hess_f32(const orc_hess_spec *h, int64_t n_pix, int32_t n_bands, const float *mag,
                 uint32_t *hess, orc_hess_stats *st);

/* Per-pixel bin index of orc_hess / orc_hess_f32 (-1 outside the window, -2 NaN) and, for the fp64
 * form, near[i]: bit 0 = x within tol_x of a bin edge, bit 1 = y within tol_y (NULL: not wanted). */
int orc_hess_pixels(const orc_hess_spec *h, int64_t n_pix, int32_t n_bands, const double *mag,
                    double tol_x, double tol_y, int32_t *bin, uint8_t *near);
int orc_hess_pixels_f32(const orc_hess_spec *h, int64_t n_pix, int32_t n_bands, const float *mag, int32_t *bin);

/* ---- stage 7 log-likelihood ---------------------------------------------- */
/* Poisson lnL (north_star; DESIGN.md R-Q15). */
double orc_loglike_poisson(const uint32_t *hess_model, const uint32_t *hess_data, int64_t n_bins,
                           double m_floor);
/* Eq. 2-4 Gaussian lnL (DESIGN.md R-Q14).  literal=1: Eq. 3 as printed. */
double orc_loglike_gauss(const uint32_t *hess_model, const orc_hess_stats *sm,
                         const uint32_t *hess_data, const orc_hess_stats *sd,
                         int64_t n_bins, int literal);

int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
