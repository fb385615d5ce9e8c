/*
 * pcmd.h -- C ABI of libpcmd.so: the pCMD Monte Carlo forward model, Hess diagram and
 * log-likelihood of Cook, Conroy, van Dokkum & Speagle (arXiv:1904.00011; PAPER.md), as
 * hand-written sm_100a CUDA kernels.  No torch types, no C++ types: plain pointers (each
 * marked HOST or DEVICE) and sizes.  Readings of the paper (R-C1..R-Q17) are in DESIGN.md.
 *
 * Conventions for every entry point
 *   - returns PCMD_OK (0) or a negative PCMD_E* code; never throws, never aborts;
 *   - work is ENQUEUED on `cuda_stream` (a cudaStream_t passed as void*, NULL = default
 *     stream) and outputs are valid once that stream reaches the call.  No host
 *     synchronisation happens, except inside pcmd_create/pcmd_destroy, when ctx scratch has to
 *     grow (first call at a larger n_models / larger star counts), in the *_host entry points
 *     (which return results to the host) and in pcmd_status / pcmd_debug_* (which read back);
 *   - the caller owns every d_* / h_* buffer; the ctx owns device copies of the isochrone
 *     table, PSFs, sampler tables and scratch;
 *   - one ctx per stream; a ctx is not thread-safe;
 *   - image layout: [model][band][y][x] float32, pixel index p = y*n_im + x.
 */
#ifndef PCMD_H
#define PCMD_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PCMD_OK       0
#define PCMD_EINVAL  -1   /* bad shape, NULL pointer, NaN / negative weight, sigma <= 0        */
#define PCMD_ERANGE  -2   /* an expected star count lambda_j exceeds 2^22 (R-C2)               */
#define PCMD_ENOMEM  -3   /* host or device allocation failed                                  */
#define PCMD_ECUDA   -4   /* a CUDA call failed; pcmd_last_cuda_error(ctx) gives the code      */
#define PCMD_ELIMIT  -5   /* the request exceeds the fixed scratch of a no-allocation entry point */

#define PCMD_MAX_BANDS 4
#define PCMD_MAX_HESS  4

#define PCMD_LIKE_POISSON        0  /* north_star / R-Q15                                       */
#define PCMD_LIKE_GAUSS          1  /* PAPER.md:218-233 Eq. 2-4, reading R-Q14                   */
#define PCMD_LIKE_GAUSS_LITERAL  2  /* Eq. 3 exactly as printed                                  */

typedef struct pcmd_ctx pcmd_ctx;   /* opaque */

/* One Hess diagram: x = mag[band_plus] - mag[band_minus], y = mag[band_y];
 * nx x ny half-open bins over [x_lo,x_hi) x [y_lo,y_hi) in apparent magnitudes (R-Q13). */
typedef struct {
    int32_t band_plus, band_minus, band_y;
    double  x_lo, x_hi, y_lo, y_hi;
    int32_t nx, ny;
} pcmd_hess_spec;

/* Per (model, hess): pixels inside the window, outside it, with a NaN magnitude; sums of x and
 * y over the inside pixels (used by Eq. 4). */
typedef struct {
    uint32_t n_in, n_out, n_bad, _pad;
    double   sum_x, sum_y;
} pcmd_hess_stats;

/* Hyper-parameters fixed for a fit (Table 2) and the isochrone table
 * (PAPER.md:69-71).  All pointers are HOST arrays, copied during pcmd_create. */
typedef struct {
    int32_t n_im, n_bands, n_age, n_feh, n_points;  /* N, B<=PCMD_MAX_BANDS, A, Z, J            */
    const int32_t *age_idx;     /* [J] age index a(j) of isochrone point j                       */
    const int32_t *feh_idx;     /* [J] [Fe/H] grid index z(j)                                    */
    const double  *imf_w;       /* [J] IMF weight, sum = 1 within each isochrone (R-Q2)          */
    const double  *absmag;      /* [J][B] absolute magnitudes                                    */
    const double  *feh_grid;    /* [Z]                                                           */
    const double  *zp;          /* [B] magnitude that gives 1 electron over the exposure         */
    const double  *dust_coef;   /* [B] A_b per unit of the dust parameter         */
    const float   *psf;         /* psf_separable=0: [B][K][K], centre (r,r), r=(K-1)/2, sum 1;
                                   psf_separable=1: [B][2][K] (row factor, column factor), the
                                   2-D PSF being column (x) row (R-Q10)                          */
    int32_t        psf_k;       /* K, odd, 1 <= K <= 63                                          */
    int32_t        psf_separable;
    const double  *sky;         /* [B] electrons                                  */
    const double  *read_sigma;  /* [B] electrons (R-Q11)                                         */
    int32_t        shot_noise;  /* 0/1                                             */
    int32_t        poisson_sky; /* 0/1 (R-Q11)                                                   */
    double         like_floor;  /* m_floor of the Poisson lnL (R-Q15), e.g. 0.1                  */
    int32_t        n_hess;      /* <= PCMD_MAX_HESS                                              */
    const pcmd_hess_spec *hess; /* [n_hess]                                                      */
    double         dust_frac;   /* F_dust                                         */
    int32_t        dust_mode;   /* 0 none, 1 star fraction, 2 pixel mixture (R-Q7)               */
    double         mdf_cut;     /* 0.01                                           */
    int32_t        psf_grid;    /* G: 0 or 1: one PSF per band.  2..8: sub-pixel PSF grid (PAPER.md:180,
                                   R-Q19): psf is [B][G*G][K][K] (psf_separable must be 0), the image is
                                   divided into G x G cells of ceil(N/G) pixels and an output pixel is
                                   convolved with the PSF of its cell (index gy*G + gx)              */
    int32_t        sampler_mode;/* 0: one Poisson draw per (pixel, isochrone point) (R-C1/R-C2);
                                   1: aggregated sampler (PAPER.md:75 footnote 3, DESIGN.md R-A1): the pixel's
                                   number of stars is one Poisson(N_pix) draw and every star is placed on a
                                   point with probability lambda_j / N_pix -- O(N_pix) instead of O(J) random
                                   numbers per pixel, a different random stream (R-C1 stream 4)        */
} pcmd_config;

/* One model = the paper's free parameters (Table 1). */
typedef struct {
    const double *sfh;          /* HOST [A] stars per pixel per age, linear; N_pix = sum (R-Q5)  */
    double feh_mean, feh_sigma; /* M2/M3 Gaussian MDF; sigma > 0              */
    double dmod;                /* D2 distance modulus                        */
    double dust_med, dust_sigma;/* E1-E3: median and ln-width of the log-normal (R-Q8)           */
} pcmd_params;

int  pcmd_create(pcmd_ctx **out, const pcmd_config *cfg);
void pcmd_destroy(pcmd_ctx *ctx);

/* Stages 1-5: isochrone weighting, Poisson star counts summed into pixel
 * fluxes, dust, PSF convolution, noise and magnitudes, for n_models parameter vectors.
 *   params        HOST [n_models]; read during the call
 *   seed          Philox key (R-C1); model i uses counter word model_index0 + i
 *   d_mag         DEVICE out [n_models][B][N][N] float32 apparent magnitudes (NaN: flux <= 0)
 *   d_flux_raw    DEVICE out, same shape, stage-2 flux in electrons; may be NULL
 *   d_count_hash  DEVICE out [n_models][P] uint64, sum_j n_pj*(splitmix64(j)|1) mod 2^64;
 *   d_count_total DEVICE out [n_models][P] uint32, sum_j n_pj.  Both NULL (production) or both
 *                 non-NULL (parity build of the same kernel, which also tracks integer counts).
 * With cfg.sampler_mode = 1 the star counts come from the aggregated sampler (R-A1); every output keeps
 * its meaning.  Errors: PCMD_EINVAL (NULL / non-finite / negative parameters, sigma <= 0), PCMD_ERANGE (an
 * expected count above 2^22; raised on the host when it can be seen there, else by the device: pcmd_status),
 * PCMD_ENOMEM, PCMD_ECUDA. */
int  pcmd_simulate(pcmd_ctx *ctx, const pcmd_params *params, int32_t n_models,
                   uint64_t seed, uint32_t model_index0,
                   float *d_mag, float *d_flux_raw,
                   uint64_t *d_count_hash, uint32_t *d_count_total, void *cuda_stream);

/* Repeated realisations of ONE parameter vector (Appendix A: "we recompute the
 * likelihood of the best fit model 100 times"; the likelihood is stochastic):
 * identical to pcmd_simulate with n_repeats copies of params[0] -- realisation r uses counter word
 * model_index0 + r -- but stage 1 runs once.  Outputs are [n_repeats][...] like pcmd_simulate's. */
int  pcmd_simulate_repeat(pcmd_ctx *ctx, const pcmd_params *params, int32_t n_repeats,
                          uint64_t seed, uint32_t model_index0,
                          float *d_mag, float *d_flux_raw,
                          uint64_t *d_count_hash, uint32_t *d_count_total, void *cuda_stream);

/* Stage 6: Hess diagrams of d_mag.
 *   d_hess   DEVICE out [n_models][hess_bins_total] uint32, the n_hess diagrams of a model one
 *            after another, each [ny][nx]; overwritten
 *   d_stats  DEVICE out [n_models][n_hess]; may be NULL */
int  pcmd_hess(pcmd_ctx *ctx, const float *d_mag, int32_t n_models,
               uint32_t *d_hess, pcmd_hess_stats *d_stats, void *cuda_stream);

/* Stage 6 for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same kernels, launch geometry, arguments and results as
 * pcmd_hess (bit-identical diagrams and statistics), but the per-block partial statistics go to a
 * fixed array in the library's device image instead of the ctx's grow-on-demand scratch.  The call
 * makes no cudaMalloc / cudaFree / allocating library call.
 *   limit   n_models * n_hess * (blocks per diagram) <= PCMD_HESS_NOALLOC_MAX_PARTS (32 bytes each:
 *           256 KB that every GPU which loads the library holds until exit); a larger request returns
 *           PCMD_ELIMIT and launches nothing.  pcmd_hess_noalloc_parts(ctx, n_models) returns the
 *           number a call would need (blocks per diagram = 1 once n_models * n_hess >= 8 * SMs).
 *   sharing the array is ONE per device and process, shared by every ctx and every call; it keeps the
 *           last call's contents (nothing in it has to start at zero: every slot a call reads it has
 *           written first).  Two calls that overlap on the GPU (different streams, or graphs replayed
 *           concurrently) race on it: serialise them.
 *   set-up  the array's device address is looked up once per device on the first call, or by
 *           pcmd_hess_noalloc_setup() (no arguments: the CURRENT device) -- call that before starting
 *           a graph capture.  Returns PCMD_OK or PCMD_ECUDA. */
#define PCMD_HESS_NOALLOC_MAX_PARTS 8192
int     pcmd_hess_noalloc_setup(void);
int64_t pcmd_hess_noalloc_parts(const pcmd_ctx *ctx, int32_t n_models);
int     pcmd_hess_noalloc(pcmd_ctx *ctx, const float *d_mag, int32_t n_models,
                          uint32_t *d_hess, pcmd_hess_stats *d_stats, void *cuda_stream);

/* Stage 7: log-likelihood of the data Hess given each model Hess, summed over the n_hess
 * diagrams.  like_mode: PCMD_LIKE_*.  d_stats / d_data_stats are needed by the GAUSS modes
 * only (may be NULL for POISSON).  d_hess_data: DEVICE [hess_bins_total], one fixed data set.
 *   d_loglike DEVICE out [n_models] float64 */
int  pcmd_loglike(pcmd_ctx *ctx, const uint32_t *d_hess_model, const pcmd_hess_stats *d_stats,
                  int32_t n_models, const uint32_t *d_hess_data,
                  const pcmd_hess_stats *d_data_stats, int32_t like_mode,
                  double *d_loglike, void *cuda_stream);

/* The whole path with HOST buffers: params -> simulate -> hess -> loglike, the data Hess copied
 * host->device and the model Hess / lnL copied device->host inside the call (it synchronises
 * the stream before returning).  h_hess_out / h_stats_out may be NULL. */
int  pcmd_evaluate_host(pcmd_ctx *ctx, const pcmd_params *params, int32_t n_models,
                        uint64_t seed, uint32_t model_index0,
                        const uint32_t *h_hess_data, const pcmd_hess_stats *h_data_stats,
                        int32_t like_mode, double *h_loglike, uint32_t *h_hess_out,
                        pcmd_hess_stats *h_stats_out, void *cuda_stream);

/* Number of uint32 bins of one model's Hess block (sum of nx*ny over the n_hess specs). */
int64_t pcmd_hess_bins_total(const pcmd_ctx *ctx);

/* Stage-1 parity taps for model `model` of the LAST pcmd_simulate call (synchronises).
 * Any pointer may be NULL.  h_lambda[J] float64; h_flux[J][B] float32; h_k0[J], h_len[J]:
 * first count and number of stored thresholds of each sampler table (R-C2); h_tables:
 * concatenated stored thresholds T (values 1..2^32-1) in point order, at most cap entries;
 * *n_tables receives the total number. */
int  pcmd_debug_weights(pcmd_ctx *ctx, int32_t model, double *h_lambda, float *h_flux,
                        uint32_t *h_k0, uint32_t *h_len, uint32_t *h_tables, int64_t cap,
                        int64_t *n_tables);
/* Optional DEVICE outputs of stages 3 and 4 for the following pcmd_simulate calls
 * ([n_models][B][N][N] float32 each; NULL switches a tap off). */
int  pcmd_debug_taps(pcmd_ctx *ctx, float *d_flux_dust, float *d_flux_conv);

/* Raw Philox4x32-10 words (R-C1) for n counters, computed on the device with the same
 * routine the kernels use: h_ctr HOST [n][4], h_out HOST [n][4] (synchronises). */
int  pcmd_debug_philox(uint64_t seed, const uint32_t *h_ctr, int64_t n, uint32_t *h_out);

/* Device-side status of the last calls on this ctx (synchronises the stream): PCMD_OK, or
 * PCMD_ERANGE / PCMD_ENOMEM raised by a kernel (lambda too large, sampler-table scratch full). */
int  pcmd_status(pcmd_ctx *ctx, void *cuda_stream);
int  pcmd_last_cuda_error(const pcmd_ctx *ctx);
/* Per-stage device timing.  pcmd_profile(ctx, 1) makes the following pcmd_simulate / pcmd_hess /
 * pcmd_loglike calls record CUDA events on the caller's stream around each stage;
 * pcmd_stage_ms waits for the events of the LAST such calls and writes h_ms[5] HOST float32
 * milliseconds: stage 1 (weights + sampler tables), stage 2 (+ dust epilogue), stages 4-5
 * (convolution + noise + magnitudes), stage 6, stage 7; -1 for a stage not run since enabling. */
int  pcmd_profile(pcmd_ctx *ctx, int32_t enable);
int  pcmd_stage_ms(pcmd_ctx *ctx, float *h_ms);
/* Kernels launched on behalf of this ctx since pcmd_create (bench.py's gpu_launches). */
int64_t pcmd_launch_count(const pcmd_ctx *ctx);
const char *pcmd_strerror(int code);

/* HOST-only convenience: the paper's free parameters (Table 1) -> the linear fields of
 * pcmd_params.  log10_sfh[n_age]: log10 of the stars per pixel formed in each age bin (model S5; the
 * parametric models S1-S4 are spread over the age grid by the caller, paper_1904_00011_b200/sfh.py);
 * feh, sigma_feh: mean and width of the Gaussian MDF (M2/M3); log10_ebv: log10 of the median extinction
 * parameter, sigma_dust its dimensionless log-normal width (E1-E3; E1 = width 0); dmod: distance modulus
 * (D1/D2).  Writes sfh_out[n_age] (caller's storage, which out->sfh then points to) with libm pow.  Both
 * the library and any reference implementation consume this OUTPUT, so no transcendental sits between
 * the caller's numbers and the expected star counts.  Returns PCMD_EINVAL on NULL / non-finite input. */
int  pcmd_params_from_paper(int32_t n_age, const double *log10_sfh, double feh, double sigma_feh,
                            double log10_ebv, double sigma_dust, double dmod, double *sfh_out,
                            pcmd_params *out);

/* Instruction-pipe micro-benchmarks on the current device (measurement support for the stage-2
 * roofline of DESIGN.md "Rooflines"; nothing of the method runs here).  Test `test` (0 <=
 * test < n, pcmd_pipe_bench_name(test) != NULL) runs `iters` iterations of an unrolled stream of
 * one instruction kind in ctas_per_sm x SMs CTAs of `threads` threads and writes h_out[4] HOST
 * float64: [0] warp-instructions (Philox test: warp-calls) per clock per scheduler, from the
 * slowest CTA's clock64 span; [1] that span in SM clocks; [2] kernel milliseconds (CUDA events);
 * [3] thread-steps (Philox test: calls) per second over the whole GPU.  Synchronises. */
int  pcmd_pipe_bench(int32_t test, int32_t ctas_per_sm, int32_t threads, int32_t iters, double *h_out);
const char *pcmd_pipe_bench_name(int32_t test);

#ifdef __cplusplus
}
#endif
#endif
