// api.cu -- the C ABI of include/pcmd.h: argument checks, ctx ownership, launch sequencing.
// No arithmetic of the method runs on the host: the host only validates, sizes scratch and
// enqueues kernels.
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include "pcmd_internal.cuh"

static uint64_t splitmix64_host(uint64_t j) {  // R-C4 checksum multiplier (debug counts only)
    uint64_t z = j + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

template <typename T>
static int upload(pcmd_ctx *c, T **dst, const T *src, size_t n) {
    PCMD_CUDA(c, cudaMalloc((void **)dst, (n ? n : 1) * sizeof(T)));
    if (n) PCMD_CUDA(c, cudaMemcpy(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice));
    return PCMD_OK;
}

int pcmd_pdl_enabled() {
    static int on = -1;
    if (on < 0) { const char *e = getenv("PCMD_NO_PDL"); on = (e && e[0] == '1') ? 0 : 1; }
    return on;
}

extern "C" const char *pcmd_strerror(int code) {
    switch (code) {
        case PCMD_OK: return "ok";
        case PCMD_EINVAL: return "invalid argument";
        case PCMD_ERANGE: return "expected star count of an isochrone point exceeds 2^22";
        case PCMD_ENOMEM: return "out of memory";
        case PCMD_ECUDA: return "CUDA error";
        case PCMD_ELIMIT: return "request exceeds the fixed scratch of a no-allocation entry point";
        default: return "unknown error";
    }
}

static void free_scratch(pcmd_ctx *c) {
    cudaFree(c->d_sfh); cudaFree(c->d_model); cudaFree(c->d_mdfw); cudaFree(c->d_lambda);
    cudaFree(c->d_q);
    cudaFree(c->d_tab); cudaFree(c->d_rec); cudaFree(c->d_grp); cudaFree(c->d_plan);
    cudaFree(c->d_gcls); cudaFree(c->d_arena); cudaFree(c->d_gpos); cudaFree(c->d_alloc); c->d_alloc = nullptr;
    c->d_grp = nullptr; c->d_plan = nullptr; c->d_gcls = nullptr; c->d_arena = nullptr; c->d_gpos = nullptr;
    cudaFree(c->d_agg_lam); cudaFree(c->d_agg_C); cudaFree(c->d_agg_G); cudaFree(c->d_agg_rawcnt); cudaFree(c->d_agg_klo);
    cudaFree(c->d_agg_stcnt); cudaFree(c->d_agg_tab); cudaFree(c->d_agg_q); cudaFree(c->d_agg_rec);
    c->d_agg_lam = nullptr; c->d_agg_C = nullptr; c->d_agg_G = nullptr; c->d_agg_rawcnt = nullptr; c->d_agg_klo = nullptr;
    c->d_agg_stcnt = nullptr; c->d_agg_tab = nullptr; c->d_agg_q = nullptr; c->d_agg_rec = nullptr;
    c->agg_tcap = 0; c->agg_models = 0;
    if (c->h_stage) cudaFreeHost(c->h_stage);
    c->d_sfh = nullptr; c->d_model = nullptr; c->d_mdfw = nullptr; c->d_lambda = nullptr;
    c->d_q = nullptr;
    c->d_tab = nullptr; c->d_rec = nullptr; c->h_stage = nullptr;
    c->cap_models = 0; c->cap_raw = 0;
}

// Scratch for n_models models whose sampler tables need at most cap_raw raw entries each.
static int ensure_scratch(pcmd_ctx *c, int n_models, int64_t cap_raw, int64_t agg_tcap) {
    if (n_models <= c->cap_models && cap_raw <= c->cap_raw && (c->sampler_mode != 1 || agg_tcap <= c->agg_tcap)) return PCMD_OK;
    if (agg_tcap < c->agg_tcap) agg_tcap = c->agg_tcap;
    const int nm = n_models > c->cap_models ? n_models : c->cap_models;
    const int64_t cr = cap_raw > c->cap_raw ? cap_raw : c->cap_raw;
    cudaDeviceSynchronize();
    free_scratch(c);
    const size_t J = c->J, Jp = c->Jpad;
    PCMD_CUDA(c, cudaMalloc(&c->d_sfh, (size_t)nm * c->A * sizeof(double)));
    PCMD_CUDA(c, cudaMalloc(&c->d_model, (size_t)nm * sizeof(DevModel)));
    PCMD_CUDA(c, cudaMalloc(&c->d_mdfw, (size_t)nm * c->Z * sizeof(double)));
    PCMD_CUDA(c, cudaMalloc(&c->d_lambda, (size_t)nm * J * sizeof(double)));
    PCMD_CUDA(c, cudaMalloc(&c->d_alloc, (size_t)nm * 2 * sizeof(uint32_t)));
    PCMD_CUDA(c, cudaMalloc(&c->d_q, (size_t)nm * cr * sizeof(double)));
    PCMD_CUDA(c, cudaMalloc(&c->d_tab, (size_t)nm * cr * sizeof(uint32_t)));
    PCMD_CUDA(c, cudaMalloc(&c->d_rec, (size_t)nm * Jp * sizeof(PointRec)));
    PCMD_CUDA(c, cudaMalloc(&c->d_grp, (size_t)nm * (Jp / 4) * sizeof(GroupRec)));
    PCMD_CUDA(c, cudaMalloc(&c->d_plan, (size_t)nm * sizeof(ModelPlan)));
    PCMD_CUDA(c, cudaMalloc(&c->d_gcls, (size_t)nm * (Jp / 4)));
    PCMD_CUDA(c, cudaMalloc(&c->d_gpos, (size_t)nm * (Jp / 4) * sizeof(uint32_t)));
    {   // padded search tables: room for every group in D9 (8 KB), capped at 1 GiB over all models
        int64_t words = (int64_t)(Jp / 4) * 2048, lim = ((int64_t)1 << 28) / nm;
        lim &= ~(int64_t)31;          // every model's arena starts 128-byte aligned (bulk copies need 16 B)
        if (words > lim) words = lim;
        if (words < (int64_t)(Jp / 4) * 128) words = (int64_t)(Jp / 4) * 128;   // D5 always fits
        c->arena_cap = words;
        PCMD_CUDA(c, cudaMalloc(&c->d_arena, (size_t)nm * words * sizeof(uint32_t)));
    }
    if (c->sampler_mode == 1) {
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_lam, (size_t)nm * sizeof(double)));
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_C, (size_t)nm * (J + 1) * sizeof(uint64_t)));
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_G, (size_t)nm * 4098 * sizeof(uint32_t)));
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_rawcnt, (size_t)nm * 2 * sizeof(uint32_t)));
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_stcnt, (size_t)nm * 2 * sizeof(uint32_t)));
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_klo, (size_t)nm * sizeof(uint32_t)));
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_q, (size_t)nm * agg_tcap * sizeof(double)));
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_tab, (size_t)nm * agg_tcap * sizeof(uint32_t)));
        PCMD_CUDA(c, cudaMalloc(&c->d_agg_rec, (size_t)nm * sizeof(PointRec)));
        PCMD_CUDA(c, cudaMemset(c->d_agg_rec, 0, (size_t)nm * sizeof(PointRec)));
        c->agg_tcap = agg_tcap; c->agg_models = nm;
    }
    c->h_stage_bytes = (size_t)nm * (c->A * sizeof(double) + sizeof(DevModel));
    PCMD_CUDA(c, cudaMallocHost(&c->h_stage, 2 * c->h_stage_bytes));
    c->cap_models = nm; c->cap_raw = cr;
    return PCMD_OK;
}

extern "C" int pcmd_create(pcmd_ctx **out, const pcmd_config *cfg) {
    if (!out || !cfg) return PCMD_EINVAL;
    *out = nullptr;
    if (cfg->n_im < 1 || cfg->n_im > 32768 || cfg->n_bands < 1 || cfg->n_bands > PCMD_MAX_BANDS ||
        cfg->n_age < 1 || cfg->n_feh < 1 || cfg->n_points < 1 || cfg->psf_k < 1 || cfg->psf_k > 63 ||
        (cfg->psf_k & 1) == 0 || cfg->n_hess < 0 || cfg->n_hess > PCMD_MAX_HESS ||
        cfg->dust_mode < 0 || cfg->dust_mode > 2 || cfg->psf_grid < 0 || cfg->psf_grid > 8 ||
        cfg->sampler_mode < 0 || cfg->sampler_mode > 1 ||
        (cfg->psf_grid > 1 && cfg->psf_separable))
        return PCMD_EINVAL;
    if (!cfg->age_idx || !cfg->feh_idx || !cfg->imf_w || !cfg->absmag || !cfg->feh_grid || !cfg->zp ||
        !cfg->dust_coef || !cfg->psf || !cfg->sky || !cfg->read_sigma || (cfg->n_hess && !cfg->hess))
        return PCMD_EINVAL;
    if (!(cfg->dust_frac >= 0.0 && cfg->dust_frac <= 1.0) || !(cfg->mdf_cut >= 0.0 && cfg->mdf_cut < 1.0) ||
        !(cfg->like_floor > 0.0))
        return PCMD_EINVAL;
    const int J = cfg->n_points, B = cfg->n_bands, K = cfg->psf_k;
    for (int j = 0; j < J; ++j) {
        if (cfg->age_idx[j] < 0 || cfg->age_idx[j] >= cfg->n_age || cfg->feh_idx[j] < 0 ||
            cfg->feh_idx[j] >= cfg->n_feh || !(cfg->imf_w[j] >= 0.0) || !isfinite(cfg->imf_w[j]))
            return PCMD_EINVAL;
        for (int b = 0; b < B; ++b) if (!isfinite(cfg->absmag[(size_t)j * B + b])) return PCMD_EINVAL;
    }
    for (int b = 0; b < B; ++b)
        if (!isfinite(cfg->zp[b]) || !(cfg->sky[b] >= 0.0) || cfg->sky[b] > PCMD_LAMBDA_MAX ||
            !(cfg->read_sigma[b] >= 0.0) || !isfinite(cfg->dust_coef[b]))
            return PCMD_EINVAL;
    int64_t bins = 0;
    for (int h = 0; h < cfg->n_hess; ++h) {
        const pcmd_hess_spec &s = cfg->hess[h];
        if (s.band_plus < 0 || s.band_plus >= B || s.band_minus < 0 || s.band_minus >= B || s.band_y < 0 ||
            s.band_y >= B || s.nx < 1 || s.ny < 1 || s.nx > 4096 || s.ny > 4096 || !(s.x_hi > s.x_lo) ||
            !(s.y_hi > s.y_lo))
            return PCMD_EINVAL;
        bins += (int64_t)s.nx * s.ny;
    }
    pcmd_ctx *c = new (std::nothrow) pcmd_ctx;
    if (!c) return PCMD_ENOMEM;
    memset(c, 0, sizeof(*c));
    c->N = cfg->n_im; c->B = B; c->A = cfg->n_age; c->Z = cfg->n_feh; c->J = J; c->Jpad = (J + 3) & ~3;
    c->sampler_mode = cfg->sampler_mode;
    c->K = K; c->psf_sep = cfg->psf_separable; c->shot_noise = cfg->shot_noise != 0;
    c->poisson_sky = cfg->poisson_sky != 0; c->n_hess = cfg->n_hess; c->dust_mode = cfg->dust_mode;
    c->P = (int64_t)cfg->n_im * cfg->n_im; c->hess_bins = bins;
    c->like_floor = cfg->like_floor; c->dust_frac = cfg->dust_frac; c->mdf_cut = cfg->mdf_cut;
    for (int b = 0; b < B; ++b) {
        c->zp[b] = cfg->zp[b]; c->dust_coef[b] = cfg->dust_coef[b]; c->sky[b] = cfg->sky[b];
        c->read_sigma[b] = cfg->read_sigma[b];
    }
    for (int h = 0; h < cfg->n_hess; ++h) c->hess[h] = cfg->hess[h];
    int dev = 0, rc = PCMD_OK;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
    c->h_imf_w = (double *)malloc((size_t)J * sizeof(double));
    if (!c->h_imf_w) { delete c; return PCMD_ENOMEM; }
    memcpy(c->h_imf_w, cfg->imf_w, (size_t)J * sizeof(double));
    for (int j = 0; j < J; ++j) {
        c->imf_sqrt_sum += sqrt(cfg->imf_w[j]);
        if (cfg->imf_w[j] > c->imf_w_max) c->imf_w_max = cfg->imf_w[j];
    }
#define TRY(x) do { rc = (x); if (rc) { pcmd_destroy(c); return rc; } } while (0)
    TRY(upload(c, &c->d_age_idx, cfg->age_idx, (size_t)J));
    TRY(upload(c, &c->d_feh_idx, cfg->feh_idx, (size_t)J));
    TRY(upload(c, &c->d_imf_w, cfg->imf_w, (size_t)J));
    TRY(upload(c, &c->d_absmag, cfg->absmag, (size_t)J * B));
    TRY(upload(c, &c->d_feh_grid, cfg->feh_grid, (size_t)cfg->n_feh));
    {   // PSF: kept as [B][G*G][K][K]; a separable PSF is expanded (column factor (x) row factor)
        const int G2 = cfg->psf_grid > 1 ? cfg->psf_grid * cfg->psf_grid : 1;
        c->psf_grid = cfg->psf_grid > 1 ? cfg->psf_grid : 1;
        float *p2 = (float *)malloc((size_t)B * G2 * K * K * sizeof(float));
        if (!p2) { pcmd_destroy(c); return PCMD_ENOMEM; }
        if (G2 > 1) memcpy(p2, cfg->psf, (size_t)B * G2 * K * K * sizeof(float));
        else
            for (int b = 0; b < B; ++b)
                for (int y = 0; y < K; ++y)
                    for (int x = 0; x < K; ++x)
                        p2[((size_t)b * K + y) * K + x] = cfg->psf_separable
                            ? (float)((double)cfg->psf[((size_t)b * 2 + 1) * K + y] * (double)cfg->psf[((size_t)b * 2) * K + x])
                            : cfg->psf[((size_t)b * K + y) * K + x];
        rc = upload(c, &c->d_psf, p2, (size_t)B * G2 * K * K);
        free(p2);
        if (rc) { pcmd_destroy(c); return rc; }
        if (cfg->psf_separable) {
            TRY(upload(c, &c->d_psf_sep, cfg->psf, (size_t)B * 2 * K));
            c->h_psf_sep = (float *)malloc((size_t)B * 2 * K * sizeof(float));
            if (!c->h_psf_sep) { pcmd_destroy(c); return PCMD_ENOMEM; }
            memcpy(c->h_psf_sep, cfg->psf, (size_t)B * 2 * K * sizeof(float));
        }
    }
    {
        uint64_t *mult = (uint64_t *)malloc((size_t)c->Jpad * sizeof(uint64_t));
        if (!mult) { pcmd_destroy(c); return PCMD_ENOMEM; }
        for (int j = 0; j < c->Jpad; ++j) mult[j] = splitmix64_host((uint64_t)j) | 1ull;
        rc = upload(c, &c->d_mult, mult, (size_t)c->Jpad);
        free(mult);
        if (rc) { pcmd_destroy(c); return rc; }
    }
    {
        DevHess dh[PCMD_MAX_HESS];
        int64_t off = 0;
        for (int h = 0; h < cfg->n_hess; ++h) {
            const pcmd_hess_spec &s = cfg->hess[h];
            dh[h].band_plus = s.band_plus; dh[h].band_minus = s.band_minus; dh[h].band_y = s.band_y;
            dh[h].nx = s.nx; dh[h].ny = s.ny; dh[h].x_lo = (float)s.x_lo; dh[h].y_lo = (float)s.y_lo;
            dh[h].inv_dx = (float)((double)s.nx / (s.x_hi - s.x_lo));
            dh[h].inv_dy = (float)((double)s.ny / (s.y_hi - s.y_lo));
            dh[h].bin_off = off; off += (int64_t)s.nx * s.ny;
        }
        TRY(upload(c, &c->d_hess_spec, dh, (size_t)cfg->n_hess));
    }
    {
        cudaError_t e = cudaMalloc(&c->d_status, 2 * sizeof(int32_t));   // [status, stage-2 unit counter]
        if (e == cudaSuccess) e = cudaMemset(c->d_status, 0, 2 * sizeof(int32_t));
        if (e != cudaSuccess) { c->last_cuda = (int)e; pcmd_destroy(c); return PCMD_ECUDA; }
    }
    TRY(pcmd_build_sky_tables(c));
    TRY(pcmd_build_lfact(c));
    TRY(pcmd_stage2_occupancy(c));
    TRY(pcmd_conv_setup(c));
#undef TRY
    cudaDeviceSynchronize();
    *out = c;
    return PCMD_OK;
}

extern "C" void pcmd_destroy(pcmd_ctx *c) {
    if (!c) return;
    cudaDeviceSynchronize();
    free_scratch(c);
    cudaFree(c->d_age_idx); cudaFree(c->d_feh_idx); cudaFree(c->d_imf_w); cudaFree(c->d_absmag);
    cudaFree(c->d_feh_grid); cudaFree(c->d_psf); cudaFree(c->d_psf_sep); cudaFree(c->d_mult); cudaFree(c->d_lfact); cudaFree(c->d_hess_spec);
    cudaFree(c->d_sky_tab); cudaFree(c->d_status); cudaFree(c->d_hpart); cudaFree(c->d_part); cudaFree(c->d_fdust);
    cudaFree(c->d_mag); cudaFree(c->d_hessbuf); cudaFree(c->d_statbuf); cudaFree(c->d_lnl);
    cudaFree(c->d_hess_data); cudaFree(c->d_data_stats);
    if (c->h_pin) cudaFreeHost(c->h_pin);
    if (c->stage_ev_valid) { cudaEventDestroy(c->stage_ev[0]); cudaEventDestroy(c->stage_ev[1]); }
    if (c->prof_made) for (int i = 0; i < 8; ++i) cudaEventDestroy(c->prof_ev[i]);
    free(c->h_imf_w); free(c->h_psf_sep);
    delete c;
}

// ---------------------------------------------------------------------------------------------


// n_models parameter vectors (tables), n_real realisations (images): n_real = n_models, or
// n_models = 1 and n_real repeats of it (pcmd_simulate_repeat).
static int stage_params(pcmd_ctx *c, const pcmd_params *params, int n_models, int n_real, cudaStream_t s) {
    // upper bound of the raw sampler-table size of one model (sizing only, no method arithmetic):
    // lambda_j <= max_a sfh_a * imf_w_j, and a table spans fewer than 20 sqrt(lambda) + 96 counts.
    int64_t cap = 0;
    double npix_max = 0.0;          // largest N_pix = sum of the SFH (sizes the Poisson(N_pix) table of the aggregated sampler)
    for (int i = 0; i < n_models; ++i) {
        const pcmd_params &p = params[i];
        if (!p.sfh || !(p.feh_sigma > 0.0) || !isfinite(p.feh_mean) || !isfinite(p.feh_sigma) ||
            !isfinite(p.dmod) || !(p.dust_med >= 0.0) || !isfinite(p.dust_med) || !(p.dust_sigma >= 0.0) ||
            !isfinite(p.dust_sigma))
            return PCMD_EINVAL;
        double smax = 0.0, ssum = 0.0;
        for (int a = 0; a < c->A; ++a) {
            if (!(p.sfh[a] >= 0.0) || !isfinite(p.sfh[a])) return PCMD_EINVAL;
            if (p.sfh[a] > smax) smax = p.sfh[a];
            ssum += p.sfh[a];
        }
        if (ssum > npix_max) npix_max = ssum;
        double tot = 0.0;
        if (smax * c->imf_w_max <= PCMD_LAMBDA_MAX) {
            tot = 20.0 * sqrt(smax) * c->imf_sqrt_sum + 96.0 * c->J;   // sum_j 20 sqrt(smax w_j) + 96
        } else {
            for (int j = 0; j < c->J; ++j) {
                const double lb = smax * c->h_imf_w[j];
                // the bound may be loose (MDF weight < 1); the kernel raises ERANGE on the true value
                tot += (lb > PCMD_LAMBDA_MAX) ? 20.0 * 2048.0 + 96.0 : 20.0 * sqrt(lb) + 96.0;
            }
        }
        if ((int64_t)tot > cap) cap = (int64_t)tot;
    }
    if (cap > 0xFFFFFFF0ll) return PCMD_ERANGE;
    if (c->sampler_mode == 1 && npix_max * 1.0001 > PCMD_LAMBDA_MAX) return PCMD_ERANGE;   // R-C2 covers means up to 2^22
    const int64_t agg_tcap = (int64_t)(20.0 * sqrt(npix_max * 1.0001 + 1.0) + 96.0);
    int rc = ensure_scratch(c, n_models, c->sampler_mode == 1 ? 16 : cap, agg_tcap);
    if (rc) return rc;
    c->n_seg = c->sampler_mode == 1 ? 1 : pcmd_stage2_segments(c, n_real);
    const int64_t need_img = (int64_t)n_real * c->B * c->P;
    if (need_img > c->fdust_elems) {
        cudaDeviceSynchronize();
        cudaFree(c->d_fdust); c->d_fdust = nullptr; c->fdust_elems = 0;
        PCMD_CUDA(c, cudaMalloc(&c->d_fdust, (size_t)need_img * sizeof(float)));
        c->fdust_elems = need_img;
    }
    const int64_t need = (int64_t)n_real * c->n_seg * c->B * c->P;
    if (need > c->part_elems) {
        cudaDeviceSynchronize();
        cudaFree(c->d_part); c->d_part = nullptr; c->part_elems = 0;
        PCMD_CUDA(c, cudaMalloc(&c->d_part, (size_t)need * sizeof(float)));
        c->part_elems = need;
    }
    // the half of the pinned staging area the previous call did not use: wait only for the call before that
    c->stage_flip ^= 1;
    if (c->stage_ev_valid) PCMD_CUDA(c, cudaEventSynchronize(c->stage_ev[c->stage_flip]));
    double *hs = reinterpret_cast<double *>(reinterpret_cast<char *>(c->h_stage) + (size_t)c->stage_flip * c->h_stage_bytes);
    DevModel *hm = reinterpret_cast<DevModel *>(hs + (size_t)n_models * c->A);
    for (int i = 0; i < n_models; ++i) {
        memcpy(hs + (size_t)i * c->A, params[i].sfh, c->A * sizeof(double));
        hm[i].feh_mean = params[i].feh_mean; hm[i].feh_sigma = params[i].feh_sigma;
        hm[i].dmod = params[i].dmod; hm[i].dust_med = params[i].dust_med; hm[i].dust_sigma = params[i].dust_sigma;
    }
    PCMD_CUDA(c, cudaMemcpyAsync(c->d_sfh, hs, (size_t)n_models * c->A * sizeof(double), cudaMemcpyHostToDevice, s));
    PCMD_CUDA(c, cudaMemcpyAsync(c->d_model, hm, (size_t)n_models * sizeof(DevModel), cudaMemcpyHostToDevice, s));
    return PCMD_OK;
}

static int simulate_impl(pcmd_ctx *c, const pcmd_params *params, int32_t n_models, int32_t n_real, uint64_t seed,
                         uint32_t model_index0, float *d_mag, float *d_flux_raw, uint64_t *d_count_hash,
                         uint32_t *d_count_total, void *cuda_stream) {
    if (!c || !params || n_models < 1 || n_real < 1 || !d_mag) return PCMD_EINVAL;
    if ((d_count_hash == nullptr) != (d_count_total == nullptr)) return PCMD_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (!c->stage_ev_valid) {
        PCMD_CUDA(c, cudaEventCreateWithFlags(&c->stage_ev[0], cudaEventDisableTiming));
        PCMD_CUDA(c, cudaEventCreateWithFlags(&c->stage_ev[1], cudaEventDisableTiming));
        PCMD_CUDA(c, cudaEventRecord(c->stage_ev[0], s));
        PCMD_CUDA(c, cudaEventRecord(c->stage_ev[1], s));
        c->stage_ev_valid = 1;
    }
    int rc = stage_params(c, params, n_models, n_real, s);
    if (rc) return rc;
    PCMD_CUDA(c, cudaEventRecord(c->stage_ev[c->stage_flip], s));
    PCMD_CUDA(c, cudaMemsetAsync(c->d_status, 0, 2 * sizeof(int32_t), s));
    c->last_models = n_models;
    c->tab_stride = (n_models == n_real) ? 1 : 0;     // 0: every realisation reads model 0's tables
    PCMD_PROF(c, 0, s);
    if ((rc = pcmd_launch_stage1(c, n_models, s))) return rc;
    PCMD_PROF(c, 1, s);
    if ((rc = pcmd_launch_stage2(c, n_real, seed, model_index0, d_flux_raw, d_count_hash, d_count_total, s))) return rc;
    PCMD_PROF(c, 2, s);
    if (c->tap_dust)
        PCMD_CUDA(c, cudaMemcpyAsync(c->tap_dust, c->d_fdust, (size_t)n_real * c->B * c->P * sizeof(float),
                                     cudaMemcpyDeviceToDevice, s));
    if ((rc = pcmd_launch_conv_noise(c, n_real, seed, model_index0, d_mag, s))) return rc;
    PCMD_PROF(c, 3, s);
    return PCMD_OK;
}

extern "C" int pcmd_simulate(pcmd_ctx *c, const pcmd_params *params, int32_t n_models, uint64_t seed,
                             uint32_t model_index0, float *d_mag, float *d_flux_raw,
                             uint64_t *d_count_hash, uint32_t *d_count_total, void *cuda_stream) {
    return simulate_impl(c, params, n_models, n_models, seed, model_index0, d_mag, d_flux_raw, d_count_hash,
                         d_count_total, cuda_stream);
}

extern "C" int pcmd_simulate_repeat(pcmd_ctx *c, const pcmd_params *params, int32_t n_repeats, uint64_t seed,
                                    uint32_t model_index0, float *d_mag, float *d_flux_raw,
                                    uint64_t *d_count_hash, uint32_t *d_count_total, void *cuda_stream) {
    return simulate_impl(c, params, 1, n_repeats, seed, model_index0, d_mag, d_flux_raw, d_count_hash,
                         d_count_total, cuda_stream);
}

extern "C" int pcmd_hess(pcmd_ctx *c, const float *d_mag, int32_t n_models, uint32_t *d_hess,
                         pcmd_hess_stats *d_stats, void *cuda_stream) {
    if (!c || !d_mag || !d_hess || n_models < 1 || c->n_hess < 1) return PCMD_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    PCMD_PROF(c, 4, s);
    int rc = pcmd_launch_hess(c, d_mag, n_models, d_hess, d_stats, s);
    if (rc) return rc;
    PCMD_PROF(c, 5, s);
    return PCMD_OK;
}

extern "C" int pcmd_loglike(pcmd_ctx *c, const uint32_t *d_hess_model, const pcmd_hess_stats *d_stats,
                            int32_t n_models, const uint32_t *d_hess_data,
                            const pcmd_hess_stats *d_data_stats, int32_t like_mode, double *d_loglike,
                            void *cuda_stream) {
    if (!c || !d_hess_model || !d_hess_data || !d_loglike || n_models < 1 || c->n_hess < 1) return PCMD_EINVAL;
    if (like_mode < PCMD_LIKE_POISSON || like_mode > PCMD_LIKE_GAUSS_LITERAL) return PCMD_EINVAL;
    if (like_mode != PCMD_LIKE_POISSON && (!d_stats || !d_data_stats)) return PCMD_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    PCMD_PROF(c, 6, s);
    int rc = pcmd_launch_loglike(c, d_hess_model, d_stats, n_models, d_hess_data, d_data_stats, like_mode,
                                 d_loglike, s);
    if (rc) return rc;
    PCMD_PROF(c, 7, s);
    return PCMD_OK;
}

extern "C" int64_t pcmd_hess_bins_total(const pcmd_ctx *c) { return c ? c->hess_bins : 0; }

extern "C" int pcmd_evaluate_host(pcmd_ctx *c, const pcmd_params *params, int32_t n_models, uint64_t seed,
                                  uint32_t model_index0, const uint32_t *h_hess_data,
                                  const pcmd_hess_stats *h_data_stats, int32_t like_mode, double *h_loglike,
                                  uint32_t *h_hess_out, pcmd_hess_stats *h_stats_out, void *cuda_stream) {
    if (!c || !params || n_models < 1 || !h_hess_data || !h_loglike || c->n_hess < 1) return PCMD_EINVAL;
    if (like_mode != PCMD_LIKE_POISSON && !h_data_stats) return PCMD_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t hb = (size_t)c->hess_bins, nh = (size_t)c->n_hess;
    if (n_models > c->eval_cap) {
        cudaDeviceSynchronize();
        cudaFree(c->d_mag); cudaFree(c->d_hessbuf); cudaFree(c->d_statbuf); cudaFree(c->d_lnl);
        cudaFree(c->d_hess_data); cudaFree(c->d_data_stats);
        if (c->h_pin) cudaFreeHost(c->h_pin);
        c->d_mag = nullptr; c->d_hessbuf = nullptr; c->d_statbuf = nullptr; c->d_lnl = nullptr;
        c->d_hess_data = nullptr; c->d_data_stats = nullptr; c->h_pin = nullptr; c->eval_cap = 0;
        PCMD_CUDA(c, cudaMalloc(&c->d_mag, (size_t)n_models * c->B * c->P * sizeof(float)));
        PCMD_CUDA(c, cudaMalloc(&c->d_hessbuf, (size_t)n_models * hb * sizeof(uint32_t)));
        PCMD_CUDA(c, cudaMalloc(&c->d_statbuf, (size_t)n_models * nh * sizeof(pcmd_hess_stats)));
        PCMD_CUDA(c, cudaMalloc(&c->d_lnl, (size_t)n_models * sizeof(double)));
        PCMD_CUDA(c, cudaMalloc(&c->d_hess_data, hb * sizeof(uint32_t)));
        PCMD_CUDA(c, cudaMalloc(&c->d_data_stats, nh * sizeof(pcmd_hess_stats)));
        c->h_pin_bytes = hb * sizeof(uint32_t) + nh * sizeof(pcmd_hess_stats) +
                         (size_t)n_models * (hb * sizeof(uint32_t) + nh * sizeof(pcmd_hess_stats) + sizeof(double));
        PCMD_CUDA(c, cudaMallocHost(&c->h_pin, c->h_pin_bytes));
        c->eval_cap = n_models;
    }
    // pinned layout: [data hess][data stats][model hess][model stats][lnl]
    char *pin = (char *)c->h_pin;
    uint32_t *p_dh = (uint32_t *)pin; pin += hb * sizeof(uint32_t);
    pcmd_hess_stats *p_ds = (pcmd_hess_stats *)pin; pin += nh * sizeof(pcmd_hess_stats);
    uint32_t *p_mh = (uint32_t *)pin; pin += (size_t)n_models * hb * sizeof(uint32_t);
    pcmd_hess_stats *p_ms = (pcmd_hess_stats *)pin; pin += (size_t)n_models * nh * sizeof(pcmd_hess_stats);
    double *p_l = (double *)pin;
    memcpy(p_dh, h_hess_data, hb * sizeof(uint32_t));
    PCMD_CUDA(c, cudaMemcpyAsync(c->d_hess_data, p_dh, hb * sizeof(uint32_t), cudaMemcpyHostToDevice, s));
    if (h_data_stats) {
        memcpy(p_ds, h_data_stats, nh * sizeof(pcmd_hess_stats));
        PCMD_CUDA(c, cudaMemcpyAsync(c->d_data_stats, p_ds, nh * sizeof(pcmd_hess_stats), cudaMemcpyHostToDevice, s));
    }
    int rc = pcmd_simulate(c, params, n_models, seed, model_index0, c->d_mag, nullptr, nullptr, nullptr, cuda_stream);
    if (rc) return rc;
    if ((rc = pcmd_hess(c, c->d_mag, n_models, c->d_hessbuf, c->d_statbuf, cuda_stream))) return rc;
    if ((rc = pcmd_loglike(c, c->d_hessbuf, c->d_statbuf, n_models, c->d_hess_data,
                           h_data_stats ? c->d_data_stats : nullptr, like_mode, c->d_lnl, cuda_stream)))
        return rc;
    PCMD_CUDA(c, cudaMemcpyAsync(p_l, c->d_lnl, (size_t)n_models * sizeof(double), cudaMemcpyDeviceToHost, s));
    if (h_hess_out)
        PCMD_CUDA(c, cudaMemcpyAsync(p_mh, c->d_hessbuf, (size_t)n_models * hb * sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
    if (h_stats_out)
        PCMD_CUDA(c, cudaMemcpyAsync(p_ms, c->d_statbuf, (size_t)n_models * nh * sizeof(pcmd_hess_stats), cudaMemcpyDeviceToHost, s));
    int32_t st = 0;
    PCMD_CUDA(c, cudaMemcpyAsync(&st, c->d_status, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    PCMD_CUDA(c, cudaStreamSynchronize(s));
    memcpy(h_loglike, p_l, (size_t)n_models * sizeof(double));
    if (h_hess_out) memcpy(h_hess_out, p_mh, (size_t)n_models * hb * sizeof(uint32_t));
    if (h_stats_out) memcpy(h_stats_out, p_ms, (size_t)n_models * nh * sizeof(pcmd_hess_stats));
    return st;
}

// ---------------------------------------------------------------------------------------------
extern "C" int pcmd_debug_weights(pcmd_ctx *c, int32_t model, double *h_lambda, float *h_flux, uint32_t *h_k0,
                                  uint32_t *h_len, uint32_t *h_tables, int64_t cap, int64_t *n_tables) {
    if (!c || model < 0 || model >= c->last_models) return PCMD_EINVAL;
    PCMD_CUDA(c, cudaDeviceSynchronize());
    const int J = c->J;
    if (h_lambda)
        PCMD_CUDA(c, cudaMemcpy(h_lambda, c->d_lambda + (size_t)model * J, (size_t)J * sizeof(double), cudaMemcpyDeviceToHost));
    PointRec *rec = (PointRec *)malloc((size_t)J * sizeof(PointRec));
    if (!rec) return PCMD_ENOMEM;
    cudaError_t e = cudaMemcpy(rec, c->d_rec + (size_t)model * c->Jpad, (size_t)J * sizeof(PointRec), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { free(rec); c->last_cuda = (int)e; return PCMD_ECUDA; }
    int64_t total = 0;
    for (int j = 0; j < J; ++j) {
        if (h_k0) h_k0[j] = rec[j].k0;
        if (h_len) h_len[j] = rec[j].len;
        if (h_flux) for (int b = 0; b < c->B; ++b) h_flux[(size_t)j * c->B + b] = rec[j].f[b];
        total += rec[j].len;
    }
    if (n_tables) *n_tables = total;
    if (h_tables && c->sampler_mode != 1) {
        // tables are compact but placed in completion order (k_points): gathered here in point order
        uint32_t *tmp = (uint32_t *)malloc((size_t)(c->cap_raw ? c->cap_raw : 1) * sizeof(uint32_t));
        if (!tmp) { free(rec); return PCMD_ENOMEM; }
        e = cudaMemcpy(tmp, c->d_tab + (size_t)model * c->cap_raw, (size_t)c->cap_raw * sizeof(uint32_t), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { free(tmp); free(rec); c->last_cuda = (int)e; return PCMD_ECUDA; }
        int64_t o = 0;
        for (int j = 0; j < J && o < cap; ++j)
            for (uint32_t i = 0; i < rec[j].len && o < cap; ++i) h_tables[o++] = tmp[rec[j].off + i] + 1u;  // stored minus 1 on the device
        free(tmp);
    }
    free(rec);
    return PCMD_OK;
}

extern "C" int pcmd_debug_taps(pcmd_ctx *c, float *d_flux_dust, float *d_flux_conv) {
    if (!c) return PCMD_EINVAL;
    c->tap_dust = d_flux_dust; c->tap_conv = d_flux_conv;
    return PCMD_OK;
}

__global__ void k_debug_philox(uint32_t k0, uint32_t k1, const uint32_t *__restrict__ ctr, int64_t n,
                               uint32_t *__restrict__ out) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t w[4];
    philox4x32_10(k0, k1, ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], w);
    out[4 * i] = w[0]; out[4 * i + 1] = w[1]; out[4 * i + 2] = w[2]; out[4 * i + 3] = w[3];
}

extern "C" int pcmd_debug_philox(uint64_t seed, const uint32_t *h_ctr, int64_t n, uint32_t *h_out) {
    if (!h_ctr || !h_out || n < 1) return PCMD_EINVAL;
    uint32_t *d_c = nullptr, *d_o = nullptr;
    cudaError_t e = cudaMalloc(&d_c, (size_t)n * 16);
    if (e == cudaSuccess) e = cudaMalloc(&d_o, (size_t)n * 16);
    if (e == cudaSuccess) e = cudaMemcpy(d_c, h_ctr, (size_t)n * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_debug_philox<<<(unsigned)((n + 127) / 128), 128>>>((uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32), d_c, n, d_o);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(h_out, d_o, (size_t)n * 16, cudaMemcpyDeviceToHost);
    cudaFree(d_c); cudaFree(d_o);      // freed on every path
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? PCMD_ENOMEM : PCMD_ECUDA;
    return PCMD_OK;
}

extern "C" int pcmd_params_from_paper(int32_t n_age, const double *log10_sfh, double feh, double sigma_feh,
                                      double log10_ebv, double sigma_dust, double dmod, double *sfh_out,
                                      pcmd_params *out) {
    if (n_age < 1 || !log10_sfh || !sfh_out || !out) return PCMD_EINVAL;
    if (!isfinite(feh) || !(sigma_feh > 0.0) || !isfinite(sigma_feh) || !isfinite(log10_ebv) ||
        !(sigma_dust >= 0.0) || !isfinite(sigma_dust) || !isfinite(dmod))
        return PCMD_EINVAL;
    for (int a = 0; a < n_age; ++a) {
        if (isnan(log10_sfh[a]) || log10_sfh[a] == INFINITY) return PCMD_EINVAL;
        sfh_out[a] = pow(10.0, log10_sfh[a]);        // -inf -> 0 stars in that bin
    }
    out->sfh = sfh_out;
    out->feh_mean = feh; out->feh_sigma = sigma_feh; out->dmod = dmod;
    out->dust_med = pow(10.0, log10_ebv); out->dust_sigma = sigma_dust;
    return PCMD_OK;
}

extern "C" int pcmd_status(pcmd_ctx *c, void *cuda_stream) {
    if (!c) return PCMD_EINVAL;
    PCMD_CUDA(c, cudaStreamSynchronize((cudaStream_t)cuda_stream));
    int32_t st = 0;
    PCMD_CUDA(c, cudaMemcpy(&st, c->d_status, sizeof(int32_t), cudaMemcpyDeviceToHost));
    return st;
}

extern "C" int pcmd_profile(pcmd_ctx *c, int32_t enable) {
    if (!c) return PCMD_EINVAL;
    if (enable && !c->prof_made) {
        for (int i = 0; i < 8; ++i) PCMD_CUDA(c, cudaEventCreate(&c->prof_ev[i]));
        c->prof_made = 1;
    }
    c->prof_on = enable != 0;
    c->prof_seen = 0;
    return PCMD_OK;
}

extern "C" int pcmd_stage_ms(pcmd_ctx *c, float *h_ms) {
    if (!c || !h_ms || !c->prof_made) return PCMD_EINVAL;
    static const int span[5][2] = {{0, 1}, {1, 2}, {2, 3}, {4, 5}, {6, 7}};
    for (int i = 0; i < 5; ++i) {
        h_ms[i] = -1.f;
        const uint32_t need = (1u << span[i][0]) | (1u << span[i][1]);
        if ((c->prof_seen & need) != need) continue;
        PCMD_CUDA(c, cudaEventSynchronize(c->prof_ev[span[i][1]]));
        PCMD_CUDA(c, cudaEventElapsedTime(&h_ms[i], c->prof_ev[span[i][0]], c->prof_ev[span[i][1]]));
    }
    return PCMD_OK;
}

extern "C" int pcmd_last_cuda_error(const pcmd_ctx *c) { return c ? c->last_cuda : 0; }
extern "C" int64_t pcmd_launch_count(const pcmd_ctx *c) { return c ? c->launches : 0; }
