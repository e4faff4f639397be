/*
 * api.cu -- the C ABI of include/shwfs.h: handle life cycle, argument checking, algorithm choice and
 * the host-buffer pipeline.  No arithmetic of the method lives here; see wk.cu and literal.cu.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "internal.h"
#include "tma.cuh"

namespace {

thread_local char g_cuda_err[256] = "";

#define CU_TRY(call, where)                                \
    do {                                                   \
        cudaError_t e_ = (call);                           \
        if (e_ != cudaSuccess) {                           \
            shwfs_note_cuda_error(e_, where);              \
            rc = (e_ == cudaErrorMemoryAllocation) ? SHWFS_ENOMEM : SHWFS_ECUDA; \
            goto fail;                                     \
        }                                                  \
    } while (0)

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

void free_handle(shwfs_handle *h)
{
    if (!h) return;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != h->device) cudaSetDevice(h->device);
    cudaFree(h->d_amp);
    cudaFree(h->d_valid);
    cudaFree(h->d_patch);
    cudaFree(h->d_sched);
    cudaFree(h->d_kernels);
    cudaFree(h->d_wk_table);
    cudaFree(h->d_khat);
    cudaFree(h->d_sod_g);
    cudaFree(h->d_dm_modes);
    cudaFree(h->d_dm_patch);
    cudaFree(h->d_um_modes);
    cudaFree(h->d_um_coef);
    for (int k = 0; k < 2; ++k) {
        if (h->h_pin[k]) cudaFreeHost(h->h_pin[k]);
        cudaFree(h->d_phase[k]);
        if (h->ev_h2d[k]) cudaEventDestroy(h->ev_h2d[k]);
        if (h->ev_done[k]) cudaEventDestroy(h->ev_done[k]);
    }
    cudaFree(h->d_slopes);
    if (h->st_copy) cudaStreamDestroy(h->st_copy);
    if (h->st_comp) cudaStreamDestroy(h->st_comp);
    free(h->h_valid);
    free(h->h_runs);
    if (prev >= 0 && prev != h->device) cudaSetDevice(prev);
    delete h;
    cudaGetLastError();
}

int pick_auto(const shwfs_handle *h)
{
    /* without kernels one P x P FFT is cheaper than the autocorrelation once
     * n >= 16; with kernels the lag-domain form always wins.  Fall back along the chain. */
    const bool wk = shwfs_wk_supported(h, 0), lit = shwfs_literal_supported(h);
    if (shwfs_pruned_fft_supported(h) && (h->n >= 16 || !wk)) return SHWFS_ALGO_PRUNED_FFT;
    if (!h->has_kernels && lit && (h->n >= 16 || !wk)) return SHWFS_ALGO_LITERAL;
    if (shwfs_wk_fft_supported(h)) return SHWFS_ALGO_WK_FFT;           /* n >= 12: 80 line FFTs beat n^4 complex MACs */
    if (wk) return SHWFS_ALGO_WK;
    if (shwfs_wk_supported(h, 1)) return SHWFS_ALGO_WK_GENERIC;
    if (lit) return SHWFS_ALGO_LITERAL;
    return -1;
}

int ensure_khat(shwfs_handle *h)
{
    if (!h->has_kernels || h->d_khat) return SHWFS_OK;
    cudaError_t e = cudaMalloc(&h->d_khat, sizeof(float2) * (size_t)h->nsub * h->P * h->P);
    if (e != cudaSuccess) { h->d_khat = nullptr; shwfs_note_cuda_error(e, "cudaMalloc(khat)"); return SHWFS_ENOMEM; }
    e = shwfs_literal_build_khat(h, 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(0);
    if (e != cudaSuccess) {
        shwfs_note_cuda_error(e, "literal_build_khat");
        cudaFree(h->d_khat); h->d_khat = nullptr;
        return SHWFS_ECUDA;
    }
    return SHWFS_OK;
}

}  // namespace

#ifndef SHWFS_TMA_L2PROMO
#define SHWFS_TMA_L2PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_128B
#endif

/* tma.cuh: the driver's encoder is fetched through the runtime, so the library links against cudart only */
bool shwfs_tma_patch_map(CUtensorMap *out, const float *base, int N, long long frames, int n)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    static bool looked = false;
    if (!looked) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            encode = (encode_fn)fn;
        else
            cudaGetLastError();
        looked = true;
    }
    if (!encode || !base || frames <= 0 || N <= 0 || (N & 3) || (n & 3) || n > 256) return false;
    if (reinterpret_cast<uintptr_t>(base) & 15) return false;
    const cuuint64_t dim[3] = {(cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)frames};
    const cuuint64_t stride[2] = {(cuuint64_t)N * 4, (cuuint64_t)N * (cuuint64_t)N * 4};
    const cuuint32_t box[3] = {(cuuint32_t)n, (cuuint32_t)n, 1};
    const cuuint32_t one[3] = {1, 1, 1};
    const CUtensorMapSwizzle sw = n == 16 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE;
    return encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float *>(base), dim, stride, box, one,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, sw, SHWFS_TMA_L2PROMO,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

void shwfs_note_cuda_error(cudaError_t e, const char *where)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", where, cudaGetErrorString(e));
    cudaGetLastError();   /* clear the sticky-free error state */
}

extern "C" {

int shwfs_version(void) { return 100; }

const char *shwfs_strerror(int code)
{
    switch (code) {
    case SHWFS_OK: return "ok";
    case SHWFS_EINVAL: return "invalid argument";
    case SHWFS_EUNSUPPORTED: return "sizes not supported by any kernel instance";
    case SHWFS_ENOMEM: return "out of memory";
    case SHWFS_ECUDA: return "CUDA error (see shwfs_last_cuda_error)";
    default: return "unknown error code";
    }
}

const char *shwfs_last_cuda_error(void) { return g_cuda_err; }

int shwfs_create(const shwfs_geometry *g, float lambda_m, int32_t pad, int32_t bin,
                 const float *elong_kernels, shwfs_handle **out)
{
    if (!g || !out || !g->amplitude) return SHWFS_EINVAL;
    const int N = g->n_pupil, S = g->n_sub_side, n = g->n_pix, P = pad, b = bin;
    if (N <= 0 || S <= 0 || n <= 0 || (long long)S * n != N) return SHWFS_EINVAL;
    if (!is_pow2(P) || P < n || P > 64 || b <= 0 || P % b || (P / 2) % b) return SHWFS_EINVAL;
    if (!(lambda_m > 0.f) || !(g->pixel_size_m > 0.f)) return SHWFS_EINVAL;
    if (!(g->threshold_frac >= 0.f && g->threshold_frac < 1.f)) return SHWFS_EINVAL;
    if (g->threshold_mode != 0 && g->threshold_mode != 1) return SHWFS_EINVAL;
    if (!isfinite(g->phase_to_rad) || !isfinite(g->min_illum)) return SHWFS_EINVAL;
    if (g->valid_yx && g->n_valid <= 0) return SHWFS_EINVAL;

    /* H0: valid-subaperture list (reading A2), row-major over (sy,sx) */
    int32_t *valid = (int32_t *)malloc(sizeof(int32_t) * 2 * (size_t)S * S);
    if (!valid) return SHWFS_ENOMEM;
    int nsub = 0;
    if (g->valid_yx) {
        if (g->n_valid > S * S) { free(valid); return SHWFS_EINVAL; }
        for (int i = 0; i < g->n_valid; ++i) {
            const int sy = g->valid_yx[2 * i], sx = g->valid_yx[2 * i + 1];
            if (sy < 0 || sy >= S || sx < 0 || sx >= S) { free(valid); return SHWFS_EINVAL; }
            valid[2 * i] = sy; valid[2 * i + 1] = sx;
        }
        nsub = g->n_valid;
    } else {
        for (int sy = 0; sy < S; ++sy)
            for (int sx = 0; sx < S; ++sx) {
                double s = 0.0;
                for (int j = 0; j < n; ++j)
                    for (int k = 0; k < n; ++k) s += (double)g->amplitude[(size_t)(sy * n + j) * N + sx * n + k];
                if (s / ((double)n * n) >= (double)g->min_illum) { valid[2 * nsub] = sy; valid[2 * nsub + 1] = sx; ++nsub; }
            }
    }
    if (nsub == 0) { free(valid); return SHWFS_EINVAL; }

    shwfs_handle *h = new (std::nothrow) shwfs_handle();
    if (!h) { free(valid); return SHWFS_ENOMEM; }
    memset(h, 0, sizeof(*h));
    h->N = N; h->S = S; h->n = n; h->P = P; h->b = b; h->D = P / b; h->nsub = nsub;
    h->dx = g->pixel_size_m; h->lambda_m = lambda_m; h->tau = g->threshold_frac; h->c_phi = g->phase_to_rad;
    h->mode = g->threshold_mode; h->has_kernels = elong_kernels != nullptr;
    h->h_valid = valid;
    h->chunk_frames = 0;
    {   /* bounding column extent of the valid subapertures of each lenslet row; consecutive rows with the same
         * extent merge into one band = {first lenslet row, rows, first column, width in pixels} */
        int *lo = (int *)malloc(sizeof(int) * (size_t)S), *hi = (int *)malloc(sizeof(int) * (size_t)S);
        int *runs = (int *)malloc(sizeof(int) * 4 * (size_t)S);
        if (lo && hi && runs) {
            for (int sy = 0; sy < S; ++sy) { lo[sy] = S; hi[sy] = -1; }
            for (int i = 0; i < nsub; ++i) {
                const int sy = valid[2 * i], sx = valid[2 * i + 1];
                if (sx < lo[sy]) lo[sy] = sx;
                if (sx > hi[sy]) hi[sy] = sx;
            }
            int nr = 0;
            long long px = 0;
            for (int sy = 0; sy < S; ++sy) {
                if (hi[sy] < 0) continue;
                if (nr > 0 && runs[4 * (nr - 1)] + runs[4 * (nr - 1) + 1] == sy && runs[4 * (nr - 1) + 2] == lo[sy] * n &&
                    runs[4 * (nr - 1) + 3] == (hi[sy] - lo[sy] + 1) * n) {
                    runs[4 * (nr - 1) + 1] += 1;
                } else {
                    runs[4 * nr] = sy; runs[4 * nr + 1] = 1; runs[4 * nr + 2] = lo[sy] * n; runs[4 * nr + 3] = (hi[sy] - lo[sy] + 1) * n;
                    ++nr;
                }
                px += (long long)(hi[sy] - lo[sy] + 1) * n * n;
            }
            /* worth it only if it saves a tenth of the bytes */
            if (px * 10 <= (long long)N * N * 9) { h->h_runs = runs; h->n_runs = nr; h->run_pixels = px; runs = nullptr; }
        }
        free(lo); free(hi); free(runs);
    }

    int rc = SHWFS_OK;
    CU_TRY(cudaGetDevice(&h->device), "cudaGetDevice");
    CU_TRY(cudaDeviceGetAttribute(&h->sms, cudaDevAttrMultiProcessorCount, h->device), "cudaDeviceGetAttribute");
    h->no_tma = getenv("SHWFS_NO_TMA") != nullptr;
    h->force_persistent = getenv("SHWFS_FORCE_PERSISTENT") != nullptr;
    if (!shwfs_wk_supported(h, 0) && !shwfs_wk_supported(h, 1) && !shwfs_literal_supported(h) && !shwfs_pruned_fft_supported(h)) { rc = SHWFS_EUNSUPPORTED; goto fail; }
    h->algo = pick_auto(h);
    h->algo_explicit = 0;
    if (h->algo < 0) { rc = SHWFS_EUNSUPPORTED; goto fail; }

    CU_TRY(cudaMalloc(&h->d_amp, sizeof(float) * (size_t)N * N), "cudaMalloc(amplitude)");
    CU_TRY(cudaMemcpy(h->d_amp, g->amplitude, sizeof(float) * (size_t)N * N, cudaMemcpyHostToDevice), "cudaMemcpy(amplitude)");
    CU_TRY(cudaMalloc(&h->d_valid, sizeof(int2) * (size_t)nsub), "cudaMalloc(valid)");
    CU_TRY(cudaMemcpy(h->d_valid, valid, sizeof(int2) * (size_t)nsub, cudaMemcpyHostToDevice), "cudaMemcpy(valid)");
    {   /* patch table: origin of each valid subaperture in pixels, flagged when its amplitudes are all exactly 1 */
        int2 *patch = (int2 *)malloc(sizeof(int2) * (size_t)nsub);
        if (!patch) { rc = SHWFS_ENOMEM; goto fail; }
        for (int i = 0; i < nsub; ++i) {
            const int y0 = valid[2 * i] * n, x0 = valid[2 * i + 1] * n;
            bool lit = true;
            for (int j = 0; j < n && lit; ++j)
                for (int k = 0; k < n; ++k)
                    if (g->amplitude[(size_t)(y0 + j) * N + x0 + k] != 1.0f) { lit = false; break; }
            patch[i] = make_int2(x0 | (lit ? SHWFS_PATCH_LIT : 0), y0);
        }
        cudaError_t e1 = cudaMalloc(&h->d_patch, sizeof(int2) * (size_t)nsub);
        if (e1 == cudaSuccess) e1 = cudaMemcpy(h->d_patch, patch, sizeof(int2) * (size_t)nsub, cudaMemcpyHostToDevice);
        free(patch);
        CU_TRY(e1, "patch table");
        CU_TRY(cudaMalloc(&h->d_sched, 2 * sizeof(int)), "cudaMalloc(sched)");
        CU_TRY(cudaMemset(h->d_sched, 0, 2 * sizeof(int)), "cudaMemset(sched)");
    }
    if (h->has_kernels) {
        const size_t kb = sizeof(float) * (size_t)nsub * P * P;
        CU_TRY(cudaMalloc(&h->d_kernels, kb), "cudaMalloc(kernels)");
        CU_TRY(cudaMemcpy(h->d_kernels, elong_kernels, kb, cudaMemcpyHostToDevice), "cudaMemcpy(kernels)");
    }
    if (shwfs_wk_supported(h, 1) || shwfs_wk_supported(h, 0)) {
        const int per = n * (2 * n - 1);
        h->wk_table_stride = h->has_kernels ? per : 0;
        CU_TRY(cudaMalloc(&h->d_wk_table, sizeof(float2) * (size_t)per * (h->has_kernels ? nsub : 1)), "cudaMalloc(wk table)");
        CU_TRY(shwfs_wk_build_table(h, 0), "wk_build_table");
    }
    CU_TRY(cudaStreamSynchronize(0), "create sync");
    if (h->algo == SHWFS_ALGO_LITERAL) { rc = ensure_khat(h); if (rc) goto fail; }
    *out = h;
    return SHWFS_OK;
fail:
    free_handle(h);
    return rc;
}

int shwfs_destroy(shwfs_handle *h)
{
    if (!h) return SHWFS_OK;
    if (h->st_comp) cudaStreamSynchronize(h->st_comp);
    if (h->st_copy) cudaStreamSynchronize(h->st_copy);
    free_handle(h);
    return SHWFS_OK;
}

int shwfs_num_subaps(const shwfs_handle *h, int32_t *nsub)
{
    if (!h || !nsub) return SHWFS_EINVAL;
    *nsub = h->nsub;
    return SHWFS_OK;
}

int shwfs_valid_list(const shwfs_handle *h, int32_t *yx_host)
{
    if (!h || !yx_host) return SHWFS_EINVAL;
    memcpy(yx_host, h->h_valid, sizeof(int32_t) * 2 * (size_t)h->nsub);
    return SHWFS_OK;
}

int shwfs_pixel_scale(const shwfs_handle *h, double *rad_per_detector_px)
{
    if (!h || !rad_per_detector_px) return SHWFS_EINVAL;
    *rad_per_detector_px = (double)h->b * (double)h->lambda_m / ((double)h->P * (double)h->dx);
    return SHWFS_OK;
}

int shwfs_set_algorithm(shwfs_handle *h, int32_t algo)
{
    if (!h) return SHWFS_EINVAL;
    int a = algo;
    if (a == SHWFS_ALGO_AUTO) a = pick_auto(h);
    switch (a) {
    case SHWFS_ALGO_LITERAL:
        if (!shwfs_literal_supported(h)) return SHWFS_EUNSUPPORTED;
        { int rc = ensure_khat(h); if (rc) return rc; }
        break;
    case SHWFS_ALGO_WK: if (!shwfs_wk_supported(h, 0)) return SHWFS_EUNSUPPORTED; break;
    case SHWFS_ALGO_WK_GENERIC: if (!shwfs_wk_supported(h, 1)) return SHWFS_EUNSUPPORTED; break;
    case SHWFS_ALGO_WK_FFT: if (!shwfs_wk_fft_supported(h)) return SHWFS_EUNSUPPORTED; break;
    case SHWFS_ALGO_PRUNED_FFT: if (!shwfs_pruned_fft_supported(h)) return SHWFS_EUNSUPPORTED; break;
    default: return SHWFS_EINVAL;
    }
    h->algo = a;
    h->algo_explicit = algo != SHWFS_ALGO_AUTO;
    return SHWFS_OK;
}

int shwfs_get_algorithm(const shwfs_handle *h, int32_t *algo)
{
    if (!h || !algo) return SHWFS_EINVAL;
    *algo = h->algo;
    return SHWFS_OK;
}

int shwfs_host_bytes_per_frame(const shwfs_handle *h, int64_t *bytes)
{
    if (!h || !bytes) return SHWFS_EINVAL;
    *bytes = (int64_t)sizeof(float) * (h->n_runs > 0 ? h->run_pixels : (long long)h->N * h->N);
    return SHWFS_OK;
}

int shwfs_launch_count(const shwfs_handle *h, int64_t *count)
{
    if (!h || !count) return SHWFS_EINVAL;
    *count = h->launches;
    return SHWFS_OK;
}

int shwfs_last_kernel(const shwfs_handle *h, char *name, int32_t len)
{
    if (!h || !name || len <= 0) return SHWFS_EINVAL;
    snprintf(name, (size_t)len, "%s", h->last_kernel ? h->last_kernel : "");
    return SHWFS_OK;
}

int shwfs_set_sodium(shwfs_handle *h, const shwfs_sodium *sd)
{
    if (!h) return SHWFS_EINVAL;
    if (!sd) { h->sod_L = 0; h->sod_shared = 0; return SHWFS_OK; }
    const int L = sd->n_layers;
    if (L < 1 || L > SHWFS_MAX_LAYERS || !sd->weight || !sd->defocus) return SHWFS_EINVAL;
    if (!isfinite(sd->centre_x_m) || !isfinite(sd->centre_y_m)) return SHWFS_EINVAL;
    for (int l = 0; l < L; ++l) {
        if (!(sd->weight[l] >= 0.f) || !isfinite(sd->weight[l]) || !isfinite(sd->defocus[l])) return SHWFS_EINVAL;
        if ((sd->tilt_x && !isfinite(sd->tilt_x[l])) || (sd->tilt_y && !isfinite(sd->tilt_y[l]))) return SHWFS_EINVAL;
    }
    if (!shwfs_wk_supported(h, 0) && !shwfs_wk_supported(h, 1)) return SHWFS_EUNSUPPORTED;
    /* reading B1, expanded about each subaperture centre r_i (float64 on the host): over the patch the
     * sub-layer's analytic phase is piston + (2 a (r_i - r_c) + g) . d + a |d|^2, d = offset from r_i.   */
    const size_t cnt = (size_t)L * h->nsub;
    float2 *g = (float2 *)malloc(sizeof(float2) * cnt);
    if (!g) return SHWFS_ENOMEM;
    const double two_pi = 6.283185307179586476925286766559, dx = (double)h->dx;
    for (int l = 0; l < L; ++l) {
        const double a = (double)sd->defocus[l];
        const double tx = sd->tilt_x ? (double)sd->tilt_x[l] : 0.0, ty = sd->tilt_y ? (double)sd->tilt_y[l] : 0.0;
        for (int i = 0; i < h->nsub; ++i) {
            const double yc = (((double)h->h_valid[2 * i] + 0.5) * h->n - 0.5 * h->N) * dx;
            const double xc = (((double)h->h_valid[2 * i + 1] + 0.5) * h->n - 0.5 * h->N) * dx;
            double gx = (2.0 * a * (xc - (double)sd->centre_x_m) + tx) * dx / two_pi;
            double gy = (2.0 * a * (yc - (double)sd->centre_y_m) + ty) * dx / two_pi;
            /* whole turns per pixel alias to a piston on the half-integer pixel offsets: drop them */
            gx -= nearbyint(gx); gy -= nearbyint(gy);
            g[(size_t)l * h->nsub + i] = make_float2((float)gx, (float)gy);
        }
    }
    int rc = SHWFS_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != h->device) cudaSetDevice(h->device);
    float2 *d_new = nullptr;
    cudaError_t e = cudaMalloc(&d_new, sizeof(float2) * cnt);
    if (e == cudaSuccess) e = cudaMemcpy(d_new, g, sizeof(float2) * cnt, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        shwfs_note_cuda_error(e, "shwfs_set_sodium");
        cudaFree(d_new);
        rc = (e == cudaErrorMemoryAllocation) ? SHWFS_ENOMEM : SHWFS_ECUDA;
    } else {
        cudaDeviceSynchronize();                 /* nothing in flight may still read the old table */
        cudaFree(h->d_sod_g);
        h->d_sod_g = d_new;
        h->sod_L = L; h->sod_shared = sd->shared_phase != 0;
        for (int l = 0; l < SHWFS_MAX_LAYERS; ++l) {
            h->sod_q[l] = l < L ? (float)((double)sd->defocus[l] * dx * dx / two_pi) : 0.f;
            h->sod_sw[l] = l < L ? (float)sqrt((double)sd->weight[l]) : 0.f;
        }
    }
    if (prev >= 0 && prev != h->device) cudaSetDevice(prev);
    free(g);
    return rc;
}

int shwfs_set_noise(shwfs_handle *h, const shwfs_noise *nz)
{
    if (!h) return SHWFS_EINVAL;
    if (!nz || !(nz->flux > 0.f)) { h->nz_flux = 0.f; return SHWFS_OK; }
    if (!isfinite(nz->flux) || !(nz->read_noise >= 0.f) || !isfinite(nz->read_noise)) return SHWFS_EINVAL;
    if (nz->photon_model != 0 && nz->photon_model != 1) return SHWFS_EINVAL;
    if (!shwfs_wk_supported(h, 0) && !shwfs_wk_supported(h, 1)) return SHWFS_EUNSUPPORTED;
    h->nz_flux = nz->flux; h->nz_ron = nz->read_noise; h->nz_seed = nz->seed; h->nz_first_frame = nz->first_frame;
    h->nz_model = nz->photon_model;
    return SHWFS_OK;
}

int shwfs_set_dm(shwfs_handle *h, const float *modes_dev, int32_t M)
{
    if (!h || M < 0) return SHWFS_EINVAL;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != h->device) cudaSetDevice(h->device);
    int rc = SHWFS_OK;
    cudaDeviceSynchronize();                     /* nothing in flight may still read the old tables */
    cudaFree(h->d_dm_modes); h->d_dm_modes = nullptr;
    cudaFree(h->d_dm_patch); h->d_dm_patch = nullptr; h->dm_patch_cap = 0;
    cudaFree(h->d_um_modes); h->d_um_modes = nullptr;
    cudaFree(h->d_um_coef); h->d_um_coef = nullptr; h->um_coef_cap = 0;
    h->dm_M = 0;
    if (M > 0 && modes_dev) {
        if (!shwfs_wk_supported(h, 0) && !shwfs_wk_supported(h, 1)) { rc = SHWFS_EUNSUPPORTED; goto done; }
        CU_TRY(cudaMalloc(&h->d_dm_modes, sizeof(float) * (size_t)h->nsub * M * h->n * h->n), "cudaMalloc(dm modes)");
        h->dm_patch_cap = (size_t)h->nsub * h->n * h->n;          /* one frame: enough for the loop */
        CU_TRY(cudaMalloc(&h->d_dm_patch, sizeof(float) * h->dm_patch_cap), "cudaMalloc(dm patch)");
        CU_TRY(shwfs_loop_relayout_modes(h, modes_dev, M, 0), "relayout_modes");
        h->dm_M = M;
        h->dm_fp32 = getenv("SHWFS_DM_FP32") != nullptr;   /* A/B runs: keep the FP32 SIMT GEMM for batches too */
        if (shwfs_umma_np(h) > 0) {
            /* tensor-core operand tiles (hi|lo split, canonical layout); best effort: without them the FP32
             * SIMT GEMM of loop.cu serves every batch size */
            if (cudaMalloc(&h->d_um_modes, sizeof(float) * shwfs_umma_modes_floats(h, M)) == cudaSuccess) {
                CU_TRY(shwfs_umma_build_modes(h, 0), "umma_build_modes");
            } else {
                h->d_um_modes = nullptr;
                cudaGetLastError();
            }
        }
        CU_TRY(cudaStreamSynchronize(0), "set_dm sync");
    }
    goto done;
fail:
    cudaFree(h->d_dm_modes); h->d_dm_modes = nullptr;
    cudaFree(h->d_dm_patch); h->d_dm_patch = nullptr; h->dm_patch_cap = 0;
    h->dm_M = 0;
done:
    if (prev >= 0 && prev != h->device) cudaSetDevice(prev);
    return rc;
}

/* the enqueue-only entry points launch on the current device: it has to be the handle's */
static bool on_device(const shwfs_handle *h)
{
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == h->device;
}

/* include/shwfs.h: frames are 16-byte aligned (vector loads and TMA boxes start on their first pixel) */
static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

static bool ext_on(const shwfs_handle *h) { return h->sod_L > 0 || h->nz_flux > 0.f; }

/* frames of phase per time step t: L when every sub-layer has its own wavefront */
static int frames_per_step(const shwfs_handle *h) { return (h->sod_L > 0 && !h->sod_shared) ? h->sod_L : 1; }

/* call_T: frames of the whole API call (== T unless the host pipeline feeds it in chunks), see shwfs_wk_launch */
static int run_path(shwfs_handle *h, const float *phase_dev, int T, int call_T, float *slopes_dev, int stage, float *img,
                    unsigned t_base, cudaStream_t st, const float *dm_patch = nullptr)
{
    if ((long long)T * h->nsub > 0x7fffffffLL / 2) return SHWFS_EINVAL;
    cudaError_t e;
    if (stage == 3 && !(h->nz_flux > 0.f)) stage = 2;      /* no noise: the final image is the binned one */
    if (ext_on(h) || dm_patch) {
        /* sub-layers / noise / DM live in the lag-domain kernels only (shwfs_set_sodium made sure one exists) */
        if (stage == 0 || stage == 1) return SHWFS_EUNSUPPORTED;
        const int generic = (h->algo == SHWFS_ALGO_WK_GENERIC) || !(shwfs_wk_supported(h, 0) || shwfs_wk_fft_supported(h));
        e = shwfs_wk_launch(h, phase_dev, T, call_T, slopes_dev, stage == 2 ? img : nullptr, stage == 3 ? img : nullptr,
                            t_base, dm_patch, generic, st);
    } else if (stage == 0 || stage == 1) {
        int rc = ensure_khat(h);
        if (rc) return rc;
        if (!shwfs_literal_supported(h)) return SHWFS_EUNSUPPORTED;
        e = shwfs_literal_launch(h, phase_dev, T, slopes_dev, stage, img, st);
    } else if (h->algo == SHWFS_ALGO_LITERAL) {
        e = shwfs_literal_launch(h, phase_dev, T, slopes_dev, stage == 3 ? 2 : stage, img, st);
    } else if (h->algo == SHWFS_ALGO_PRUNED_FFT) {
        e = shwfs_pruned_fft_launch(h, phase_dev, T, slopes_dev, (stage == 2 || stage == 3) ? img : nullptr, st);
    } else {
        if (stage == 3) stage = 2;
        e = shwfs_wk_launch(h, phase_dev, T, call_T, slopes_dev, stage == 2 ? img : nullptr, nullptr, t_base, nullptr,
                            h->algo == SHWFS_ALGO_WK_GENERIC, st);
    }
    if (e != cudaSuccess) { shwfs_note_cuda_error(e, "kernel launch"); return SHWFS_ECUDA; }
    return SHWFS_OK;
}

int shwfs_measure(shwfs_handle *h, const float *phase_dev, int32_t T, float *slopes_dev, void *cuda_stream)
{
    if (!h || T < 0) return SHWFS_EINVAL;
    if (T == 0) return SHWFS_OK;
    if (!phase_dev || !slopes_dev || !on_device(h) || !aligned16(phase_dev)) return SHWFS_EINVAL;
    return run_path(h, phase_dev, T, T, slopes_dev, -1, nullptr, 0u, (cudaStream_t)cuda_stream);
}

int shwfs_measure_residual(shwfs_handle *h, const float *phase_dev, const float *coef_dev, int32_t T,
                           float *slopes_dev, void *cuda_stream)
{
    if (!h || T < 0 || h->dm_M <= 0) return SHWFS_EINVAL;
    if (T == 0) return SHWFS_OK;
    if (!phase_dev || !coef_dev || !slopes_dev || !on_device(h) || !aligned16(phase_dev)) return SHWFS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t need = (size_t)T * h->nsub * h->n * h->n;
    if (h->dm_patch_cap < need) {
        cudaStreamSynchronize(st);
        cudaFree(h->d_dm_patch); h->d_dm_patch = nullptr; h->dm_patch_cap = 0;
        cudaError_t e = cudaMalloc(&h->d_dm_patch, sizeof(float) * need);
        if (e != cudaSuccess) { shwfs_note_cuda_error(e, "cudaMalloc(dm patch)"); return SHWFS_ENOMEM; }
        h->dm_patch_cap = need;
    }
    if (h->d_um_modes && T > 8) {
        const size_t cneed = shwfs_umma_coef_floats(T, h->dm_M);
        if (h->um_coef_cap < cneed) {
            cudaStreamSynchronize(st);
            cudaFree(h->d_um_coef); h->d_um_coef = nullptr; h->um_coef_cap = 0;
            cudaError_t e2 = cudaMalloc(&h->d_um_coef, sizeof(float) * cneed);
            if (e2 != cudaSuccess) { shwfs_note_cuda_error(e2, "cudaMalloc(um coef)"); return SHWFS_ENOMEM; }
            h->um_coef_cap = cneed;
        }
    }
    cudaError_t e = shwfs_loop_dm_phase(h, coef_dev, h->dm_M, T, h->d_dm_patch, st);
    if (e != cudaSuccess) { shwfs_note_cuda_error(e, "dm_phase"); return SHWFS_ECUDA; }
    h->launches += (h->d_um_modes && T > 8 && h->d_um_coef && !h->dm_fp32) ? 2 : 1;
    return run_path(h, phase_dev, T, T, slopes_dev, -1, nullptr, 0u, st, h->d_dm_patch);
}

int shwfs_reconstruct(shwfs_handle *h, const float *R_dev, const float *slopes_dev, int32_t T, float gain,
                      float *coef_dev, void *cuda_stream)
{
    if (!h || T < 0 || h->dm_M <= 0 || !isfinite(gain)) return SHWFS_EINVAL;
    if (T == 0) return SHWFS_OK;
    if (!R_dev || !slopes_dev || !coef_dev || !on_device(h)) return SHWFS_EINVAL;
    cudaError_t e = shwfs_loop_reconstruct(R_dev, slopes_dev, T, 2 * h->nsub, h->dm_M, gain, coef_dev, h->dm_M,
                                           nullptr, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) { shwfs_note_cuda_error(e, "reconstruct"); return SHWFS_ECUDA; }
    h->launches += 1;
    return SHWFS_OK;
}

int shwfs_closed_loop(shwfs_handle *h, const float *phase_dev, const float *R_dev, float gain, float *coef_dev,
                      int32_t T, float *slopes_dev, float *coef_hist_dev, void *cuda_stream)
{
    if (!h || T < 0 || h->dm_M <= 0 || !isfinite(gain)) return SHWFS_EINVAL;
    if (T == 0) return SHWFS_OK;
    if (!phase_dev || !R_dev || !coef_dev || !slopes_dev || !on_device(h) || !aligned16(phase_dev)) return SHWFS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t step = (size_t)h->N * h->N * frames_per_step(h);
    const int K = 2 * h->nsub;
    /* per frame: DM phase of c_t on the valid patches, sensor on the residual, c_{t+1} = c_t + gain R s_t */
    cudaError_t e = cudaSuccess;
    for (int t = 0; t < T && e == cudaSuccess; ++t) {
        e = shwfs_loop_dm_phase(h, coef_dev, h->dm_M, 1, h->d_dm_patch, st);
        if (e != cudaSuccess) break;
        h->launches += 1;
        int rc = run_path(h, phase_dev + (size_t)t * step, 1, 1, slopes_dev + (size_t)t * K, -1, nullptr, (unsigned)t,
                          st, h->d_dm_patch);
        if (rc) return rc;
        e = shwfs_loop_reconstruct(R_dev, slopes_dev + (size_t)t * K, 1, K, h->dm_M, gain, coef_dev, h->dm_M,
                                   coef_hist_dev ? coef_hist_dev + (size_t)t * h->dm_M : nullptr, st);
        h->launches += 1;
    }
    if (e != cudaSuccess) { shwfs_note_cuda_error(e, "closed_loop"); return SHWFS_ECUDA; }
    return SHWFS_OK;
}

int shwfs_debug_spots(shwfs_handle *h, const float *phase_dev, int32_t T, int32_t stage, float *out_dev,
                      void *cuda_stream)
{
    if (!h || T < 0 || stage < 0 || stage > 3) return SHWFS_EINVAL;
    if (T == 0) return SHWFS_OK;
    if (!phase_dev || !out_dev || !on_device(h) || !aligned16(phase_dev)) return SHWFS_EINVAL;
    /* the debug path needs somewhere to put the slopes it also computes */
    const size_t need = 2 * (size_t)T * h->nsub;
    if (h->d_slopes_cap < need) {
        cudaStreamSynchronize((cudaStream_t)cuda_stream);
        cudaFree(h->d_slopes); h->d_slopes = nullptr; h->d_slopes_cap = 0;
        cudaError_t e = cudaMalloc(&h->d_slopes, sizeof(float) * need);
        if (e != cudaSuccess) { shwfs_note_cuda_error(e, "cudaMalloc(debug slopes)"); return SHWFS_ENOMEM; }
        h->d_slopes_cap = need;
    }
    return run_path(h, phase_dev, T, T, h->d_slopes, stage, out_dev, 0u, (cudaStream_t)cuda_stream);
}

}  // extern "C"

/* ------------------------------------------------------------------------------------------------
 * Host-buffer entry point: frames are cut into chunks of ~128 MiB, copied on st_copy into one of two
 * device buffers and measured on st_comp, so the H2D copy of chunk c+1 overlaps the kernels of
 * chunk c.  A pinned (cudaHostAlloc / cudaHostRegister) caller buffer is copied from directly; a
 * pageable one goes through the handle's own two pinned staging buffers.
 * ---------------------------------------------------------------------------------------------- */
namespace {

int host_init(shwfs_handle *h)
{
    if (h->host_ready) return SHWFS_OK;
    int rc = SHWFS_OK;
    /* one "frame" of the pipeline = one time step = up to SHWFS_MAX_LAYERS wavefronts, so that a later
     * shwfs_set_sodium never outgrows the buffers */
    const size_t frame_bytes = sizeof(float) * (size_t)h->N * h->N;
    size_t chunk = ((size_t)128 << 20) / frame_bytes;
    if (chunk < SHWFS_MAX_LAYERS) chunk = SHWFS_MAX_LAYERS;
    if (chunk > 256) chunk = 256;
    h->chunk_frames = (int)chunk;
    CU_TRY(cudaStreamCreateWithFlags(&h->st_copy, cudaStreamNonBlocking), "cudaStreamCreate");
    CU_TRY(cudaStreamCreateWithFlags(&h->st_comp, cudaStreamNonBlocking), "cudaStreamCreate");
    for (int k = 0; k < 2; ++k) {
        CU_TRY(cudaEventCreateWithFlags(&h->ev_h2d[k], cudaEventDisableTiming), "cudaEventCreate");
        CU_TRY(cudaEventCreateWithFlags(&h->ev_done[k], cudaEventDisableTiming), "cudaEventCreate");
        CU_TRY(cudaMalloc(&h->d_phase[k], frame_bytes * chunk), "cudaMalloc(frame chunk)");
    }
    h->host_ready = 1;
    return SHWFS_OK;
fail:
    return rc;   /* partial allocations are released by shwfs_destroy */
}

bool is_pinned(const void *p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeHost;
}

}  // namespace

static int measure_host_impl(shwfs_handle *h, const float *phase_host, int32_t T, float *slopes_host, bool wait)
{
    if (!h || T < 0) return SHWFS_EINVAL;
    if (T == 0) return SHWFS_OK;
    if (!phase_host || !slopes_host) return SHWFS_EINVAL;
    if ((long long)T * h->nsub > 0x7fffffffLL / 2) return SHWFS_EINVAL;
    int rc = SHWFS_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != h->device) cudaSetDevice(h->device);
    {
        rc = host_init(h);
        if (rc) goto fail;
        const int fps = frames_per_step(h);
        const int chunk_steps = h->chunk_frames / fps;          /* >= 1: chunk_frames >= SHWFS_MAX_LAYERS */
        const size_t frame_elems = (size_t)h->N * h->N * fps, frame_bytes = sizeof(float) * frame_elems;
        const size_t n_slopes = 2 * (size_t)T * h->nsub;
        if (h->d_slopes_cap < n_slopes) {
            cudaStreamSynchronize(h->st_comp);
            cudaFree(h->d_slopes); h->d_slopes = nullptr; h->d_slopes_cap = 0;
            CU_TRY(cudaMalloc(&h->d_slopes, sizeof(float) * n_slopes), "cudaMalloc(slopes)");
            h->d_slopes_cap = n_slopes;
        }
        const bool pinned_in = is_pinned(phase_host);
        if (!wait && !(pinned_in && is_pinned(slopes_host))) { rc = SHWFS_EINVAL; goto fail; }   /* async: pinned only */
        if (!pinned_in)
            for (int k = 0; k < 2; ++k)
                if (!h->h_pin[k]) CU_TRY(cudaHostAlloc(&h->h_pin[k], sizeof(float) * (size_t)h->N * h->N * h->chunk_frames, cudaHostAllocDefault), "cudaHostAlloc");
        int c = 0;
        for (int t0 = 0; t0 < T; t0 += chunk_steps, ++c) {
            const int k = c & 1;
            const int tc = (T - t0 < chunk_steps) ? T - t0 : chunk_steps;
            const float *src = phase_host + (size_t)t0 * frame_elems;
            if (!pinned_in) {
                CU_TRY(cudaEventSynchronize(h->ev_h2d[k]), "cudaEventSynchronize");   /* staging buffer free again */
                memcpy(h->h_pin[k], src, frame_bytes * tc);
                src = h->h_pin[k];
            }
            CU_TRY(cudaStreamWaitEvent(h->st_copy, h->ev_done[k], 0), "cudaStreamWaitEvent");
            if (h->n_runs > 0) {
                /* one strided 3-D copy per run: width x n rows x (frames of the chunk); the rest of the frame
                 * (outside the pupil, central obstruction) never crosses the bus */
                cudaMemcpy3DParms p;
                memset(&p, 0, sizeof(p));
                p.srcPtr = make_cudaPitchedPtr((void *)src, sizeof(float) * (size_t)h->N, (size_t)h->N, (size_t)h->N);
                p.dstPtr = make_cudaPitchedPtr((void *)h->d_phase[k], sizeof(float) * (size_t)h->N, (size_t)h->N, (size_t)h->N);
                p.kind = cudaMemcpyHostToDevice;
                for (int q = 0; q < h->n_runs; ++q) {
                    const int sy = h->h_runs[4 * q], rows = h->h_runs[4 * q + 1], x0 = h->h_runs[4 * q + 2], w = h->h_runs[4 * q + 3];
                    p.srcPos = make_cudaPos(sizeof(float) * (size_t)x0, (size_t)sy * h->n, 0);
                    p.dstPos = p.srcPos;
                    p.extent = make_cudaExtent(sizeof(float) * (size_t)w, (size_t)rows * h->n, (size_t)tc * fps);
                    CU_TRY(cudaMemcpy3DAsync(&p, h->st_copy), "cudaMemcpy3DAsync(H2D)");
                }
            } else {
                CU_TRY(cudaMemcpyAsync(h->d_phase[k], src, frame_bytes * tc, cudaMemcpyHostToDevice, h->st_copy), "cudaMemcpyAsync(H2D)");
            }
            CU_TRY(cudaEventRecord(h->ev_h2d[k], h->st_copy), "cudaEventRecord");
            CU_TRY(cudaStreamWaitEvent(h->st_comp, h->ev_h2d[k], 0), "cudaStreamWaitEvent");
            /* the chunks are parts of one call of T frames: same kernel instance for all */
            rc = run_path(h, h->d_phase[k], tc, T, h->d_slopes + 2 * (size_t)t0 * h->nsub, -1, nullptr, (unsigned)t0, h->st_comp);
            if (rc) goto fail;
            CU_TRY(cudaEventRecord(h->ev_done[k], h->st_comp), "cudaEventRecord");
        }
        CU_TRY(cudaMemcpyAsync(slopes_host, h->d_slopes, sizeof(float) * n_slopes, cudaMemcpyDeviceToHost, h->st_comp), "cudaMemcpyAsync(D2H)");
        if (wait) CU_TRY(cudaStreamSynchronize(h->st_comp), "cudaStreamSynchronize");
    }
fail:
    if (rc && h->st_comp) { cudaStreamSynchronize(h->st_comp); cudaStreamSynchronize(h->st_copy); }
    if (prev >= 0 && prev != h->device) cudaSetDevice(prev);
    return rc;
}

extern "C" int shwfs_measure_host(shwfs_handle *h, const float *phase_host, int32_t T, float *slopes_host)
{
    return measure_host_impl(h, phase_host, T, slopes_host, true);
}

extern "C" int shwfs_measure_host_async(shwfs_handle *h, const float *phase_host, int32_t T, float *slopes_host)
{
    return measure_host_impl(h, phase_host, T, slopes_host, false);
}

extern "C" int shwfs_host_wait(shwfs_handle *h)
{
    if (!h) return SHWFS_EINVAL;
    if (!h->st_comp) return SHWFS_OK;
    cudaError_t e = cudaStreamSynchronize(h->st_comp);
    if (e != cudaSuccess) { shwfs_note_cuda_error(e, "shwfs_host_wait"); return SHWFS_ECUDA; }
    return SHWFS_OK;
}
