/*
 * internal.h -- private declarations shared by the translation units of libshwfs.so.
 * Not part of the ABI (include/shwfs.h is) and never included by anything under oracle/.
 *
 * Notation follows SURVEY.md section 8 / DESIGN.md: N pupil side, S subapertures per side, n phase
 * pixels per subaperture side, P padded FFT side, b binning, D = P/b detector side, nsub valid
 * subapertures, T frames.
 */
#ifndef SHWFS_INTERNAL_H_
#define SHWFS_INTERNAL_H_

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/shwfs.h"

#define SHWFS_PATCH_LIT (1 << 30)

struct shwfs_handle {
    /* geometry */
    int N, S, n, P, b, D, nsub;
    float dx, lambda_m, tau, c_phi;
    int mode;              /* threshold mode */
    int device;
    int has_kernels;
    int algo;              /* resolved SHWFS_ALGO_* used by shwfs_measure */
    int algo_explicit;     /* 1: chosen by shwfs_set_algorithm (non-AUTO): no per-call choice between instances */
    int sms;               /* multiprocessors of `device` (grid sizing, per-call instance choice)              */
    int dm_fp32;           /* SHWFS_DM_FP32 was set when shwfs_set_dm ran: keep the FP32 SIMT GEMM for batches    */
    int64_t launches;
    const char *last_kernel;   /* name of the sensor kernel instance of the most recent launch (static storage) */

    /* device tables (owned) */
    float  *d_amp;         /* [N*N] amplitude mask                                             */
    int2   *d_valid;       /* [nsub] (x = sy, y = sx)                                          */
    int2   *d_patch;       /* [nsub] (x = sx*n | SHWFS_PATCH_LIT, y = sy*n): patch origin in pixels; the flag says
                              every amplitude of the patch is exactly 1 (the kernel then reads no amplitude) */
    int    *d_sched;       /* [2] chunk counters of the persistent kernels' dynamic sweep (sweep.cuh), zero between launches */
    int     force_persistent; /* SHWFS_FORCE_PERSISTENT was set at create: the persistent TMA instances whatever the call size
                                 (sanitizer runs on small inputs, tests/sanitizer_workloads.py) */
    int     no_tma;        /* SHWFS_NO_TMA was set at create: register-gather instances only (A/B runs)   */
    float  *d_kernels;     /* [nsub*P*P] spatial elongation kernels (kept for lazy tables)     */
    float2 *d_wk_table;    /* lag-domain table M: [nsub][2n-1][n] (or [1][2n-1][n] w/o kernels) */
    int     wk_table_stride; /* elements between subapertures: n*(2n-1), or 0 when shared      */
    float2 *d_khat;        /* literal chain: DFT of the re-centred kernel, [nsub][P][P]; lazy  */

    /* paper's full LGS model (shwfs_set_sodium / shwfs_set_noise); sod_L == 0: plain single-layer sensor */
    int     sod_L, sod_shared;
    float   sod_q[SHWFS_MAX_LAYERS];    /* a_l dx^2 / 2pi, turns/pixel^2 */
    float   sod_sw[SHWFS_MAX_LAYERS];   /* sqrt(w_l) */
    float2 *d_sod_g;                    /* [L][nsub] (2 a_l (r_i - r_c) + g_l) dx / 2pi, turns/pixel */
    float   nz_flux, nz_ron;
    int     nz_model;                   /* shwfs_noise.photon_model */
    uint64_t nz_seed;
    uint32_t nz_first_frame;

    /* closed-loop neighbours (shwfs_set_dm ...): modes re-laid per subaperture, padded coefficient buffers */
    float  *d_dm_modes;                 /* [nsub][M][n*n] modes re-laid per subaperture */
    int     dm_M;
    float  *d_um_modes;                 /* tensor-core operand B: split (hi|lo) canonical tiles, dm_umma.cu; or null */
    float  *d_um_coef;                  /* tensor-core operand A of the current call (split coefficient tiles)       */
    size_t  um_coef_cap;                /* floats */
    int     um_nkb;                     /* k-blocks of 16 modes */
    float  *d_dm_patch;                 /* [cap_T][nsub][n*n] DM phase of the current call, patch layout */
    size_t  dm_patch_cap;               /* floats */

    /* host copies for queries */
    int32_t *h_valid;      /* [nsub*2] (sy,sx) */

    /* shwfs_measure_host staging (lazy) */
    float *h_pin[2];       /* pinned staging for pageable callers */
    float *d_phase[2];     /* device frame chunks */
    float *d_slopes;       /* device slopes for the whole call, grown on demand */
    size_t d_slopes_cap;   /* floats */
    /* bands of lenslet rows with one bounding column extent of their valid subapertures: the host pipeline
     * copies only these (H1 never reads anything else).  band = {first lenslet row, rows, first column,
     * width in pixels}; n_runs == 0: copy whole frames.                                                */
    int   *h_runs;
    int    n_runs;
    long long run_pixels;  /* pixels per frame covered by the runs */
    int    chunk_frames;
    cudaStream_t st_copy, st_comp;
    cudaEvent_t ev_h2d[2], ev_done[2];
    int host_ready;
};

/* ---- launchers: each enqueues on `st` and returns the CUDA status of the launch ---------------- */

/* Lag-domain table M, built once at create in float64 on the device. */
cudaError_t shwfs_wk_build_table(shwfs_handle *h, cudaStream_t st);

/* Wiener-Khinchin path: slopes (and optionally the binned image B, [T*nsub*D*D]).  call_T = frames of the
 * whole API call this launch is a part of (== T unless the host pipeline feeds the call in chunks): the
 * per-call choice between kernel instances is made on it, so every chunk of one call takes the same instance. */
cudaError_t shwfs_wk_launch(shwfs_handle *h, const float *phase, int T, int call_T, float *slopes,
                            float *binned_or_null, float *noisy_or_null, unsigned t_base,
                            const float *dm_patch_or_null, int generic, cudaStream_t st);

/* loop.cu: closed-loop neighbours */
cudaError_t shwfs_loop_relayout_modes(shwfs_handle *h, const float *modes_dev, int M, cudaStream_t st);
/* dm_umma.cu: the DM-phase GEMM on tcgen05 (3xTF32) */
int shwfs_umma_np(const shwfs_handle *h);                         /* padded n*n, 0 if the size has no instance */
size_t shwfs_umma_modes_floats(const shwfs_handle *h, int M);
size_t shwfs_umma_coef_floats(int T, int M);
cudaError_t shwfs_umma_build_modes(shwfs_handle *h, cudaStream_t st);
cudaError_t shwfs_umma_dm_phase(shwfs_handle *h, const float *coef, int ldc, int T, float *out, cudaStream_t st);

cudaError_t shwfs_loop_dm_phase(shwfs_handle *h, const float *coef, int ldc, int T, float *out, cudaStream_t st);
cudaError_t shwfs_loop_reconstruct(const float *R, const float *slopes, int T, int K, int M, float gain,
                                   float *coef, int ldc, float *hist_or_null, cudaStream_t st);
int shwfs_wk_supported(const shwfs_handle *h, int generic);
int shwfs_wk_fft_supported(const shwfs_handle *h);   /* wk_fft.cu: autocorrelation by FFT (n = 16) */

/* Literal chain: P x P FFT(s) in shared memory/registers.  stage < 0: slopes only.
 * stage 0/1/2 also writes that image to `img`.                                              */
cudaError_t shwfs_literal_launch(shwfs_handle *h, const float *phase, int T, float *slopes,
                                 int stage, float *img, cudaStream_t st);
cudaError_t shwfs_literal_build_khat(shwfs_handle *h, cudaStream_t st);
int shwfs_literal_supported(const shwfs_handle *h);

/* Pruned-FFT path (no elongation kernels, D = 16): slopes and optionally the binned image */
cudaError_t shwfs_pruned_fft_launch(shwfs_handle *h, const float *phase, int T, float *slopes,
                                    float *binned_or_null, cudaStream_t st);
int shwfs_pruned_fft_supported(const shwfs_handle *h);

void shwfs_note_cuda_error(cudaError_t e, const char *where);

/* cudaFuncSetAttribute is per device: a launcher keeps one of these per kernel instance and sets the
 * attribute the first time it runs on each device (a handle's calls arrive with h->device current).  */
struct shwfs_once_per_device {
    bool done[64];
    /* true if `set` still has to run on the current device; mark() after it succeeded */
    bool pending(int *dev_out)
    {
        int dev = 0;
        cudaGetDevice(&dev);
        *dev_out = dev;
        return dev < 0 || dev >= 64 || !done[dev];
    }
    void mark(int dev) { if (dev >= 0 && dev < 64) done[dev] = true; }
};

#endif /* SHWFS_INTERNAL_H_ */
