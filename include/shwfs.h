/*
 * shwfs.h -- C ABI of the B200-native Shack-Hartmann wavefront-sensor hot path.
 *
 * The operation is the LGS/NGS Shack-Hartmann sensor module of PAPER.md:91 (section 4):
 *   "The WF is split into sub-apertures and the spot computed by FFT for each sensor sub-aperture.
 *    [...] We consider the physical extension of the projection of the laser on the sodium layer
 *    through a convolution for a gaussian of the desired properties. [...] the centroid computed on
 *    the final [...] image to retrieve the slopes."
 * and its output is the "X- and Y- slopes" vector of PAPER.md:76.  The call set follows
 * BASELINE.json:north_star: shwfs_create(geometry, lambda, pad, binning, elongation kernels),
 * shwfs_measure(phase[T,N,N] fp32 device ptr -> slopes[T,nsub,2], stream), shwfs_destroy.
 * The paper gives no formula; the conventions (steps H1..H8, readings A1..A15) are those of
 * SURVEY.md section 8 and DESIGN.md sections 2-4.
 *
 * Per (frame t, valid subaperture i):
 *   H1 gather   p[j,k] = phase[t, sy*n+j, sx*n+k],  a[j,k] = amplitude[sy*n+j, sx*n+k]
 *   H2 field    e[j,k] = a * exp(i*(phase_to_rad*p - pi*(j+k)/P)), zero padded to P x P
 *   H3 DFT      E[v,u] = sum e[j,k] exp(-2*pi*i*(v*j+u*k)/P)
 *   H4          I = |E|^2 / P^2
 *   H5          C = I (*) K_i, circular on P x P, kernel centre at (P/2,P/2)   (only if kernels given)
 *   H6 centre   Sh[r,c] = C[(r-P/2) mod P, (c-P/2) mod P];  bin  B[R,C] = sum of b x b blocks
 *   H7          m = max B;  Wt = max(B - tau*m, 0)  (mode 0)  |  B*[B >= tau*m]  (mode 1)
 *   H8          slope_x = sum Wt*(C-(D-1)/2) / sum Wt,  slope_y with R;  sum Wt == 0 -> (0,0)
 * All arithmetic is fp32 on the device.  How the library reaches that result (lag-domain form,
 * pruned transforms) is an implementation matter: DESIGN.md section 6.
 *
 * Conventions
 *   - Every function returns 0 (SHWFS_OK) or a negative error code; nothing throws, aborts or exits;
 *     output arguments are untouched on failure.
 *   - "HOST" pointers are ordinary host memory, "DEVICE" pointers are CUDA device memory of the
 *     device that was current at shwfs_create.  shwfs_create copies every HOST array it is given.
 *   - shwfs_measure only enqueues work on `cuda_stream` (a cudaStream_t passed as void*, NULL = default
 *     stream): no allocation, no synchronisation, no host<->device copy.  Results are valid once the
 *     caller has synchronised that stream.  (shwfs_debug_spots, a test hook, may allocate its scratch and
 *     synchronise the stream the first time it is called, see there.)
 *   - The enqueue-only calls (shwfs_measure, _measure_residual, _reconstruct, _closed_loop, _debug_spots)
 *     must be made with the handle's device current (the one that was current at shwfs_create) and return
 *     SHWFS_EINVAL otherwise; the other calls switch to it and back themselves.
 *   - A handle is not thread-safe; distinct handles are independent (one handle = one WFS).  Calls on ONE handle
 *     must also not overlap on the GPU: enqueue them on one stream, or order the streams with events.  The handle
 *     owns device state that a call uses while it runs (the chunk counter from which the persistent kernels are
 *     dealt their spots, the DM-phase scratch of shwfs_measure_residual); two calls of one handle running at the
 *     same time on different streams would share it.  Different handles may run concurrently (bench.py runs the six
 *     LGS sensors that way).
 */
#ifndef SHWFS_H_
#define SHWFS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SHWFS_OK            0
#define SHWFS_EINVAL       (-1)  /* null pointer, inconsistent sizes, T < 0, no valid subaperture      */
#define SHWFS_EUNSUPPORTED (-2)  /* sizes are consistent but no kernel instance covers them            */
#define SHWFS_ENOMEM       (-3)  /* host or device allocation failed                                   */
#define SHWFS_ECUDA        (-4)  /* a CUDA call failed; shwfs_last_cuda_error gives the CUDA text      */

/* Algorithms.  Both give the H1..H8 result to fp32 rounding. */
#define SHWFS_ALGO_AUTO     0    /* the fastest instance for the handle's sizes (default)              */
                                 /* (for n = 8, 10 also per call: calls of under ~64 spots per SM, i.e.  */
                                 /* the one-frame closed-loop step, take the SHWFS_ALGO_WK_FFT instance) */
#define SHWFS_ALGO_LITERAL  1    /* P x P shared-memory FFT chain, exactly the H3..H6 order             */
#define SHWFS_ALGO_WK       2    /* Wiener-Khinchin lag-domain form: autocorrelation of the field, x   */
                                 /* precomputed (kernel MTF x bin x centre) table, D x D real transform */
#define SHWFS_ALGO_WK_GENERIC 3  /* same form, size-generic unspecialised kernel                       */
#define SHWFS_ALGO_PRUNED_FFT 4  /* no elongation kernels, D = 16: one input-pruned P x P FFT per spot,   */
                                 /* half-warp per spot, bin + threshold + CoG in registers             */
#define SHWFS_ALGO_WK_FFT   5    /* the lag-domain form with the field's autocorrelation taken by FFT on  */
                                 /* a 32 x 32 grid instead of by direct sums (n = 12, 14, 16; D = 16)    */

#define SHWFS_MAX_LAYERS 8        /* sodium sub-layers per LGS ("1 to 5 typically")            */

typedef struct shwfs_handle shwfs_handle;              /* opaque */

typedef struct {
  int32_t n_pupil;          /* N  : phase frames are N x N, row-major, x (columns) fastest             */
  int32_t n_sub_side;       /* S  : S x S lenslet grid, S * n_pix == N                                 */
  int32_t n_pix;            /* n  : phase pixels per subaperture side                                  */
  float   pixel_size_m;     /* dx : metres per pupil pixel (> 0; only used by shwfs_pixel_scale)       */
  const float   *amplitude; /* HOST [N*N] pupil amplitude mask (any finite values, normally 0..1)      */
  float   min_illum;        /* subaperture valid if mean(amplitude over its patch) >= min_illum        */
  const int32_t *valid_yx;  /* optional HOST [n_valid*2] explicit (sy,sx) list; overrides the rule     */
  int32_t n_valid;          /* length of valid_yx (ignored when valid_yx is NULL)                      */
  float   threshold_frac;   /* tau in [0,1): fraction of the per-spot peak; 0 = plain CoG              */
  int32_t threshold_mode;   /* 0 = subtract-and-clip (default), 1 = hard mask                          */
  float   phase_to_rad;     /* c_phi: multiplies the input to give radians at lambda (1 if already)    */
} shwfs_geometry;

/* Build one WFS.  lambda_m > 0; pad = P (power of two, n <= P <= 64); bin = b (b | P, (P/2) % b == 0).
 * elong_kernels: HOST [nsub*P*P] fp32 spatial kernels at unbinned resolution, centre at (P/2,P/2),
 * index order of the valid list, used as given (no renormalisation) -- or NULL for no elongation (H5
 * skipped).  The valid list is row-major over (sy,sx) (sy outer).  On success *out receives the handle.
 * Errors: EINVAL (null g/out/amplitude, N != S*n, bad P/b/lambda/dx/tau/mode, valid_yx entry out of range
 * or n_valid <= 0, no valid subaperture), EUNSUPPORTED (n > 32 or P/b > 32), ENOMEM, ECUDA.             */
int shwfs_create(const shwfs_geometry *g, float lambda_m, int32_t pad, int32_t bin,
                 const float *elong_kernels, shwfs_handle **out);

/* phase_dev: DEVICE [T*N*N] fp32 (16-byte aligned); slopes_dev: DEVICE [T*nsub*2] fp32,
 * slopes[t][i][0] = x-slope, [1] = y-slope, in binned detector pixels about the detector centre;
 * i indexes the valid list.  Positive x-slope <=> phase increasing with x (the column index).
 * T == 0 is a successful no-op.  Non-finite phase values are not checked: they reach only that spot's
 * slopes.  Errors: EINVAL (null h, null pointers with T > 0, T < 0, phase_dev not 16-byte aligned, another
 * device current), ECUDA (launch failure).                                                               */
int shwfs_measure(shwfs_handle *h, const float *phase_dev, int32_t T, float *slopes_dev,
                  void *cuda_stream);

/* Same measurement from HOST buffers: phase_host [T*N*N] -> slopes_host [T*nsub*2].  The library copies
 * in frame chunks through its own pinned staging buffers and device scratch (allocated on first use,
 * owned by the handle), overlaps copies with compute on two internal streams, and returns after the
 * slopes have landed in slopes_host.  This is the end-to-end entry point timed as "e2e" by bench.py.   */
int shwfs_measure_host(shwfs_handle *h, const float *phase_host, int32_t T, float *slopes_host);

/* The same, returning once everything is enqueued on the handle's own streams: both buffers must be pinned host
 * memory (EINVAL otherwise) and stay untouched until shwfs_host_wait(h) returns.  Several handles (the six LGS
 * sensors of a system) can so keep the bus busy back to back.  One call in flight per handle.            */
int shwfs_measure_host_async(shwfs_handle *h, const float *phase_host, int32_t T, float *slopes_host);
int shwfs_host_wait(shwfs_handle *h);

/* Bytes of one N x N wavefront that shwfs_measure_host actually moves to the device: only the bounding column
 * extent of the valid subapertures of each lenslet row is copied (strided 3-D copies, rows of equal extent
 * merged) when that saves at least a tenth of the frame; the rest is never read by H1.                  */
int shwfs_host_bytes_per_frame(const shwfs_handle *h, int64_t *bytes);

/* Frees everything the handle owns.  shwfs_destroy(NULL) returns 0. */
int shwfs_destroy(shwfs_handle *h);

/* ---- queries ---------------------------------------------------------------------------------- */
int shwfs_num_subaps(const shwfs_handle *h, int32_t *nsub);
int shwfs_valid_list(const shwfs_handle *h, int32_t *yx_host /* HOST [nsub*2] */);
/* radians of wavefront tilt angle per binned detector pixel: b * lambda / (P * dx) */
int shwfs_pixel_scale(const shwfs_handle *h, double *rad_per_detector_px);

/* Select the algorithm used by shwfs_measure (SHWFS_ALGO_*).  EUNSUPPORTED if that algorithm has no
 * instance for the handle's sizes.  shwfs_get_algorithm reports the resolved (never AUTO) choice.    */
int shwfs_set_algorithm(shwfs_handle *h, int32_t algo);
int shwfs_get_algorithm(const shwfs_handle *h, int32_t *algo);

/* Number of kernels this handle has launched since shwfs_create (bench.py's gpu_launches). */
int shwfs_launch_count(const shwfs_handle *h, int64_t *count);

/* Name of the sensor kernel instance that the handle's most recent measurement launched, e.g.
 * "wk_measure_kernel<10,0,0>" (n, threshold mode, extension kind) or "wkf_kernel<16,0,0,tma>": under
 * SHWFS_ALGO_AUTO the instance is chosen per call (size of the call, alignment of the frames), so the
 * algorithm id alone does not say what ran.  Copies at most len - 1 characters into name (HOST) and
 * terminates it; "" before the first launch.  Errors: EINVAL.                                          */
int shwfs_last_kernel(const shwfs_handle *h, char *name, int32_t len);

/* ---- the paper's full LGS model ------------------------
 * "In the code a laser guide star WF is the results of different, 1 to 5 typically, projections of the beam
 *  on as many sub-layers of the sodium layer [...] For each sub-layer the proper phase shift in Tip Tilt and
 *  Defocus is considered and the spot array multiplied by the corresponding value of the sodium thickness
 *  level profile. [...] Finally the sub-layer arrays are piled-up and the centroid computed on the final
 *  noise-added image to retrieve the slopes."
 * With a sodium model set, H2..H4 run once per sub-layer l on the pupil phase
 *      phase_to_rad * phase_l(r) + defocus[l] * |r - r_c|^2 + tilt[l] . r        (r = pixel centre, metres
 *      from the pupil centre, x = (column + 1/2 - N/2) * dx),
 * the intensities are summed with weights weight[l] >= 0, then H5 (one Gaussian per subaperture), H6, the
 * optional noise, H7 and H8 follow.  A source at altitude h_l seen by a sensor conjugated to h_0 from a
 * launch telescope at r_c has defocus[l] = (pi / lambda) (1/h_0 - 1/h_l).  Requires the lag-domain
 * algorithm (EUNSUPPORTED if the handle's sizes have no such instance); selects it if needed.          */
typedef struct {
  int32_t n_layers;         /* L in [1, SHWFS_MAX_LAYERS]                                             */
  int32_t shared_phase;     /* 0: shwfs_measure reads phase as [T,L,N,N]; 1: [T,N,N] shared by all l  */
  const float *weight;      /* HOST [L] sodium profile value w_l >= 0, used as given                  */
  const float *defocus;     /* HOST [L] a_l, rad / m^2                                                */
  const float *tilt_x;      /* HOST [L] rad / m, or NULL for zeros (uplink tip-tilt)                  */
  const float *tilt_y;      /* HOST [L] rad / m, or NULL                                              */
  float centre_x_m;         /* r_c: centre of the quadratic (launch telescope), metres from the       */
  float centre_y_m;         /*      pupil centre                                                      */
} shwfs_sodium;
/* s == NULL returns to the single-layer sensor.  Arrays are copied.  Errors: EINVAL, EUNSUPPORTED, ENOMEM. */
int shwfs_set_sodium(shwfs_handle *h, const shwfs_sodium *s);

/* Detector noise on the binned image B before H7.  photon_model 0 (reading B4):
 *      counts = flux * B + sqrt(max(flux * B, 0) + read_noise^2) * z,   z ~ N(0,1)
 * (photon noise in its Gaussian limit plus read noise), z from Philox4x32-10 with key = seed and counter =
 * (p/4, i, first_frame + t, 0), p = C*D + R the column-major pixel index, Box-Muller on the output pairs
 * (csrc/noise.cuh).  photon_model 1 (reading B4'): true photon statistics,
 *      counts = k + read_noise * z,   k ~ Poisson(max(flux * B, 0)),
 * k drawn from the uniforms of the blocks with counter = (p/2, i, first_frame + t, 1 + attempt) by inversion for
 * rates under 30 and by the transformed-rejection method PTRS (Hoermann 1993) above; z as in model 0.
 * flux = photo-electrons per unit of B (a fully lit subaperture of unit amplitude and
 * unit weights has sum B = n^2 sum K).  nz == NULL or flux <= 0 switches the noise off.  first_frame lets
 * successive calls continue one noise stream.  Requires the lag-domain algorithm, as shwfs_set_sodium.
 * Errors: EINVAL (negative or non-finite read_noise, photon_model not 0 or 1), EUNSUPPORTED.                 */
typedef struct {
  float    flux;
  float    read_noise;      /* electrons rms, >= 0 */
  uint64_t seed;
  uint32_t first_frame;
  int32_t  photon_model;    /* 0: Gaussian limit of the photon noise; 1: Poisson counts */
} shwfs_noise;
int shwfs_set_noise(shwfs_handle *h, const shwfs_noise *nz);

/* ---- closed-loop neighbours of the path -------------------------
 * "The WFS modules compute the vector signals (X-and Y- slopes) from the residual phase (the open loop
 *  wavefront subtracted by the DM).  Vector slopes multiplied by the control matrix returns the vector
 *  coefficients for the modal base linear composition, in the form of the differential coefficients to be
 *  added to the one defining the existing mirror shape. [...] a pure integrator scheme".
 * DM phase of frame t = sum_m coef[t][m] * modes[m] (units of the wavefront input); residual = wavefront - DM.
 * Requires the lag-domain algorithm (EUNSUPPORTED otherwise), like shwfs_set_sodium; with sub-layers the
 * same DM phase is subtracted from every sub-layer's wavefront.
 *
 * shwfs_set_dm: modes_dev DEVICE [M*N*N] fp32; the library keeps its own per-subaperture re-layouts (nsub * M *
 * n*n floats for the frame-by-frame loop, and -- for n*n in {64, 100, 256} -- about 2.3x that as hi|lo TF32
 * operand tiles of the tcgen05 GEMM that serves batches of more than 8 frames) and does not reference modes_dev
 * after the call returns (it synchronises).
 * M == 0 or modes_dev == NULL drops the DM.  Errors: EINVAL, EUNSUPPORTED, ENOMEM, ECUDA.               */
int shwfs_set_dm(shwfs_handle *h, const float *modes_dev, int32_t M);

/* shwfs_measure on the residual phase: coef_dev DEVICE [T*M].  Two kernels: the DM phase on the valid
 * subapertures (a batched GEMM into a T*nsub*n*n scratch in patch layout: tensor cores with a 3-term TF32 split,
 * fp32-like accuracy, for T > 8; an fp32 matrix-vector kernel below), then the sensor kernel, whose
 * gather subtracts it: the full-frame residual is never written to memory.  Enqueues on cuda_stream; may
 * (re)allocate the scratch the first time a larger T is seen (that call synchronises the stream once).
 * Errors: EINVAL (no DM set, null pointers, T < 0), ENOMEM, ECUDA.                                      */
int shwfs_measure_residual(shwfs_handle *h, const float *phase_dev, const float *coef_dev, int32_t T,
                           float *slopes_dev, void *cuda_stream);

/* coef[t][m] += gain * sum_k R[m][k] * slopes[t][k],  k = 2*i + axis  (the layout of slopes[t][i][:]).
 * R_dev DEVICE [M * 2*nsub] row-major, slopes_dev DEVICE [T*nsub*2], coef_dev DEVICE [T*M] in/out.
 * M is the count given to shwfs_set_dm.  Enqueues on cuda_stream.  Errors: EINVAL, ECUDA.               */
int shwfs_reconstruct(shwfs_handle *h, const float *R_dev, const float *slopes_dev, int32_t T, float gain,
                      float *coef_dev, void *cuda_stream);

/* T sequential frames of the pure-integrator loop, all enqueued on cuda_stream (three kernels per frame):
 *     s_t = slopes(phase[t] - DM(c_t));  hist[t] = c_t;  c_{t+1} = c_t + gain * R s_t
 * coef_dev DEVICE [M]: c_0 on entry, c_T on exit.  slopes_dev DEVICE [T*nsub*2].  coef_hist_dev DEVICE [T*M]
 * or NULL.  With a noise model, frame t uses counter first_frame + t.  Errors: EINVAL, ECUDA.           */
int shwfs_closed_loop(shwfs_handle *h, const float *phase_dev, const float *R_dev, float gain, float *coef_dev,
                      int32_t T, float *slopes_dev, float *coef_hist_dev, void *cuda_stream);

/* ---- debug (parity on images; not on the timed path) ------------------------------------------- */
/* Enqueues on cuda_stream like shwfs_measure, except that the first call (and a later call with a larger T,
 * and the first call of stage 0 or 1 on a handle with elongation kernels, which builds the literal chain's
 * transformed kernels) allocates handle-owned scratch and synchronises the stream once.
 * stage 0: centred intensity  roll(I)  DEVICE out [T*nsub*P*P]
 * stage 1: centred image after elongation  Sh  [T*nsub*P*P]  (== stage 0 without kernels)
 * stage 2: binned image B  [T*nsub*D*D], D = P/b -- produced by the handle's CURRENT algorithm, so it
 *          is the image the timed path thresholds; stages 0 and 1 exist only in the literal chain
 *          (single-layer sensor only).
 * stage 3: binned image after the detector noise  [T*nsub*D*D]  (== stage 2 when the noise is off).   */
int shwfs_debug_spots(shwfs_handle *h, const float *phase_dev, int32_t T, int32_t stage,
                      float *out_dev, void *cuda_stream);

const char *shwfs_strerror(int code);
/* Text of the last CUDA error seen by the calling thread's calls into the library ("" if none). */
const char *shwfs_last_cuda_error(void);
int shwfs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SHWFS_H_ */
