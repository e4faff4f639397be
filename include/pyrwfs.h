/*
 * pyrwfs.h -- C ABI of the B200-native pyramid wavefront sensor, exported by the same
 * library as include/shwfs.h (libshwfs.so) with the same conventions: every function returns 0 or a negative
 * SHWFS_E* code (shwfs_strerror / shwfs_last_cuda_error apply), nothing throws or exits, "HOST"/"DEVICE" say
 * where a pointer lives, pyrwfs_measure only enqueues work on the caller's stream (and, like shwfs_measure,
 * must be called with the handle's device current: SHWFS_EINVAL otherwise).
 *
 * The operation is the pyramid sensor module of PAPER.md:92 (section 4): "We follow the scheme presented in
 * (Verinaud 2004) [...] This module makes a large use of the GPU computing power for the whole computation
 * including matrix-matrix complex array multiplications, Fast Fourier Transform and other operations on
 * arrays", with the circular modulation of PAPER.md:96 ("a modulated (3 lambda/D) pyramid").  The paper gives
 * no formula; the steps are the Fourier-optics model of that reference (readings D1..D7).
 *
 * Per frame t (pupil N x N in the corner of an Np x Np grid, K modulation points th_k = 2 pi (k + 1/2) / K):
 *   Q1 field     e_k[y,x] = a[y,x] exp(i (phase_to_rad * phase[t,y,x] + 2 pi r_mod (x cos th_k + y sin th_k) / D_pix))
 *   Q2 focal     F_k = DFT2(e_k)                                  (forward, exp(-2 pi i ...), Np x Np)
 *   Q3 pyramid   F_k *= exp(-2 pi i s (|u~| + |v~|) / Np),  u~ = signed frequency index
 *   Q4 pupil     G_k = IDFT2(F_k) / Np^2,  I_k = |G_k|^2
 *   Q5 modulate  I = (1/K) sum_k I_k
 *   Q6 quadrants Q[a][b][y,x] = I[(y + a s) mod Np, (x + b s) mod Np], a, b = +1 (index 0), -1 (index 1),
 *                binned by bp x bp block sums to Sp x Sp detector pixels (N = Sp * bp)
 *   Q7 signals   over the valid detector pixels i = (Y,X) (mean pupil amplitude over the block >= min_illum,
 *                row-major):  I0 = mean_i (Q++ + Q+- + Q-+ + Q--),
 *                s_x[i] = (Q[+][+] + Q[-][+] - Q[+][-] - Q[-][-]) / I0,  s_y[i] likewise with a.
 *                A phase growing with x gives s_x > 0.
 * All device arithmetic is fp32; the transforms are hand-written four-step FFTs (csrc/pyramid.cu).
 */
#ifndef PYRWFS_H_
#define PYRWFS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pyrwfs_handle pyrwfs_handle;            /* opaque */

typedef struct {
  int32_t n_pupil;          /* N : phase frames are N x N, row-major, x fastest; N % bin == 0             */
  const float *amplitude;   /* HOST [N*N] pupil amplitude mask; copied                                     */
  float   min_illum;        /* detector pixel valid if mean(amplitude over its block) >= min_illum         */
  int32_t pad;              /* Np: 256 or 1024 (= R*R, R = 16 or 32); N <= Np/2                            */
  int32_t separation;       /* s : pixels between the pupil and each of its four copies; s >= N/2 and      */
                            /*     s + N <= Np - s (the copies neither overlap nor wrap onto one another)  */
  int32_t bin;              /* bp: pupil pixels per detector pixel side                                    */
  float   mod_radius;       /* r_mod in lambda/D (0: no modulation)                                        */
  int32_t mod_points;       /* K >= 0 (0: no modulation); K is used as given                               */
  float   pupil_diameter_px;/* D_pix > 0: pupil diameter in pixels (sets lambda/D)                         */
  float   phase_to_rad;     /* multiplies the input to give radians at the sensing wavelength              */
} pyrwfs_config;

/* Errors: EINVAL (null pointers, sizes violating the constraints above, no valid pixel), EUNSUPPORTED (pad not
 * 256 or 1024), ENOMEM, ECUDA.  *out untouched on failure.                                                */
int pyrwfs_create(const pyrwfs_config *cfg, pyrwfs_handle **out);
int pyrwfs_destroy(pyrwfs_handle *h);                     /* NULL is a no-op returning 0 */

int pyrwfs_num_pixels(const pyrwfs_handle *h, int32_t *nvalid);
int pyrwfs_valid_list(const pyrwfs_handle *h, int32_t *yx_host /* HOST [nvalid*2] (Y,X) */);
int pyrwfs_launch_count(const pyrwfs_handle *h, int64_t *count);

/* phase_dev DEVICE [T*N*N] fp32 -> signals_dev DEVICE [T*nvalid*2] fp32 ([.][0] = s_x, [.][1] = s_y).
 * Frames are processed in chunks through scratch owned by the handle (sized at create: no allocation here).
 * T == 0 is a no-op.  Errors: EINVAL, ECUDA.                                                              */
int pyrwfs_measure(pyrwfs_handle *h, const float *phase_dev, int32_t T, float *signals_dev, void *cuda_stream);

/* Parity aid: the binned quadrant images Q, DEVICE out [T*2*2*Sp*Sp] (index order [t][a][b][Y][X]). */
int pyrwfs_debug_quadrants(pyrwfs_handle *h, const float *phase_dev, int32_t T, float *out_dev, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PYRWFS_H_ */
