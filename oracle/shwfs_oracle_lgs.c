/*
 * shwfs_oracle_lgs.c -- float64 CPU oracle for the paper's full LGS Shack-Hartmann model
 * (SURVEY.md 8(f) rows f1 "sodium sub-layer sum" and f2 "detector noise before the centroid").
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT (same rules as shwfs_oracle.c, whose stage functions it calls:
 * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call it; nothing is shared with the CUDA library).
 *
 * Passage followed, PAPER.md:91 (section 4, "LGS Shack Hartmann wavefront sensor"), in its order:
 *   "We divided the sodium layer into different sub-layers.  The LGS wavefront sensor module has as input
 *    the WFs [...] for each sodium sub-layer and the directions and positions of the launching telescopes.
 *    [...] The WF is split into sub-apertures and the spot computed by FFT for each sensor sub-aperture.
 *    For each sub-layer the proper phase shift in Tip Tilt and Defocus is considered and the spot array
 *    multiplied by the corresponding value of the sodium thickness level profile.  [...] We consider the
 *    physical extension of the projection of the laser on the sodium layer through a convolution for a
 *    gaussian of the desired properties.  [...] Finally the sub-layer arrays are piled-up and the centroid
 *    computed on the final noise-added image to retrieve the slopes."
 * The paper gives no formula.  Readings (B1..B6):
 *   L1  per sub-layer l the pupil phase is  c_phi*phase_l(r) + a_l*|r - r_c|^2 + g_l . r   with r the pixel
 *       centre in metres from the pupil centre, r_c the centre of the quadratic (the launch telescope
 *       position: a source at altitude h_l seen by a sensor focused at h_0 has a_l = (pi/lambda)(1/h_0 -
 *       1/h_l)), g_l an extra uniform tilt (uplink tip-tilt); a_l [rad/m^2], g_l [rad/m] are inputs.
 *   L2  spot array I_l = |DFT(e_l)|^2 / P^2 (O2..O4 of shwfs_oracle.c), times the profile value w_l.
 *   L3  the sub-layer arrays are summed, THEN convolved with the subaperture's Gaussian (the convolution is
 *       linear, so this equals convolving each and summing), centred and binned (O5..O7).
 *   L4  noise on the binned image: counts = F*B + sqrt(max(F*B,0) + ron^2) * z, z ~ N(0,1): photon noise in
 *       its Gaussian limit plus read noise, one normal deviate per pixel (F = photo-electrons per unit of
 *       B, ron = read noise in electrons rms).  Continuous in B, so GPU/oracle parity is by tolerance.
 *   L5  z comes from the counter-based generator Philox4x32-10 (Salmon et al., SC'11): key = (seed lo,
 *       seed hi), counter = (p / 4, i, t, 0) with p = C*D + R the column-major pixel index, i the valid-list
 *       index, t the frame; the four 32-bit outputs x0..x3 give, by Box-Muller on (x0,x1) and (x2,x3)
 *       with u = ((x >> 9) + 0.5) * 2^-23, the deviates of pixels 4*(p/4) .. 4*(p/4)+3:
 *       z0 = rho1 cos(2 pi u1), z1 = rho1 sin(2 pi u1), z2 = rho2 cos(2 pi u3), z3 = rho2 sin(2 pi u3),
 *       rho1 = sqrt(-2 ln u0), rho2 = sqrt(-2 ln u2).
 *   L6  threshold + centre of gravity (O8, O9) on the noisy image.
 *   (photon_model = 1 replaces L4 by true Poisson counts plus read noise: steps N1..N5 of shwfs_oracle_poisson.c.)
 *
 * Pins (tests/test_oracle_lgs_pins.py, -m "not gpu"): J1 one layer with w=1, a=0, g=0 equals
 * shwfs_oracle_measure; J2 the binned image is the weighted sum of single-layer binned images; J3 a tilt
 * of 2*pi*m/P per pixel shifts the spot by m pixels exactly; J4 a defocus on a flat wavefront displaces
 * each spot by the local gradient 2 a (r_i - r_c) (closed form, linear range); J5 layers (+a,+g) and
 * (-a,-g) with equal weights on a flat wavefront give zero slopes; J6 Philox4x32-10 known-answer vectors
 * of the Random123 distribution; J7 the deviates are standard normal (moments, Kolmogorov-Smirnov) and
 * uncorrelated between pixels, spots and frames; J8 counts have mean F*B and variance F*B + ron^2;
 * J9 F -> infinity recovers the noise-free slopes.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* stage functions of shwfs_oracle.c (O3..O9) */
int shwfs_oracle_dft2(const double *in, double *out, int P, int sign);
void shwfs_oracle_intensity(const double *E, int P, double *I);
int shwfs_oracle_convolve_fft(const double *I, const float *K, int P, double *C);
void shwfs_oracle_centre(const double *C, int P, double *Sh);
void shwfs_oracle_bin(const double *Sh, int P, int b, double *B);
void shwfs_oracle_add_noise_poisson(const double *B, int D, double F, double ron, uint64_t seed, uint32_t t,
                                    uint32_t i, double *counts, double *margin_out);   /* shwfs_oracle_poisson.c */
void shwfs_oracle_threshold_cog(const double *B, int D, double tau, int mode, double *slope_xy);

/* ------------------------------------------------------------------ L1
 * Field of one sodium sub-layer on the P x P grid (patch in the corner):
 *   e[j,k] = a[j,k] * exp(i*(c_phi*p[j,k] + defocus*((x-cx)^2+(y-cy)^2) + tilt_x*x + tilt_y*y - pi*(j+k)/P))
 * with x = (sx*n + k + 1/2 - N/2)*dx, y = (sy*n + j + 1/2 - N/2)*dx (pixel centres, metres).          */
void shwfs_oracle_field_layer(const float *phase_frame, const float *amplitude, int N, int n, int P,
                              int sy, int sx, double c_phi, double dx, double defocus, double cx,
                              double cy, double tilt_x, double tilt_y, double *e /* [P*P*2] */)
{
    memset(e, 0, sizeof(double) * 2 * (size_t)P * P);
    for (int j = 0; j < n; ++j)
        for (int k = 0; k < n; ++k) {
            size_t src = (size_t)(sy * n + j) * N + (size_t)(sx * n + k);
            double x = ((double)(sx * n + k) + 0.5 - 0.5 * (double)N) * dx;
            double y = ((double)(sy * n + j) + 0.5 - 0.5 * (double)N) * dx;
            double th = c_phi * (double)phase_frame[src]
                      + defocus * ((x - cx) * (x - cx) + (y - cy) * (y - cy))
                      + tilt_x * x + tilt_y * y
                      - M_PI * (double)(j + k) / (double)P;
            double a = (double)amplitude[src];
            e[2 * (j * P + k) + 0] = a * cos(th);
            e[2 * (j * P + k) + 1] = a * sin(th);
        }
}

/* ------------------------------------------------------------------ L5
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11):
 * ten rounds of  (c0,c1,c2,c3) <- (hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0)),
 * the key bumped by the Weyl constants (W0, W1) between rounds.                                       */
void shwfs_oracle_philox4x32(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += W0; k1 += W1; }
        uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* u = ((x >> 9) + 1/2) * 2^-23 in (0,1): 23 bits, exactly representable in fp32 as well */
static double unit_open(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

/* The four standard-normal deviates of Philox block `blk` of spot (t, i): Box-Muller on (x0,x1), (x2,x3). */
void shwfs_oracle_normal4(uint64_t seed, uint32_t t, uint32_t i, uint32_t blk, double z[4])
{
    uint32_t ctr[4] = {blk, i, t, 0u}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, x[4];
    shwfs_oracle_philox4x32(ctr, key, x);
    double r1 = sqrt(-2.0 * log(unit_open(x[0]))), a1 = 2.0 * M_PI * unit_open(x[1]);
    double r2 = sqrt(-2.0 * log(unit_open(x[2]))), a2 = 2.0 * M_PI * unit_open(x[3]);
    z[0] = r1 * cos(a1); z[1] = r1 * sin(a1);
    z[2] = r2 * cos(a2); z[3] = r2 * sin(a2);
}

/* ------------------------------------------------------------------ L4
 * counts[R,C] = F*B[R,C] + sqrt(max(F*B[R,C],0) + ron^2) * z_p,  p = C*D + R (column-major), z_p the
 * (p mod 4)-th deviate of block p/4.  F <= 0 means "no noise": counts = B.                            */
void shwfs_oracle_add_noise(const double *B, int D, double F, double ron, uint64_t seed, uint32_t t,
                            uint32_t i, double *counts)
{
    if (!(F > 0.0)) { memcpy(counts, B, sizeof(double) * (size_t)D * D); return; }
    for (int C = 0; C < D; ++C)
        for (int R = 0; R < D; ++R) {
            uint32_t p = (uint32_t)(C * D + R);
            double z[4];
            shwfs_oracle_normal4(seed, t, i, p / 4u, z);
            double m = F * B[R * D + C];
            counts[R * D + C] = m + sqrt((m > 0.0 ? m : 0.0) + ron * ron) * z[p % 4u];
        }
}

/* ------------------------------------------------------------------ one spot, L1..L6
 * phase_layers[l] points at the N x N frame of sub-layer l (the same pointer L times when the sub-layers
 * share one wavefront).  Optional outputs: img2 = binned image before noise [D*D], img3 = after noise.  */
int shwfs_oracle_spot_lgs(const float *const *phase_layers, int L, const double *weight,
                          const double *defocus, const double *tilt_x, const double *tilt_y, double cx,
                          double cy, const float *amplitude, int N, int n, int P, int b, int sy, int sx,
                          double c_phi, double dx, double tau, int mode, const float *K, double F,
                          double ron, uint64_t seed, uint32_t t, uint32_t i, double *slope_xy,
                          double *img2, double *img3, int photon_model, double *margin3)
{
    size_t PP = (size_t)P * P;
    int D = P / b;
    double *e = (double *)malloc(sizeof(double) * 2 * PP);
    double *I = (double *)malloc(sizeof(double) * PP);
    double *S = (double *)calloc(PP, sizeof(double));
    double *C = (double *)malloc(sizeof(double) * PP);
    double *Sh = (double *)malloc(sizeof(double) * PP);
    double *B = (double *)malloc(sizeof(double) * (size_t)D * D);
    double *Bn = (double *)malloc(sizeof(double) * (size_t)D * D);
    int rc = (e && I && S && C && Sh && B && Bn) ? 0 : -1;
    for (int l = 0; l < L && !rc; ++l) {
        shwfs_oracle_field_layer(phase_layers[l], amplitude, N, n, P, sy, sx, c_phi, dx, defocus[l], cx, cy,
                                 tilt_x ? tilt_x[l] : 0.0, tilt_y ? tilt_y[l] : 0.0, e);          /* L1 */
        rc = shwfs_oracle_dft2(e, e, P, -1);
        if (rc) break;
        shwfs_oracle_intensity(e, P, I);                                                         /* L2 */
        for (size_t q = 0; q < PP; ++q) S[q] += weight[l] * I[q];                                 /* L3 */
    }
    if (!rc) {
        if (K) rc = shwfs_oracle_convolve_fft(S, K, P, C);
        else memcpy(C, S, sizeof(double) * PP);
    }
    if (!rc) {
        shwfs_oracle_centre(C, P, Sh);
        shwfs_oracle_bin(Sh, P, b, B);
        if (img2) memcpy(img2, B, sizeof(double) * (size_t)D * D);
        if (photon_model == 1) shwfs_oracle_add_noise_poisson(B, D, F, ron, seed, t, i, Bn, margin3);    /* N1..N5 */
        else shwfs_oracle_add_noise(B, D, F, ron, seed, t, i, Bn);                                /* L4, L5 */
        if (img3) memcpy(img3, Bn, sizeof(double) * (size_t)D * D);
        shwfs_oracle_threshold_cog(Bn, D, tau, mode, slope_xy);                                   /* L6 */
    }
    free(e); free(I); free(S); free(C); free(Sh); free(B); free(Bn);
    return rc;
}

/* ------------------------------------------------------------------ whole call
 * phase: [T,L,N,N] fp32 (shared_phase == 0) or [T,N,N] used by every sub-layer (shared_phase != 0).
 * stage: -1 none, 2 = binned image before noise, 3 = after noise ([T,nsub,D,D]).
 * Returns 0, -1 (no memory) or -2 (bad argument).                                                    */
int shwfs_oracle_measure_lgs(const float *phase, int T, int L, int shared_phase, int N, int n, int P, int b,
                             const float *amplitude, const int32_t *valid_yx, int nsub, double c_phi,
                             double dx, const double *weight, const double *defocus, const double *tilt_x,
                             const double *tilt_y, double cx, double cy, double tau, int mode,
                             const float *kernels, double F, double ron, uint64_t seed, double *slopes,
                             int stage, double *images, int nthreads, int photon_model, double *margins)
{
    if (!phase || !amplitude || !valid_yx || !slopes || !weight || !defocus || T < 0 || L < 1 || L > 64 ||
        n <= 0 || n > P || b <= 0 || P % b || N % n || (stage >= 0 && !images) || (stage >= 0 && stage < 2) ||
        stage > 3)
        return -2;
    int D = P / b;
    size_t img_sz = (size_t)D * D, fr = (size_t)N * N;
    long total = (long)T * nsub;
    int fail = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
    for (long w = 0; w < total; ++w) {
        int t = (int)(w / nsub), i = (int)(w % nsub);
        const float *layers[64];
        for (int l = 0; l < L; ++l)
            layers[l] = shared_phase ? phase + (size_t)t * fr : phase + ((size_t)t * L + l) * fr;
        double *im = (stage >= 0) ? images + (size_t)w * img_sz : NULL;
        double *mg = margins ? margins + (size_t)w * img_sz : NULL;      /* [T,nsub,D,D], photon_model 1 only */
        int rc = shwfs_oracle_spot_lgs(layers, L, weight, defocus, tilt_x, tilt_y, cx, cy, amplitude, N, n, P,
                                       b, valid_yx[2 * i], valid_yx[2 * i + 1], c_phi, dx, tau, mode,
                                       kernels ? kernels + (size_t)i * P * P : NULL, F, ron, seed,
                                       (uint32_t)t, (uint32_t)i, slopes + 2 * (size_t)w,
                                       stage == 2 ? im : NULL, stage == 3 ? im : NULL, photon_model, mg);
        if (rc) {
#pragma omp atomic write
            fail = 1;
        }
    }
    return fail ? -1 : 0;
}
