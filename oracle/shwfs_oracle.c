/*
 * shwfs_oracle.c -- float64 CPU oracle for the Shack-Hartmann WFS hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this
 * file.  It shares no code, header, table or constant with the CUDA library
 * under paper_1408_0698_b200/csrc/ and neither includes the other.
 *
 * What it computes: the plain definition of the LGS/NGS Shack-Hartmann sensor
 * of PAPER.md:91 (section 4, "LGS Shack Hartmann wavefront sensor"):
 *   "The WF is split into sub-apertures and the spot computed by FFT for each
 *    sensor sub-aperture. [...] We consider the physical extension of the
 *    projection of the laser on the sodium layer through a convolution for a
 *    gaussian of the desired properties. [...] the centroid computed on the
 *    final [...] image to retrieve the slopes."
 * The paper gives no formula; the steps O1..O9 below are SURVEY.md section
 * 8(c)'s reading (standard Fraunhofer model), restated in DESIGN.md section 3.
 * Everything is done spot by spot, step by step, in float64, with no blocking,
 * fusion or pruning: every transform is the full P x P one.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): invariants I1..I17 of
 * flat wavefront => zero slope, integer tilt => exact
 * circular shift, linear-range tilt closed form, Parseval, FFT == brute-force
 * DFT, FFT convolution == direct O(P^4) sum, Wiener-Khinchin, symmetry,
 * single-pixel centroid, and a numpy fft2 restatement of the whole chain.
 * Parity unpinned (conventions fixed by SURVEY.md, not by the paper; listed in
 * DESIGN.md section 4): threshold semantics (A7), kernel parameterisation
 * (A9, A11-A13), phase units (A3), validity rule (A2), tau defaults (A8).
 *
 * Complex arrays are interleaved (re, im) doubles, row-major, x fastest.
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

/* ------------------------------------------------------------------ O1+O2
 * O1 patch:  p[j,k] = phi[sy*n+j, sx*n+k], a[j,k] likewise   (PAPER.md:91
 *            "The WF is split into sub-apertures")
 * O2 field:  e[j,k] = a[j,k] * exp(i*(c_phi*p[j,k] - pi*(j+k)/P)), j,k < n,
 *            zero elsewhere on the P x P grid (patch in the corner).
 *            The -pi(j+k)/P ramp is reading A5 (half-pixel centring).      */
void shwfs_oracle_field(const float *phase_frame, const float *amplitude,
                        int N, int n, int P, int sy, int sx, double c_phi,
                        double *e /* [P*P*2] */)
{
    memset(e, 0, sizeof(double) * 2 * (size_t)P * P);
    for (int j = 0; j < n; ++j)
        for (int k = 0; k < n; ++k) {
            size_t src = (size_t)(sy * n + j) * N + (size_t)(sx * n + k);
            double p = (double)phase_frame[src];
            double a = (double)amplitude[src];
            double th = c_phi * p - M_PI * (double)(j + k) / (double)P;
            e[2 * (j * P + k) + 0] = a * cos(th);
            e[2 * (j * P + k) + 1] = a * sin(th);
        }
}

/* ------------------------------------------------------------------ O3
 * 1-D DFT of a strided line, X[v] = sum_j x[j] exp(sign*2*pi*i*v*j/L).
 * L <= 16: the naive O(L^2) sum.  L >= 32: iterative radix-2 decimation in
 * time.  Twiddles come from cos/sin of the exact index (no recurrences).
 * sign = -1 is the forward transform of O3, +1 the unnormalised inverse.   */
static void dft1_naive(const double *in, double *out, int L, int sign)
{
    for (int v = 0; v < L; ++v) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < L; ++j) {
            int m = (int)(((long)v * j) % L);
            double ang = sign * 2.0 * M_PI * (double)m / (double)L;
            double c = cos(ang), s = sin(ang);
            sr += in[2 * j] * c - in[2 * j + 1] * s;
            si += in[2 * j] * s + in[2 * j + 1] * c;
        }
        out[2 * v] = sr;
        out[2 * v + 1] = si;
    }
}

static void fft1_radix2(const double *in, double *out, int L, int sign)
{
    int bits = 0;
    while ((1 << bits) < L) ++bits;
    for (int i = 0; i < L; ++i) {           /* bit-reversal permutation */
        int r = 0;
        for (int q = 0; q < bits; ++q)
            if (i & (1 << q)) r |= 1 << (bits - 1 - q);
        out[2 * r] = in[2 * i];
        out[2 * r + 1] = in[2 * i + 1];
    }
    for (int len = 2; len <= L; len <<= 1) { /* butterflies */
        int half = len >> 1;
        for (int base = 0; base < L; base += len)
            for (int q = 0; q < half; ++q) {
                double ang = sign * 2.0 * M_PI * (double)q / (double)len;
                double c = cos(ang), s = sin(ang);
                double *u = out + 2 * (base + q);
                double *w = out + 2 * (base + q + half);
                double tr = w[0] * c - w[1] * s;
                double ti = w[0] * s + w[1] * c;
                w[0] = u[0] - tr; w[1] = u[1] - ti;
                u[0] = u[0] + tr; u[1] = u[1] + ti;
            }
    }
}

/* 1-D transform of a contiguous line of L complex numbers. */
void shwfs_oracle_dft1(const double *in, double *out, int L, int sign)
{
    if (L <= 16) dft1_naive(in, out, L, sign);
    else fft1_radix2(in, out, L, sign);
}

/* 2-D transform, rows then columns: X[v,u] = sum_j sum_k x[j,k]
 * exp(sign*2*pi*i*(v*j+u*k)/P).  in and out may alias.  P must be a power of
 * two when P > 16.  Returns 0, or -1 on allocation failure.                */
int shwfs_oracle_dft2(const double *in, double *out, int P, int sign)
{
    double *line = (double *)malloc(sizeof(double) * 4 * (size_t)P);
    double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)P * P);
    if (!line || !tmp) { free(line); free(tmp); return -1; }
    double *lin = line, *lout = line + 2 * P;
    for (int j = 0; j < P; ++j)                       /* along x (k -> u) */
        shwfs_oracle_dft1(in + 2 * (size_t)j * P, tmp + 2 * (size_t)j * P, P, sign);
    for (int u = 0; u < P; ++u) {                     /* along y (j -> v) */
        for (int j = 0; j < P; ++j) {
            lin[2 * j] = tmp[2 * ((size_t)j * P + u)];
            lin[2 * j + 1] = tmp[2 * ((size_t)j * P + u) + 1];
        }
        shwfs_oracle_dft1(lin, lout, P, sign);
        for (int v = 0; v < P; ++v) {
            out[2 * ((size_t)v * P + u)] = lout[2 * v];
            out[2 * ((size_t)v * P + u) + 1] = lout[2 * v + 1];
        }
    }
    free(line); free(tmp);
    return 0;
}

/* Brute-force O(P^4) 2-D DFT straight from the double sum (pin I5). */
void shwfs_oracle_dft2_brute(const double *in, double *out, int P, int sign)
{
    for (int v = 0; v < P; ++v)
        for (int u = 0; u < P; ++u) {
            double sr = 0.0, si = 0.0;
            for (int j = 0; j < P; ++j)
                for (int k = 0; k < P; ++k) {
                    int m = (int)(((long)v * j + (long)u * k) % P);
                    double ang = sign * 2.0 * M_PI * (double)m / (double)P;
                    double c = cos(ang), s = sin(ang);
                    double xr = in[2 * (j * P + k)], xi = in[2 * (j * P + k) + 1];
                    sr += xr * c - xi * s;
                    si += xr * s + xi * c;
                }
            out[2 * (v * P + u)] = sr;
            out[2 * (v * P + u) + 1] = si;
        }
}

/* ------------------------------------------------------------------ O4
 * I[v,u] = |E[v,u]|^2 / P^2  (reading A6: sum I = sum a^2 by Parseval).    */
void shwfs_oracle_intensity(const double *E, int P, double *I /* [P*P] */)
{
    double inv = 1.0 / ((double)P * (double)P);
    for (int i = 0; i < P * P; ++i)
        I[i] = (E[2 * i] * E[2 * i] + E[2 * i + 1] * E[2 * i + 1]) * inv;
}

/* ------------------------------------------------------------------ O5
 * C[v,u] = sum_{v',u'} I[v',u'] * K[(v-v'+P/2) mod P, (u-u'+P/2) mod P]
 * circular convolution, kernel centre at index (P/2,P/2) (PAPER.md:91
 * "a convolution for a gaussian of the desired properties"; circularity and
 * centre convention: readings A9/A10).  Direct O(P^4) form of the definition. */
void shwfs_oracle_convolve_direct(const double *I, const float *K, int P, double *C)
{
    int h = P / 2;
    for (int v = 0; v < P; ++v)
        for (int u = 0; u < P; ++u) {
            double s = 0.0;
            for (int vp = 0; vp < P; ++vp)
                for (int up = 0; up < P; ++up) {
                    int ky = ((v - vp + h) % P + P) % P;
                    int kx = ((u - up + h) % P + P) % P;
                    s += I[vp * P + up] * (double)K[ky * P + kx];
                }
            C[v * P + u] = s;
        }
}

/* Same result through the convolution theorem with the oracle's own
 * transforms: C = IDFT( DFT(I) * DFT(Kc) ) / P^2,  Kc[d] = K[(d+P/2) mod P].
 * (Pin I12 checks it against the direct sum.)                              */
int shwfs_oracle_convolve_fft(const double *I, const float *K, int P, double *C)
{
    size_t PP = (size_t)P * P;
    double *a = (double *)malloc(sizeof(double) * 2 * PP);
    double *k = (double *)malloc(sizeof(double) * 2 * PP);
    if (!a || !k) { free(a); free(k); return -1; }
    int h = P / 2;
    for (int y = 0; y < P; ++y)
        for (int x = 0; x < P; ++x) {
            a[2 * (y * P + x)] = I[y * P + x];
            a[2 * (y * P + x) + 1] = 0.0;
            k[2 * (y * P + x)] = (double)K[((y + h) % P) * P + ((x + h) % P)];
            k[2 * (y * P + x) + 1] = 0.0;
        }
    int rc = shwfs_oracle_dft2(a, a, P, -1);
    if (!rc) rc = shwfs_oracle_dft2(k, k, P, -1);
    if (!rc) {
        for (size_t i = 0; i < PP; ++i) {
            double re = a[2 * i] * k[2 * i] - a[2 * i + 1] * k[2 * i + 1];
            double im = a[2 * i] * k[2 * i + 1] + a[2 * i + 1] * k[2 * i];
            a[2 * i] = re; a[2 * i + 1] = im;
        }
        rc = shwfs_oracle_dft2(a, a, P, +1);
    }
    if (!rc) {
        double inv = 1.0 / (double)PP;
        for (size_t i = 0; i < PP; ++i) C[i] = a[2 * i] * inv;
    }
    free(a); free(k);
    return rc;
}

/* ------------------------------------------------------------------ O6
 * Sh[r,c] = C[(r-P/2) mod P, (c-P/2) mod P]  (zero tilt lands on the corner
 * shared by pixels P/2-1 and P/2, reading A5).                             */
void shwfs_oracle_centre(const double *C, int P, double *Sh)
{
    int h = P / 2;
    for (int r = 0; r < P; ++r)
        for (int c = 0; c < P; ++c)
            Sh[r * P + c] = C[(((r - h) % P + P) % P) * P + (((c - h) % P + P) % P)];
}

/* ------------------------------------------------------------------ O7
 * B[R,Cc] = sum_{alpha,beta<b} Sh[b*R+alpha, b*Cc+beta], D = P/b.          */
void shwfs_oracle_bin(const double *Sh, int P, int b, double *B)
{
    int D = P / b;
    for (int R = 0; R < D; ++R)
        for (int Cc = 0; Cc < D; ++Cc) {
            double s = 0.0;
            for (int al = 0; al < b; ++al)
                for (int be = 0; be < b; ++be)
                    s += Sh[(b * R + al) * P + (b * Cc + be)];
            B[R * D + Cc] = s;
        }
}

/* ------------------------------------------------------------------ O8+O9
 * O8: m = max B; Wt = max(B - tau*m, 0) (mode 0, reading A7) or
 *     Wt = B*[B >= tau*m] (mode 1).
 * O9: s_x = sum Wt*(Cc-(D-1)/2)/sum Wt, s_y with R; sum Wt == 0 => (0,0).
 * ("the centroid computed on the final [...] image to retrieve
 *  the slopes"; "X- and Y- slopes".)                          */
void shwfs_oracle_threshold_cog(const double *B, int D, double tau, int mode,
                                double *slope_xy /* [2] */)
{
    double m = B[0];
    for (int i = 1; i < D * D; ++i) if (B[i] > m) m = B[i];
    double thr = tau * m;
    double sw = 0.0, sx = 0.0, sy = 0.0, ref = 0.5 * (double)(D - 1);
    for (int R = 0; R < D; ++R)
        for (int Cc = 0; Cc < D; ++Cc) {
            double v = B[R * D + Cc], w;
            if (mode == 0) { w = v - thr; if (w < 0.0) w = 0.0; }
            else w = (v >= thr) ? v : 0.0;
            sw += w;
            sx += w * ((double)Cc - ref);
            sy += w * ((double)R - ref);
        }
    if (sw == 0.0) { slope_xy[0] = 0.0; slope_xy[1] = 0.0; }
    else { slope_xy[0] = sx / sw; slope_xy[1] = sy / sw; }   /* NaN propagates */
}

/* ------------------------------------------------------------------ one spot
 * O1..O9 for frame `phase_frame`, subaperture (sy,sx).  K is that
 * subaperture's P x P kernel or NULL.  conv_direct != 0 uses the O(P^4) sum.
 * Optional outputs (any may be NULL): img0 = centred I [P*P], img1 = centred
 * convolved image Sh [P*P], img2 = B [D*D].  Returns 0 or -1 (no memory).   */
int shwfs_oracle_spot(const float *phase_frame, const float *amplitude, int N,
                      int n, int P, int b, int sy, int sx, double c_phi,
                      double tau, int mode, const float *K, int conv_direct,
                      double *slope_xy, double *img0, double *img1, double *img2)
{
    size_t PP = (size_t)P * P;
    int D = P / b;
    double *e = (double *)malloc(sizeof(double) * 2 * PP);
    double *I = (double *)malloc(sizeof(double) * PP);
    double *C = (double *)malloc(sizeof(double) * PP);
    double *Sh = (double *)malloc(sizeof(double) * PP);
    double *B = (double *)malloc(sizeof(double) * (size_t)D * D);
    int rc = (e && I && C && Sh && B) ? 0 : -1;
    if (!rc) {
        shwfs_oracle_field(phase_frame, amplitude, N, n, P, sy, sx, c_phi, e);  /* O1,O2 */
        rc = shwfs_oracle_dft2(e, e, P, -1);                                    /* O3 */
    }
    if (!rc) {
        shwfs_oracle_intensity(e, P, I);                                        /* O4 */
        if (img0) shwfs_oracle_centre(I, P, img0);
        if (K) {                                                                /* O5 */
            if (conv_direct) shwfs_oracle_convolve_direct(I, K, P, C);
            else rc = shwfs_oracle_convolve_fft(I, K, P, C);
        } else memcpy(C, I, sizeof(double) * PP);
    }
    if (!rc) {
        shwfs_oracle_centre(C, P, Sh);                                          /* O6 */
        if (img1) memcpy(img1, Sh, sizeof(double) * PP);
        shwfs_oracle_bin(Sh, P, b, B);                                          /* O7 */
        if (img2) memcpy(img2, B, sizeof(double) * (size_t)D * D);
        shwfs_oracle_threshold_cog(B, D, tau, mode, slope_xy);                  /* O8,O9 */
    }
    free(e); free(I); free(C); free(Sh); free(B);
    return rc;
}

/* ------------------------------------------------------------------ H0
 * Valid-subaperture rule (reading A2): subaperture (sy,sx) is valid if the
 * mean of the amplitude over its n x n patch is >= min_illum; list order is
 * row-major (sy outer).  yx may be NULL to count only.  Returns the count.  */
int shwfs_oracle_valid_list(const float *amplitude, int N, int n, double min_illum,
                            int32_t *yx /* [S*S*2] or NULL */)
{
    int S = N / n, cnt = 0;
    for (int sy = 0; sy < S; ++sy)
        for (int sx = 0; sx < S; ++sx) {
            double s = 0.0;
            for (int j = 0; j < n; ++j)
                for (int k = 0; k < n; ++k)
                    s += (double)amplitude[(size_t)(sy * n + j) * N + (sx * n + k)];
            if (s / ((double)n * n) >= min_illum) {
                if (yx) { yx[2 * cnt] = sy; yx[2 * cnt + 1] = sx; }
                ++cnt;
            }
        }
    return cnt;
}

/* ------------------------------------------------------------------ whole call
 * slopes[t,i,:] for every frame t < T and valid subaperture i < nsub
 * (OpenMP over spots; nthreads <= 0 means the OpenMP default).
 * kernels: [nsub,P,P] fp32 or NULL.  stage in {-1,0,1,2}: if >= 0, `images`
 * receives that stage for every spot ([T,nsub,P,P] for 0/1, [T,nsub,D,D] for 2).
 * Returns 0, -1 (no memory) or -2 (bad argument).                          */
int shwfs_oracle_measure(const float *phase, int T, int N, int n, int P, int b,
                         const float *amplitude, const int32_t *valid_yx, int nsub,
                         double c_phi, double tau, int mode, const float *kernels,
                         int conv_direct, double *slopes, int stage, double *images,
                         int nthreads)
{
    if (!phase || !amplitude || !valid_yx || !slopes || T < 0 || n <= 0 || n > P ||
        b <= 0 || P % b || N % n || (stage >= 0 && !images) || stage > 2)
        return -2;
    int D = P / b;
    size_t img_sz = (stage == 2) ? (size_t)D * D : (size_t)P * P;
    long total = (long)T * nsub;
    int fail = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 16)
    for (long w = 0; w < total; ++w) {
        int t = (int)(w / nsub), i = (int)(w % nsub);
        double *im = (stage >= 0) ? images + (size_t)w * img_sz : NULL;
        int rc = shwfs_oracle_spot(phase + (size_t)t * N * N, amplitude, N, n, P, b,
                                   valid_yx[2 * i], valid_yx[2 * i + 1], c_phi, tau, mode,
                                   kernels ? kernels + (size_t)i * P * P : NULL, conv_direct,
                                   slopes + 2 * (size_t)w,
                                   stage == 0 ? im : NULL, stage == 1 ? im : NULL,
                                   stage == 2 ? im : NULL);
        if (rc) {
#pragma omp atomic write
            fail = 1;
        }
    }
    return fail ? -1 : 0;
}

int shwfs_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
