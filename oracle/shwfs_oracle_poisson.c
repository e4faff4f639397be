/*
 * shwfs_oracle_poisson.c -- float64 CPU oracle for detector noise with true Poisson photon statistics
 * ("photon (Poisson) + read (Gaussian) noise on the binned image, counter-based RNG
 * (Philox) so the oracle can reproduce it bit-for-bit per (seed, t, i, pixel)").
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT (same rules as shwfs_oracle.c and shwfs_oracle_lgs.c, whose Philox and
 * normal-deviate functions it calls; nothing is shared with the CUDA library).
 *
 * Passage followed: "Finally the sub-layer arrays are piled-up and the centroid computed on the
 * final noise-added image to retrieve the slopes."  The paper says no more about the noise; reading B4'
 * (DESIGN.md section 12), photon_model = 1:
 *   N1  rate of pixel p = C*D + R (column-major, as in L5):  lambda = max(F * B[R,C], 0)   photo-electrons
 *   N2  uniforms: Philox4x32-10 block with key = seed and counter = (p / 2, i, t, 1 + j), j = 0, 1, ... the
 *       attempt; pixel p takes the output words (x[2 (p mod 2)], x[2 (p mod 2) + 1]) as
 *       u1, u2 = ((x >> 9) + 1/2) 2^-23 in (0,1).  (Counter word 3 = 0 is the block of normal deviates of L5.)
 *   N3  lambda < 30: inversion by sequential search on u1 (attempt 0 only):
 *           k = 0, q = exp(-lambda), s = q;  while (u1 > s and k < kmax): k += 1, q *= lambda / k, s += q
 *       kmax = floor(lambda + 12 sqrt(lambda) + 30) only ends the search when rounding keeps s below a u1 that
 *       is within an ulp of 1 (it is far beyond every quantile a 23-bit uniform can ask for)
 *   N4  lambda >= 30: the transformed-rejection method PTRS of W. Hoermann, "The transformed rejection method
 *       for generating Poisson random variables", Insurance: Mathematics and Economics 12 (1993) 39-45:
 *           sm = sqrt(lambda), b = 0.931 + 2.53 sm, a = -0.059 + 0.02483 b,
 *           1/alpha = 1.1239 + 1.1328 / (b - 3.4), v_r = 0.9277 - 3.6224 / (b - 2)
 *           attempt j: U = u1 - 1/2, V = u2, us = 1/2 - |U|, k = floor((2 a / us + b) U + lambda + 0.43)
 *             accept k if us >= 0.07 and V <= v_r
 *             next attempt if k < 0, or if us < 0.013 and V > us
 *             accept k if ln V + ln(1/alpha) - ln(a / us^2 + b) <= -lambda + k ln lambda - lgamma(k + 1)
 *           (at most 64 attempts, then k = round(lambda): probability < 1e-60).
 *   N5  counts[R,C] = k + ron * z_p, z_p the normal deviate of L5 (block p / 4, deviate p mod 4).
 * Each draw also returns a MARGIN: the smallest distance by which any comparison it took was decided (|u1 - s|
 * of every step of N3; in N4 the distance of the floor argument to an integer and of every inequality to
 * equality; |lambda - 30| / 30 for the choice between N3 and N4).  The fp32 device path decides the same
 * comparisons on rates that differ from the oracle's by rounding; where the margin is larger than that, the
 * integer must be the same on both sides (tests/test_lgs_gpu.py), elsewhere it may differ.
 *
 * Every function below is pinned; what no pin can reach are this build's conventions (the paper says only
 * "noise-added"): the counter layout of N2, the rate of 30 at which N3 hands over to N4, noise on the binned image.
 * Pins (tests/test_oracle_poisson_pins.py, -m "not gpu"): P1 N3 equals the quantile function of the Poisson
 * distribution (scipy.stats.poisson.ppf) for every u1 clear of a step; P2 mean = variance = lambda and a chi^2
 * test against the Poisson pmf at lambda = 0.3, 3, 29.9 (N3) and 30, 300 (N4); P3 (k - lambda) / sqrt(lambda)
 * is standard normal for lambda = 1e4 (Kolmogorov-Smirnov): the Gaussian limit of reading B4; P4 lambda = 0
 * gives 0, a negative rate is clipped; P5 pixels, spots and frames draw independently (counter layout N2);
 * P6 with ron > 0 the variance is lambda + ron^2 and the read-noise term is the deviate of L5.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

void shwfs_oracle_philox4x32(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void shwfs_oracle_normal4(uint64_t seed, uint32_t t, uint32_t i, uint32_t blk, double z[4]);

static double unit_open(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }
static void keep_min(double *m, double d) { if (d < 0) d = -d; if (d < *m) *m = d; }

/* N2: the two uniforms of pixel p, attempt j */
void shwfs_oracle_poisson_uniforms(uint64_t seed, uint32_t t, uint32_t i, uint32_t p, uint32_t j, double u[2])
{
    uint32_t ctr[4] = {p / 2u, i, t, 1u + j}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, x[4];
    shwfs_oracle_philox4x32(ctr, key, x);
    u[0] = unit_open(x[2 * (p & 1u)]);
    u[1] = unit_open(x[2 * (p & 1u) + 1]);
}

/* N3: inversion by sequential search */
long shwfs_oracle_poisson_inversion(double lambda, double u1, double *margin)
{
    long k = 0;
    const long kmax = (long)floor(lambda + 12.0 * sqrt(lambda) + 30.0);
    double q = exp(-lambda), s = q, m = 1.0;
    keep_min(&m, u1 - s);
    while (u1 > s && k < kmax) {
        k += 1;
        q *= lambda / (double)k;
        s += q;
        keep_min(&m, u1 - s);
    }
    if (margin) *margin = m;
    return k;
}

/* N4: PTRS; the attempts draw their own uniforms (N2) */
long shwfs_oracle_poisson_ptrs(double lambda, uint64_t seed, uint32_t t, uint32_t i, uint32_t p, double *margin,
                               int *attempts)
{
    const double sm = sqrt(lambda), b = 0.931 + 2.53 * sm, a = -0.059 + 0.02483 * b;
    const double inv_alpha = 1.1239 + 1.1328 / (b - 3.4), v_r = 0.9277 - 3.6224 / (b - 2.0);
    double m = 1.0;
    long k = (long)floor(lambda + 0.5);
    int j;
    for (j = 0; j < 64; ++j) {
        double u[2];
        shwfs_oracle_poisson_uniforms(seed, t, i, p, (uint32_t)j, u);
        const double U = u[0] - 0.5, V = u[1], us = 0.5 - fabs(U);
        const double x = (2.0 * a / us + b) * U + lambda + 0.43;
        const double kf = floor(x);
        keep_min(&m, x - kf);
        keep_min(&m, kf + 1.0 - x);
        keep_min(&m, us - 0.07);
        keep_min(&m, V - v_r);
        if (us >= 0.07 && V <= v_r) { k = (long)kf; break; }
        if (kf < 0.0) continue;
        keep_min(&m, us - 0.013);
        keep_min(&m, V - us);
        if (us < 0.013 && V > us) continue;
        const double lhs = log(V) + log(inv_alpha) - log(a / (us * us) + b);
        const double rhs = -lambda + kf * log(lambda) - lgamma(kf + 1.0);
        keep_min(&m, lhs - rhs);
        if (lhs <= rhs) { k = (long)kf; break; }
    }
    if (margin) *margin = m;
    if (attempts) *attempts = j + 1;
    return k;
}

/* N1 + N3/N4 for one pixel */
long shwfs_oracle_poisson_draw(double lambda, uint64_t seed, uint32_t t, uint32_t i, uint32_t p, double *margin)
{
    double m = 1.0, m2 = 1.0;
    long k;
    if (!(lambda > 0.0)) { if (margin) *margin = 1.0; return 0; }
    keep_min(&m, (lambda - 30.0) / 30.0);
    if (lambda < 30.0) {
        double u[2];
        shwfs_oracle_poisson_uniforms(seed, t, i, p, 0u, u);
        k = shwfs_oracle_poisson_inversion(lambda, u[0], &m2);
    } else {
        k = shwfs_oracle_poisson_ptrs(lambda, seed, t, i, p, &m2, NULL);
    }
    if (margin) *margin = m < m2 ? m : m2;
    return k;
}

/* N1..N5 on a D x D binned image (row-major B[R*D + C]); margin_out (or NULL) receives the margin of each pixel.
 * F <= 0 means "no noise": counts = B. */
void shwfs_oracle_add_noise_poisson(const double *B, int D, double F, double ron, uint64_t seed, uint32_t t,
                                    uint32_t i, double *counts, double *margin_out)
{
    if (!(F > 0.0)) {
        memcpy(counts, B, sizeof(double) * (size_t)D * D);
        if (margin_out) for (int q = 0; q < D * D; ++q) margin_out[q] = 1.0;
        return;
    }
    for (int C = 0; C < D; ++C)
        for (int R = 0; R < D; ++R) {
            const uint32_t p = (uint32_t)(C * D + R);
            double z[4], m;
            const double lam = F * B[R * D + C];
            const long k = shwfs_oracle_poisson_draw(lam > 0.0 ? lam : 0.0, seed, t, i, p, &m);
            shwfs_oracle_normal4(seed, t, i, p / 4u, z);
            counts[R * D + C] = (double)k + ron * z[p % 4u];
            if (margin_out) margin_out[R * D + C] = m;
        }
}
