/*
 * noise.cuh -- detector noise on the binned image before the centroid ("the centroid computed
 * on the final noise-added image", readings B4/B4'/B5 of DESIGN.md).  photon_model 0:
 *     counts = F*B + sqrt(max(F*B, 0) + ron^2) * z,   z ~ N(0,1),
 * z drawn from the counter-based generator Philox4x32-10 (Salmon et al., SC'11) so that any (seed, frame,
 * subaperture, pixel) can be reproduced independently: key = (seed lo, seed hi), counter = (p/4, i, t, 0)
 * with p = C*D + R the column-major pixel index; Box-Muller on the output pairs (x0,x1), (x2,x3) with
 * u = ((x >> 9) + 1/2) * 2^-23 (exact in fp32) gives the deviates of pixels 4*(p/4) .. 4*(p/4)+3.
 * photon_model 1 (SURVEY.md 8(f) f2 as written: "photon (Poisson) + read (Gaussian) noise"):
 *     counts = k + ron * z,   k ~ Poisson(max(F*B, 0)),
 * k drawn from the uniforms of the Philox blocks with counter = (p/2, i, t, 1 + attempt) -- pixel p takes words
 * 2 (p mod 2) and 2 (p mod 2) + 1 -- by inversion (sequential search) below a rate of 30 and by Hoermann's
 * transformed rejection PTRS (Insurance: Mathematics and Economics 12 (1993) 39) from 30 up, in fp32.  An integer
 * decided by floating-point comparisons cannot agree with a float64 evaluation on every pixel; it does wherever the
 * comparison is not within rounding of equality, which is how the parity test states it (tests/test_lgs_gpu.py).
 */
#ifndef SHWFS_NOISE_CUH_
#define SHWFS_NOISE_CUH_

#include <stdint.h>

namespace shwfs {

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k)
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k.x += W0; k.y += W1; }
        const uint32_t h0 = __umulhi(M0, c.x), l0 = M0 * c.x;
        const uint32_t h1 = __umulhi(M1, c.z), l1 = M1 * c.z;
        c = make_uint4(h1 ^ c.y ^ k.x, l1, h0 ^ c.w ^ k.y, l0);
    }
    return c;
}

__device__ __forceinline__ float unit_open(uint32_t x) { return ((float)(x >> 9) + 0.5f) * (1.0f / 8388608.0f); }

/* Box-Muller radius sqrt(-2 ln u) with the hardware log2 (absolute error of ln u ~ 4e-7: the deviate is good
 * to ~1e-6, far below the 1e-4-of-peak image tolerance once scaled by the noise sigma) */
__device__ __forceinline__ float bm_radius(float u) { return sqrtf(fmaxf(-2.0f * __logf(u), 0.f)); }

/* the four deviates of block `blk` of spot (frame t, subaperture i) */
__device__ __forceinline__ void normal4(uint2 key, uint32_t t, uint32_t i, uint32_t blk, float (&z)[4])
{
    const uint4 x = philox4x32_10(make_uint4(blk, i, t, 0u), key);
    const float r1 = bm_radius(unit_open(x.x)), r2 = bm_radius(unit_open(x.z));
    /* angle 2 pi u = pi + 2 pi (u - 1/2): the fast sincos is evaluated on (-pi, pi) and negated */
    float s1, c1, s2, c2;
    __sincosf((unit_open(x.y) - 0.5f) * 6.283185307179586f, &s1, &c1);
    __sincosf((unit_open(x.w) - 0.5f) * 6.283185307179586f, &s2, &c2);
    z[0] = -r1 * c1; z[1] = -r1 * s1; z[2] = -r2 * c2; z[3] = -r2 * s2;
}

__device__ __forceinline__ float noisy_count(float B, float F, float ron2, float z)
{
    const float m = F * B;
    return fmaf(sqrtf(fmaxf(m, 0.f) + ron2), z, m);
}

/* ---- photon_model 1: Poisson counts ---- */

/* sequential search on u1: the smallest k with CDF(k) >= u1 (kmax: see the oracle's note, never reached by a
 * 23-bit uniform unless rounding keeps the sum below a u1 within an ulp of 1) */
__device__ __forceinline__ float poisson_inversion(float lam, float u1)
{
    const float kmax = floorf(lam + 12.0f * sqrtf(lam) + 30.0f);
    float k = 0.f, q = expf(-lam), s = q;
    while (u1 > s && k < kmax) {
        k += 1.0f;
        q *= lam / k;
        s += q;
    }
    return k;
}

/* transformed rejection (PTRS), rate >= 30; x holds the attempt-0 block of the pixel's pair, later attempts
 * draw their own */
static __device__ __noinline__ float poisson_ptrs(float lam, uint4 x, uint2 key, uint32_t t, uint32_t i, uint32_t p)
{
    const float sm = sqrtf(lam), b = 0.931f + 2.53f * sm, a = -0.059f + 0.02483f * b;
    const float inv_alpha = 1.1239f + 1.1328f / (b - 3.4f), v_r = 0.9277f - 3.6224f / (b - 2.0f);
    for (uint32_t j = 0; j < 64u; ++j) {
        if (j > 0) x = philox4x32_10(make_uint4(p >> 1, i, t, 1u + j), key);
        const float U = unit_open((p & 1u) ? x.z : x.x) - 0.5f, V = unit_open((p & 1u) ? x.w : x.y);
        const float us = 0.5f - fabsf(U);
        const float kf = floorf((2.0f * a / us + b) * U + lam + 0.43f);
        if (us >= 0.07f && V <= v_r) return kf;
        if (kf < 0.f || (us < 0.013f && V > us)) continue;
        if (logf(V) + logf(inv_alpha) - logf(a / (us * us) + b) <= -lam + kf * logf(lam) - lgammaf(kf + 1.0f)) return kf;
    }
    return floorf(lam + 0.5f);
}

/* pixel p of spot (t, i) at rate F*B; x = Philox block (p/2, i, t, 1) of the pixel's pair */
__device__ __forceinline__ float poisson_count(float B, float F, uint4 x, uint2 key, uint32_t t, uint32_t i, uint32_t p)
{
    const float lam = fmaxf(F * B, 0.f);
    if (!(lam > 0.f)) return 0.f;
    if (lam < 30.0f) return poisson_inversion(lam, unit_open((p & 1u) ? x.z : x.x));
    return poisson_ptrs(lam, x, key, t, i, p);
}

/* The Poisson model on one detector column (lane = column C, pixels p = 16 C + R): the eight pair blocks
 * 8C .. 8C+7 of uniforms and the four blocks 4C .. 4C+3 of normal deviates.  Kept out of line, with the column
 * passed through memory, so that the sensor kernels that carry it pay for it only when it is switched on. */
static __device__ __noinline__ void add_poisson_col16(float *col, int C, uint2 key, uint32_t t, uint32_t i, float F, float ron)
{
#pragma unroll 1
    for (int q = 0; q < 4; ++q) {
        float z[4];
        normal4(key, t, i, (uint32_t)(4 * C + q), z);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t p0 = (uint32_t)(16 * C + 4 * q + 2 * h);
            const uint4 x = philox4x32_10(make_uint4(p0 >> 1, i, t, 1u), key);
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int r = 4 * q + 2 * h + e;
                col[r] = fmaf(ron, z[2 * h + e], poisson_count(col[r], F, x, key, t, i, p0 + (uint32_t)e));
            }
        }
    }
}

/* One detector column (16 pixels, lane = column C) of a 16 x 16 image: blocks 4C .. 4C+3 of normal deviates. */
__device__ __forceinline__ void add_noise_col16(float (&bcol)[16], int C, uint2 key, uint32_t t, uint32_t i,
                                                float F, float ron2, int photon_model)
{
    if (photon_model == 1) {
        float col[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) col[r] = bcol[r];
        add_poisson_col16(col, C, key, t, i, F, sqrtf(ron2));
#pragma unroll
        for (int r = 0; r < 16; ++r) bcol[r] = col[r];
        return;
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        float z[4];
        normal4(key, t, i, (uint32_t)(4 * C + q), z);
#pragma unroll
        for (int r = 0; r < 4; ++r) bcol[4 * q + r] = noisy_count(bcol[4 * q + r], F, ron2, z[r]);
    }
}

}  // namespace shwfs
#endif
