/*
 * noise.cuh -- detector noise on the binned image before the centroid ("the centroid computed
 * on the final noise-added image", readings B4/B5 of DESIGN.md):
 *     counts = F*B + sqrt(max(F*B, 0) + ron^2) * z,   z ~ N(0,1),
 * z drawn from the counter-based generator Philox4x32-10 (Salmon et al., SC'11) so that any (seed, frame,
 * subaperture, pixel) can be reproduced independently: key = (seed lo, seed hi), counter = (p/4, i, t, 0)
 * with p = C*D + R the column-major pixel index; Box-Muller on the output pairs (x0,x1), (x2,x3) with
 * u = ((x >> 9) + 1/2) * 2^-23 (exact in fp32) gives the deviates of pixels 4*(p/4) .. 4*(p/4)+3.
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

/* One detector column (16 pixels, lane = column C) of a 16 x 16 image: blocks 4C .. 4C+3. */
__device__ __forceinline__ void add_noise_col16(float (&bcol)[16], int C, uint2 key, uint32_t t, uint32_t i,
                                                float F, float ron2)
{
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
