/*
 * cog.cuh -- H7 (peak + threshold) and H8 (centre of gravity) of include/shwfs.h on a 16 x 16 detector held
 * one column per lane by a half-warp ("the centroid computed on the final image to retrieve
 * the slopes").  Shared by the lag-domain path (wk.cu) and the pruned-FFT path (pruned_fft.cu).
 */
#ifndef SHWFS_COG_CUH_
#define SHWFS_COG_CUH_

namespace shwfs {

/* H7 + H8 on a half-warp: lane C (0..15) holds column C of B as bcol[R].  Returns slopes in lane 0
 * of the half-warp.  Shuffles use xor offsets < 16, so the two halves of a warp stay separate.    */
template <int MODE>
__device__ __forceinline__ float2 cog16(const float (&bcol)[16], int C, float tau)
{
    float mx = bcol[0];
#pragma unroll
    for (int R = 1; R < 16; ++R) mx = fmaxf(mx, bcol[R]);
#pragma unroll
    for (int o = 8; o >= 1; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    const float thr = tau * mx;
    float sw = 0.f, sy = 0.f;
#pragma unroll
    for (int R = 0; R < 16; ++R) {
        const float v = bcol[R];
        const float w = MODE == 0 ? fmaxf(v - thr, 0.f) : (v >= thr ? v : 0.f);
        sw += w;
        sy = fmaf(w, (float)R - 7.5f, sy);
    }
    float sx = sw * ((float)C - 7.5f);
#pragma unroll
    for (int o = 8; o >= 1; o >>= 1) {
        sw += __shfl_xor_sync(0xffffffffu, sw, o);
        sx += __shfl_xor_sync(0xffffffffu, sx, o);
        sy += __shfl_xor_sync(0xffffffffu, sy, o);
    }
    if (sw == 0.f) return make_float2(0.f, 0.f);
    const float inv = 1.0f / sw;
    return make_float2(sx * inv, sy * inv);
}

}  // namespace shwfs
#endif
