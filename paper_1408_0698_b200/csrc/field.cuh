/*
 * field.cuh -- H2 of include/shwfs.h: the complex field of one pupil pixel ("the spot
 * computed by FFT for each sensor sub-aperture": the transform is taken of a*exp(i*phi)).
 * Shared by the lag-domain path (wk.cu) and the literal FFT chain (literal.cu).
 */
#ifndef SHWFS_FIELD_CUH_
#define SHWFS_FIELD_CUH_

namespace shwfs {

/* turns = phase_to_rad / (2*pi); ramp = (j+k) / (2P) in turns (reading A5: half-pixel centring).  The
 * argument is reduced to [-1/2, 1/2] turns before the fast sincos so that the +-60 rad open-loop phases
 * of the MAORY pupil keep ~1e-6 absolute accuracy.                                                   */
__device__ __forceinline__ float2 field_value(float ph, float amp, float turns, float ramp)
{
    float u = fmaf(ph, turns, -ramp);
    u -= rintf(u);
    float s, c;
    __sincosf(u * 6.283185307179586f, &s, &c);
    return make_float2(amp * c, amp * s);
}

/* the same under unit amplitude (fully lit subapertures) */
__device__ __forceinline__ float2 field_unit(float ph, float turns, float ramp)
{
    float u = fmaf(ph, turns, -ramp);
    u -= rintf(u);
    float s, c;
    __sincosf(u * 6.283185307179586f, &s, &c);
    return make_float2(c, s);
}

}  // namespace shwfs
#endif
