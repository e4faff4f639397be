/*
 * wk_common.cuh -- what the two lag-domain kernels (wk.cu: autocorrelation by direct sums; wk_fft.cu: by FFT on a
 * 2n x 2n grid) share: the argument block, and the table product + x-transform of one lag row (H5 + the
 * x half of H6 of include/shwfs.h in Fourier form; wk.cu's header has the identity).
 */
#ifndef SHWFS_WK_COMMON_CUH_
#define SHWFS_WK_COMMON_CUH_

#include "internal.h"
#include "fft_regs.cuh"

namespace shwfs {

struct WkArgs {
    const float *phase;
    const float *amp;
    const int2 *valid;
    const float2 *M;
    float *slopes;
    float *binned;
    long long frame_stride;
    int T, N, nsub, mstride, total, mode;
    float tau, turns, ramp_unit;
    /* paper's full LGS model (EXT instances only): sodium sub-layers and detector noise */
    const float2 *sod_g;         /* [L][nsub] local gradient of the sub-layer's analytic phase, turns/pixel */
    float *noisy;                /* stage-3 debug image (binned, after noise) or null                       */
    long long layer_stride;      /* elements between sub-layers of one frame (0: shared wavefront)          */
    int L;
    float sod_q[SHWFS_MAX_LAYERS];   /* curvature a_l dx^2 / 2pi, turns/pixel^2                             */
    float sod_sw[SHWFS_MAX_LAYERS];  /* sqrt(w_l): folded into the amplitude                                */
    float flux, ron2;
    uint2 key;
    unsigned t0;
    /* closed-loop neighbour (EXT instances only): residual = wavefront - DM phase.  The DM
     * phase sum_m coef[t][m] * mode[m] arrives in patch layout from dm_phase_kernel (loop.cu).          */
    const float *dm_patch;       /* [T][nsub][n*n] or null */
};

/* S = G * M aliased onto lx mod 16, 16-point x-transform, H[ly][0..15] -> shared memory */
template <int n, bool F2 = false>
__device__ __forceinline__ void finish_row(const float2 (&acc)[2 * n - 1], const float2 *__restrict__ Mrow,
                                           float *__restrict__ hrow)
{
    float sr[16], si[16];
#pragma unroll
    for (int m = 0; m < 16; ++m) {
        bool first = true;
        sr[m] = 0.f; si[m] = 0.f;
#pragma unroll
        for (int pass = 0; pass < 2; ++pass) {
            const int lx = pass == 0 ? m : m - 16;
            if (lx > n - 1 || lx < -(n - 1)) continue;
            const int a = lx + n - 1;
            const float2 mv = __ldg(Mrow + a);
            const float gr = acc[a].x, gi = acc[a].y;
            if (first) {
                sr[m] = fmaf(gr, mv.x, -gi * mv.y);
                si[m] = fmaf(gr, mv.y, gi * mv.x);
                first = false;
            } else {
                sr[m] = fmaf(gr, mv.x, fmaf(-gi, mv.y, sr[m]));
                si[m] = fmaf(gr, mv.y, fmaf(gi, mv.x, si[m]));
            }
        }
    }
    fft_fma<16, +1>(sr, si);                     /* H[C] = sum_m s'[m] w_16^(C m) */
#pragma unroll
    for (int C = 0; C < 16; C += 2) {
        const int p0 = fft_out_index<16>(C), p1 = fft_out_index<16>(C + 1);
        if (F2) {                                /* 8-byte aligned row (multi-layer instances) */
            reinterpret_cast<float2 *>(hrow)[C] = make_float2(sr[p0], si[p0]);
            reinterpret_cast<float2 *>(hrow)[C + 1] = make_float2(sr[p1], si[p1]);
        } else {
            reinterpret_cast<float4 *>(hrow)[C / 2] = make_float4(sr[p0], si[p0], sr[p1], si[p1]);
        }
    }
}

}  // namespace shwfs

/* wk_fft.cu: even n = 8 .. 16, D = 16 */
cudaError_t shwfs_wk_fft_launch(const shwfs::WkArgs &A, int n, cudaStream_t st);

#endif
