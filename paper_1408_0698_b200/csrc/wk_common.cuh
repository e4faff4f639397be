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
    int photon_model;            /* 0 Gaussian limit of the photon noise, 1 Poisson counts (noise.cuh) */
    uint2 key;
    unsigned t0;
    /* closed-loop neighbour (EXT instances only): residual = wavefront - DM phase.  The DM
     * phase sum_m coef[t][m] * mode[m] arrives in patch layout from dm_phase_kernel (loop.cu).          */
    const float *dm_patch;       /* [T][nsub][n*n] or null */
    int *sched;                  /* chunk counters of the dynamic sweep (sweep.cuh), persistent instances */
    const int2 *patch;           /* [nsub] patch table of the handle (internal.h): origin in pixels + fully-lit flag */
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
            const float2 mv = __ldg(Mrow + a * n);          /* M[a][ly]: lag row ly is a column of the table */
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


/* The table product S[m] = sum over the lags lx = m (mod 16) of G[ly,lx] M_i[ly,lx] visits the 2n-1 lags in the
 * order m = 0..15, lx = m before lx = m - 16.  term_lag<n>(k): index a = lx + n - 1 of the k-th lag in that order,
 * term_m<n>(k): the m it belongs to, term_first<n>(k): whether it opens the sum of its m.                      */
template <int n>
__host__ __device__ constexpr int term_lag(int k)
{
    int c = 0;
    for (int m = 0; m < 16; ++m)
        for (int pass = 0; pass < 2; ++pass) {
            const int lx = pass == 0 ? m : m - 16;
            if (lx > n - 1 || lx < -(n - 1)) continue;
            if (c == k) return lx + n - 1;
            ++c;
        }
    return -1;
}
template <int n>
__host__ __device__ constexpr int term_m(int k) { return (term_lag<n>(k) - (n - 1)) & 15; }
template <int n>
__host__ __device__ constexpr bool term_first(int k) { return k == 0 || term_m<n>(k - 1) != term_m<n>(k); }

/* Staging of one table row in shared memory (wk_fft.cu): the 2n-1 entries M_i[.][ly] of lag row ly go, in the
 * order the product visits them, to `dst` by 8-byte cp.async -- no registers, and the copies fly during the
 * transform that produces G.  Left to plain loads the compiler puts each entry's load a few instructions before
 * its use (the kernel has no registers to spare) and every one of the 2n-1 exposes an L1 round trip: 15 % of the
 * stall samples of wkf_kernel<16> (profiles/r02_wkf16.md).  The thread that stages a row is the one that reads
 * it, so cp.async.wait_group is all the synchronisation there is.                                             */
template <int n>
__device__ __forceinline__ void mrow_stage(const float2 *__restrict__ Mcol, float *dst)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
#pragma unroll
    for (int k = 0; k < 2 * n - 1; ++k)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d + 8u * k), "l"(Mcol + term_lag<n>(k) * n) : "memory");
    asm volatile("cp.async.commit_group;" ::: "memory");
}
__device__ __forceinline__ void mrow_wait() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

/* S = G * M aliased onto lx mod 16 and the 16-point x-transform on packed complex registers (FP32x2,
 * fft_regs.cuh): a complex product is two FFMA2 with the scalar halves of G broadcast,
 * g m = g_r (m_r, m_i) + g_i (-m_i, m_r).  mrow: the table row in visiting order (mrow_stage), 16-byte aligned;
 * H[ly][0..15] -> hrow, which may be the same memory (everything is read before anything is written).       */
template <int n, bool F2 = false>
__device__ __forceinline__ void finish_row2(const float2 (&acc)[2 * n - 1], const float *mrow, float *hrow)
{
    constexpr int LX = 2 * n - 1;
    float2 mv[LX + 1];
#pragma unroll
    for (int k = 0; k < LX + 1; k += 2) {
        const float4 v = reinterpret_cast<const float4 *>(mrow)[k / 2];
        mv[k] = make_float2(v.x, v.y);
        mv[k + 1] = make_float2(v.z, v.w);
    }
    float2 s[16];
#pragma unroll
    for (int m = 0; m < 16; ++m) s[m] = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < LX; ++k) {
        const int a = term_lag<n>(k), m = term_m<n>(k);
        const float2 g = acc[a];
        s[m] = term_first<n>(k) ? __fmul2_rn(bc2(g.x), mv[k]) : __ffma2_rn(bc2(g.x), mv[k], s[m]);
        s[m] = __ffma2_rn(bc2(g.y), rot_pi2(mv[k]), s[m]);
    }
    fft_fma2<16, +1>(s);                         /* H[C] = sum_m s'[m] w_16^(C m) */
#pragma unroll
    for (int C = 0; C < 16; C += 2) {
        const int p0 = fft_out_index<16>(C), p1 = fft_out_index<16>(C + 1);
        if (F2) {                                /* 8-byte aligned row (multi-layer instances) */
            reinterpret_cast<float2 *>(hrow)[C] = s[p0];
            reinterpret_cast<float2 *>(hrow)[C + 1] = s[p1];
        } else {
            reinterpret_cast<float4 *>(hrow)[C / 2] = make_float4(s[p0].x, s[p0].y, s[p1].x, s[p1].y);
        }
    }
}

/* B[R,C] = Re sum_m H[m][C] w_16^(R m) for one detector column C: the y half of H6 in Fourier form.  hm(m) returns
 * H[m][C], m < n.                                                                                         */
template <int n, typename F>
__device__ __forceinline__ void ytransform16(F hm, float (&bcol)[16])
{
    float2 y[16];
#pragma unroll
    for (int m = 0; m < 16; ++m) y[m] = m < n ? hm(m) : make_float2(0.f, 0.f);
    fft_fma2<16, +1, n>(y);
#pragma unroll
    for (int R = 0; R < 16; ++R) bcol[R] = y[fft_out_index<16>(R)].x;
}

}  // namespace shwfs

/* wk_fft.cu: even n = 8 .. 16, D = 16 */
cudaError_t shwfs_wk_fft_launch(shwfs_handle *h, const shwfs::WkArgs &A, int n, cudaStream_t st);

#endif
