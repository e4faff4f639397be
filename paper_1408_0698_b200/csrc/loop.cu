/*
 * loop.cu -- the closed-loop neighbours of the Shack-Hartmann path, sm_100a.
 *
 * "The WFS modules compute the vector signals (X-and Y- slopes) from the residual phase (the
 * open loop wavefront subtracted by the DM).  Vector slopes multiplied by the control matrix returns the
 * vector coefficients for the modal base linear composition, in the form of the differential coefficients
 * to be added to the one defining the existing mirror shape.  [...] a pure integrator scheme".
 *
 *   before the path   residual = wavefront - sum_m c[t,m] mode[m]: evaluated INSIDE the sensor kernel's
 *                     gather (wk.cu, EXT instances) from a per-subaperture re-layout of the modes built
 *                     here once per shwfs_set_dm, so the residual never exists in HBM;
 *   after the path    d[t,m] = sum_k R[m,k] s[t,k] (k = 2 i + axis), c += gain * d: recon_kernel, one warp
 *                     per mode, the slope vector streamed with 8-byte loads, warp-shuffle reduction.
 * shwfs_closed_loop chains the two, frame after frame, on the caller's stream (readings C1..C4 of DESIGN.md).
 */
#include "internal.h"

namespace {

/* modes[M][N][N] -> out[nsub][Mp][n*n] (zero for m >= M): block = (subaperture, mode) */
__global__ void relayout_modes_kernel(const float *__restrict__ modes, const int2 *__restrict__ valid, int N,
                                      int n, int M, int Mp, float *__restrict__ out)
{
    const int i = blockIdx.x, m = blockIdx.y;
    const int2 yx = valid[i];
    float *dst = out + ((size_t)i * Mp + m) * (n * n);
    for (int q = threadIdx.x; q < n * n; q += blockDim.x) {
        const int j = q / n, k = q - j * n;
        dst[q] = m < M ? modes[(size_t)m * N * N + (size_t)(yx.x * n + j) * N + yx.y * n + k] : 0.f;
    }
}

__global__ void pad_coef_kernel(const float *__restrict__ coef, int T, int M, int Mp, float *__restrict__ out)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= T * Mp) return;
    const int t = idx / Mp, m = idx - t * Mp;
    out[idx] = m < M ? coef[(size_t)t * M + m] : 0.f;
}

__global__ void copy_kernel(const float *__restrict__ in, int n, float *__restrict__ out)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < n) out[idx] = in[idx];
}

/* coef[t][m] += gain * sum_k R[m][k] * s[t][k].  One warp per mode m; frames in tiles of TT so that a row of
 * R is read once per tile.  hist (optional, T == 1 only): hist[m] = coef[m] BEFORE the update (reading C4). */
constexpr int RC_WARPS = 4;
constexpr int RC_TT = 8;

__global__ void __launch_bounds__(32 * RC_WARPS) recon_kernel(const float *__restrict__ R,
                                                              const float *__restrict__ s, int T, int K, int M,
                                                              float gain, float *__restrict__ coef, int ldc,
                                                              float *__restrict__ hist)
{
    const int lane = threadIdx.x & 31;
    const int m = blockIdx.x * RC_WARPS + (threadIdx.x >> 5);
    if (m >= M) return;
    const float2 *row = reinterpret_cast<const float2 *>(R + (size_t)m * K);
    const int K2 = K >> 1;                                   /* K = 2 * nsub is even */
    for (int t0 = 0; t0 < T; t0 += RC_TT) {
        float acc[RC_TT];
#pragma unroll
        for (int q = 0; q < RC_TT; ++q) acc[q] = 0.f;
        for (int k = lane; k < K2; k += 32) {
            const float2 r = __ldg(row + k);
#pragma unroll
            for (int q = 0; q < RC_TT; ++q) {
                if (t0 + q < T) {
                    const float2 v = __ldg(reinterpret_cast<const float2 *>(s + (size_t)(t0 + q) * K) + k);
                    acc[q] = fmaf(r.x, v.x, fmaf(r.y, v.y, acc[q]));
                }
            }
        }
#pragma unroll
        for (int q = 0; q < RC_TT; ++q) {
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
        }
        if (lane == 0) {
#pragma unroll
            for (int q = 0; q < RC_TT; ++q) {
                if (t0 + q < T) {
                    float *c = coef + (size_t)(t0 + q) * ldc + m;
                    const float old = *c;
                    if (hist) hist[(size_t)(t0 + q) * M + m] = old;
                    *c = fmaf(gain, acc[q], old);
                }
            }
        }
    }
}

}  // namespace

cudaError_t shwfs_loop_relayout_modes(shwfs_handle *h, const float *modes_dev, int M, cudaStream_t st)
{
    dim3 grid((unsigned)h->nsub, (unsigned)h->dm_Mp);
    relayout_modes_kernel<<<grid, 128, 0, st>>>(modes_dev, h->d_valid, h->N, h->n, M, h->dm_Mp, h->d_dm_modes);
    return cudaGetLastError();
}

cudaError_t shwfs_loop_pad_coef(const float *coef, int T, int M, int Mp, float *out, cudaStream_t st)
{
    const int total = T * Mp;
    pad_coef_kernel<<<(total + 255) / 256, 256, 0, st>>>(coef, T, M, Mp, out);
    return cudaGetLastError();
}

cudaError_t shwfs_loop_unpad_coef(const float *padded, int M, float *out, cudaStream_t st)
{
    copy_kernel<<<(M + 255) / 256, 256, 0, st>>>(padded, M, out);
    return cudaGetLastError();
}

cudaError_t shwfs_loop_reconstruct(const float *R, const float *slopes, int T, int K, int M, float gain,
                                   float *coef, int ldc, float *hist, cudaStream_t st)
{
    recon_kernel<<<(M + RC_WARPS - 1) / RC_WARPS, 32 * RC_WARPS, 0, st>>>(R, slopes, T, K, M, gain, coef, ldc, hist);
    return cudaGetLastError();
}
