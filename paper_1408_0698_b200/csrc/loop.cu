/*
 * loop.cu -- the closed-loop neighbours of the Shack-Hartmann path, sm_100a.
 *
 * "The WFS modules compute the vector signals (X-and Y- slopes) from the residual phase (the
 * open loop wavefront subtracted by the DM).  Vector slopes multiplied by the control matrix returns the
 * vector coefficients for the modal base linear composition, in the form of the differential coefficients
 * to be added to the one defining the existing mirror shape.  [...] a pure integrator scheme".
 *
 *   before the path   DM phase sum_m c[t,m] mode[m] on the valid subapertures only, in patch layout
 *                     [T][nsub][n*n]: dm_phase_kernel, a batched FP32 GEMM C_i[T x n^2] = c[T x M] *
 *                     modes_i[M x n^2] over a per-subaperture re-layout of the modes built once per
 *                     shwfs_set_dm (contiguous, coalesced, L2-friendly); the sensor kernel's gather (wk.cu,
 *                     EXT instances) subtracts it from the wavefront, so the full-frame residual never
 *                     exists in memory;
 *   after the path    d[t,m] = sum_k R[m,k] s[t,k] (k = 2 i + axis), c += gain * d: recon_kernel, one warp
 *                     per mode, the slope vector streamed with 8-byte loads, warp-shuffle reduction.
 * shwfs_closed_loop chains the two, frame after frame, on the caller's stream (readings C1..C4 of DESIGN.md).
 */
#include "internal.h"

namespace {

/* modes[M][N][N] -> out[nsub][M][n*n]: block = (subaperture, mode) */
__global__ void relayout_modes_kernel(const float *__restrict__ modes, const int2 *__restrict__ valid, int N,
                                      int n, int M, float *__restrict__ out)
{
    const int i = blockIdx.x, m = blockIdx.y;
    const int2 yx = valid[i];
    float *dst = out + ((size_t)i * M + m) * (n * n);
    for (int q = threadIdx.x; q < n * n; q += blockDim.x) {
        const int j = q / n, k = q - j * n;
        dst[q] = modes[(size_t)m * N * N + (size_t)(yx.x * n + j) * N + yx.y * n + k];
    }
}

/* DM phase in patch layout: out[t][i][q] = sum_m coef[t*ldc + m] * modes_sub[i][m][q], q < n*n (n*n % 4 == 0).
 * CTA = (subaperture i, tile of TT = 8*FT frames), 256 threads = 8 frame groups x 32 float4 columns; modes
 * of MC at a time go through shared memory (one contiguous, coalesced block of the re-laid table), the
 * coefficient tile transposed so that a thread's FT frames are one 16-byte broadcast load.  FT = 4 for
 * batches (register tile 4 frames x 4 pixels, 16 FFMA per two LDS.128), FT = 1 for the T = 1 loop step,
 * which is bound by streaming the mode table.                                                          */
constexpr int DM_MC = 16;

template <int FT>
__global__ void __launch_bounds__(256) dm_phase_kernel(const float *__restrict__ coef, int ldc,
                                                       const float *__restrict__ modes_sub, int T, int nsub, int nn,
                                                       int M, float *__restrict__ out)
{
    constexpr int TT = 8 * FT;
    extern __shared__ __align__(16) float dm_smem[];
    float *sm_modes = dm_smem;                      /* [DM_MC][nn]  */
    float *sm_coef = dm_smem + DM_MC * nn;          /* [DM_MC][TT]  */
    const int i = blockIdx.x, t0 = blockIdx.y * TT;
    const int tid = threadIdx.x, fy = tid >> 5, lane = tid & 31;
    const int NQ = nn >> 2;
    constexpr int MAXQ = 2;                         /* columns per lane: nn <= 256 */
    float4 acc[MAXQ][FT];
#pragma unroll
    for (int c = 0; c < MAXQ; ++c)
#pragma unroll
        for (int f = 0; f < FT; ++f) acc[c][f] = make_float4(0.f, 0.f, 0.f, 0.f);
    const float *mi = modes_sub + (size_t)i * M * nn;
    for (int m0 = 0; m0 < M; m0 += DM_MC) {
        const int mc = min(DM_MC, M - m0);
        __syncthreads();
        {
            const float4 *src = reinterpret_cast<const float4 *>(mi + (size_t)m0 * nn);
            float4 *dst = reinterpret_cast<float4 *>(sm_modes);
            for (int q = tid; q < mc * NQ; q += 256) dst[q] = __ldg(src + q);
            for (int q = tid; q < DM_MC * TT; q += 256) {
                const int k = q / TT, f = q - k * TT;
                sm_coef[q] = (k < mc && t0 + f < T) ? __ldg(coef + (size_t)(t0 + f) * ldc + m0 + k) : 0.f;
            }
        }
        __syncthreads();
#pragma unroll 4
        for (int k = 0; k < mc; ++k) {
            float a[FT];
            if (FT == 4) {
                const float4 v = *reinterpret_cast<const float4 *>(sm_coef + k * TT + fy * FT);
                a[0] = v.x; a[1 % FT] = v.y; a[2 % FT] = v.z; a[3 % FT] = v.w;
            } else {
#pragma unroll
                for (int f = 0; f < FT; ++f) a[f] = sm_coef[k * TT + fy * FT + f];
            }
#pragma unroll
            for (int c = 0; c < MAXQ; ++c) {
                const int cq = lane + 32 * c;
                if (cq < NQ) {
                    const float4 b = *reinterpret_cast<const float4 *>(sm_modes + k * nn + 4 * cq);
#pragma unroll
                    for (int f = 0; f < FT; ++f) {
                        acc[c][f].x = fmaf(a[f], b.x, acc[c][f].x); acc[c][f].y = fmaf(a[f], b.y, acc[c][f].y);
                        acc[c][f].z = fmaf(a[f], b.z, acc[c][f].z); acc[c][f].w = fmaf(a[f], b.w, acc[c][f].w);
                    }
                }
            }
        }
    }
#pragma unroll
    for (int c = 0; c < MAXQ; ++c) {
        const int cq = lane + 32 * c;
        if (cq < NQ) {
#pragma unroll
            for (int f = 0; f < FT; ++f) {
                const int t = t0 + fy * FT + f;
                if (t < T) reinterpret_cast<float4 *>(out + ((size_t)t * nsub + i) * nn)[cq] = acc[c][f];
            }
        }
    }
}

/* any n (n*n not a multiple of 4, or > 256): one thread per output element */
__global__ void dm_phase_simple_kernel(const float *__restrict__ coef, int ldc, const float *__restrict__ modes_sub,
                                       int T, int nsub, int nn, int M, float *__restrict__ out)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)T * nsub * nn) return;
    const int q = (int)(idx % nn), i = (int)((idx / nn) % nsub), t = (int)(idx / ((size_t)nn * nsub));
    const float *mp = modes_sub + (size_t)i * M * nn + q;
    float acc = 0.f;
    for (int m = 0; m < M; ++m) acc = fmaf(coef[(size_t)t * ldc + m], mp[(size_t)m * nn], acc);
    out[idx] = acc;
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
    dim3 grid((unsigned)h->nsub, (unsigned)M);
    relayout_modes_kernel<<<grid, 128, 0, st>>>(modes_dev, h->d_valid, h->N, h->n, M, h->d_dm_modes);
    return cudaGetLastError();
}

cudaError_t shwfs_loop_dm_phase(shwfs_handle *h, const float *coef, int ldc, int T, float *out, cudaStream_t st)
{
    const int nn = h->n * h->n, M = h->dm_M;
    if (nn % 4 == 0 && nn <= 256) {
        if (T <= 8) {
            const size_t smem = sizeof(float) * (size_t)(DM_MC * nn + DM_MC * 8);
            dm_phase_kernel<1><<<dim3((unsigned)h->nsub, (unsigned)((T + 7) / 8)), 256, smem, st>>>(
                coef, ldc, h->d_dm_modes, T, h->nsub, nn, M, out);
        } else {
            const size_t smem = sizeof(float) * (size_t)(DM_MC * nn + DM_MC * 32);
            dm_phase_kernel<4><<<dim3((unsigned)h->nsub, (unsigned)((T + 31) / 32)), 256, smem, st>>>(
                coef, ldc, h->d_dm_modes, T, h->nsub, nn, M, out);
        }
    } else {
        const size_t total = (size_t)T * h->nsub * nn;
        dm_phase_simple_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(coef, ldc, h->d_dm_modes, T, h->nsub,
                                                                               nn, M, out);
    }
    return cudaGetLastError();
}

cudaError_t shwfs_loop_reconstruct(const float *R, const float *slopes, int T, int K, int M, float gain,
                                   float *coef, int ldc, float *hist, cudaStream_t st)
{
    recon_kernel<<<(M + RC_WARPS - 1) / RC_WARPS, 32 * RC_WARPS, 0, st>>>(R, slopes, T, K, M, gain, coef, ldc, hist);
    return cudaGetLastError();
}
