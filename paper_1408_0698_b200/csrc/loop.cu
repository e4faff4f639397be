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
 *   after the path    d[t,m] = sum_k R[m,k] s[t,k] (k = 2 i + axis), c += gain * d: recon_kernel, one CTA
 *                     per mode, the row of R split over its threads, shuffle + shared-memory reduction.
 * shwfs_closed_loop chains the two, frame after frame, on the caller's stream (readings C1..C4 of DESIGN.md).
 */
#include <cuda_pipeline.h>
#include <stdlib.h>

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
 * coefficient tile transposed so that a thread's FT frames are one 16-byte broadcast load; two stages filled
 * by cp.async so that the loads of chunk c+1 overlap the arithmetic of chunk c.  FT = 8 for
 * batches (register tile 8 frames x 4 pixels, FT = 4 up to 32 frames; n*n is a template parameter so that every shared-memory
 * offset is an immediate and the k loop is branch-free), FT = 1 for the T = 1 loop step,
 * which is bound by streaming the mode table.                                                          */
constexpr int DM_MC = 16;

template <int FT, int NN>
__global__ void __launch_bounds__(256) dm_phase_kernel(const float *__restrict__ coef, int ldc,
                                                       const float *__restrict__ modes_sub, int T, int nsub, int M,
                                                       float *__restrict__ out)
{
    constexpr int TT = 8 * FT, NQ = NN / 4, MAXQ = (NQ + 31) / 32;
    constexpr int TS = TT + 4;                              /* padded row of the transposed coefficient tile */
    constexpr int STAGE = DM_MC * NN + DM_MC * TS;          /* [DM_MC][NN] modes, then [DM_MC][TS] coefficients */
    extern __shared__ __align__(16) float dm_smem[];
    const int i = blockIdx.y, t0 = blockIdx.x * TT;        /* frame tiles of one subaperture are neighbours: */
    const int tid = threadIdx.x, fy = tid >> 5, lane = tid & 31;   /* its mode slice is re-read from L2       */
    float4 acc[MAXQ][FT];
#pragma unroll
    for (int c = 0; c < MAXQ; ++c)
#pragma unroll
        for (int f = 0; f < FT; ++f) acc[c][f] = make_float4(0.f, 0.f, 0.f, 0.f);
    const float *mi = modes_sub + (size_t)i * M * NN;

    /* cp.async (LDGSTS) one chunk of modes and the transposed coefficient tile into stage `st`; rows past M
     * and frames past T are zero-filled so that the arithmetic below needs no bounds */
    auto issue = [&](int st, int m0) {
        float *sm_modes = dm_smem + st * STAGE, *sm_coef = sm_modes + DM_MC * NN;
        const int mc = min(DM_MC, M - m0);
        const float4 *src = reinterpret_cast<const float4 *>(mi + (size_t)m0 * NN);
        for (int q = tid; q < DM_MC * NQ; q += 256) {
            const bool ok = q < mc * NQ;
            __pipeline_memcpy_async(reinterpret_cast<float4 *>(sm_modes) + q, ok ? src + q : src, 16, ok ? 0 : 16);
        }
        for (int q = tid; q < DM_MC * TT; q += 256) {
            const int f = q / DM_MC, k = q - f * DM_MC;      /* consecutive threads: consecutive modes of a frame */
            const bool ok = k < mc && t0 + f < T;
            __pipeline_memcpy_async(sm_coef + k * TS + f, ok ? coef + (size_t)(t0 + f) * ldc + m0 + k : coef, 4,
                                    ok ? 0 : 4);
        }
        __pipeline_commit();
    };

    const int nchunk = (M + DM_MC - 1) / DM_MC;
    issue(0, 0);
    for (int ch = 0; ch < nchunk; ++ch) {
        if (ch + 1 < nchunk) { issue((ch + 1) & 1, (ch + 1) * DM_MC); __pipeline_wait_prior(1); }
        else __pipeline_wait_prior(0);
        __syncthreads();
        const float *sm_modes = dm_smem + (ch & 1) * STAGE, *sm_coef = sm_modes + DM_MC * NN;
#pragma unroll
        for (int k = 0; k < DM_MC; ++k) {
            float a[FT];
            if (FT % 4 == 0) {
#pragma unroll
                for (int f4 = 0; f4 < FT / 4; ++f4) {
                    const float4 v = *reinterpret_cast<const float4 *>(sm_coef + k * TS + fy * FT + 4 * f4);
                    a[(4 * f4) % FT] = v.x; a[(4 * f4 + 1) % FT] = v.y; a[(4 * f4 + 2) % FT] = v.z; a[(4 * f4 + 3) % FT] = v.w;
                }
            } else {
#pragma unroll
                for (int f = 0; f < FT; ++f) a[f] = sm_coef[k * TS + fy * FT + f];
            }
#pragma unroll
            for (int c = 0; c < MAXQ; ++c) {
                const int cq = lane + 32 * c;
                if ((c + 1) * 32 <= NQ || cq < NQ) {
                    const float4 b = *reinterpret_cast<const float4 *>(sm_modes + k * NN + 4 * cq);
#pragma unroll
                    for (int f = 0; f < FT; ++f) {
                        acc[c][f].x = fmaf(a[f], b.x, acc[c][f].x); acc[c][f].y = fmaf(a[f], b.y, acc[c][f].y);
                        acc[c][f].z = fmaf(a[f], b.z, acc[c][f].z); acc[c][f].w = fmaf(a[f], b.w, acc[c][f].w);
                    }
                }
            }
        }
        __syncthreads();                                    /* stage (ch & 1) is refilled two chunks later */
    }
#pragma unroll
    for (int c = 0; c < MAXQ; ++c) {
        const int cq = lane + 32 * c;
        if (cq < NQ) {
#pragma unroll
            for (int f = 0; f < FT; ++f) {
                const int t = t0 + fy * FT + f;
                if (t < T) reinterpret_cast<float4 *>(out + ((size_t)t * nsub + i) * NN)[cq] = acc[c][f];
            }
        }
    }
}

template <int FT, int NN>
void launch_dm_phase(shwfs_handle *h, const float *coef, int ldc, int T, float *out, cudaStream_t st)
{
    constexpr int TT = 8 * FT;
    const size_t smem = 2 * sizeof(float) * (size_t)(DM_MC * NN + DM_MC * (TT + 4));
    dm_phase_kernel<FT, NN><<<dim3((unsigned)((T + TT - 1) / TT), (unsigned)h->nsub), 256, smem, st>>>(
        coef, ldc, h->d_dm_modes, T, h->nsub, h->dm_M, out);
}

template <int NN, int FMAX>
__global__ void dm_phase_gemv_kernel(const float *__restrict__ coef, int ldc, const float *__restrict__ modes_sub,
                                     int T, int nsub, int M, float *__restrict__ out);

template <int NN, int FMAX>
void launch_dm_gemv(shwfs_handle *h, const float *coef, int ldc, int T, float *out, cudaStream_t st)
{
    dm_phase_gemv_kernel<NN, FMAX><<<(unsigned)((h->nsub + 7) / 8), 256, sizeof(float) * FMAX * (size_t)h->dm_M, st>>>(
        coef, ldc, h->d_dm_modes, T, h->nsub, h->dm_M, out);
}

template <int NN>
void launch_dm_phase_n(shwfs_handle *h, const float *coef, int ldc, int T, float *out, cudaStream_t st)
{
    if (T <= 8 && (size_t)h->dm_M * 8 * sizeof(float) <= 48 * 1024) {
        /* accumulators for exactly as many frames as needed: the T = 1 loop step keeps 1 + 8 float4 live and
         * fits five CTAs per SM, i.e. the whole table in one wave */
        if (T == 1) launch_dm_gemv<NN, 1>(h, coef, ldc, T, out, st);
        else if (T == 2) launch_dm_gemv<NN, 2>(h, coef, ldc, T, out, st);
        else if (T <= 4) launch_dm_gemv<NN, 4>(h, coef, ldc, T, out, st);
        else launch_dm_gemv<NN, 8>(h, coef, ldc, T, out, st);
    } else if (T <= 8) launch_dm_phase<1, NN>(h, coef, ldc, T, out, st);
    else if (T <= 32) launch_dm_phase<4, NN>(h, coef, ldc, T, out, st);
    else launch_dm_phase<8, NN>(h, coef, ldc, T, out, st);
}

/* any other n: one thread per output element */
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

/* Few frames (the T = 1 loop step): the product is a matrix-vector one, bound by streaming the mode table
 * once.  One warp per subaperture, lane = float4 column, eight independent 16-byte loads in flight per lane,
 * the coefficients of the <= 8 frames broadcast from shared memory.                                      */
template <int NN, int FMAX>
__global__ void __launch_bounds__(256) dm_phase_gemv_kernel(const float *__restrict__ coef, int ldc,
                                                            const float *__restrict__ modes_sub, int T, int nsub,
                                                            int M, float *__restrict__ out)
{
    constexpr int NQ = NN / 4, MAXQ = (NQ + 31) / 32, UN = 8;
    extern __shared__ float gv_coef[];                       /* [M][FMAX] */
    for (int q = threadIdx.x; q < M * FMAX; q += 256) {
        const int m = q / FMAX, f = q - m * FMAX;
        gv_coef[q] = f < T ? __ldg(coef + (size_t)f * ldc + m) : 0.f;
    }
    __syncthreads();
    const int i = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (i >= nsub) return;
    const float4 *mi = reinterpret_cast<const float4 *>(modes_sub + (size_t)i * M * NN);
#pragma unroll
    for (int c = 0; c < MAXQ; ++c) {
        const int cq = lane + 32 * c;
        if (cq >= NQ) continue;
        float4 acc[FMAX];
#pragma unroll
        for (int f = 0; f < FMAX; ++f) acc[f] = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int m0 = 0; m0 < M; m0 += UN) {
            float4 b[UN];
#pragma unroll
            for (int u = 0; u < UN; ++u)
                b[u] = m0 + u < M ? __ldg(mi + (size_t)(m0 + u) * NQ + cq) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                if (m0 + u < M) {
                    const float *a = gv_coef + (m0 + u) * FMAX;
#pragma unroll
                    for (int f = 0; f < FMAX; ++f) {
                        if (f < T) {
                            acc[f].x = fmaf(a[f], b[u].x, acc[f].x); acc[f].y = fmaf(a[f], b[u].y, acc[f].y);
                            acc[f].z = fmaf(a[f], b[u].z, acc[f].z); acc[f].w = fmaf(a[f], b[u].w, acc[f].w);
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int f = 0; f < FMAX; ++f)
            if (f < T) reinterpret_cast<float4 *>(out + ((size_t)f * nsub + i) * NN)[cq] = acc[f];
    }
}

/* coef[t][m] += gain * sum_k R[m][k] * s[t][k].  One CTA per mode m, its 256 threads split the row of R
 * (8-byte loads, frames in register tiles of RC_TT so that the row is read once per tile), warp-shuffle then
 * shared-memory reduction.  hist (optional): hist[t][m] = coef[t][m] BEFORE the update (reading C4).     */
constexpr int RC_TT = 8;

template <int RC_THREADS>
__global__ void __launch_bounds__(RC_THREADS) recon_kernel(const float *__restrict__ R, const float *__restrict__ s,
                                                           int T, int K, int M, float gain,
                                                           float *__restrict__ coef, int ldc, float *__restrict__ hist)
{
    __shared__ float part[RC_THREADS / 32][RC_TT];
    const int m = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float2 *row = reinterpret_cast<const float2 *>(R + (size_t)m * K);
    const int K2 = K >> 1;                                   /* K = 2 * nsub is even */
    for (int t0 = 0; t0 < T; t0 += RC_TT) {
        float acc[RC_TT];
#pragma unroll
        for (int q = 0; q < RC_TT; ++q) acc[q] = 0.f;
#pragma unroll 4
        for (int k = tid; k < K2; k += RC_THREADS) {
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
        __syncthreads();                                     /* previous tile's partials are consumed */
        if (lane == 0) {
#pragma unroll
            for (int q = 0; q < RC_TT; ++q) part[warp][q] = acc[q];
        }
        __syncthreads();
        if (tid < RC_TT && t0 + tid < T) {
            float d = 0.f;
#pragma unroll
            for (int w = 0; w < RC_THREADS / 32; ++w) d += part[w][tid];
            float *c = coef + (size_t)(t0 + tid) * ldc + m;
            const float old = *c;
            if (hist) hist[(size_t)(t0 + tid) * M + m] = old;
            *c = fmaf(gain, d, old);
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
    /* batches go to the tensor cores (dm_umma.cu) when the split operand tiles exist; SHWFS_DM_FP32=1 keeps the
     * FP32 SIMT GEMM below (A/B comparisons) */
    if (T > 8 && h->d_um_modes && h->d_um_coef && h->um_coef_cap >= shwfs_umma_coef_floats(T, M) &&
        !h->dm_fp32)
        return shwfs_umma_dm_phase(h, coef, ldc, T, out, st);
    if (h->nsub <= 65535 && (nn == 64 || nn == 100 || nn == 256)) {
        switch (nn) {
        case 64: launch_dm_phase_n<64>(h, coef, ldc, T, out, st); break;
        case 100: launch_dm_phase_n<100>(h, coef, ldc, T, out, st); break;
        default: launch_dm_phase_n<256>(h, coef, ldc, T, out, st); break;
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
    /* the loop step (a frame or two): 1024 threads put the whole row of R in flight at once -- the kernel is one
     * L2 round trip deep instead of five; batches reuse each row element over 8 frames and are fine with 256 */
    if (T <= 2) recon_kernel<1024><<<M, 1024, 0, st>>>(R, slopes, T, K, M, gain, coef, ldc, hist);
    else recon_kernel<256><<<M, 256, 0, st>>>(R, slopes, T, K, M, gain, coef, ldc, hist);
    return cudaGetLastError();
}
