/*
 * pruned_fft.cu -- the Shack-Hartmann chain WITHOUT elongation kernels (NGS case: "The WF is
 * split into sub-apertures and the spot computed by FFT for each sensor sub-aperture ... the centroid
 * computed on the final image to retrieve the slopes"), as one input-pruned P x P FFT per spot, sm_100a.
 *
 * Steps H1 gather, H2 field, H3 zero-padded P x P DFT, H4 |.|^2/P^2, H6 centre + b x b bin, H7 threshold,
 * H8 centre of gravity of include/shwfs.h, D = P/b = 16 detector pixels per side.
 *
 * Thread mapping: 16 threads (a half-warp) per spot, 8 spots per tile, persistent CTAs striding over the tiles
 * (the gather of the next tile is issued before the column pass of the current one), no CTA-wide barrier.
 *   row pass     thread r < n owns patch row r: 8-byte gathers, sincos, one P-point DIF FFT in registers
 *                whose inputs >= NZ are known zeros (first stage free); the n x P result goes to shared
 *                memory with the columns permuted (u -> (u mod b) * 16 + u / b) so that the column pass
 *                reads conflict-free.  Rows >= n are zero and are never transformed.
 *   column pass  thread c owns the b adjacent columns b*c .. b*c+b-1 = detector column c ^ 8: for each, an
 *                NZ-input P-point FFT down the column, |.|^2, and the row half of the b x b bin
 *                accumulated in registers at compile-time positions (the roll by P/2 is an xor, the
 *                bit reversal of the DIF output a renaming).  The thread ends with one detector column.
 *   H7 + H8      cog16 (cog.cuh): max / sums by xor shuffles inside the half-warp; lane 0 writes 8 bytes.
 * Only the phase patch is read from and the two slopes written to HBM.
 */
#include "internal.h"
#include "fft_regs.cuh"
#include "field.cuh"
#include "cog.cuh"

namespace {

using namespace shwfs;

constexpr int PF_THREADS = 128;
constexpr int PF_SPOTS = PF_THREADS / 16;

struct PfArgs {
    const float *phase;
    const float *amp;
    const int2 *valid;
    float *slopes;
    float *binned;            /* stage-2 debug image [T*nsub*16*16] or null */
    long long frame_stride;
    int T, N, nsub, total, n;
    float tau, turns, ramp_unit;
};

template <int P, int NZ>
struct PfCfg {
    static constexpr int b = P / 16;
    static constexpr int LD = 2 * P + 4;                 /* floats per stored row; LD/4 odd => STS.128 conflict-free */
    static constexpr int TILE = NZ * LD;                 /* floats per spot */
    static constexpr size_t SMEM = sizeof(float) * (size_t)PF_SPOTS * TILE;
    static_assert(P == 16 || P == 32 || P == 64, "P must be 16, 32 or 64 (D = 16)");
    static_assert(NZ <= 16 && NZ <= P && NZ % 2 == 0, "at most 16 non-zero rows, one per thread");
};

/* position of column u in a stored row: the b columns of one detector column are P/b apart */
template <int P>
__host__ __device__ constexpr int col_pos(int u) { return (u % (P / 16)) * 16 + u / (P / 16); }

/* H1 of one spot row: the NZ/2 pixel pairs of patch row r of spot g (zeros when the row does not exist) */
template <int NZ>
__device__ __forceinline__ void pf_gather(const PfArgs &A, int off, int t, float2 (&ph)[NZ / 2], float2 (&am)[NZ / 2])
{
#pragma unroll
    for (int q = 0; q < NZ / 2; ++q) { ph[q] = make_float2(0.f, 0.f); am[q] = make_float2(0.f, 0.f); }
    if (off >= 0) {                         /* off: pixel offset of this thread's patch row, -1 if there is none */
        const float2 *pp = reinterpret_cast<const float2 *>(A.phase + (size_t)t * A.frame_stride + off);
        const float2 *pa = reinterpret_cast<const float2 *>(A.amp + off);
#pragma unroll
        for (int q = 0; q < NZ / 2; ++q)
            if (2 * q < A.n) { ph[q] = __ldg(pp + q); am[q] = __ldg(pa + q); }
    }
}


template <int P, int NZ, int MODE>
__global__ void __launch_bounds__(PF_THREADS, P == 64 ? 2 : 4) pruned_fft_kernel(const PfArgs A)
{
    using Cfg = PfCfg<P, NZ>;
    constexpr int b = Cfg::b, LD = Cfg::LD, HP = P / 2;
    extern __shared__ __align__(16) float pf_smem[];
    const int tid = threadIdx.x, sp = tid >> 4, r = tid & 15;
    float *tile = pf_smem + sp * Cfg::TILE;

    /* persistent CTAs: CTA b takes tiles b, b + gridDim.x, ... (the host sizes the grid to the resident CTAs of
     * the device, so a launch has no ragged last wave).  Two tiles of look-ahead: the valid-list lookup (the
     * only dependent load of the gather) of tile k+2 and the gather of tile k+1 fly during tile k. */
    const int ntiles = (A.total + PF_SPOTS - 1) / PF_SPOTS;
    auto row_offset = [&](int tile_id, int &tt) {
        const int g = tile_id * PF_SPOTS + sp;
        tt = 0;
        if (tile_id >= ntiles || g >= A.total || r >= A.n) return -1;
        const int i = g / A.T;
        const int2 yx = __ldg(A.valid + i);
        tt = g - i * A.T;
        return (yx.x * A.n + r) * A.N + yx.y * A.n;
    };
    int tt0, tt1;
    int off0 = row_offset(blockIdx.x, tt0);
    int off1 = row_offset(blockIdx.x + gridDim.x, tt1);
    float2 ph[NZ / 2], am[NZ / 2];
    pf_gather<NZ>(A, off0, tt0, ph, am);

#pragma unroll 1
    for (int tile_id = blockIdx.x; tile_id < ntiles; tile_id += gridDim.x) {
        const int g = tile_id * PF_SPOTS + sp;
        const bool live = g < A.total;
        int i = 0, t = 0;
        if (live) { i = g / A.T; t = g - i * A.T; }

        float re[P], im[P];

        /* ---- row pass: H2 field, P-point FFT of row r (inputs >= NZ are zero) ---- */
        if (r < NZ) {
            if (live && r < A.n) {
#pragma unroll
                for (int q = 0; q < NZ / 2; ++q) {
                    const float ramp = (float)(r + 2 * q) * A.ramp_unit;
                    const float2 e0 = field_value(ph[q].x, am[q].x, A.turns, ramp);
                    const float2 e1 = field_value(ph[q].y, am[q].y, A.turns, ramp + A.ramp_unit);
                    re[2 * q] = e0.x; im[2 * q] = e0.y;
                    re[2 * q + 1] = e1.x; im[2 * q + 1] = e1.y;
                }
#pragma unroll
                for (int k = NZ; k < P; ++k) { re[k] = 0.f; im[k] = 0.f; }
                fft_fma<P, -1, NZ>(re, im);
            } else {
#pragma unroll
                for (int k = 0; k < P; ++k) { re[k] = 0.f; im[k] = 0.f; }
            }
            float4 *row = reinterpret_cast<float4 *>(tile + r * LD);
#pragma unroll
            for (int q = 0; q < P / 2; ++q) {
                /* stored positions 2q, 2q+1 hold columns u0, u1 (inverse of col_pos) */
                const int p0 = 2 * q, p1 = 2 * q + 1;
                const int u0 = (p0 % 16) * b + p0 / 16, u1 = (p1 % 16) * b + p1 / 16;
                const int x0 = fft_out_index<P>(u0), x1 = fft_out_index<P>(u1);
                row[q] = make_float4(re[x0], im[x0], re[x1], im[x1]);
            }
        }
        __syncwarp();
        /* H1 of the next tile: in flight during the column pass */
        pf_gather<NZ>(A, off1, tt1, ph, am);
        off1 = row_offset(tile_id + 2 * gridDim.x, tt1);

        /* ---- column pass: b columns per thread, |.|^2 and the row half of the bin in registers ---- */
        float acc[16];
#pragma unroll
        for (int R = 0; R < 16; ++R) acc[R] = 0.f;
#pragma unroll
        for (int be = 0; be < b; ++be) {
            const float2 *colp = reinterpret_cast<const float2 *>(tile) + be * 16 + r;
#pragma unroll
            for (int v = 0; v < NZ; ++v) {
                const float2 f = colp[v * (LD / 2)];
                re[v] = f.x; im[v] = f.y;
            }
#pragma unroll
            for (int v = NZ; v < P; ++v) { re[v] = 0.f; im[v] = 0.f; }
            fft_fma<P, -1, NZ>(re, im);
#pragma unroll
            for (int R = 0; R < 16; ++R) {
#pragma unroll
                for (int al = 0; al < b; ++al) {
                    const int x = fft_out_index<P>((R * b + al) ^ HP);      /* H6: roll by P/2, then bin */
                    acc[R] = fmaf(re[x], re[x], fmaf(im[x], im[x], acc[R]));
                }
            }
        }
        constexpr float inv_pp = 1.0f / ((float)P * (float)P);
#pragma unroll
        for (int R = 0; R < 16; ++R) acc[R] *= inv_pp;

        /* ---- H7 + H8: thread r holds detector column C = r ^ 8 ---- */
        const int C = r ^ 8;
        const float2 sl = cog16<MODE>(acc, C, A.tau);
        if (live) {
            const size_t o = (size_t)t * A.nsub + i;
            if (r == 0) reinterpret_cast<float2 *>(A.slopes)[o] = sl;
            if (A.binned) {
#pragma unroll
                for (int R = 0; R < 16; ++R) A.binned[(o * 16 + R) * 16 + C] = acc[R];
            }
        }
        __syncwarp();                                      /* the tile is rewritten by the next row pass */
    }
}

template <int P, int NZ, int MODE>
cudaError_t launch_pf_mode(const PfArgs &A, cudaStream_t st)
{
    using Cfg = PfCfg<P, NZ>;
    if (Cfg::SMEM > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(pruned_fft_kernel<P, NZ, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
    }
    const int ntiles = (A.total + PF_SPOTS - 1) / PF_SPOTS;
    static int resident = 0;                       /* CTAs the device holds at once */
    if (resident == 0) {
        int dev = 0, sms = 0, per_sm = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pruned_fft_kernel<P, NZ, MODE>, PF_THREADS, Cfg::SMEM);
        resident = sms * (per_sm > 0 ? per_sm : 1);
    }
    const int grid = ntiles < resident ? ntiles : resident;
    pruned_fft_kernel<P, NZ, MODE><<<grid, PF_THREADS, Cfg::SMEM, st>>>(A);
    return cudaGetLastError();
}

template <int P, int NZ>
cudaError_t launch_pf(const PfArgs &A, int mode, cudaStream_t st)
{
    return mode == 0 ? launch_pf_mode<P, NZ, 0>(A, st) : launch_pf_mode<P, NZ, 1>(A, st);
}

}  // namespace

int shwfs_pruned_fft_supported(const shwfs_handle *h)
{
    return !h->has_kernels && h->D == 16 && (h->P == 16 || h->P == 32 || h->P == 64) && h->n <= 16 && h->n % 2 == 0;
}

cudaError_t shwfs_pruned_fft_launch(shwfs_handle *h, const float *phase, int T, float *slopes, float *binned,
                                    cudaStream_t st)
{
    PfArgs A;
    A.phase = phase; A.amp = h->d_amp; A.valid = h->d_valid; A.slopes = slopes; A.binned = binned;
    A.frame_stride = (long long)h->N * h->N;
    A.T = T; A.N = h->N; A.nsub = h->nsub; A.total = T * h->nsub; A.n = h->n;
    A.tau = h->tau;
    A.turns = (float)((double)h->c_phi / 6.283185307179586476925286766559);
    A.ramp_unit = 0.5f / (float)h->P;
    if (A.total == 0) return cudaSuccess;
    h->launches += 1;
    switch (h->P) {
    case 16: return h->n <= 8 ? launch_pf<16, 8>(A, h->mode, st) : launch_pf<16, 16>(A, h->mode, st);
    case 32: return launch_pf<32, 16>(A, h->mode, st);
    case 64: return launch_pf<64, 16>(A, h->mode, st);
    default: return cudaErrorInvalidValue;
    }
}
