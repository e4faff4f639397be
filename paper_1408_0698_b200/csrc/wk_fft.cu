/*
 * wk_fft.cu -- the lag-domain (Wiener-Khinchin) form of the Shack-Hartmann hot path for n = 12, 14, 16, with the
 * autocorrelation of the field computed by FFT instead of by direct sums, sm_100a.
 *
 * Same operation as wk.cu (H1..H8 of include/shwfs.h; "the spot computed by FFT for each sensor
 * sub-aperture ... a convolution for a gaussian ... the centroid computed on the final image"), same table M,
 * same result to fp32 rounding.  What differs is how G[ly,lx] = sum_{j,k} e[j,k] conj(e[j+ly,k+lx]) is
 * obtained: the direct sums cost n^2 (n+1)/2 * n = 32.9 k complex MACs per spot at n = 16 (92 k instructions,
 * profiles/r01_wk16_full_v4.md); on a Q x Q grid with Q = 2n = 32 >= 2n-1 the aperiodic autocorrelation is
 * the periodic one, G = DFT_Q(|DFT_Q(e)|^2) / Q^2, i.e. 80 line transforms of 32 points (~50 k instructions
 * with everything around them).  The grid size is independent of the sensor's padding P: the identity of
 * wk.cu's header holds for any P, and P enters only through the table M.  n = 12 and 14, which have no
 * direct-sum instance, run the same code with the rows, lag rows and table width of their size (threads
 * r >= n idle in steps A, D, E).  n = 8 and 10 are instantiated too: under SHWFS_ALGO_AUTO calls of one or two frames
 * (the closed-loop step, less than a wave of wk.cu's 32-spot CTAs) come here; on batches the direct sums win.
 *
 * Thread mapping: a half-warp per spot, 8 spots per CTA, no CTA-wide barrier; one 16 x 32 complex tile of
 * shared memory per spot is reused by every exchange.
 *   A  thread r owns patch row r: H1 gather (16-byte loads), H2 field (scaled by 2^-5.5 so that the
 *      unnormalised transforms below need no further factor), 32-point FFT of the row (inputs >= 16 are zero)
 *      -> tile[r][u]
 *   B  thread c owns columns c and c + 16: 32-point FFT down each (16 non-zero inputs), S[v][u] = |.|^2; the
 *      two columns run through one copy of the code (a rolled loop): the kernel is straight-line code of
 *      ~3 k instructions per thread and stalls on instruction fetch (ncu: no_instructions first), so code
 *      size counts -- rolling the two columns is worth 4 %, rolling A with B or C with D costs spills
 *   C  the two real columns go through ONE complex transform z = S[.][c] + i S[.][c+16]; the transforms
 *      g_u[ly] of the two columns are separated by the Hermitian symmetry of each (ly = 0..15 is all that
 *      is needed: G[-l] = conj G[l] is folded into M) -> tile[ly][u]
 *   D  thread ly owns lag row ly: 32-point FFT over u -> G[ly][lx], lx = -15..15
 *   E  table product with M_i[ly][.], alias lx mod 16, 16-point x-transform (finish_row of wk_common.cuh)
 *      -> tile[ly][0..15]
 *   F  thread C owns detector column C: 16-point y-transform (real part), optional detector noise, H7 + H8
 *      (cog16) with half-warp shuffles; lane 0 writes the two slopes.
 * The extensions of wk.cu are carried: detector noise, DM residual, sodium sub-layers (several: steps A-C per
 * sub-layer, the separated transforms of S pile up in a second tile per spot, D-F once).
 */
#include "wk_common.cuh"
#include "field.cuh"
#include "cog.cuh"
#include "noise.cuh"

namespace {

using namespace shwfs;

constexpr int WF_ROWS = 16;                    /* tile rows (threads per spot): n <= 16              */
constexpr int WF_Q = 32;                       /* transform grid side                                */
constexpr int WF_THREADS = 128;
constexpr int WF_SPOTS = WF_THREADS / 16;
constexpr int WF_LD = 2 * WF_Q + 4;            /* floats per tile row; LD/4 odd => 16-byte row accesses conflict-free */
constexpr int WF_TILE = WF_ROWS * WF_LD;
constexpr size_t WF_SMEM = sizeof(float) * (size_t)WF_SPOTS * WF_TILE;

__device__ __forceinline__ constexpr int xq(int k) { return fft_out_index<WF_Q>(k & (WF_Q - 1)); }

/* EXTK as in wk.cu: 0 plain sensor, 1 extensions on one (sub-)layer, 2 several sodium sub-layers (S is linear in the
 * sub-layer intensities: steps A-C run per sub-layer and the separated column transforms pile up in a second
 * tile per spot, each element owned by one thread; D-F run once) */
template <int n, int MODE, int EXTK>
__global__ void __launch_bounds__(WF_THREADS, EXTK == 2 ? 3 : 4) wkf_kernel(const WkArgs A)
{
    constexpr bool EXT = EXTK > 0, ML = EXTK == 2;
    static_assert(n % 2 == 0 && n <= WF_ROWS && 2 * n - 1 <= WF_Q, "even n <= 16: one thread per patch row, grid 32 >= 2n-1");
    constexpr int Q = WF_Q, LD = WF_LD, LX = 2 * n - 1;
    extern __shared__ __align__(16) float wf_smem[];
    const int tid = threadIdx.x, sp = tid >> 4, r = tid & 15;
    float *tile = wf_smem + sp * WF_TILE;
    float *gtile = ML ? wf_smem + (WF_SPOTS + sp) * WF_TILE : tile;      /* where step C leaves g_u[ly] */

    const int g = blockIdx.x * WF_SPOTS + sp;
    const bool live = g < A.total;
    int i = 0, t = 0;
    if (live) { i = g / A.T; t = g - i * A.T; }

    float re[Q], im[Q];

    const int n_layers = ML ? A.L : 1;
#pragma unroll 1
    for (int layer = 0; layer < n_layers; ++layer) {
    /* ---- A: gather, field, row transform (threads r < n) ---- */
    if (r < n) {
        float pv[n], av[n];
#pragma unroll
        for (int k = 0; k < n; ++k) { pv[k] = 0.f; av[k] = 0.f; }
        if (live) {
            const int2 yx = __ldg(A.valid + i);
            const int off = (yx.x * n + r) * A.N + yx.y * n;
            const float *pp = A.phase + (size_t)t * A.frame_stride + (ML ? (size_t)layer * A.layer_stride : 0) + off;
            const float *pa = A.amp + off;
            /* PAPER.md:76 "the residual phase (the open loop wavefront subtracted by the DM)" */
            const float *pd = EXT && A.dm_patch != nullptr ? A.dm_patch + ((size_t)t * A.nsub + i) * (n * n) + r * n : nullptr;
            if constexpr (n % 4 == 0) {          /* rows start on 16 bytes */
#pragma unroll
                for (int q = 0; q < n / 4; ++q) {
                    const float4 v = __ldg(reinterpret_cast<const float4 *>(pp) + q);
                    const float4 w = __ldg(reinterpret_cast<const float4 *>(pa) + q);
                    pv[4 * q] = v.x; pv[4 * q + 1] = v.y; pv[4 * q + 2] = v.z; pv[4 * q + 3] = v.w;
                    av[4 * q] = w.x; av[4 * q + 1] = w.y; av[4 * q + 2] = w.z; av[4 * q + 3] = w.w;
                }
                if (EXT && pd != nullptr) {
#pragma unroll
                    for (int q = 0; q < n / 4; ++q) {
                        const float4 d = __ldg(reinterpret_cast<const float4 *>(pd) + q);
                        pv[4 * q] -= d.x; pv[4 * q + 1] -= d.y; pv[4 * q + 2] -= d.z; pv[4 * q + 3] -= d.w;
                    }
                }
            } else {
#pragma unroll
                for (int q = 0; q < n / 2; ++q) {
                    const float2 v = __ldg(reinterpret_cast<const float2 *>(pp) + q);
                    const float2 w = __ldg(reinterpret_cast<const float2 *>(pa) + q);
                    pv[2 * q] = v.x; pv[2 * q + 1] = v.y; av[2 * q] = w.x; av[2 * q + 1] = w.y;
                }
                if (EXT && pd != nullptr) {
#pragma unroll
                    for (int q = 0; q < n / 2; ++q) {
                        const float2 d = __ldg(reinterpret_cast<const float2 *>(pd) + q);
                        pv[2 * q] -= d.x; pv[2 * q + 1] -= d.y;
                    }
                }
            }
        }
        /* 2^-5.5 on the field = 1/2048 on the intensity: 1/Q^2 of the two unnormalised transforms of S and the
         * 1/2 of the real-pair separation of step C */
        float sc = 0.02209708691207961f;
        float lin0 = 0.f, gx = 0.f, lq = 0.f, dj2 = 0.f;
        const bool sodium = EXT && A.L > 0;
        if (sodium) {
            /* the sub-layer's analytic phase in turns (reading B1): g . d + q |d|^2, d from the patch centre */
            const float2 gr = __ldg(A.sod_g + (size_t)layer * A.nsub + i);
            const float dj = (float)r - 0.5f * (float)(n - 1);
            lq = A.sod_q[layer];
            gx = gr.x;
            lin0 = fmaf(gr.y, dj, gr.x * (-0.5f * (float)(n - 1)));
            dj2 = dj * dj;
            sc *= A.sod_sw[layer];
        }
#pragma unroll
        for (int k = 0; k < n; ++k) {
            float ramp = (float)(r + k) * A.ramp_unit;
            if (sodium) {
                const float dk = (float)k - 0.5f * (float)(n - 1);
                ramp -= fmaf(gx, (float)k, lin0) + lq * (dj2 + dk * dk);
            }
            const float2 e = field_value(pv[k], av[k] * sc, A.turns, ramp);
            re[k] = e.x; im[k] = e.y;
        }
#pragma unroll
        for (int k = n; k < Q; ++k) { re[k] = 0.f; im[k] = 0.f; }
        fft_fma<Q, -1, n>(re, im);
        float4 *row = reinterpret_cast<float4 *>(tile + r * LD);
#pragma unroll
        for (int q = 0; q < Q / 2; ++q)
            row[q] = make_float4(re[xq(2 * q)], im[xq(2 * q)], re[xq(2 * q + 1)], im[xq(2 * q + 1)]);
    }
    __syncwarp();

    /* ---- B: column transforms of columns r and r + 16, intensity ---- */
    float zr[Q], zi[Q];
#pragma unroll 1                                 /* one copy of the transform's code: the kernel is instruction-fetch bound */
    for (int col = 0; col < 2; ++col) {
        const float2 *colp = reinterpret_cast<const float2 *>(tile) + r + 16 * col;
#pragma unroll
        for (int v = 0; v < n; ++v) {
            const float2 f = colp[v * (LD / 2)];
            re[v] = f.x; im[v] = f.y;
        }
#pragma unroll
        for (int v = n; v < Q; ++v) { re[v] = 0.f; im[v] = 0.f; }
        fft_fma<Q, -1, n>(re, im);
#pragma unroll
        for (int v = 0; v < Q; ++v) {
            const float s = fmaf(re[xq(v)], re[xq(v)], im[xq(v)] * im[xq(v)]);
            zi[v] = s;
        }
        if (col == 0) {
#pragma unroll
            for (int v = 0; v < Q; ++v) zr[v] = zi[v];
        }
    }
    __syncwarp();                                /* every thread has read its columns: the tile can be rewritten */

    /* ---- C: both real columns in one complex transform over v, separated by symmetry ---- */
    fft_fma<Q, -1>(zr, zi);
    {
        float2 *colp = reinterpret_cast<float2 *>(gtile) + r;
#pragma unroll
        for (int ly = 0; ly < n; ++ly) {
            const int a = xq(ly), b = xq(Q - ly);
            /* Z[ly] = g1[ly] + i g2[ly], conj Z[-ly] = g1[ly] - i g2[ly]  (the 1/2 is in the field's scale) */
            float2 g1 = make_float2(zr[a] + zr[b], zi[a] - zi[b]);
            float2 g2 = make_float2(zi[a] + zi[b], zr[b] - zr[a]);
            if (ML && layer > 0) {
                const float2 p1 = colp[ly * (LD / 2)], p2 = colp[ly * (LD / 2) + 16];
                g1.x += p1.x; g1.y += p1.y; g2.x += p2.x; g2.y += p2.y;
            }
            colp[ly * (LD / 2)] = g1;
            colp[ly * (LD / 2) + 16] = g2;
        }
    }
    }   /* sub-layers */
    __syncwarp();

    /* ---- D: lag row r < n: transform over u ---- */
    if (r < n) {
        const float4 *row = reinterpret_cast<const float4 *>(gtile + r * LD);
#pragma unroll
        for (int q = 0; q < Q / 2; ++q) {
            const float4 f = row[q];
            re[2 * q] = f.x; im[2 * q] = f.y; re[2 * q + 1] = f.z; im[2 * q + 1] = f.w;
        }
        fft_fma<Q, -1>(re, im);
        /* ---- E: table product, alias, x-transform; H[r][0..15] takes the place of the row this thread read ---- */
        float2 acc[LX];
#pragma unroll
        for (int a = 0; a < LX; ++a) acc[a] = make_float2(re[xq(a - (n - 1))], im[xq(a - (n - 1))]);
        const float2 *Mi = A.M + (size_t)i * A.mstride;
        finish_row<n>(acc, Mi + r * LX, tile + r * LD);
    }
    __syncwarp();

    /* ---- F: y-transform (real part), noise, threshold, centre of gravity ---- */
    {
        const int C = r;
        float yr[16], yi[16];
#pragma unroll
        for (int m = 0; m < 16; ++m) {
            if (m < n) {
                const float2 v = *reinterpret_cast<const float2 *>(tile + m * LD + 2 * C);
                yr[m] = v.x; yi[m] = v.y;
            } else { yr[m] = 0.f; yi[m] = 0.f; }
        }
        fft_fma<16, +1, n>(yr, yi);               /* B[R,C] = Re sum_m H[m][C] w_16^(R m) */
        float bcol[16];
#pragma unroll
        for (int R = 0; R < 16; ++R) bcol[R] = yr[fft_out_index<16>(R)];
        const size_t o = (size_t)t * A.nsub + i;
        if (live && A.binned) {
#pragma unroll
            for (int R = 0; R < 16; ++R) A.binned[(o * 16 + R) * 16 + C] = bcol[R];
        }
        if (EXT && A.flux > 0.f) {
            add_noise_col16(bcol, C, A.key, A.t0 + (unsigned)t, (unsigned)i, A.flux, A.ron2);
            if (live && A.noisy) {
#pragma unroll
                for (int R = 0; R < 16; ++R) A.noisy[(o * 16 + R) * 16 + C] = bcol[R];
            }
        }
        const float2 sl = cog16<MODE>(bcol, C, A.tau);
        if (live && C == 0) reinterpret_cast<float2 *>(A.slopes)[o] = sl;
    }
}

template <int n, int MODE, int EXTK>
cudaError_t launch_wkf_mode(const WkArgs &A, cudaStream_t st)
{
    constexpr size_t smem = EXTK == 2 ? 2 * WF_SMEM : WF_SMEM;
    static bool attr_set[64] = {false};             /* per device, as in wk.cu */
    int dev = 0;
    cudaGetDevice(&dev);
    if (smem > 48 * 1024 && dev >= 0 && dev < 64 && !attr_set[dev]) {
        cudaError_t e = cudaFuncSetAttribute(wkf_kernel<n, MODE, EXTK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set[dev] = true;
    }
    const int grid = (A.total + WF_SPOTS - 1) / WF_SPOTS;
    wkf_kernel<n, MODE, EXTK><<<grid, WF_THREADS, smem, st>>>(A);
    return cudaGetLastError();
}

template <int n>
cudaError_t launch_wkf(const WkArgs &A, cudaStream_t st)
{
    if (A.L > 1) return A.mode == 0 ? launch_wkf_mode<n, 0, 2>(A, st) : launch_wkf_mode<n, 1, 2>(A, st);
    if (A.L > 0 || A.flux > 0.f || A.dm_patch != nullptr)
        return A.mode == 0 ? launch_wkf_mode<n, 0, 1>(A, st) : launch_wkf_mode<n, 1, 1>(A, st);
    return A.mode == 0 ? launch_wkf_mode<n, 0, 0>(A, st) : launch_wkf_mode<n, 1, 0>(A, st);
}

}  // namespace

int shwfs_wk_fft_supported(const shwfs_handle *h)
{
    return h->D == 16 && (h->n == 12 || h->n == 14 || h->n == 16);
}

cudaError_t shwfs_wk_fft_launch(const shwfs::WkArgs &A, int n, cudaStream_t st)
{
    static_assert(WF_SMEM <= 48 * 1024, "static limit of dynamic shared memory");
    switch (n) {
    case 8: return launch_wkf<8>(A, st);
    case 10: return launch_wkf<10>(A, st);
    case 12: return launch_wkf<12>(A, st);
    case 14: return launch_wkf<14>(A, st);
    case 16: return launch_wkf<16>(A, st);
    default: return cudaErrorInvalidValue;
    }
}
