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
 * shared memory per spot is reused by every exchange.  Every line transform runs on packed (re, im) registers
 * with FP32x2 butterflies (fft_fma2, fft_regs.cuh).
 *   A  thread r owns patch row r: H1 gather, H2 field (scaled by 2^-5.5 so that the unnormalised transforms
 *      below need no further factor), 32-point FFT of the row (inputs >= 16 are zero) -> tile[r][u].
 *      The plain n = 16 instance (config 5) is persistent and takes its patches by TMA (tma.cuh, sweep.cuh):
 *      one 16 x 16 box per spot into a 1 KB slot, requested for the CTA's next tile as soon as step A has read
 *      the slot, so that it lands during steps B-F; fully lit subapertures read no amplitude.  The other
 *      instances gather with 16- or 8-byte loads at the head of the CTA, one tile per CTA.
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
#include "tma.cuh"
#include "sweep.cuh"

#include <stdio.h>
#include <string.h>

namespace {

using namespace shwfs;

constexpr int WF_ROWS = 16;                    /* tile rows (threads per spot): n <= 16              */
constexpr int WF_Q = 32;                       /* transform grid side                                */
constexpr int WF_THREADS = 128;
constexpr int WF_SPOTS = WF_THREADS / 16;
constexpr int WF_LD = 2 * WF_Q + 4;            /* floats per tile row; LD/4 odd => 16-byte row accesses conflict-free */
constexpr int WF_TILE = WF_ROWS * WF_LD;
constexpr size_t WF_SMEM = sizeof(float) * (size_t)WF_SPOTS * WF_TILE;
constexpr int WF_SLOT = 1024;                  /* bytes of one staged 16 x 16 fp32 patch (TMA instance) */
constexpr size_t WF_STAGE = (size_t)WF_SPOTS * WF_SLOT + 64;      /* slots + one mbarrier per half-warp */

__device__ __forceinline__ constexpr int xq(int k) { return fft_out_index<WF_Q>(k & (WF_Q - 1)); }

/* EXTK as in wk.cu: 0 plain sensor, 1 extensions on one (sub-)layer, 2 several sodium sub-layers (S is linear in the
 * sub-layer intensities: steps A-C run per sub-layer and the separated column transforms pile up in a second
 * tile per spot, each element owned by one thread; D-F run once) */
template <int n, int MODE, int EXTK, bool TMA>
__global__ void __launch_bounds__(WF_THREADS, EXTK == 2 ? 3 : 4) wkf_kernel(const WkArgs A, const __grid_constant__ CUtensorMap tmap)
{
    constexpr bool EXT = EXTK > 0, ML = EXTK == 2;
    static_assert(n % 2 == 0 && n <= WF_ROWS && 2 * n - 1 <= WF_Q, "even n <= 16: one thread per patch row, grid 32 >= 2n-1");
    static_assert(!TMA || (n == 16 && EXTK == 0), "the TMA box is 16 x 16; extensions gather in registers");
    constexpr int Q = WF_Q, LD = WF_LD, LX = 2 * n - 1;
    extern __shared__ __align__(16) unsigned char wf_smem[];
    const int tid = threadIdx.x, sp = tid >> 4, r = tid & 15;
    unsigned char *base = wf_smem;
    if (TMA) base += (1024u - (smem_addr(wf_smem) & 1023u)) & 1023u;      /* the swizzle pattern is in address bits */
    unsigned char *slot = base + sp * WF_SLOT;
    uint64_t *bar = reinterpret_cast<uint64_t *>(base + WF_SPOTS * WF_SLOT) + sp;
    float *tiles = reinterpret_cast<float *>(base + (TMA ? WF_STAGE : 0));
    float *tile = tiles + sp * WF_TILE;
    float *gtile = ML ? tiles + (WF_SPOTS + sp) * WF_TILE : tile;        /* where step C leaves g_u[ly] */

    /* TMA instance: persistent CTAs striding over the tiles; the others are launched one tile per CTA and run
     * the loop once */
    Sweep sw_(A.patch, TMA ? A.sched : nullptr, A.T, A.nsub, A.total, SWEEP_CHUNK);
    auto request = [&](const Spot &s) {
        if (r == 0 && sw_.live(s)) {
            mbar_expect_tx(bar, WF_SLOT);
            tma_load_patch(slot, &tmap, s.col0(), s.row0(), s.t, bar);
        }
    };
    Spot cur = sw_.first();
    Spot nxt = cur;
    uint32_t parity = 0;
    if constexpr (TMA) {
        sw_.advance(nxt);
        sw_.lookup(nxt);
        if (r == 0) {
            tma_prefetch_map(&tmap);
            mbar_init(bar, 1);
            mbar_init_fence();
        }
        __syncwarp();
        request(cur);
    }

#pragma unroll 1
    for (; sw_.mine(cur); ) {
    const bool live = sw_.live(cur);
    const int i = live ? cur.i : 0, t = live ? cur.t : 0;

    float2 z[Q];

    const int n_layers = ML ? A.L : 1;
#pragma unroll 1
    for (int layer = 0; layer < n_layers; ++layer) {
    /* ---- A: gather, field, row transform (threads r < n) ---- */
    if (r < n) {
        /* 2^-5.5 on the field = 1/2048 on the intensity: 1/Q^2 of the two unnormalised transforms of S and the
         * 1/2 of the real-pair separation of step C */
        float sc = 0.02209708691207961f;
        if constexpr (TMA) {
            const float nramp_r = -(float)r * A.ramp_unit;      /* ramp in two steps: see pruned_fft.cu */
            const float4 *srow = reinterpret_cast<const float4 *>(slot + r * 64);
            const int sw = (r >> 1) & 3;                        /* 64-byte swizzle: chunk q of row r at chunk q ^ sw */
            float4 av[n / 4];
#pragma unroll
            for (int q = 0; q < n / 4; ++q) av[q] = make_float4(sc, sc, sc, sc);
            if (live && !cur.lit()) {                           /* partially lit subaperture: its amplitude row */
                const float4 *pa = reinterpret_cast<const float4 *>(A.amp + (size_t)(cur.row0() + r) * A.N + cur.col0());
#pragma unroll
                for (int q = 0; q < n / 4; ++q) {
                    const float4 w = __ldg(pa + q);
                    av[q] = make_float4(w.x * sc, w.y * sc, w.z * sc, w.w * sc);
                }
            }
            if (live) {
                mbar_wait(bar, parity);
                parity ^= 1u;
#pragma unroll
                for (int q = 0; q < n / 4; ++q) {
                    const float4 v = srow[q ^ sw];
                    const float pv[4] = {v.x, v.y, v.z, v.w};
                    const float aa[4] = {av[q].x, av[q].y, av[q].z, av[q].w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int k = 4 * q + e;
                        z[k] = field_value(fmaf(-(float)k, A.ramp_unit, fmaf(pv[e], A.turns, nramp_r)), aa[e], 1.0f, 0.f);
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < n; ++k) z[k] = make_float2(0.f, 0.f);
            }
        } else {
        float pv[n], av[n];
#pragma unroll
        for (int k = 0; k < n; ++k) { pv[k] = 0.f; av[k] = 0.f; }
        if (live) {
            const int off = (cur.row0() + r) * A.N + cur.col0();
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
            z[k] = field_value(pv[k], av[k] * sc, A.turns, ramp);
        }
        }
#pragma unroll
        for (int k = n; k < Q; ++k) z[k] = make_float2(0.f, 0.f);
        fft_fma2<Q, -1, n>(z);
        float4 *row = reinterpret_cast<float4 *>(tile + r * LD);
#pragma unroll
        for (int q = 0; q < Q / 2; ++q)
            row[q] = make_float4(z[xq(2 * q)].x, z[xq(2 * q)].y, z[xq(2 * q + 1)].x, z[xq(2 * q + 1)].y);
    }
    __syncwarp();
    if constexpr (TMA) request(nxt);             /* the slot has been read: the next tile's patch lands during B-F */

    /* ---- B: column transforms of columns r and r + 16, intensity: s0[v] = S[v][r], s1[v] = S[v][r + 16] ---- */
    float s0[Q], s1[Q];
#pragma unroll 1                                 /* one copy of the transform's code: the kernel is instruction-fetch bound */
    for (int col = 0; col < 2; ++col) {
        const float2 *colp = reinterpret_cast<const float2 *>(tile) + r + 16 * col;
#pragma unroll
        for (int v = 0; v < n; ++v) z[v] = colp[v * (LD / 2)];
#pragma unroll
        for (int v = n; v < Q; ++v) z[v] = make_float2(0.f, 0.f);
        fft_fma2<Q, -1, n>(z);
#pragma unroll
        for (int v = 0; v < Q; ++v) {
            const float2 sq = __fmul2_rn(z[xq(v)], z[xq(v)]);
            s1[v] = sq.x + sq.y;
        }
        if (col == 0) {
#pragma unroll
            for (int v = 0; v < Q; ++v) s0[v] = s1[v];
        }
    }
    __syncwarp();                                /* every thread has read its columns: the tile can be rewritten */

    /* ---- C: both real columns in one complex transform over v, separated by symmetry ---- */
    float2 zc[Q];
    fft_fma2_split<Q, -1>(s0, s1, zc);           /* scalar first stage: s0, s1 need not sit in register pairs */
    {
        float2 *colp = reinterpret_cast<float2 *>(gtile) + r;
#pragma unroll
        for (int ly = 0; ly < n; ++ly) {
            const float2 za = zc[xq(ly)], zb = zc[xq(Q - ly)];
            /* Z[ly] = g1[ly] + i g2[ly], conj Z[-ly] = g1[ly] - i g2[ly]  (the 1/2 is in the field's scale):
             * g1 = Z[ly] + conj Z[-ly], g2 = -i (Z[ly] - conj Z[-ly]) */
            float2 g1 = __fadd2_rn(za, make_float2(zb.x, -zb.y));
            float2 g2 = __fadd2_rn(rot_mi2(za), make_float2(zb.y, zb.x));
            if (ML && layer > 0) {
                g1 = __fadd2_rn(g1, colp[ly * (LD / 2)]);
                g2 = __fadd2_rn(g2, colp[ly * (LD / 2) + 16]);
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
            z[2 * q] = make_float2(f.x, f.y); z[2 * q + 1] = make_float2(f.z, f.w);
        }
        /* the thread's row of the tile is free from here to the end of step E: the table row M_i[.][ly = r] is
         * staged in it while the transform runs */
        mrow_stage<n>(A.M + (size_t)i * A.mstride + r, tile + r * LD);
        fft_fma2<Q, -1>(z);
        /* ---- E: table product, alias, x-transform; H[r][0..15] takes the place of the row this thread read ---- */
        float2 acc[LX];
#pragma unroll
        for (int a = 0; a < LX; ++a) acc[a] = z[xq(a - (n - 1))];
        mrow_wait();
        finish_row2<n>(acc, tile + r * LD, tile + r * LD);
    }
    __syncwarp();

    /* ---- F: y-transform (real part), noise, threshold, centre of gravity ---- */
    {
        const int C = r;
        float bcol[16];
        ytransform16<n>([&](int m) { return *reinterpret_cast<const float2 *>(tile + m * LD + 2 * C); }, bcol);
        const size_t o = (size_t)t * A.nsub + i;
        if (live && A.binned) {
#pragma unroll
            for (int R = 0; R < 16; ++R) A.binned[(o * 16 + R) * 16 + C] = bcol[R];
        }
        if (EXT && A.flux > 0.f) {
            add_noise_col16(bcol, C, A.key, A.t0 + (unsigned)t, (unsigned)i, A.flux, A.ron2, A.photon_model);
            if (live && A.noisy) {
#pragma unroll
                for (int R = 0; R < 16; ++R) A.noisy[(o * 16 + R) * 16 + C] = bcol[R];
            }
        }
        const float2 sl = cog16<MODE>(bcol, C, A.tau);
        if (live && C == 0) reinterpret_cast<float2 *>(A.slopes)[o] = sl;
    }
    __syncwarp();                                /* the tile is rewritten by the next step A */
    if constexpr (TMA) {
        cur = nxt;
        sw_.advance(nxt);
        sw_.lookup(nxt);                         /* has the whole next step A to arrive */
    } else {
        sw_.advance(cur);                        /* one tile per CTA: past the end */
    }
    }
    sw_.leave();
}

template <int n, int MODE, int EXTK, bool TMA>
cudaError_t launch_wkf_inst(shwfs_handle *h, const WkArgs &A, const CUtensorMap &map, cudaStream_t st)
{
    constexpr size_t smem = (EXTK == 2 ? 2 * WF_SMEM : WF_SMEM) + (TMA ? WF_STAGE + 1024 : 0);
    static shwfs_once_per_device attr;
    static int resident[64];                        /* CTAs each device holds at once (persistent instance) */
    int dev;
    if (attr.pending(&dev)) {
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(wkf_kernel<n, MODE, EXTK, TMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        int per_sm = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, wkf_kernel<n, MODE, EXTK, TMA>, WF_THREADS, smem);
        if (dev >= 0 && dev < 64) resident[dev] = h->sms * (per_sm > 0 ? per_sm : 1);
        attr.mark(dev);
    }
    static char name[64];
    if (!name[0]) snprintf(name, sizeof(name), "wkf_kernel<%d,%d,%d,%s>", n, MODE, EXTK, TMA ? "tma" : "ldg");
    h->last_kernel = name;
    int grid = (A.total + WF_SPOTS - 1) / WF_SPOTS;         /* one tile per CTA */
    if (TMA) {                                              /* persistent: one chunk of the sweep per warp at least */
        const int nchunks = (A.total + SWEEP_CHUNK - 1) / SWEEP_CHUNK;
        const int res = (dev >= 0 && dev < 64 && resident[dev] > 0) ? resident[dev] : h->sms;
        grid = (nchunks + WF_THREADS / 32 - 1) / (WF_THREADS / 32);
        if (grid > res) grid = res;
    }
    wkf_kernel<n, MODE, EXTK, TMA><<<grid, WF_THREADS, smem, st>>>(A, map);
    return cudaGetLastError();
}

template <int n, int MODE, int EXTK>
cudaError_t launch_wkf_mode(shwfs_handle *h, const WkArgs &A, cudaStream_t st)
{
    CUtensorMap map;
    if constexpr (n == 16 && EXTK == 0) {
        /* the persistent instance deals chunks of SWEEP_CHUNK spots dynamically: worth it from ~8 chunks per resident
         * warp (16 warps per SM) up; smaller calls spread over one-tile CTAs */
        if (!h->no_tma && (h->force_persistent || (long long)A.total >= 8LL * SWEEP_CHUNK * 16 * h->sms) &&
            shwfs_tma_patch_map(&map, A.phase, A.N, A.T, 16))
            return launch_wkf_inst<n, MODE, EXTK, true>(h, A, map, st);
    }
    memset(&map, 0, sizeof(map));
    return launch_wkf_inst<n, MODE, EXTK, false>(h, A, map, st);
}

template <int n>
cudaError_t launch_wkf(shwfs_handle *h, const WkArgs &A, cudaStream_t st)
{
    if (A.L > 1) return A.mode == 0 ? launch_wkf_mode<n, 0, 2>(h, A, st) : launch_wkf_mode<n, 1, 2>(h, A, st);
    if (A.L > 0 || A.flux > 0.f || A.dm_patch != nullptr)
        return A.mode == 0 ? launch_wkf_mode<n, 0, 1>(h, A, st) : launch_wkf_mode<n, 1, 1>(h, A, st);
    return A.mode == 0 ? launch_wkf_mode<n, 0, 0>(h, A, st) : launch_wkf_mode<n, 1, 0>(h, A, st);
}

}  // namespace

int shwfs_wk_fft_supported(const shwfs_handle *h)
{
    return h->D == 16 && (h->n == 12 || h->n == 14 || h->n == 16);
}

cudaError_t shwfs_wk_fft_launch(shwfs_handle *h, const shwfs::WkArgs &A, int n, cudaStream_t st)
{
    static_assert(WF_SMEM <= 48 * 1024, "static limit of dynamic shared memory");
    switch (n) {
    case 8: return launch_wkf<8>(h, A, st);
    case 10: return launch_wkf<10>(h, A, st);
    case 12: return launch_wkf<12>(h, A, st);
    case 14: return launch_wkf<14>(h, A, st);
    case 16: return launch_wkf<16>(h, A, st);
    default: return cudaErrorInvalidValue;
    }
}
