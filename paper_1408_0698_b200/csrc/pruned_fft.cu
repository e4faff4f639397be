/*
 * pruned_fft.cu -- the Shack-Hartmann chain WITHOUT elongation kernels (NGS case: "The WF is
 * split into sub-apertures and the spot computed by FFT for each sensor sub-aperture ... the centroid
 * computed on the final image to retrieve the slopes"), as one input-pruned P x P FFT per spot, sm_100a.
 *
 * Steps H1 gather, H2 field, H3 zero-padded P x P DFT, H4 |.|^2/P^2, H6 centre + b x b bin, H7 threshold,
 * H8 centre of gravity of include/shwfs.h, D = P/b = 16 detector pixels per side.
 *
 * Thread mapping: 16 threads (a half-warp) per spot, two spots per warp and step, persistent warps that are dealt
 * chunks of four spots from a counter (sweep.cuh; small calls: a strided deal), no CTA-wide barrier (a half-warp
 * never waits for another).
 *   H1           TMA instances (n = 16, 16-byte aligned frames): lane 0 of the half-warp issues ONE
 *                cp.async.bulk.tensor box (16 x 16 fp32, 64-byte swizzle) per spot into a 1 KB staging slot,
 *                completion on the half-warp's own mbarrier; the box of the warp's next step is requested as soon
 *                as the row pass of this step has read the slot, and lands during the column pass.  The gather costs
 *                no registers and no L1 data-pipe wavefronts (tma.cuh).  Other sizes: thread r gathers patch
 *                row r by 8-byte loads one tile ahead, in registers.
 *                Amplitude: subapertures whose n x n amplitudes are all exactly 1 (93 % of config 2) are
 *                flagged in the patch table at create and read no amplitude at all.
 *   row pass     thread r < n owns patch row r: sincos, one P-point FFT in registers whose inputs >= NZ are
 *                known zeros (first stage free); the n x P result goes to shared memory with the columns
 *                permuted (u -> (u mod b) * 16 + u / b) so that the column pass reads conflict-free.
 *                Rows >= n are zero and are never transformed.
 *   column pass  thread c owns the b adjacent columns b*c .. b*c+b-1 = detector column c ^ 8: for each, an
 *                NZ-input P-point FFT down the column, |.|^2, and the row half of the b x b bin
 *                accumulated in registers at compile-time positions (the roll by P/2 is an xor, the
 *                bit reversal of the output a renaming).  The thread ends with one detector column.
 *   H7 + H8      cog16 (cog.cuh): max / sums by xor shuffles inside the half-warp; lane 0 writes 8 bytes.
 * Only the phase patch is read from and the two slopes written to HBM.
 *
 * The table lookup of a spot (the only dependent load of the gather) is issued a step ahead and nothing is
 * computed from it before the step it belongs to: in the round-1 kernel the offset arithmetic sat right
 * behind the lookup and held 18 % of all stall samples (profiles/r02_pf32.md).
 */
#include <stdio.h>
#include <string.h>

#include "internal.h"
#include "fft_regs.cuh"
#include "field.cuh"
#include "cog.cuh"
#include "tma.cuh"
#include "sweep.cuh"

namespace {

using namespace shwfs;

constexpr int PF_THREADS = 128;
constexpr int PF_SPOTS = PF_THREADS / 16;
constexpr int PF_SLOT = 1024;                  /* bytes of one staged 16 x 16 fp32 patch */
constexpr int PF_CHUNK = 4;                    /* spots per chunk of the dynamic deal: two warp steps */

struct PfArgs {
    const float *phase;
    const float *amp;
    const int2 *patch;        /* [nsub] {first column of the patch | SHWFS_PATCH_LIT, first row of the patch} */
    float *slopes;
    float *binned;            /* stage-2 debug image [T*nsub*16*16] or null */
    int *sched;               /* chunk counters of the dynamic deal (sweep.cuh) */
    int chunk;                /* spots per chunk of the dynamic deal, 0 = strided deal */
    long long frame_stride;
    int T, N, nsub, total, n;
    float tau, turns, ramp_unit;
};

template <int P, int NZ, bool TMA>
struct PfCfg {
    static constexpr int b = P / 16;
    static constexpr int LD = 2 * P + 4;                 /* floats per stored row; LD/4 odd => STS.128 conflict-free */
    static constexpr int TILE = NZ * LD;                 /* floats per spot */
    static constexpr size_t TILES = sizeof(float) * (size_t)PF_SPOTS * TILE;
    /* TMA: [slack to a 1 KB boundary][8 staging slots][8 mbarriers][tiles] */
    static constexpr size_t STAGE = TMA ? (size_t)PF_SPOTS * PF_SLOT + 64 : 0;
    static constexpr size_t SMEM = TILES + STAGE + (TMA ? 1024 : 0);
#ifndef PF_TMA_CTAS
#define PF_TMA_CTAS 4
#endif
    static constexpr int MIN_CTAS = P == 64 ? 2 : (TMA ? PF_TMA_CTAS : 4);
    static_assert(P == 16 || P == 32 || P == 64, "P must be 16, 32 or 64 (D = 16)");
    static_assert(NZ <= 16 && NZ <= P && NZ % 2 == 0, "at most 16 non-zero rows, one per thread");
    static_assert(!TMA || NZ == 16, "the TMA box is 16 x 16");
};

/* position of column u in a stored row: the b columns of one detector column are P/b apart */
template <int P>
__host__ __device__ constexpr int col_pos(int u) { return (u % (P / 16)) * 16 + u / (P / 16); }

/* H1 of one spot row without TMA: the NZ/2 pixel pairs of patch row r (zeros when the row does not exist) */
template <int NZ>
__device__ __forceinline__ void pf_gather(const PfArgs &A, const Spot &s, bool live, int r, float2 (&ph)[NZ / 2], float2 (&am)[NZ / 2])
{
    const bool lit = s.lit();
#pragma unroll
    for (int q = 0; q < NZ / 2; ++q) { ph[q] = make_float2(0.f, 0.f); am[q] = make_float2(0.f, 0.f); }
    if (live && r < A.n) {
        const int off = (s.row0() + r) * A.N + s.col0();
        const float2 *pp = reinterpret_cast<const float2 *>(A.phase + (size_t)s.t * A.frame_stride + off);
        const float2 *pa = reinterpret_cast<const float2 *>(A.amp + off);
#pragma unroll
        for (int q = 0; q < NZ / 2; ++q)
            if (2 * q < A.n) {
                ph[q] = __ldg(pp + q);
                am[q] = lit ? make_float2(1.f, 1.f) : __ldg(pa + q);
            }
    }
}

template <int P, int NZ, int MODE, bool TMA>
__global__ void __launch_bounds__(PF_THREADS, PfCfg<P, NZ, TMA>::MIN_CTAS)
pruned_fft_kernel(const PfArgs A, const __grid_constant__ CUtensorMap tmap)
{
    using Cfg = PfCfg<P, NZ, TMA>;
    constexpr int b = Cfg::b, LD = Cfg::LD, HP = P / 2;
    extern __shared__ __align__(16) unsigned char pf_smem[];
    const int tid = threadIdx.x, sp = tid >> 4, r = tid & 15;

    unsigned char *base = pf_smem;
    if (TMA) base += (1024u - (smem_addr(pf_smem) & 1023u)) & 1023u;        /* the swizzle pattern is in address bits */
    unsigned char *slot = base + sp * PF_SLOT;
    uint64_t *bar = reinterpret_cast<uint64_t *>(base + PF_SPOTS * PF_SLOT) + sp;
    float *tile = reinterpret_cast<float *>(base + Cfg::STAGE) + sp * Cfg::TILE;

    /* persistent CTAs (sweep.cuh): the host sizes the grid to the resident CTAs of the device, so a launch has no
     * ragged last wave */
    Sweep sw_(A.patch, A.chunk ? A.sched : nullptr, A.T, A.nsub, A.total, A.chunk);      /* chunk 0: strided deal */
    auto request = [&](const Spot &s) {                   /* TMA: one box per spot, issued by the half-warp's lane 0 */
        if (r == 0 && sw_.live(s)) {
            mbar_expect_tx(bar, PF_SLOT);
            tma_load_patch(slot, &tmap, s.col0(), s.row0(), s.t, bar);
        }
    };

    Spot cur = sw_.first();
    Spot nxt = cur;
    sw_.advance(nxt);
    sw_.lookup(nxt);

    float2 ph[TMA ? 1 : NZ / 2], am[TMA ? 1 : NZ / 2];
    uint32_t parity = 0;
    if constexpr (TMA) {
        if (r == 0) {
            tma_prefetch_map(&tmap);
            mbar_init(bar, 1);
            mbar_init_fence();
        }
        __syncwarp();
        request(cur);
    } else {
        pf_gather<NZ>(A, cur, sw_.live(cur), r, ph, am);
    }

#pragma unroll 1
    for (; sw_.mine(cur); ) {
        const bool live = sw_.live(cur);
        const bool lit = cur.lit();
        const int o_cur = live ? cur.t * A.nsub + cur.i : -1;     /* all that is left of `cur` after the row pass */

        float2 z[P];                                       /* packed (re, im): FP32x2 butterflies, fft_regs.cuh */

        /* ---- row pass: H2 field, P-point FFT of row r (inputs >= NZ are zero) ---- */
        if (r < NZ) {
            if (live && r < A.n) {
                if constexpr (TMA) {
                    /* the ramp -(r + k)/(2P) in two steps, -r/(2P) before and the compile-time k/(2P) after the
                     * data-dependent product: written as one term per pixel the compiler hoists 16 loop-invariant
                     * ramps out of the tile loop and spills them */
                    const float nramp_r = -(float)r * (0.5f / (float)P);
                    const int sw = (r >> 1) & 3;    /* 64-byte swizzle: chunk q of row r sits at chunk q ^ sw */
                    const float4 *srow = reinterpret_cast<const float4 *>(slot + r * 64);
                    if (lit) {                      /* every amplitude of the patch is 1: nothing else to read */
                        mbar_wait(bar, parity);
#pragma unroll
                        for (int q = 0; q < NZ / 4; ++q) {
                            const float4 v = srow[q ^ sw];
                            const float pv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const int k = 4 * q + e;
                                z[k] = field_unit(fmaf(pv[e], A.turns, nramp_r), 1.0f, (float)k * (0.5f / (float)P));
                            }
                        }
                    } else {                        /* partially lit subaperture: its amplitude row, 16-byte loads */
                        const float4 *pa = reinterpret_cast<const float4 *>(
                            A.amp + (size_t)(cur.row0() + r) * A.N + cur.col0());
                        float4 av[NZ / 4];
#pragma unroll
                        for (int q = 0; q < NZ / 4; ++q) av[q] = __ldg(pa + q);
                        mbar_wait(bar, parity);
#pragma unroll
                        for (int q = 0; q < NZ / 4; ++q) {
                            const float4 v = srow[q ^ sw];
                            const float pv[4] = {v.x, v.y, v.z, v.w};
                            const float aa[4] = {av[q].x, av[q].y, av[q].z, av[q].w};
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const int k = 4 * q + e;
                                z[k] = field_value(fmaf(pv[e], A.turns, nramp_r), aa[e], 1.0f, (float)k * (0.5f / (float)P));
                            }
                        }
                    }
                    parity ^= 1u;
                } else {
#pragma unroll
                    for (int q = 0; q < NZ / 2; ++q) {
                        const float ramp = (float)(r + 2 * q) * A.ramp_unit;
                        z[2 * q] = field_value(ph[q].x, am[q].x, A.turns, ramp);
                        z[2 * q + 1] = field_value(ph[q].y, am[q].y, A.turns, ramp + A.ramp_unit);
                    }
                }
#pragma unroll
                for (int k = NZ; k < P; ++k) z[k] = make_float2(0.f, 0.f);
                fft_fma2<P, -1, NZ>(z);
            } else {
#pragma unroll
                for (int k = 0; k < P; ++k) z[k] = make_float2(0.f, 0.f);
            }
            float4 *row = reinterpret_cast<float4 *>(tile + r * LD);
#pragma unroll
            for (int q = 0; q < P / 2; ++q) {
                /* stored positions 2q, 2q+1 hold columns u0, u1 (inverse of col_pos) */
                const int p0 = 2 * q, p1 = 2 * q + 1;
                const int u0 = (p0 % 16) * b + p0 / 16, u1 = (p1 % 16) * b + p1 / 16;
                const int x0 = fft_out_index<P>(u0), x1 = fft_out_index<P>(u1);
                row[q] = make_float4(z[x0].x, z[x0].y, z[x1].x, z[x1].y);
            }
        }
        __syncwarp();                                      /* rows visible; the staging slot has been read */
        /* H1 of the next tile: in flight during the column pass */
        if constexpr (TMA) request(nxt);
        else pf_gather<NZ>(A, nxt, sw_.live(nxt), r, ph, am);

        /* ---- column pass: b columns per thread, |.|^2 and the row half of the bin in registers ---- */
        float acc[16];                                     /* one register per detector row between two columns */
#pragma unroll
        for (int be = 0; be < b; ++be) {
            const float2 *colp = reinterpret_cast<const float2 *>(tile) + be * 16 + r;
#pragma unroll
            for (int v = 0; v < NZ; ++v) z[v] = colp[v * (LD / 2)];
#pragma unroll
            for (int v = NZ; v < P; ++v) z[v] = make_float2(0.f, 0.f);
            fft_fma2<P, -1, NZ>(z);
#pragma unroll
            for (int R = 0; R < 16; ++R) {
                /* (sum re^2, sum im^2) of the b rows of detector row R, one FFMA2 per value */
                float2 a2 = be == 0 ? make_float2(0.f, 0.f) : make_float2(acc[R], 0.f);
#pragma unroll
                for (int al = 0; al < b; ++al) {
                    const int x = fft_out_index<P>((R * b + al) ^ HP);      /* H6: roll by P/2, then bin */
                    a2 = (be == 0 && al == 0) ? __fmul2_rn(z[x], z[x]) : __ffma2_rn(z[x], z[x], a2);
                }
                acc[R] = a2.x + a2.y;
            }
        }
        constexpr float inv_pp = 1.0f / ((float)P * (float)P);
#pragma unroll
        for (int R = 0; R < 16; ++R) acc[R] *= inv_pp;

        /* ---- H7 + H8: thread r holds detector column C = r ^ 8 ---- */
        const int C = r ^ 8;
        const float2 sl = cog16<MODE>(acc, C, A.tau);
        if (o_cur >= 0) {
            const size_t o = (size_t)o_cur;
            if (r == 0) reinterpret_cast<float2 *>(A.slopes)[o] = sl;
            if (A.binned) {
#pragma unroll
                for (int R = 0; R < 16; ++R) A.binned[(o * 16 + R) * 16 + C] = acc[R];
            }
        }
        __syncwarp();                                      /* the tile is rewritten by the next row pass */
        /* table lookup of the tile after the next: it has the whole next row pass to arrive (the table is a few KB,
         * L1/L2 resident), and nothing of it is live across a column pass */
        cur = nxt;
        sw_.advance(nxt);
        sw_.lookup(nxt);
    }
    sw_.leave();
}

template <int P, int NZ, int MODE, bool TMA>
cudaError_t launch_pf_inst(shwfs_handle *h, const PfArgs &A, const CUtensorMap &map, cudaStream_t st)
{
    using Cfg = PfCfg<P, NZ, TMA>;
    static shwfs_once_per_device attr;
    static int resident[64];                        /* CTAs each device holds at once */
    int dev;
    if (attr.pending(&dev)) {
        cudaError_t e = cudaFuncSetAttribute(pruned_fft_kernel<P, NZ, MODE, TMA>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
        int per_sm = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pruned_fft_kernel<P, NZ, MODE, TMA>, PF_THREADS, Cfg::SMEM);
        if (dev >= 0 && dev < 64) resident[dev] = h->sms * (per_sm > 0 ? per_sm : 1);
        attr.mark(dev);
    }
    static char name[64];
    if (!name[0]) snprintf(name, sizeof(name), "pruned_fft_kernel<%d,%d,%d,%s>", P, NZ, MODE, TMA ? "tma" : "ldg");
    h->last_kernel = name;
    const int need = (A.total + PF_SPOTS - 1) / PF_SPOTS;
    const int res = (dev >= 0 && dev < 64 && resident[dev] > 0) ? resident[dev] : h->sms;
    const int grid = need < res ? need : res;
    /* calls of at least four steps per resident warp: chunks of PF_CHUNK spots dealt from the handle's counter
     * (1.15e9 against 1.09e9 spots/s on config 2: the warps of an SM do not run at the same speed and a static deal
     * ends with 3.2 of 4 warps per scheduler resident; chunks of 2 / 8 spots: 1.09 / 1.13e9); smaller calls:
     * strided */
    PfArgs B = A;
    B.chunk = (long long)A.total >= 4LL * PF_SPOTS * res ? PF_CHUNK : 0;
    pruned_fft_kernel<P, NZ, MODE, TMA><<<grid, PF_THREADS, Cfg::SMEM, st>>>(B, map);
    return cudaGetLastError();
}

template <int P, int NZ>
cudaError_t launch_pf(shwfs_handle *h, const PfArgs &A, cudaStream_t st)
{
    CUtensorMap map;
    if constexpr (NZ == 16) {
        /* TMA instance when a patch is a legal box: n = 16, frames 16-byte aligned with a 16-byte row pitch */
        if (h->n == 16 && !h->no_tma && shwfs_tma_patch_map(&map, A.phase, h->N, A.T, 16))
            return h->mode == 0 ? launch_pf_inst<P, NZ, 0, true>(h, A, map, st) : launch_pf_inst<P, NZ, 1, true>(h, A, map, st);
    }
    memset(&map, 0, sizeof(map));
    return h->mode == 0 ? launch_pf_inst<P, NZ, 0, false>(h, A, map, st) : launch_pf_inst<P, NZ, 1, false>(h, A, map, st);
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
    A.phase = phase; A.amp = h->d_amp; A.patch = h->d_patch; A.slopes = slopes; A.binned = binned; A.sched = h->d_sched; A.chunk = 0;
    A.frame_stride = (long long)h->N * h->N;
    A.T = T; A.N = h->N; A.nsub = h->nsub; A.total = T * h->nsub; A.n = h->n;
    A.tau = h->tau;
    A.turns = (float)((double)h->c_phi / 6.283185307179586476925286766559);
    A.ramp_unit = 0.5f / (float)h->P;
    if (A.total == 0) return cudaSuccess;
    h->launches += 1;
    switch (h->P) {
    case 16: return h->n <= 8 ? launch_pf<16, 8>(h, A, st) : launch_pf<16, 16>(h, A, st);
    case 32: return launch_pf<32, 16>(h, A, st);
    case 64: return launch_pf<64, 16>(h, A, st);
    default: return cudaErrorInvalidValue;
    }
}
