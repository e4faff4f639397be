/*
 * dm_umma.cu -- the DM phase of the closed-loop neighbours on the
 * 5th-generation tensor cores: the one dense contraction of the widened path,
 *     C_i[T x n^2] = coef[T x M] . modes_i[M x n^2]        for every valid subaperture i,
 * as tcgen05.mma (kind::tf32, accumulator in TMEM) with the 3-term split that keeps fp32 accuracy:
 *     x = hi + lo,  hi = tf32(x),  lo = tf32(x - hi);   C = A_hi B_hi + A_hi B_lo + A_lo B_hi
 * (the dropped A_lo B_lo term is 2^-22 relative; DESIGN.md 6.5 measures 1.7e-7 of peak for this split where a
 * single TF32 pass gives 4.9e-4).
 *
 * Operands live in memory already in the tensor core's canonical K-major no-swizzle layout -- 8-row x 16-byte
 * core matrices, [k/4][row/8][row%8][k%4] -- so that a stage is filled by two contiguous bulk copies
 * (cp.async.bulk, completion on an mbarrier) and described by a 64-bit shared-memory descriptor
 * (LBO = bytes between the two 16-byte K chunks of one MMA, SBO = 128 bytes between 8-row groups):
 *     B = modes: [nsub][k-block][hi|lo][KB/4][NP/8][8][4]   built once per shwfs_set_dm (umma_split_modes_kernel)
 *     A = coef : [frame tile][k-block][hi|lo][KB/4][16][8][4] built per call              (umma_split_coef_kernel)
 * CTA = (subaperture, tile of 128 frames), 128 threads: thread 0 issues the bulk copies (3-stage ring of 8-mode
 * stages: 46 KB, four CTAs and 4 x 128 TMEM columns per SM) and the MMAs (three per stage: the split terms,
 * M = 128, N = NP, K = 8), tcgen05.commit frees a stage /
 * signals the epilogue; then every warp reads its 32 TMEM lanes (= frames) with tcgen05.ld and writes 16-byte
 * rows of the patch-layout output.  Used for T > 8; the T <= 8 loop step is the bandwidth-bound GEMV of loop.cu.
 */
#include "internal.h"

namespace {

constexpr int UM_KB = 8;                   /* modes per stage */
constexpr int UM_STAGES = 3;
constexpr int UM_MT = 128;                 /* frames per CTA = UMMA M */

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ float tf32_rn(float x)
{
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}

/* position (in floats) of element (row, k) inside one canonical [KB/4][rows/8][8][4] tile */
__device__ __forceinline__ int canon_index(int row, int k, int rows) { return (k >> 2) * (rows * 4) + (row >> 3) * 32 + (row & 7) * 4 + (k & 3); }

/* modes_sub [nsub][M][NN] (the plain re-layout of loop.cu) -> split canonical tiles; grid (nsub, nkb) */
__global__ void umma_split_modes_kernel(const float *__restrict__ modes_sub, int M, int NN, int NP, int nkb,
                                        float *__restrict__ out)
{
    const int i = blockIdx.x, kb = blockIdx.y;
    float *hi = out + ((size_t)i * nkb + kb) * 2 * UM_KB * NP, *lo = hi + UM_KB * NP;
    for (int e = threadIdx.x; e < UM_KB * NP; e += blockDim.x) {
        const int k = e / NP, px = e - k * NP, m = kb * UM_KB + k;
        const float x = (m < M && px < NN) ? modes_sub[((size_t)i * M + m) * NN + px] : 0.f;
        const float h = tf32_rn(x);
        const int o = canon_index(px, k, NP);
        hi[o] = h;
        lo[o] = tf32_rn(x - h);
    }
}

/* coef [T][ldc] -> split canonical tiles [mtile][kb][hi|lo][KB/4][16][8][4]; grid (ceil(T/128), nkb) */
__global__ void umma_split_coef_kernel(const float *__restrict__ coef, int ldc, int T, int M, int nkb,
                                       float *__restrict__ out)
{
    const int mt = blockIdx.x, kb = blockIdx.y;
    float *hi = out + ((size_t)mt * nkb + kb) * 2 * UM_KB * UM_MT, *lo = hi + UM_KB * UM_MT;
    for (int e = threadIdx.x; e < UM_KB * UM_MT; e += blockDim.x) {
        const int row = e / UM_KB, k = e - row * UM_KB, t = mt * UM_MT + row, m = kb * UM_KB + k;
        const float x = (t < T && m < M) ? coef[(size_t)t * ldc + m] : 0.f;
        const float h = tf32_rn(x);
        const int o = canon_index(row, k, UM_MT);
        hi[o] = h;
        lo[o] = tf32_rn(x - h);
    }
}

__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    uint64_t d = (uint64_t)((addr >> 4) & 0x3FFF);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;                 /* descriptor version 1 (sm_100); layout type 0 = no swizzle */
    return d;
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done = 0;
    while (!done)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
}

template <int NP>
struct UmCfg {
    static constexpr int A_BYTES = 2 * UM_KB * UM_MT * 4;         /* hi + lo */
    static constexpr int B_BYTES = 2 * UM_KB * NP * 4;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int TMEM_COLS = NP <= 64 ? 64 : NP <= 128 ? 128 : 256;
    static constexpr size_t SMEM = (size_t)UM_STAGES * STAGE_BYTES + 128;
    static_assert(NP % 16 == 0 && NP >= 16 && NP <= 256, "UMMA N for M = 128 is a multiple of 16 up to 256");
};

/* grid (frame tiles, nsub); out[t][i][q], q < NN */
template <int NP>
__global__ void __launch_bounds__(128) dm_umma_kernel(const float *__restrict__ a_tiles, const float *__restrict__ b_tiles,
                                                      int T, int nsub, int NN, int nkb, float *__restrict__ out)
{
    using Cfg = UmCfg<NP>;
    extern __shared__ __align__(128) unsigned char um_smem[];
    __shared__ __align__(8) uint64_t full_bar[UM_STAGES], empty_bar[UM_STAGES], done_bar;
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5;
    const int mt = blockIdx.x, i = blockIdx.y;
    const uint32_t smem0 = (smem_u32(um_smem) + 127u) & ~127u;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < UM_STAGES; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&full_bar[s])));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&empty_bar[s])));
        }
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&done_bar)));
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(Cfg::TMEM_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = tmem_base_s;

    if (tid == 0) {
        const char *a_src = reinterpret_cast<const char *>(a_tiles) + (size_t)mt * nkb * Cfg::A_BYTES;
        const char *b_src = reinterpret_cast<const char *>(b_tiles) + (size_t)i * nkb * Cfg::B_BYTES;
        auto load = [&](int kb) {
            const int s = kb % UM_STAGES;
            const uint32_t bar = smem_u32(&full_bar[s]), dst = smem0 + s * Cfg::STAGE_BYTES;
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(Cfg::STAGE_BYTES) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(dst), "l"(a_src + (size_t)kb * Cfg::A_BYTES), "r"(Cfg::A_BYTES), "r"(bar) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(dst + Cfg::A_BYTES), "l"(b_src + (size_t)kb * Cfg::B_BYTES), "r"(Cfg::B_BYTES), "r"(bar) : "memory");
        };
        /* instruction descriptor: D = F32, A = B = TF32, both K-major, N = NP, M = 128 */
        constexpr uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(NP >> 3) << 17) | ((uint32_t)(UM_MT >> 4) << 24);
        for (int kb = 0; kb < UM_STAGES && kb < nkb; ++kb) load(kb);
        for (int kb = 0; kb < nkb; ++kb) {
            const int s = kb % UM_STAGES;
            mbar_wait(smem_u32(&full_bar[s]), (uint32_t)((kb / UM_STAGES) & 1));
            asm volatile("tcgen05.fence::after_thread_sync;");
            const uint32_t a_hi = smem0 + s * Cfg::STAGE_BYTES, a_lo = a_hi + UM_KB * UM_MT * 4;
            const uint32_t b_hi = a_hi + Cfg::A_BYTES, b_lo = b_hi + UM_KB * NP * 4;
#pragma unroll
            for (int ks = 0; ks < UM_KB / 8; ++ks) {
                /* one MMA eats K = 8 = two 16-byte chunks, UM_MT*16 (NP*16) bytes apart; 8-row groups 128 bytes apart */
                const uint32_t ao = ks * 2 * UM_MT * 16, bo = ks * 2 * NP * 16;
                const uint64_t dah = umma_desc(a_hi + ao, UM_MT * 16, 128), dal = umma_desc(a_lo + ao, UM_MT * 16, 128);
                const uint64_t dbh = umma_desc(b_hi + bo, NP * 16, 128), dbl = umma_desc(b_lo + bo, NP * 16, 128);
                const uint32_t acc0 = (kb > 0 || ks > 0) ? 1u : 0u;
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                             "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                             ::"r"(tmem), "l"(dal), "l"(dbh), "r"(idesc), "r"(acc0) : "memory");      /* small terms first */
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                             "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                             ::"r"(tmem), "l"(dah), "l"(dbl), "r"(idesc), "r"(1u) : "memory");
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                             "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                             ::"r"(tmem), "l"(dah), "l"(dbh), "r"(idesc), "r"(1u) : "memory");
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&empty_bar[s])) : "memory");
            /* refill the stage of the PREVIOUS k-block (its MMAs are done or about to be) with the k-block that comes UM_STAGES after it */
            if (kb >= 1 && kb - 1 + UM_STAGES < nkb) {
                const int sp = (kb - 1) % UM_STAGES;
                mbar_wait(smem_u32(&empty_bar[sp]), (uint32_t)(((kb - 1) / UM_STAGES) & 1));
                load(kb - 1 + UM_STAGES);
            }
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&done_bar)) : "memory");
    }
    __syncwarp();
    mbar_wait(smem_u32(&done_bar), 0u);
    asm volatile("tcgen05.fence::after_thread_sync;");

    /* epilogue: TMEM lane = frame of the tile; 8 columns at a time -> two 16-byte stores */
    const int t = mt * UM_MT + tid;
    float *dst = out + ((size_t)t * nsub + i) * NN;
    for (int c0 = 0; c0 < NN; c0 += 8) {
        uint32_t v[8];
        const uint32_t taddr = tmem + ((uint32_t)(warp * 32) << 16) + (uint32_t)c0;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(taddr));
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (t < T) {
            reinterpret_cast<float4 *>(dst + c0)[0] = make_float4(__uint_as_float(v[0]), __uint_as_float(v[1]),
                                                                  __uint_as_float(v[2]), __uint_as_float(v[3]));
            if (c0 + 4 < NN)
                reinterpret_cast<float4 *>(dst + c0 + 4)[0] = make_float4(__uint_as_float(v[4]), __uint_as_float(v[5]),
                                                                          __uint_as_float(v[6]), __uint_as_float(v[7]));
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(Cfg::TMEM_COLS));
}

template <int NP>
cudaError_t launch_umma(shwfs_handle *h, int T, float *out, cudaStream_t st)
{
    using Cfg = UmCfg<NP>;
    static shwfs_once_per_device attr;
    int dev;
    if (attr.pending(&dev)) {
        cudaError_t e = cudaFuncSetAttribute(dm_umma_kernel<NP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
        if (e != cudaSuccess) return e;
        attr.mark(dev);
    }
    const int nn = h->n * h->n;
    dm_umma_kernel<NP><<<dim3((unsigned)((T + UM_MT - 1) / UM_MT), (unsigned)h->nsub), 128, Cfg::SMEM, st>>>(
        h->d_um_coef, h->d_um_modes, T, h->nsub, nn, h->um_nkb, out);
    return cudaGetLastError();
}

}  // namespace

int shwfs_umma_np(const shwfs_handle *h)
{
    const int nn = h->n * h->n;
    if (h->nsub > 65535) return 0;
    return nn == 64 ? 64 : nn == 100 ? 112 : nn == 256 ? 256 : 0;
}

size_t shwfs_umma_modes_floats(const shwfs_handle *h, int M)
{
    const int nkb = (M + UM_KB - 1) / UM_KB;
    return (size_t)h->nsub * nkb * 2 * UM_KB * shwfs_umma_np(h);
}

size_t shwfs_umma_coef_floats(int T, int M)
{
    const int nkb = (M + UM_KB - 1) / UM_KB, mt = (T + UM_MT - 1) / UM_MT;
    return (size_t)mt * nkb * 2 * UM_KB * UM_MT;
}

/* build the split mode tiles from the plain per-subaperture table (shwfs_set_dm) */
cudaError_t shwfs_umma_build_modes(shwfs_handle *h, cudaStream_t st)
{
    const int nn = h->n * h->n, NP = shwfs_umma_np(h);
    h->um_nkb = (h->dm_M + UM_KB - 1) / UM_KB;
    umma_split_modes_kernel<<<dim3((unsigned)h->nsub, (unsigned)h->um_nkb), 256, 0, st>>>(h->d_dm_modes, h->dm_M, nn, NP,
                                                                                        h->um_nkb, h->d_um_modes);
    return cudaGetLastError();
}

/* DM phase of T frames through the tensor cores: split the coefficients, then the GEMM (two launches) */
cudaError_t shwfs_umma_dm_phase(shwfs_handle *h, const float *coef, int ldc, int T, float *out, cudaStream_t st)
{
    umma_split_coef_kernel<<<dim3((unsigned)((T + UM_MT - 1) / UM_MT), (unsigned)h->um_nkb), 256, 0, st>>>(
        coef, ldc, T, h->dm_M, h->um_nkb, h->d_um_coef);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    switch (shwfs_umma_np(h)) {
    case 64: return launch_umma<64>(h, T, out, st);
    case 112: return launch_umma<112>(h, T, out, st);
    case 256: return launch_umma<256>(h, T, out, st);
    default: return cudaErrorInvalidValue;
    }
}
