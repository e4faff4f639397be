/*
 * tma.cuh -- H1 (gather) of include/shwfs.h through the Tensor Memory Accelerator: one subaperture's n x n
 * phase patch ("The WF is split into sub-apertures") is one box of a 3-D tensor map over
 * phase[T][N][N], copied global -> shared memory by cp.async.bulk.tensor and signalled on an mbarrier.
 * BASELINE.json:north_star: "float4/TMA-staged loads of the phase patches".
 *
 * Why it matters here (profiles/r02_pf32.md): with one thread per patch row the per-thread vector loads
 * of a 16 x 16 patch touch 32 different 128-byte lines per warp instruction; the L1 data pipe ran at 88 % of
 * its wavefront peak on config 2 and was the bound of the kernel.  A TMA box does not pass through the LSU
 * data pipe at all and needs no address registers.
 *
 * Legal only where a patch row is a multiple of 16 bytes on a 16-byte-aligned address: n % 4 == 0, N % 4 == 0,
 * 16-byte-aligned frames.  The 64-byte-swizzle instance below is for n = 16 (64-byte rows): 16-byte chunk q of
 * patch row r lands at chunk q ^ ((r >> 1) & 3) of that row, so that 16 threads reading one row each (64 bytes
 * apart) hit 8 different 16-byte bank groups per quarter-warp instead of 2.
 */
#ifndef SHWFS_TMA_CUH_
#define SHWFS_TMA_CUH_

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

/* host: tensor map over phase[frames][N][N] (fp32) with an n x n x 1 box, 64-byte swizzle (n == 16) or none.
 * Returns false if the driver entry point is missing or the arguments are not encodable (the caller then
 * takes its register-gather instance). */
bool shwfs_tma_patch_map(CUtensorMap *out, const float *base, int N, long long frames, int n);

namespace shwfs {

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count));
}
/* makes the initialised barriers visible to the async proxy (the TMA unit) */
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_addr(bar)), "r"(parity) : "memory");
    } while (!done);
}

/* one box of the 3-D map at (x = column, y = row, z = frame) -> dst (shared), completion bytes on bar */
__device__ __forceinline__ void tma_load_patch(void *dst, const CUtensorMap *map, int x, int y, int z, uint64_t *bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_addr(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_addr(bar)), "r"(x), "r"(y), "r"(z)
                 : "memory");
}

__device__ __forceinline__ void tma_prefetch_map(const CUtensorMap *map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}

}  // namespace shwfs
#endif
