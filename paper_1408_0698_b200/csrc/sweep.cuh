/*
 * sweep.cuh -- how the warps of the half-warp-per-spot kernels (pruned_fft.cu, wk_fft.cu) are dealt their spots
 * g = i*T + t (frame fastest; "for each sensor sub-aperture", every frame).
 *
 * A warp never synchronises with another warp in these kernels, so the warp is the scheduling unit; it works on
 * two spots (one per half-warp) per step.  Two deals:
 *   strided (counter == nullptr)  warp w of the launch takes the spot pairs w, w + W, w + 2W, ... (W = warps of
 *            the launch): balanced to one step whatever the size of the call, no shared state.  The kernels
 *            without a per-subaperture table (pruned_fft.cu) and every one-tile-per-CTA launch use it.
 *   dynamic  the spots are cut into chunks of `chunk_spots` consecutive spots; a warp works through a chunk and
 *            then takes the next free chunk from a global counter (atomicAdd by lane 0, one grab per chunk,
 *            issued a chunk ahead and not waited for until that chunk is entered).  The first chunk of a warp is its own global warp index, the counter hands
 *            out the rest.  For large launches of the kernels that read a table row per spot (wk_fft.cu).
 * Why dynamic: with a static split (strided or contiguous) the CTAs of an SM do not run at the
 * same speed -- the warp scheduler prefers some warp slots -- and the slowest CTA of each SM ran on alone at the
 * end: wkf_kernel<16> had 3.1 of 4 warps per scheduler resident on average (profiles/r02_wkf16.md).  Why chunks
 * of consecutive spots: they belong to one or two subapertures, whose table rows M_i and amplitude patch then
 * come from L1; dealt tile by tile with a stride every table row came from L2 (26 % of the stall samples).
 * Inside a chunk (i, t) advance by a fixed step; the spot's entry of the patch table -- the only dependent load
 * of the gather H1 -- is looked up well before anything is computed from it.
 *
 * The counter pair {next chunk, warps done} lives in the handle (zero at create); the last warp to leave the
 * kernel puts both back to zero, so launches that follow one another on a stream need no host-side reset.
 */
#ifndef SHWFS_SWEEP_CUH_
#define SHWFS_SWEEP_CUH_

#include "internal.h"

namespace shwfs {

constexpr int SWEEP_CHUNK = 16;      /* spots per chunk of the persistent kernels: 8 warp steps */

struct Spot {
    int g, i, t;
    int2 pe;                  /* {first column of the patch | SHWFS_PATCH_LIT, first row of the patch} */
    __device__ __forceinline__ bool lit() const { return (pe.x & SHWFS_PATCH_LIT) != 0; }
    __device__ __forceinline__ int col0() const { return pe.x & ~SHWFS_PATCH_LIT; }
    __device__ __forceinline__ int row0() const { return pe.y; }
};

struct Sweep {
    const int2 *patch;
    int *counter;             /* [0] chunks handed out beyond the first one of each warp, [1] warps done; or null */
    int T, nsub, total, dq, dr;
    int chunk_spots;          /* dynamic deal: spots per chunk (even) */
    int half;                 /* 0 / 1: which spot of the warp's pair this thread works on */
    int c_end;                /* first spot past the chunk the look-ahead spot is in */
    int pending;              /* lane 0: the counter value the atomicAdd for the chunk after that returned -- read
                                 (and so waited for) only when that chunk is entered, a whole chunk later */
    int n_warps;

    /* counter == nullptr: static deal, warp w of the launch takes chunks w, w + n_warps, ... */
    __device__ __forceinline__ Sweep(const int2 *patch_, int *counter_, int T_, int nsub_, int total_, int chunk_spots_)
        : patch(patch_), counter(counter_), T(T_), nsub(nsub_), total(total_), chunk_spots(chunk_spots_)
    {
        half = (threadIdx.x >> 4) & 1;
        n_warps = (int)(gridDim.x * (blockDim.x >> 5));
        const int step = counter != nullptr ? 2 : 2 * n_warps;      /* spots between two steps of a warp */
        dq = step / T;
        dr = step - dq * T;
        c_end = 0x7fffffff;
        pending = 0;
    }
    __device__ __forceinline__ void enter(Spot &s, int chunk)
    {
        s.g = chunk * chunk_spots + half;
        s.i = s.g / T;
        s.t = s.g - s.i * T;
        c_end = (chunk + 1) * chunk_spots;
        if ((threadIdx.x & 31) == 0) pending = atomicAdd(counter, 1);       /* the chunk after this one */
    }
    /* the warp's first spot */
    __device__ __forceinline__ Spot first()
    {
        Spot s;
        const int w = (int)(blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5));
        if (counter != nullptr) {
            enter(s, w);
        } else {
            s.g = 2 * w + half;
            s.i = s.g / T;
            s.t = s.g - s.i * T;
        }
        lookup(s);
        return s;
    }
    /* the look-ahead spot moves on by one warp step (into the next chunk when this one is done) */
    __device__ __forceinline__ void advance(Spot &s)
    {
        s.g += counter != nullptr ? 2 : 2 * n_warps;
        s.i += dq; s.t += dr;
        if (s.t >= T) { s.t -= T; ++s.i; }
        if (s.g >= c_end) enter(s, n_warps + __shfl_sync(0xffffffffu, pending, 0));   /* dynamic deal only */
    }
    __device__ __forceinline__ void lookup(Spot &s) const { s.pe = __ldg(patch + min(s.i, nsub - 1)); }
    /* the spot's pair is work (its chunk exists); the spot itself may still lie past the last one: live() */
    __device__ __forceinline__ bool mine(const Spot &s) const { return s.g - half < total; }
    __device__ __forceinline__ bool live(const Spot &s) const { return s.g < total; }
    /* at the end of the kernel, every warp once: the last one re-arms the counters for the next launch */
    __device__ __forceinline__ void leave() const
    {
        if (counter != nullptr && (threadIdx.x & 31) == 0) {
            /* this warp's grabs (the last one is never read) are ordered before its "done", and every warp's "done"
             * before the reset: the fences make that hold by the memory model, not just by the path to L2 */
            __threadfence();
            if (atomicAdd(counter + 1, 1) == n_warps - 1) {
                __threadfence();
                counter[0] = 0; counter[1] = 0;
            }
        }
    }
};

}  // namespace shwfs
#endif
