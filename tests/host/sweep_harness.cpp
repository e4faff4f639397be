/*
 * sweep_harness.cpp -- host-side check of csrc/sweep.cuh, the deal of spots g = i*T + t to the warps of the
 * half-warp-per-spot kernels (pruned_fft.cu, wk_fft.cu).  The header is compiled AS IT IS for the host, with shims
 * for the few CUDA built-ins it uses; every warp of a launch is simulated by its two deciding lanes (lane 0 works on
 * the even spot of a pair and owns the atomics, lane 16 on the odd one) stepped in lockstep, the warps interleaved in
 * a seeded random order so that they run at unequal speeds, as on the device.  The loop is the kernels' own protocol:
 *     cur = first(); nxt = cur; advance(nxt); lookup(nxt);
 *     while (mine(cur)) { if (live(cur)) work(cur); cur = nxt; advance(nxt); lookup(nxt); }   leave();
 * Checked for both deals (strided; dynamic chunks from a counter), many ragged shapes, two launches in a row on
 * one counter: every spot visited exactly once with the right (i, t) and table entry, no table index out of range
 * on a live spot, and the counter pair back at zero after each launch.
 * Built and run by tests/test_sweep_host.py (g++, no GPU).  Test infrastructure: nothing of the product uses it.
 */
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <random>
#include <vector>

struct Dim { unsigned x, y, z; };
static Dim threadIdx, blockIdx, blockDim, gridDim;
static int g_lane0_pending;                 /* what __shfl_sync(.., pending, 0) returns: lane 0's value */
static long g_atomics;
static inline int atomicAdd(int *p, int v) { int o = *p; *p += v; ++g_atomics; return o; }
static inline int __shfl_sync(unsigned, int, int) { return g_lane0_pending; }
static inline void __threadfence() {}
static const int2 *g_patch_lo, *g_patch_hi; /* bounds of the table the lookups may touch */
static inline int2 __ldg(const int2 *p)
{
    if (p < g_patch_lo || p >= g_patch_hi) { std::printf("FAIL: table lookup out of bounds\n"); std::exit(1); }
    return *p;
}
using std::min;

#include "../../paper_1408_0698_b200/csrc/sweep.cuh"

using shwfs::Spot;
using shwfs::Sweep;

static void set_lane(int cta, int warp_in_cta, int lane, int grid, int block)
{
    threadIdx = {(unsigned)(32 * warp_in_cta + lane), 0, 0};
    blockIdx = {(unsigned)cta, 0, 0};
    blockDim = {(unsigned)block, 1, 1};
    gridDim = {(unsigned)grid, 1, 1};
}

struct Lane {
    Sweep sw;
    Spot cur, nxt;
};

struct Warp {
    int cta, wi;
    Lane *l[2];
    bool done;
};

#define CHECK(c, ...) do { if (!(c)) { std::printf("FAIL: " __VA_ARGS__); std::printf("\n"); return false; } } while (0)

/* one launch; look_ahead = the persistent kernels' protocol, false = the one-tile-per-CTA protocol of wk_fft.cu */
static bool launch(const std::vector<int2> &patch, int *counter, int T, int nsub, int chunk, int grid, int block,
                   bool look_ahead, std::mt19937 &rng, std::vector<int> &visits)
{
    const int total = T * nsub, wpc = block / 32;
    std::fill(visits.begin(), visits.end(), 0);
    g_patch_lo = patch.data(); g_patch_hi = patch.data() + nsub;
    std::vector<Warp> warps;
    for (int c = 0; c < grid; ++c)
        for (int w = 0; w < wpc; ++w) {
            Warp W{c, w, {nullptr, nullptr}, false};
            for (int h = 0; h < 2; ++h) {
                set_lane(c, w, 16 * h, grid, block);
                Lane *L = new Lane{Sweep(patch.data(), counter, T, nsub, total, chunk), Spot(), Spot()};
                L->cur = L->sw.first();
                L->nxt = L->cur;
                W.l[h] = L;
            }
            if (look_ahead) {
                g_lane0_pending = W.l[0]->sw.pending;
                for (int h = 0; h < 2; ++h) {
                    set_lane(c, w, 16 * h, grid, block);
                    W.l[h]->sw.advance(W.l[h]->nxt);
                    W.l[h]->sw.lookup(W.l[h]->nxt);
                }
            }
            warps.push_back(W);
        }
    size_t left = warps.size();
    std::vector<int> order(warps.size());
    for (size_t k = 0; k < order.size(); ++k) order[k] = (int)k;
    while (left) {
        std::shuffle(order.begin(), order.end(), rng);
        for (int k : order) {
            Warp &W = warps[k];
            if (W.done) continue;
            const int steps = 1 + (int)(rng() % 3);             /* warps run at unequal speeds */
            for (int s = 0; s < steps && !W.done; ++s) {
                set_lane(W.cta, W.wi, 0, grid, block);
                const bool m0 = W.l[0]->sw.mine(W.l[0]->cur);
                set_lane(W.cta, W.wi, 16, grid, block);
                const bool m1 = W.l[1]->sw.mine(W.l[1]->cur);
                CHECK(m0 == m1, "the two halves of a warp disagree on mine()");
                if (!m0) {
                    for (int h = 0; h < 2; ++h) { set_lane(W.cta, W.wi, 16 * h, grid, block); W.l[h]->sw.leave(); }
                    W.done = true; --left;
                    break;
                }
                g_lane0_pending = W.l[0]->sw.pending;           /* lockstep: both lanes see lane 0's value as it is now */
                for (int h = 0; h < 2; ++h) {
                    set_lane(W.cta, W.wi, 16 * h, grid, block);
                    Lane &L = *W.l[h];
                    if (L.sw.live(L.cur)) {
                        const Spot &c = L.cur;
                        CHECK(c.g >= 0 && c.g < total, "live spot %d outside [0,%d)", c.g, total);
                        CHECK(c.i == c.g / T && c.t == c.g % T, "spot %d: (i,t) = (%d,%d), T = %d", c.g, c.i, c.t, T);
                        CHECK(c.i < nsub, "spot %d: subaperture %d >= %d", c.g, c.i, nsub);
                        CHECK(c.pe.x == patch[c.i].x && c.pe.y == patch[c.i].y, "spot %d: wrong table entry", c.g);
                        CHECK((c.g & 1) == h, "spot %d on the wrong half-warp", c.g);
                        visits[c.g] += 1;
                    }
                    if (look_ahead) {
                        L.cur = L.nxt;
                        L.sw.advance(L.nxt);
                        L.sw.lookup(L.nxt);
                    } else {
                        L.sw.advance(L.cur);
                    }
                }
            }
        }
    }
    for (auto &W : warps) { delete W.l[0]; delete W.l[1]; }
    for (int g = 0; g < total; ++g)
        CHECK(visits[g] == 1, "T=%d nsub=%d chunk=%d grid=%d: spot %d visited %d times", T, nsub, chunk, grid, g, visits[g]);
    if (counter) CHECK(counter[0] == 0 && counter[1] == 0, "counter pair not re-armed: %d %d", counter[0], counter[1]);
    return true;
}

int main()
{
    std::mt19937 rng(14080698u);
    const int Ts[] = {1, 2, 3, 5, 17, 100};
    const int nsubs[] = {1, 2, 7, 80, 661, 1211};
    long cases = 0;
    for (int T : Ts)
        for (int nsub : nsubs) {
            std::vector<int2> patch(nsub);
            for (int i = 0; i < nsub; ++i) patch[i] = make_int2((int)(rng() & 0x3fffffff) | ((i & 1) << 30), (int)(rng() & 0xffff));
            const int total = T * nsub;
            std::vector<int> visits(total);
            const int tiles = (total + 7) / 8;
            /* strided deal, persistent protocol: any grid up to one tile per CTA (pruned_fft.cu sizes it so) */
            for (int grid : {1, 2, 3, 37, 148, 592, tiles}) {
                if (grid > tiles) continue;
                if (!launch(patch, nullptr, T, nsub, 0, grid, 128, true, rng, visits)) return 1;
                ++cases;
            }
            /* one tile per CTA, no look-ahead (the non-persistent instances of wk_fft.cu) */
            if (!launch(patch, nullptr, T, nsub, 0, tiles, 128, false, rng, visits)) return 1;
            ++cases;
            /* dynamic deal: chunks of 4 (pruned_fft.cu) and 16 (wk_fft.cu) spots, two launches in a row on one
             * counter pair; grids from one CTA up to more warps than there are chunks */
            for (int chunk : {4, 16}) {
                int counter[2] = {0, 0};
                const int nchunks = (total + chunk - 1) / chunk, need = (nchunks + 3) / 4;
                for (int grid : {1, 2, 5, 148, 592, need, need + 3}) {
                    if (grid < 1) continue;
                    for (int rep = 0; rep < 2; ++rep) {
                        if (!launch(patch, counter, T, nsub, chunk, grid, 128, true, rng, visits)) return 1;
                        ++cases;
                    }
                }
            }
        }
    std::printf("ok %ld launches, %ld atomics\n", cases, g_atomics);
    return 0;
}
