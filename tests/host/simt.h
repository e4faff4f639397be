/*
 * simt.h -- a small SIMT machine on the host, for running WHOLE kernels of csrc/ (cut out of their .cu files as text)
 * without a GPU.  Every CUDA thread of a launch is a coroutine (ucontext) with its own stack; a thread runs until it
 * reaches a synchronising built-in -- __syncwarp, __shfl_*_sync, __syncthreads, a wait on an mbarrier -- and is
 * switched out there until the threads it waits for have arrived.  Between two such points a thread runs alone, and
 * the ORDER in which runnable threads are picked is the caller's: ascending, descending, or seeded random.  Code that
 * needs a barrier it does not have (a shared-memory value read before its writer has run, a staging slot rewritten
 * while another lane still reads it) then gives wrong results under at least one of the orders, where a GPU, whose
 * warps mostly run in lockstep, may hide it: a poor man's racecheck beside the element-wise comparison with the oracle.
 *
 * Built-ins provided: threadIdx / blockIdx / blockDim / gridDim, __syncthreads, __syncwarp, __shfl_sync,
 * __shfl_xor_sync, __shfl_down_sync (32-bit types), __ldg, atomicAdd(int), __threadfence, the packed FP32x2
 * intrinsics (component-wise fmaf: what FFMA2 computes), __sincosf / __expf / __logf by libm, and the TMA / mbarrier
 * calls of csrc/tma.cuh: a box load is a plain copy with the 64-byte swizzle of the tensor map (16-byte chunk q of
 * row r at chunk q ^ ((r >> 1) & 3)), performed either at once or -- `lazy_tma` -- only when a thread waits on its
 * mbarrier: the earliest and the latest moment the hardware may complete it.
 *
 * Under the random order a thread may also be switched out right before an atomicAdd.  CTAs of a 1-D launch are all
 * resident from the start (launch); 2-D launches run in waves of CTAs (launch2d).  Coroutine stacks are pooled.
 *
 * Test infrastructure only (tests/test_kernels_host.py); nothing of the product uses it.
 */
#ifndef SHWFS_TEST_SIMT_H_
#define SHWFS_TEST_SIMT_H_

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <ucontext.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <map>
#include <random>
#include <vector>

namespace simt {

struct Dim { unsigned x, y, z; };

struct Warp {
    int live = 0, arrived = 0;
    unsigned gen = 0;
    uint32_t slot[2][32];            /* shuffle operands, double-buffered by the parity of the shuffle */
    unsigned shfl = 0;
};

struct Cta {
    int live = 0, arrived = 0;
    unsigned gen = 0;
    std::vector<unsigned char> smem;
    std::vector<Warp> warps;
};

struct Thread {
    ucontext_t ctx;
    unsigned char *stack = nullptr;  /* not zero-filled: most of it is never touched */
    Dim tid, bid;
    Cta *cta;
    Warp *warp;
    int lane;
    unsigned shfl_n = 0;             /* shuffles this thread has done (selects the slot buffer) */
    bool done = false;
};

enum Order { ASCENDING, DESCENDING, RANDOM };

static Thread *cur = nullptr;
static Dim g_block, g_grid;
static ucontext_t g_main;
static std::function<void()> g_body;
static long g_switches = 0;
static long g_progress = 0;             /* barriers released + threads finished */
static int g_order = 0;
static std::minstd_rand g_yield_rng(1408u);
static std::map<size_t, std::vector<unsigned char *>> g_stack_pool;

static void yield() { ++g_switches; swapcontext(&cur->ctx, &g_main); }

static void trampoline()
{
    g_body();
    Thread *t = cur;
    t->done = true;
    ++g_progress;
    /* a thread that has left no longer counts at the barriers of its warp and CTA */
    Warp *w = t->warp;
    if (--w->live > 0 && w->arrived == w->live) { w->arrived = 0; ++w->gen; ++g_progress; }
    Cta *c = t->cta;
    if (--c->live > 0 && c->arrived == c->live) { c->arrived = 0; ++c->gen; ++g_progress; }
    swapcontext(&t->ctx, &g_main);
}

static void warp_barrier()
{
    Warp *w = cur->warp;
    const unsigned g = w->gen;
    if (++w->arrived == w->live) { w->arrived = 0; ++w->gen; ++g_progress; return; }
    while (w->gen == g) yield();
}

static void cta_barrier()
{
    Cta *c = cur->cta;
    const unsigned g = c->gen;
    if (++c->arrived == c->live) { c->arrived = 0; ++c->gen; ++g_progress; return; }
    while (c->gen == g) yield();
}

/* value of lane `src` (taken modulo 32) at this shuffle */
static uint32_t shuffle(uint32_t v, int src)
{
    Thread *t = cur;
    const unsigned b = t->shfl_n++ & 1u;
    t->warp->slot[b][t->lane] = v;
    warp_barrier();
    return t->warp->slot[b][src & 31];
}

/* Runs body() once per thread of the CTAs `bids` (all resident at once) with smem_bytes of dynamic shared memory per
 * CTA (zero filled).  Returns false if the threads dead-lock (a barrier not reached by everybody). */
static bool run_ctas(const std::vector<Dim> &bids, int block, size_t smem_bytes, Order order, unsigned seed, size_t stack_bytes)
{
    const int grid = (int)bids.size();
    const int wpc = (block + 31) / 32;
    g_order = (int)order;
    g_yield_rng.seed(seed + 17u);
    std::vector<Cta> ctas(grid);
    std::vector<Thread> th((size_t)grid * block);
    for (int c = 0; c < grid; ++c) {
        ctas[c].smem.assign(smem_bytes + 16, 0);
        ctas[c].warps.resize(wpc);
        ctas[c].live = block;
        for (int t = 0; t < block; ++t) {
            Thread &T = th[(size_t)c * block + t];
            T.tid = {(unsigned)t, 0, 0};
            T.bid = bids[c];
            T.cta = &ctas[c];
            T.warp = &ctas[c].warps[t / 32];
            T.lane = t % 32;
            T.warp->live++;
            if (!g_stack_pool[stack_bytes].empty()) {      /* stacks are reused from wave to wave and launch to launch */
                T.stack = g_stack_pool[stack_bytes].back();
                g_stack_pool[stack_bytes].pop_back();
            } else {
                T.stack = static_cast<unsigned char *>(std::malloc(stack_bytes));
            }
            getcontext(&T.ctx);
            T.ctx.uc_stack.ss_sp = T.stack;
            T.ctx.uc_stack.ss_size = stack_bytes;
            T.ctx.uc_link = &g_main;
            makecontext(&T.ctx, trampoline, 0);
        }
    }
    std::mt19937 rng(seed);
    std::vector<int> idx(th.size());
    for (size_t i = 0; i < idx.size(); ++i) idx[i] = (int)i;
    size_t left = th.size();
    long idle_rounds = 0;
    while (left > 0) {
        if (order == RANDOM) std::shuffle(idx.begin(), idx.end(), rng);
        else if (order == DESCENDING) std::sort(idx.begin(), idx.end(), std::greater<int>());
        const long before = g_progress;
        size_t finished = 0;
        for (int i : idx) {
            Thread &T = th[i];
            if (T.done) continue;
            cur = &T;
            swapcontext(&g_main, &T.ctx);
            if (T.done) ++finished;
        }
        cur = nullptr;
        left -= finished;
        /* a whole round in which no barrier was released and nobody finished: every thread only re-checked the
         * barrier it sits at, and nothing can change that any more */
        if (g_progress == before) { if (++idle_rounds > 2) return false; }     /* (stacks left to the exit) */
        else idle_rounds = 0;
    }
    for (Thread &T : th) g_stack_pool[stack_bytes].push_back(T.stack);
    return true;
}

/* a 1-D launch, every CTA resident from the start (what the persistent kernels' grids are sized for) */
static bool launch(int grid, int block, size_t smem_bytes, Order order, unsigned seed, const std::function<void()> &body,
                   size_t stack_bytes = 256 * 1024)
{
    g_block = {(unsigned)block, 1, 1};
    g_grid = {(unsigned)grid, 1, 1};
    g_body = body;
    std::vector<Dim> bids(grid);
    for (int c = 0; c < grid; ++c) bids[c] = {(unsigned)c, 0, 0};
    return run_ctas(bids, block, smem_bytes, order, seed, stack_bytes);
}

/* a 2-D launch in waves of `wave` CTAs (CTAs of these kernels never wait for one another) */
static bool launch2d(int gx, int gy, int block, size_t smem_bytes, Order order, unsigned seed, const std::function<void()> &body,
                     int wave = 16, size_t stack_bytes = 256 * 1024)
{
    g_block = {(unsigned)block, 1, 1};
    g_grid = {(unsigned)gx, (unsigned)gy, 1};
    g_body = body;
    std::vector<Dim> bids;
    for (int y = 0; y < gy; ++y)
        for (int x = 0; x < gx; ++x) {
            bids.push_back({(unsigned)x, (unsigned)y, 0});
            if ((int)bids.size() == wave || (y == gy - 1 && x == gx - 1)) {
                if (!run_ctas(bids, block, smem_bytes, order, seed + (unsigned)(y * gx + x), stack_bytes)) return false;
                bids.clear();
            }
        }
    return true;
}

static unsigned char *smem()
{
    unsigned char *p = cur->cta->smem.data();
    return p + ((16 - ((uintptr_t)p & 15)) & 15);
}

/* ---- TMA / mbarrier of csrc/tma.cuh ---- */
struct TmaMap { const float *base; int N; long long frames; int n; };   /* what shwfs_tma_patch_map encodes */
struct PendingBox { void *dst; const CUtensorMap *map; int x, y, z; uint64_t *bar; };
static bool lazy_tma = false;
static std::vector<PendingBox> g_pending;
static long g_boxes = 0;

static void complete(const PendingBox &b)
{
    const TmaMap *m = reinterpret_cast<const TmaMap *>(b.map);
    unsigned char *dst = static_cast<unsigned char *>(b.dst);
    for (int r = 0; r < m->n; ++r)
        for (int q = 0; q < m->n / 4; ++q) {
            float chunk[4];
            for (int e = 0; e < 4; ++e) {
                /* elements outside the tensor read as zero (the map's out-of-bounds fill) */
                const int x = b.x + 4 * q + e, y = b.y + r;
                const bool in = x >= 0 && x < m->N && y >= 0 && y < m->N && b.z >= 0 && b.z < m->frames;
                chunk[e] = in ? m->base[((size_t)b.z * m->N + y) * m->N + x] : 0.f;
            }
            const int sw = m->n == 16 ? ((r >> 1) & 3) : 0;
            std::memcpy(dst + (size_t)r * m->n * 4 + (size_t)((q ^ sw) * 16), chunk, 16);
        }
    ++*b.bar;                        /* one box per phase (expect_tx of its bytes, arrival count 1) */
    ++g_boxes;
    ++g_progress;
}

}  // namespace simt

/* ---- the built-ins, as the kernels spell them ---- */
#undef __launch_bounds__
#define __launch_bounds__(...)
#undef __grid_constant__
#define __grid_constant__
#define threadIdx (simt::cur->tid)
#define blockIdx (simt::cur->bid)
#define blockDim (simt::g_block)
#define gridDim (simt::g_grid)

static inline void __syncthreads() { simt::cta_barrier(); }
static inline void __syncwarp(unsigned = 0xffffffffu) { simt::warp_barrier(); }
static inline void __threadfence() {}

template <class T>
static inline T simt_shfl(T v, int src)
{
    static_assert(sizeof(T) == 4, "32-bit shuffles only");
    uint32_t u;
    std::memcpy(&u, &v, 4);
    u = simt::shuffle(u, src);
    std::memcpy(&v, &u, 4);
    return v;
}
template <class T> static inline T __shfl_sync(unsigned, T v, int src) { return simt_shfl(v, src); }
template <class T> static inline T __shfl_xor_sync(unsigned, T v, int o) { return simt_shfl(v, simt::cur->lane ^ o); }
template <class T> static inline T __shfl_down_sync(unsigned, T v, int d)
{
    const int s = simt::cur->lane + d;
    return simt_shfl(v, s < 32 ? s : simt::cur->lane);
}

template <class T> static inline T __ldg(const T *p) { return *p; }
/* under the random order a thread may also be switched out right before an atomic: the warps of the dynamic deal then
 * reach the chunk counter (and its re-arming by the last warp out) in every interleaving, not only at barriers */
static inline int atomicAdd(int *p, int v)
{
    if (simt::g_order == simt::RANDOM && (simt::g_yield_rng() & 1u)) simt::yield();
    ++simt::g_progress;              /* an atomic performed is progress (dead-lock detection) */
    const int o = *p;
    *p += v;
    return o;
}
using std::max;
using std::min;

static inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
static inline float2 __fadd2_rn(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
static inline float2 __fmul2_rn(float2 a, float2 b) { return make_float2(a.x * b.x, a.y * b.y); }
extern "C" void __sincosf(float x, float *s, float *c) noexcept { *s = sinf(x); *c = cosf(x); }
extern "C" float __logf(float x) noexcept { return logf(x); }
extern "C" float __expf(float x) noexcept { return expf(x); }
static inline uint32_t __umulhi(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }
static inline void sincospi(double x, double *s, double *c) { *s = std::sin(M_PI * x); *c = std::cos(M_PI * x); }
static inline void sincospif(float x, float *s, float *c) { *s = (float)std::sin(M_PI * (double)x); *c = (float)std::cos(M_PI * (double)x); }
#undef __noinline__
#define __noinline__ __attribute__((noinline))
static inline size_t __cvta_generic_to_shared(const void *p) { return (size_t)p; }

/* csrc/tma.cuh, simulated (the header itself is inline PTX) */
#define SHWFS_TMA_CUH_
namespace shwfs {
static inline uint32_t smem_addr(const void *p) { return (uint32_t)(uintptr_t)p; }
static inline void mbar_init(uint64_t *bar, int) { *bar = 0; }       /* the word holds the number of completed phases */
static inline void mbar_init_fence() {}
static inline void mbar_expect_tx(uint64_t *, uint32_t) {}
static inline void tma_prefetch_map(const CUtensorMap *) {}
static inline void tma_load_patch(void *dst, const CUtensorMap *map, int x, int y, int z, uint64_t *bar)
{
    const simt::PendingBox b{dst, map, x, y, z, bar};
    if (simt::lazy_tma) simt::g_pending.push_back(b);
    else simt::complete(b);
}
/* try_wait.parity succeeds once the phase of that parity is over, i.e. the barrier is in a phase of the other
 * parity.  A wait for a box nobody requested never returns: the launch then counts as dead-locked, as on a GPU. */
static inline void mbar_wait(uint64_t *bar, uint32_t parity)
{
    while ((*bar & 1u) == parity) {
        bool found = false;
        for (size_t k = 0; k < simt::g_pending.size() && !found; ++k)
            if (simt::g_pending[k].bar == bar) {
                const simt::PendingBox b = simt::g_pending[k];
                simt::g_pending.erase(simt::g_pending.begin() + (long)k);
                simt::complete(b);
                found = true;
            }
        if (!found) simt::yield();
    }
}
}  // namespace shwfs

#endif
