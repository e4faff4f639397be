/*
 * loop_kernel_harness.cpp -- the FP32 kernels of csrc/loop.cu (DM phase on the valid
 * subapertures in patch layout before the sensor, control-matrix product and integrator update after it) run WHOLE on
 * the host: relayout_modes_kernel, dm_phase_kernel<FT, NN> (the cp.async double-buffered GEMM), dm_phase_gemv_kernel,
 * dm_phase_simple_kernel and recon_kernel, cut out of the .cu file as text ("loop_kernel_extract.inc", written by
 * tests/test_kernels_host.py, the launchers between the kernels removed), on the coroutine SIMT machine of simt.h.
 * The cp.async primitives of <cuda_pipeline.h> are restated as the copies they perform (size - zfill bytes copied, the
 * rest zero), done at once or -- lazy -- only when the issuing thread's __pipeline_wait_prior lets them complete.
 * (The tensor-core GEMM of dm_umma.cu, tcgen05, has no host form; its parity is tests/test_loop_gpu.py's.)
 *
 * usage: loop_kernel_harness in.bin out.bin
 *   in.bin   int32[10] {N, n, nsub, M, T, variant, order, seed, lazy, ldc}, float[1] {gain},
 *            modes[M*N*N], int32 valid[nsub*2] (sy, sx), coef[T*ldc], R[M*2*nsub], slopes[T*2*nsub]
 *            variant: 0 what launch_dm_phase_n picks for T, 1 dm_phase_kernel whatever T, 2 dm_phase_simple_kernel
 *   out.bin  dm_patch[T*nsub*n*n], coef after the update [T*ldc], hist[T*M]
 * Test infrastructure only.
 */
#include "simt.h"

#include <deque>
#include <map>

#include "../../paper_1408_0698_b200/csrc/internal.h"

/* ---- <cuda_pipeline.h>, per thread: batches of pending copies ---- */
namespace pipe {
struct Copy { void *dst; const void *src; size_t size, zfill; };
static bool lazy = false;
static std::map<simt::Thread *, std::deque<std::vector<Copy>>> q;
static void perform(const Copy &c)
{
    std::memcpy(c.dst, c.src, c.size - c.zfill);
    std::memset(static_cast<unsigned char *>(c.dst) + (c.size - c.zfill), 0, c.zfill);
}
}  // namespace pipe
static inline void __pipeline_memcpy_async(void *dst, const void *src, size_t size, size_t zfill = 0)
{
    const pipe::Copy c{dst, src, size, zfill};
    if (!pipe::lazy) { pipe::perform(c); return; }
    auto &d = pipe::q[simt::cur];                               /* d.back() is the open (uncommitted) batch */
    if (d.empty()) d.emplace_back();
    d.back().push_back(c);
}
static inline void __pipeline_commit()
{
    if (!pipe::lazy) return;
    auto &d = pipe::q[simt::cur];
    if (d.empty()) d.emplace_back();
    d.emplace_back();                                           /* closes the open batch, opens the next */
}
static inline void __pipeline_wait_prior(int n)
{
    if (!pipe::lazy) return;
    auto &d = pipe::q[simt::cur];
    while ((int)d.size() - 1 > n) {                             /* all but the newest n committed batches */
        for (const pipe::Copy &c : d.front()) pipe::perform(c);
        d.pop_front();
    }
}

namespace {
#include "loop_kernel_extract.inc"

struct Job {
    int N, n, nsub, M, T, variant, order, seed, lazy, ldc;
    float gain;
};

template <int FT, int NN>
bool dm_gemm(const Job &J, const float *coef, const float *modes_sub, float *out)
{
    constexpr int TT = 8 * FT;
    const size_t smem = 2 * sizeof(float) * (size_t)(DM_MC * NN + DM_MC * (TT + 4));
    return simt::launch2d((J.T + TT - 1) / TT, J.nsub, 256, smem, (simt::Order)J.order, (unsigned)J.seed,
                          [&]() { dm_phase_kernel<FT, NN>(coef, J.ldc, modes_sub, J.T, J.nsub, J.M, out); }, 4);
}

template <int NN, int FMAX>
bool dm_gemv(const Job &J, const float *coef, const float *modes_sub, float *out)
{
    return simt::launch2d((J.nsub + 7) / 8, 1, 256, sizeof(float) * FMAX * (size_t)J.M, (simt::Order)J.order, (unsigned)J.seed,
                          [&]() { dm_phase_gemv_kernel<NN, FMAX>(coef, J.ldc, modes_sub, J.T, J.nsub, J.M, out); }, 4);
}

/* launch_dm_phase_n of loop.cu */
template <int NN>
bool dm_phase_n(const Job &J, const float *coef, const float *modes_sub, float *out)
{
    const int T = J.T;
    if (J.variant == 0 && T <= 8 && (size_t)J.M * 8 * sizeof(float) <= 48 * 1024) {
        if (T == 1) return dm_gemv<NN, 1>(J, coef, modes_sub, out);
        if (T == 2) return dm_gemv<NN, 2>(J, coef, modes_sub, out);
        if (T <= 4) return dm_gemv<NN, 4>(J, coef, modes_sub, out);
        return dm_gemv<NN, 8>(J, coef, modes_sub, out);
    }
    if (T <= 8) return dm_gemm<1, NN>(J, coef, modes_sub, out);
    if (T <= 32) return dm_gemm<4, NN>(J, coef, modes_sub, out);
    return dm_gemm<8, NN>(J, coef, modes_sub, out);
}
}  // namespace

int main(int argc, char **argv)
{
    if (argc != 3) return 2;
    FILE *f = std::fopen(argv[1], "rb");
    if (!f) return 2;
    Job J;
    if (std::fread(&J, 4, 10, f) != 10 || std::fread(&J.gain, 4, 1, f) != 1) return 2;
    const int nn = J.n * J.n, K = 2 * J.nsub;
    std::vector<float> modes((size_t)J.M * J.N * J.N), coef((size_t)J.T * J.ldc), R((size_t)J.M * K), s((size_t)J.T * K);
    std::vector<int2> valid(J.nsub);
    if (std::fread(modes.data(), 4, modes.size(), f) != modes.size() || std::fread(valid.data(), 8, valid.size(), f) != valid.size() ||
        std::fread(coef.data(), 4, coef.size(), f) != coef.size() || std::fread(R.data(), 4, R.size(), f) != R.size() ||
        std::fread(s.data(), 4, s.size(), f) != s.size()) return 2;
    std::fclose(f);
    pipe::lazy = J.lazy != 0;
    const simt::Order o = (simt::Order)J.order;

    /* shwfs_set_dm: the per-subaperture re-layout of the modes */
    std::vector<float> modes_sub((size_t)J.nsub * J.M * nn, NAN), patch((size_t)J.T * J.nsub * nn, NAN), hist((size_t)J.T * J.M, NAN);
    if (!simt::launch2d(J.nsub, J.M, 128, 0, o, (unsigned)J.seed,
                        [&]() { relayout_modes_kernel(modes.data(), valid.data(), J.N, J.n, J.M, modes_sub.data()); }, 32)) {
        std::printf("FAIL: relayout dead-locked\n");
        return 1;
    }
    /* shwfs_loop_dm_phase, FP32 branch */
    bool ok;
    if (J.variant != 2 && (nn == 64 || nn == 100 || nn == 256)) {
        ok = nn == 64 ? dm_phase_n<64>(J, coef.data(), modes_sub.data(), patch.data())
           : nn == 100 ? dm_phase_n<100>(J, coef.data(), modes_sub.data(), patch.data())
                       : dm_phase_n<256>(J, coef.data(), modes_sub.data(), patch.data());
    } else {
        const size_t total = (size_t)J.T * J.nsub * nn;
        ok = simt::launch2d((int)((total + 255) / 256), 1, 256, 0, o, (unsigned)J.seed, [&]() {
            dm_phase_simple_kernel(coef.data(), J.ldc, modes_sub.data(), J.T, J.nsub, nn, J.M, patch.data());
        }, 8);
    }
    if (!ok) { std::printf("FAIL: the DM-phase launch dead-locked\n"); return 1; }
    for (auto &kv : pipe::q)
        for (auto &b : kv.second)
            if (!b.empty()) { std::printf("FAIL: a cp.async copy was never waited for\n"); return 1; }

    /* shwfs_loop_reconstruct */
    if (J.T <= 2)
        ok = simt::launch2d(J.M, 1, 1024, sizeof(float) * (1024 / 32) * RC_TT, o, (unsigned)J.seed + 1, [&]() {
            recon_kernel<1024>(R.data(), s.data(), J.T, K, J.M, J.gain, coef.data(), J.ldc, hist.data());
        }, 2);
    else
        ok = simt::launch2d(J.M, 1, 256, sizeof(float) * (256 / 32) * RC_TT, o, (unsigned)J.seed + 1, [&]() {
            recon_kernel<256>(R.data(), s.data(), J.T, K, J.M, J.gain, coef.data(), J.ldc, hist.data());
        }, 8);
    if (!ok) { std::printf("FAIL: the reconstructor dead-locked\n"); return 1; }

    f = std::fopen(argv[2], "wb");
    if (!f) return 2;
    std::fwrite(patch.data(), 4, patch.size(), f);
    std::fwrite(coef.data(), 4, coef.size(), f);
    std::fwrite(hist.data(), 4, hist.size(), f);
    std::fclose(f);
    std::printf("ok switches %ld\n", simt::g_switches);
    return 0;
}
