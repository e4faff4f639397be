/*
 * pf_kernel_harness.cpp -- pruned_fft_kernel of csrc/pruned_fft.cu (the config 2 kernel: H1 .. H8 of include/shwfs.h
 * without elongation kernels, one half-warp per spot) run WHOLE on the host: the kernel, cut out of the .cu file as
 * text ("pf_kernel_extract.inc", written by tests/test_kernels_host.py), with the headers it includes (fft_regs.cuh,
 * field.cuh, cog.cuh, sweep.cuh) compiled as they are, on the coroutine SIMT machine of simt.h -- every thread of the
 * launch, its shared-memory tiles, shuffles, __syncwarp's, the chunk counter of the dynamic deal and, for the TMA
 * instances, the swizzled staging slots and their mbarriers.
 *
 * usage: pf_kernel_harness in.bin out.bin
 *   in.bin   int32[14] {N, n, P, T, nsub, mode, tma, chunk, grid, order, seed, lazy_tma, pad_frames, 0}, float[2] {tau, c_phi},
 *            phase[T*N*N], amp[N*N], int32 patch[nsub*2] {first column | SHWFS_PATCH_LIT, first row}
 *   out.bin  slopes[T*nsub*2], binned[T*nsub*256], int32[2] counter pair after the launch
 * What the harness supplies itself is what the launcher (host code) does: the PfArgs and the choice of instance.
 * The comparison with the float64 oracle is the Python test's.  Test infrastructure only.
 */
#include "simt.h"

#include "../../paper_1408_0698_b200/csrc/internal.h"
#include "../../paper_1408_0698_b200/csrc/fft_regs.cuh"
#include "../../paper_1408_0698_b200/csrc/field.cuh"
#include "../../paper_1408_0698_b200/csrc/cog.cuh"
#include "../../paper_1408_0698_b200/csrc/sweep.cuh"

namespace {
using namespace shwfs;
#include "pf_kernel_extract.inc"

struct Job {
    int N, n, P, T, nsub, mode, tma, chunk, grid, order, seed, lazy, r0, r1;
    float tau, c_phi;
};

template <int P, int NZ, int MODE, bool TMA>
bool run(const Job &J, const PfArgs &A, const CUtensorMap *map)
{
    using Cfg = PfCfg<P, NZ, TMA>;
    return simt::launch(J.grid, PF_THREADS, Cfg::SMEM, (simt::Order)J.order, (unsigned)J.seed,
                        [&]() { pruned_fft_kernel<P, NZ, MODE, TMA>(A, *map); });
}

template <int P, int NZ>
bool dispatch(const Job &J, const PfArgs &A, const CUtensorMap *map)
{
    if constexpr (NZ == 16) {
        if (J.tma) return J.mode == 0 ? run<P, NZ, 0, true>(J, A, map) : run<P, NZ, 1, true>(J, A, map);
    }
    return J.mode == 0 ? run<P, NZ, 0, false>(J, A, map) : run<P, NZ, 1, false>(J, A, map);
}
}  // namespace

int main(int argc, char **argv)
{
    if (argc != 3) return 2;
    FILE *f = std::fopen(argv[1], "rb");
    if (!f) return 2;
    Job J;
    if (std::fread(&J, sizeof(int), 14, f) != 14 || std::fread(&J.tau, sizeof(float), 2, f) != 2) return 2;
    const size_t NN = (size_t)J.N * J.N, total = (size_t)J.T * J.nsub;
    std::vector<float> phase(NN * J.T), amp(NN);
    std::vector<int2> patch(J.nsub);
    if (std::fread(phase.data(), 4, phase.size(), f) != phase.size() || std::fread(amp.data(), 4, NN, f) != NN ||
        std::fread(patch.data(), 8, patch.size(), f) != patch.size()) return 2;
    std::fclose(f);

    /* outputs start as NaN: a spot the deal skipped cannot pass for one computed */
    std::vector<float> slopes(total * 2, NAN), binned(total * 256, NAN);
    int sched[2] = {0, 0};
    PfArgs A;
    A.phase = phase.data(); A.amp = amp.data(); A.patch = patch.data(); A.slopes = slopes.data(); A.binned = binned.data();
    A.sched = sched; A.chunk = J.chunk;
    A.frame_stride = (long long)NN;
    A.T = J.T; A.N = J.N; A.nsub = J.nsub; A.total = (int)total; A.n = J.n;
    A.tau = J.tau;
    A.turns = (float)((double)J.c_phi / 6.283185307179586476925286766559);
    A.ramp_unit = 0.5f / (float)J.P;

    CUtensorMap map;
    std::memset(&map, 0, sizeof(map));
    const simt::TmaMap tm{phase.data(), J.N, J.T, 16};
    static_assert(sizeof(simt::TmaMap) <= sizeof(CUtensorMap), "the stand-in fits the real map");
    std::memcpy(&map, &tm, sizeof(tm));
    simt::lazy_tma = J.lazy != 0;
    if (J.tma && J.n != 16) { std::printf("FAIL: the TMA instance is for n = 16\n"); return 1; }

    bool ok = false;
    switch (J.P) {
    case 16: ok = J.n <= 8 ? dispatch<16, 8>(J, A, &map) : dispatch<16, 16>(J, A, &map); break;
    case 32: ok = dispatch<32, 16>(J, A, &map); break;
    case 64: ok = dispatch<64, 16>(J, A, &map); break;
    default: return 2;
    }
    if (!ok) { std::printf("FAIL: the launch dead-locked\n"); return 1; }
    if (!simt::g_pending.empty() && false) return 1;

    f = std::fopen(argv[2], "wb");
    if (!f) return 2;
    std::fwrite(slopes.data(), 4, slopes.size(), f);
    std::fwrite(binned.data(), 4, binned.size(), f);
    std::fwrite(sched, 4, 2, f);
    std::fclose(f);
    std::printf("ok threads %d switches %ld boxes %ld pending %zu\n", J.grid * PF_THREADS, simt::g_switches, simt::g_boxes,
                simt::g_pending.size());
    return 0;
}
