/*
 * lit_kernel_harness.cpp -- the literal chain of csrc/literal.cu run WHOLE on the host: literal_khat_kernel (the
 * float64 transform of the re-centred elongation kernel) and literal_kernel<P, NZ> (H1 .. H8 of include/shwfs.h as
 * the paper words them: P x P FFT of the zero-padded field in shared memory, |.|^2, product with the
 * kernel's transform in the Fourier domain, inverse transform, centre, bin, threshold, centre of gravity), cut out of
 * the .cu file as text ("lit_kernel_extract.inc", written by tests/test_kernels_host.py) with the headers they include
 * compiled as they are, on the coroutine SIMT machine of simt.h.
 *
 * usage: lit_kernel_harness in.bin out.bin
 *   in.bin   int32[12] {N, n, P, b, T, nsub, mode, has_k, stage, order, seed, 0}, float[2] {tau, c_phi},
 *            phase[T*N*N], amp[N*N], int32 valid[nsub*2] (sy, sx), float K[has_k ? nsub*P*P : 0]
 *   out.bin  slopes[T*nsub*2], img[T*nsub*(stage == 2 ? D*D : P*P)]
 * What the harness supplies itself is what the launchers (host code of literal.cu) do: the LitArgs and the grids.
 * The comparison with the float64 oracle is the Python test's.  Test infrastructure only.
 */
#include "simt.h"

#include "../../paper_1408_0698_b200/csrc/internal.h"
#include "../../paper_1408_0698_b200/csrc/fft_regs.cuh"
#include "../../paper_1408_0698_b200/csrc/field.cuh"

namespace {
using namespace shwfs;
#include "lit_kernel_extract.inc"

struct Job {
    int N, n, P, b, T, nsub, mode, has_k, stage, order, seed, pad;
    float tau, c_phi;
};

template <int P, int NZ>
bool run(const Job &J, const LitArgs &A)
{
    using Cfg = LitCfg<P>;
    const int grid = (A.total + Cfg::SPB - 1) / Cfg::SPB;
    return simt::launch(grid, LIT_THREADS, Cfg::SMEM, (simt::Order)J.order, (unsigned)J.seed, [&]() { literal_kernel<P, NZ>(A); });
}

template <int P>
bool run_p(const Job &J, const LitArgs &A)
{
    return 2 * A.n <= P ? run<P, P / 2>(J, A) : run<P, P>(J, A);
}
}  // namespace

int main(int argc, char **argv)
{
    if (argc != 3) return 2;
    FILE *f = std::fopen(argv[1], "rb");
    if (!f) return 2;
    Job J;
    if (std::fread(&J, 4, 12, f) != 12 || std::fread(&J.tau, 4, 2, f) != 2) return 2;
    const int P = J.P, D = P / J.b;
    const size_t NN = (size_t)J.N * J.N, total = (size_t)J.T * J.nsub;
    std::vector<float> phase(NN * J.T), amp(NN), K(J.has_k ? (size_t)J.nsub * P * P : 0);
    std::vector<int2> valid(J.nsub);
    if (std::fread(phase.data(), 4, phase.size(), f) != phase.size() || std::fread(amp.data(), 4, NN, f) != NN ||
        std::fread(valid.data(), 8, valid.size(), f) != valid.size() || std::fread(K.data(), 4, K.size(), f) != K.size()) return 2;
    std::fclose(f);

    std::vector<float2> khat(J.has_k ? (size_t)J.nsub * P * P : 0);
    if (J.has_k && !simt::launch(J.nsub, 256, sizeof(double2) * (size_t)(P + P * P), (simt::Order)J.order, (unsigned)J.seed,
                                 [&]() { literal_khat_kernel(K.data(), P, khat.data()); })) {
        std::printf("FAIL: the K^ launch dead-locked\n");
        return 1;
    }

    const size_t per = J.stage == 2 ? (size_t)D * D : (size_t)P * P;
    std::vector<float> slopes(total * 2, NAN), img(total * per, NAN);
    LitArgs A;
    A.phase = phase.data(); A.amp = amp.data(); A.valid = valid.data();
    A.khat = J.has_k ? khat.data() : nullptr;
    A.slopes = slopes.data(); A.img = img.data();
    A.frame_stride = (long long)NN;
    A.T = J.T; A.N = J.N; A.nsub = J.nsub; A.total = (int)total; A.mode = J.mode;
    A.n = J.n; A.b = J.b; A.D = D; A.stage = J.stage;
    A.tau = J.tau;
    A.turns = (float)((double)J.c_phi / 6.283185307179586476925286766559);
    A.ramp_unit = 0.5f / (float)P;

    bool ok = false;
    switch (P) {
    case 8: ok = run_p<8>(J, A); break;
    case 16: ok = run_p<16>(J, A); break;
    case 32: ok = run_p<32>(J, A); break;
    case 64: ok = run_p<64>(J, A); break;
    default: return 2;
    }
    if (!ok) { std::printf("FAIL: the launch dead-locked\n"); return 1; }

    f = std::fopen(argv[2], "wb");
    if (!f) return 2;
    std::fwrite(slopes.data(), 4, slopes.size(), f);
    std::fwrite(img.data(), 4, img.size(), f);
    std::fclose(f);
    std::printf("ok switches %ld\n", simt::g_switches);
    return 0;
}
