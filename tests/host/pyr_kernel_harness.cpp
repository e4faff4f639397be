/*
 * pyr_kernel_harness.cpp -- the pyramid-sensor kernels of csrc/pyramid.cu (include/pyrwfs.h steps Q1 .. Q7;
 * PAPER.md:92) run WHOLE on the host: pyr_rows_kernel, pyr_cols_kernel, pyr_final_kernel (the in-CTA four-step
 * transforms of 256 / 1024 points with their shared-memory exchanges and transposed hand-overs through the scratch
 * A1 / A2), pyr_bin_kernel and pyr_signal_kernel, cut out of the .cu file as text ("pyr_kernel_extract.inc", written
 * by tests/test_kernels_host.py) with fft_regs.cuh compiled as it is, on the coroutine SIMT machine of simt.h, with
 * the 2-D grids of run_chunk (in waves of CTAs: the CTAs of these kernels never wait for one another).
 *
 * usage: pyr_kernel_harness in.bin out.bin
 *   in.bin   int32[10] {N, Np, s, bp, K, T, nvalid, order, seed, 0}, float[3] {r_mod, D_pix, c_phi},
 *            phase[T*N*N], amp[N*N], int32 valid[nvalid*2] (Y, X)
 *   out.bin  signals[T*nvalid*2], Q[T*4*Sp*Sp]
 * What the harness supplies itself is what pyrwfs_create and run_chunk (host code) do: the twiddle and modulation
 * tables, the PyArgs, the grids.  The comparison with the float64 oracle is the Python test's.  Test infrastructure.
 */
#include "simt.h"

#include <type_traits>

#include "../../paper_1408_0698_b200/csrc/internal.h"
#include "../../paper_1408_0698_b200/csrc/fft_regs.cuh"

namespace {
using namespace shwfs;
#include "pyr_kernel_extract.inc"

struct Job {
    int N, Np, s, bp, K, T, nvalid, order, seed, pad;
    float r_mod, D_pix, c_phi;
};

template <int R>
bool run_chunk(const Job &J, const PyArgs &A, const std::vector<int2> &valid, int Sp, float *I2, float *Q, float *signals)
{
    constexpr int L = R * R;
    const size_t smem = sizeof(float2) * (size_t)(L * (PY_LINES + 1) > PY_LINES * R * (R + 2) ? L * (PY_LINES + 1)
                                                                                              : PY_LINES * R * (R + 2));
    const int threads = PY_LINES * R;
    const simt::Order o = (simt::Order)J.order;
    if (!simt::launch2d((J.N + PY_LINES - 1) / PY_LINES, J.T * A.Kp, threads, smem, o, (unsigned)J.seed,
                        [&]() { pyr_rows_kernel<R>(A); })) return false;
    if (!simt::launch2d(L / PY_LINES, J.T * A.Kp, threads, smem, o, (unsigned)J.seed + 1, [&]() { pyr_cols_kernel<R>(A); }))
        return false;
    if (!simt::launch2d((2 * J.N + PY_LINES - 1) / PY_LINES, J.T, threads, smem, o, (unsigned)J.seed + 2,
                        [&]() { pyr_final_kernel<R>(A); })) return false;
    const int nq = J.T * 4 * Sp * Sp;
    if (!simt::launch2d((nq + 255) / 256, 1, 256, 0, o, (unsigned)J.seed + 3,
                        [&]() { pyr_bin_kernel(I2, J.N, J.bp, Sp, J.T, Q); })) return false;
    return simt::launch2d(J.T, 1, 256, sizeof(float) * 256, o, (unsigned)J.seed + 4,
                          [&]() { pyr_signal_kernel(Q, valid.data(), J.nvalid, Sp, signals); });
}
}  // namespace

int main(int argc, char **argv)
{
    if (argc != 3) return 2;
    FILE *f = std::fopen(argv[1], "rb");
    if (!f) return 2;
    Job J;
    if (std::fread(&J, 4, 10, f) != 10 || std::fread(&J.r_mod, 4, 3, f) != 3) return 2;
    const int N = J.N, Np = J.Np, Sp = N / J.bp;
    const size_t NN = (size_t)N * N;
    std::vector<float> phase(NN * J.T), amp(NN);
    std::vector<int2> valid(J.nvalid);
    if (std::fread(phase.data(), 4, phase.size(), f) != phase.size() || std::fread(amp.data(), 4, NN, f) != NN ||
        std::fread(valid.data(), 8, valid.size(), f) != valid.size()) return 2;
    std::fclose(f);
    if (Np != 256 && Np != 1024) return 2;

    /* pyrwfs_create: twiddles exp(+2 pi i m / Np), modulation tilts in turns per pixel */
    const bool modulated = J.K > 0 && J.r_mod > 0.f;
    const int Kp = modulated ? J.K : 1;
    std::vector<float2> tw(Np), md(Kp);
    for (int m = 0; m < Np; ++m) {
        const double a = 6.283185307179586476925286766559 * (double)m / (double)Np;
        tw[m] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    for (int k = 0; k < Kp; ++k) {
        const double th = 6.283185307179586476925286766559 * ((double)k + 0.5) / (double)Kp;
        const double r = modulated ? (double)J.r_mod / (double)J.D_pix : 0.0;
        md[k] = make_float2((float)(r * std::cos(th)), (float)(r * std::sin(th)));
    }
    /* scratch starts as NaN: an element a kernel should have written and did not cannot pass for a zero */
    const float2 nan2 = make_float2(NAN, NAN);
    std::vector<float2> A1((size_t)J.T * Kp * Np * N, nan2), A2((size_t)J.T * Kp * 2 * N * Np, nan2);
    std::vector<float> I2((size_t)J.T * 4 * N * N, NAN), Q((size_t)J.T * 4 * Sp * Sp, NAN), signals((size_t)J.T * J.nvalid * 2, NAN);

    PyArgs A;
    A.phase = phase.data(); A.amp = amp.data(); A.tw = tw.data(); A.mod = md.data();
    A.A1 = A1.data(); A.A2 = A2.data(); A.I2 = I2.data();
    A.N = N; A.Np = Np; A.s = J.s; A.Kp = Kp; A.Tc = J.T;
    A.turns = (float)((double)J.c_phi / 6.283185307179586476925286766559);
    A.scale = (float)(1.0 / ((double)Kp * std::pow((double)Np, 4.0)));

    const bool ok = Np == 1024 ? run_chunk<32>(J, A, valid, Sp, I2.data(), Q.data(), signals.data())
                               : run_chunk<16>(J, A, valid, Sp, I2.data(), Q.data(), signals.data());
    if (!ok) { std::printf("FAIL: a launch dead-locked\n"); return 1; }

    f = std::fopen(argv[2], "wb");
    if (!f) return 2;
    std::fwrite(signals.data(), 4, signals.size(), f);
    std::fwrite(Q.data(), 4, Q.size(), f);
    std::fclose(f);
    std::printf("ok switches %ld\n", simt::g_switches);
    return 0;
}
