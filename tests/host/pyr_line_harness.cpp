/*
 * pyr_line_harness.cpp -- host-side check of the in-CTA "four-step" line transform of csrc/pyramid.cu (Q2 / Q4 of
 * include/pyrwfs.h; "Fast Fourier Transform"): a line of L = R*R points owned by R threads of a warp,
 * R-point register FFT -> twiddles w_L^(j p) as powers of w_L^j (PowWalk) -> exchange through shared memory ->
 * R-point register FFT.  "pyr_line_extract.inc" is the block of pyramid.cu from unscramble() to line_fft(), cut out of
 * the .cu file AS IT IS by tests/test_pyr_line_host.py.  The R threads are run one after the other, twice: what a
 * thread writes into the exchange buffer depends on its own inputs only, so after the first pass the buffer holds
 * what the __syncwarp of the device guarantees, and the second pass reads it complete.
 * Checked against the float64 DFT X[k] = sum_x x[x] exp(SIGN 2 pi i x k / L): L = 256 and 1024, both signs, full and
 * input-pruned (upper half of the line zero, NZ = R/2), output layout z[q] = X[p + R q].  Test infrastructure only.
 */
#include <cuda_runtime.h>

#include <cmath>
#include <complex>
#include <cstdio>
#include <random>
#include <type_traits>
#include <vector>

static inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
static inline float2 __fadd2_rn(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
static inline float2 __fmul2_rn(float2 a, float2 b) { return make_float2(a.x * b.x, a.y * b.y); }
static inline float2 __ldg(const float2 *p) { return *p; }
static inline void __syncwarp() {}

#include "../../paper_1408_0698_b200/csrc/fft_regs.cuh"

namespace {
using namespace shwfs;
#include "pyr_line_extract.inc"
}

typedef std::complex<double> cd;
static std::mt19937 rng(92u);
static double worst = 0;

template <int R, int SIGN, int NZ>
static bool one_line()
{
    constexpr int L = R * R;
    std::uniform_real_distribution<float> U(-1.f, 1.f);
    std::vector<cd> x(L, 0.0);
    for (int m = 0; m < NZ; ++m)
        for (int j = 0; j < R; ++j) x[j + R * m] = cd(U(rng), U(rng));
    std::vector<float2> tw(L);                                   /* exp(+2 pi i m / L), as pyrwfs_create builds it */
    for (int m = 0; m < L; ++m) tw[m] = make_float2((float)std::cos(2 * M_PI * m / L), (float)std::sin(2 * M_PI * m / L));
    std::vector<float2> line((size_t)R * (R + 2) + 2);
    std::vector<float2> out((size_t)L);
    float2 *lp = line.data();
    if ((uintptr_t)lp & 15) ++lp;                                /* 16-byte rows, as the shared-memory buffer */
    for (int pass = 0; pass < 2; ++pass)
        for (int j = 0; j < R; ++j) {
            float2 z[R];
            for (int m = 0; m < R; ++m) z[m] = m < NZ ? make_float2((float)x[j + R * m].real(), (float)x[j + R * m].imag())
                                                      : make_float2(NAN, NAN);        /* known zeros: never read */
            line_fft<R, SIGN, NZ>(z, j, lp, tw.data());
            for (int q = 0; q < R; ++q) out[j + R * q] = z[q];   /* thread p = j holds X[p + R q] */
        }
    double scale = 0;
    std::vector<cd> X(L);
    for (int k = 0; k < L; ++k) {
        cd s = 0;
        for (int i = 0; i < L; ++i)
            if (x[i] != 0.0) s += x[i] * std::polar(1.0, SIGN * 2.0 * M_PI * (double)(((long)i * k) % L) / L);
        X[k] = s; scale = std::fmax(scale, std::abs(s));
    }
    for (int k = 0; k < L; ++k) {
        const double e = std::abs(cd(out[k].x, out[k].y) - X[k]) / scale;
        worst = std::fmax(worst, e);
        if (!(e <= 3e-6)) { std::printf("FAIL: R=%d SIGN=%d NZ=%d: X[%d] off by %.3g of the largest output\n", R, SIGN, NZ, k, e); return false; }
    }
    return true;
}

int main()
{
    for (int rep = 0; rep < 3; ++rep)
        if (!one_line<16, -1, 8>() || !one_line<16, +1, 16>() || !one_line<16, -1, 16>()
            || !one_line<32, -1, 16>() || !one_line<32, +1, 32>()) return 1;
    std::printf("ok 15 lines, worst error %.3g of the largest output\n", worst);
    return 0;
}
