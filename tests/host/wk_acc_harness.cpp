/*
 * wk_acc_harness.cpp -- host-side check of the autocorrelation accumulators of csrc/wk.cu (H3 + H4 of include/shwfs.h
 * in lag-domain form: G[ly,lx] = sum_{j,k} e[j,k] conj(e[j+ly,k+lx])), the inner loop of the headline
 * kernel.  "wk_acc_extract.inc" is the block of wk.cu from load_row() to rowself_acc() -- LagAcc and the
 * three-real-product complex MAC (one packed FFMA2 + one FFMA per product) -- cut out of the .cu file AS IT IS by
 * tests/test_wk_acc_host.py (the kernels around it use launch syntax a host compiler cannot read).  The harness drives
 * it the way phase 1 of wk_measure_kernel does (row pairs (j, j + ly); lag row 0 against itself with its Hermitian
 * fill) on the kernel's shared-memory layout of the field, and compares every lag with the plain double sums.
 * Test infrastructure only.
 */
#include <cuda_runtime.h>

#include <cmath>
#include <complex>
#include <cstdio>
#include <random>

static inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }

namespace {
#include "wk_acc_extract.inc"
}

typedef std::complex<double> cd;
static std::mt19937 rng(91u);
static double worst = 0;

template <int n>
static bool one_field()
{
    constexpr int LX = 2 * n - 1;
    alignas(16) float eb[2 * n * n];                          /* row j at eb + j * 2n: (re, im) pairs, as ebuf of the kernel */
    std::uniform_real_distribution<float> U(-1.f, 1.f);
    for (int q = 0; q < n * n; ++q) {
        const float a = U(rng) * 3.14159265f, m = U(rng) < -0.7f ? 0.f : 0.5f + 0.25f * (U(rng) + 1.f);
        eb[2 * q] = m * cosf(a); eb[2 * q + 1] = m * sinf(a);
    }
    auto E = [&](int j, int k) { return cd(eb[2 * (j * n + k)], eb[2 * (j * n + k) + 1]); };
    double scale = 0;
    for (int q = 0; q < n * n; ++q) scale += std::norm(cd(eb[2 * q], eb[2 * q + 1]));
    for (int ly = 0; ly < n; ++ly) {
        LagAcc<n> L;
        L.clear();
        if (ly == 0) for (int j = 0; j < n; ++j) rowself_acc<n>(eb + j * 2 * n, L);
        else for (int j = 0; j < n - ly; ++j) rowpair_acc<n>(eb + j * 2 * n, eb + (j + ly) * 2 * n, L);
        float2 acc[LX];
        if (ly == 0) {                                        /* as in wk_measure_kernel: G[0,-lx] = conj G[0,lx], G[0,0] real */
            acc[n - 1] = make_float2(L.xy[n - 1].x + L.xy[n - 1].y, 0.f);
            for (int lx = 1; lx < n; ++lx) {
                const float2 g = L.lag_value(n - 1 + lx);
                acc[n - 1 + lx] = g;
                acc[n - 1 - lx] = make_float2(g.x, -g.y);
            }
        } else {
            for (int a = 0; a < LX; ++a) acc[a] = L.lag_value(a);
        }
        for (int a = 0; a < LX; ++a) {
            const int lx = a - (n - 1);
            cd g = 0;
            for (int j = 0; j + ly < n; ++j)
                for (int k = 0; k < n; ++k)
                    if (k + lx >= 0 && k + lx < n) g += E(j, k) * std::conj(E(j + ly, k + lx));
            const double e = std::abs(cd(acc[a].x, acc[a].y) - g) / scale;
            worst = std::fmax(worst, e);
            if (!(e <= 2e-6)) { std::printf("FAIL: n=%d lag (%d,%d): %.3g of G[0,0]\n", n, ly, lx, e); return false; }
        }
    }
    return true;
}

int main()
{
    for (int rep = 0; rep < 200; ++rep)
        if (!one_field<8>() || !one_field<10>() || !one_field<16>()) return 1;
    std::printf("ok 600 fields, worst lag error %.3g of G[0,0]\n", worst);
    return 0;
}
