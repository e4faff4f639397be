/*
 * fft_regs_harness.cpp -- host-side check of csrc/fft_regs.cuh, the register-resident line transforms every kernel
 * of the library uses (H3 / H5 / H6 of include/shwfs.h in their various forms).  The header is compiled AS IT IS for
 * the host; the Blackwell FP32x2 intrinsics get component-wise shims (fmaf per half: what FFMA2 computes).
 * Checked, for L = 2 .. 64, both signs, full and pruned inputs:
 *   - fft_fma (scalar) and fft_fma2 (packed) against the float64 DFT  X[k] = sum_m x[m] exp(SIGN 2 pi i m k / L),
 *     output k read at fft_out_index<L>(k), inputs >= NZ never read;
 *   - fft_fma2 equals fft_fma bit for bit (the header's claim: same arithmetic and rounding, element for element);
 *   - fft_fma2_split (scalar first stage) equals fft_fma2 bit for bit.
 * Built and run by tests/test_fft_regs_host.py (g++ -ffp-contract=off, no GPU).  Test infrastructure only.
 */
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <random>

static inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
static inline float2 __fadd2_rn(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
static inline float2 __fmul2_rn(float2 a, float2 b) { return make_float2(a.x * b.x, a.y * b.y); }

#include "../../paper_1408_0698_b200/csrc/fft_regs.cuh"

using namespace shwfs;

static std::mt19937 rng(1408u);
static double worst_rel = 0.0;
static long checks = 0;

static bool same_bits(float a, float b) { return std::memcmp(&a, &b, 4) == 0; }

template <int L, int SIGN, int NZ>
static bool one_case()
{
    std::uniform_real_distribution<float> U(-1.f, 1.f);
    float re[L], im[L], xr[L], xi[L];
    float2 z[L], zs[L];
    for (int m = 0; m < L; ++m) {
        /* inputs >= NZ are "known zeros": poison them, the transform must not read them */
        re[m] = m < NZ ? U(rng) : NAN; im[m] = m < NZ ? U(rng) : NAN;
        xr[m] = m < NZ ? re[m] : 0.f; xi[m] = m < NZ ? im[m] : 0.f;
        z[m] = make_float2(re[m], im[m]);
    }
    double Xr[L], Xi[L], scale = 0.0;
    for (int k = 0; k < L; ++k) {
        double sr = 0, si = 0;
        for (int m = 0; m < NZ; ++m) {
            const double a = SIGN * 2.0 * M_PI * (double)((m * k) % L) / L;
            sr += xr[m] * std::cos(a) - xi[m] * std::sin(a);
            si += xr[m] * std::sin(a) + xi[m] * std::cos(a);
        }
        Xr[k] = sr; Xi[k] = si;
        scale = std::fmax(scale, std::hypot(sr, si));
    }
    fft_fma<L, SIGN, NZ>(re, im);
    fft_fma2<L, SIGN, NZ>(z);
    for (int k = 0; k < L; ++k) {
        const int p = fft_out_index<L>(k);
        const double e = std::fmax(std::fabs(re[p] - Xr[k]), std::fabs(im[p] - Xi[k])) / scale;
        if (!(e <= 2e-6)) { std::printf("FAIL: L=%d SIGN=%d NZ=%d k=%d: error %.3g of the largest output\n", L, SIGN, NZ, k, e); return false; }
        worst_rel = std::fmax(worst_rel, e);
        if (!same_bits(re[p], z[p].x) || !same_bits(im[p], z[p].y)) {
            std::printf("FAIL: L=%d SIGN=%d NZ=%d k=%d: packed and scalar transforms differ in the last bit\n", L, SIGN, NZ, k);
            return false;
        }
        ++checks;
    }
    if constexpr (NZ == L && L >= 4) {
        float2 z2[L];
        for (int m = 0; m < L; ++m) z2[m] = make_float2(xr[m], xi[m]);
        fft_fma2<L, SIGN, L>(z2);
        fft_fma2_split<L, SIGN>(xr, xi, zs);
        for (int p = 0; p < L; ++p)
            if (!same_bits(zs[p].x, z2[p].x) || !same_bits(zs[p].y, z2[p].y)) {
                std::printf("FAIL: L=%d SIGN=%d: fft_fma2_split differs from fft_fma2 at register %d\n", L, SIGN, p);
                return false;
            }
    }
    return true;
}

template <int L, int NZ>
static bool both_signs()
{
    for (int rep = 0; rep < 20; ++rep)
        if (!one_case<L, -1, NZ>() || !one_case<L, +1, NZ>()) return false;
    return true;
}

int main()
{
    /* bit reversal and output index are involutions on [0, L) */
    for (int k = 0; k < 64; ++k)
        if (fft_out_index<64>(fft_out_index<64>(k)) != k || fft_out_index<16>(fft_out_index<16>(k & 15)) != (k & 15)) {
            std::printf("FAIL: fft_out_index is not an involution at %d\n", k);
            return 1;
        }
    /* cos64 / sin64 against libm */
    for (int k = 0; k < 64; ++k)
        if (std::fabs(cos64(k) - std::cos(2 * M_PI * k / 64)) > 6e-8 || std::fabs(sin64(k) - std::sin(2 * M_PI * k / 64)) > 6e-8) {
            std::printf("FAIL: twiddle table entry %d\n", k);
            return 1;
        }
    /* the sizes and prunings the kernels instantiate: D = 16 (n = 8 .. 16 non-zero rows), Q = 32 (16 of 32, and the
     * n = 10 instance), P = 64 (16 of 64), plus the small ones */
    bool ok = both_signs<2, 2>() && both_signs<2, 1>() && both_signs<4, 4>() && both_signs<4, 3>()
           && both_signs<8, 8>() && both_signs<8, 5>()
           && both_signs<16, 16>() && both_signs<16, 8>() && both_signs<16, 10>()
           && both_signs<32, 32>() && both_signs<32, 16>() && both_signs<32, 10>()
           && both_signs<64, 64>() && both_signs<64, 16>();
    if (!ok) return 1;
    std::printf("ok %ld outputs, worst error %.3g of the largest output\n", checks, worst_rel);
    return 0;
}
