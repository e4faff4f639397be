/*
 * noise_harness.cpp -- host-side parity of csrc/noise.cuh (detector noise; "the
 * centroid computed on the final noise-added image") against the float64 oracle (oracle/shwfs_oracle_lgs.c,
 * oracle/shwfs_oracle_poisson.c, linked in as C objects).  The device header is compiled AS IT IS for the host; the
 * CUDA built-ins it uses get shims (__umulhi exact; __logf / __sincosf by libm's logf / sinf / cosf).
 *   - philox4x32_10 equals the oracle's Philox bit for bit on random counters and keys;
 *   - the four normal deviates of a block agree with the oracle's to 2e-6;
 *   - the Gaussian-limit count (photon_model 0) agrees to 1e-5 of sqrt(rate + ron^2);
 *   - the fp32 Poisson draw (photon_model 1: inversion below a rate of 30, PTRS above) returns the oracle's integer
 *     on every draw the oracle reports as decided by more than rounding (margin > 1e-4 + 1e-5 rate, the criterion of
 *     tests/test_lgs_gpu.py), differs by at most one count on the other inversion draws, and those are rare.
 * Built and run by tests/test_noise_host.py (gcc + g++, no GPU).  Test infrastructure only.
 */
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <random>

static inline uint32_t __umulhi(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }
/* __logf and __sincosf are declared by glibc's <math.h> (its internal names of logf / sincosf) but not exported:
 * defined here with the declared linkage */
extern "C" float __logf(float x) noexcept { return logf(x); }
extern "C" void __sincosf(float x, float *s, float *c) noexcept { *s = sinf(x); *c = cosf(x); }
#ifndef __noinline__
#define __noinline__ __attribute__((noinline))
#endif

#include "../../paper_1408_0698_b200/csrc/noise.cuh"

extern "C" {
void shwfs_oracle_philox4x32(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void shwfs_oracle_normal4(uint64_t seed, uint32_t t, uint32_t i, uint32_t blk, double z[4]);
long shwfs_oracle_poisson_draw(double lambda, uint64_t seed, uint32_t t, uint32_t i, uint32_t p, double *margin);
void shwfs_oracle_add_noise(const double *B, int D, double F, double ron, uint64_t seed, uint32_t t, uint32_t i,
                            double *counts);
}

using namespace shwfs;

#define FAIL(...) do { std::printf("FAIL: " __VA_ARGS__); std::printf("\n"); return 1; } while (0)

int main()
{
    std::mt19937_64 rng(0x14080698ull);
    /* ---- Philox: bit for bit ---- */
    for (int k = 0; k < 20000; ++k) {
        const uint32_t c[4] = {(uint32_t)rng(), (uint32_t)rng(), (uint32_t)rng(), (uint32_t)rng()};
        const uint32_t key[2] = {(uint32_t)rng(), (uint32_t)rng()};
        uint32_t want[4];
        shwfs_oracle_philox4x32(c, key, want);
        const uint4 got = philox4x32_10(make_uint4(c[0], c[1], c[2], c[3]), make_uint2(key[0], key[1]));
        if (got.x != want[0] || got.y != want[1] || got.z != want[2] || got.w != want[3]) FAIL("philox block %d", k);
    }
    /* ---- normal deviates and the Gaussian-limit count ---- */
    const uint64_t seed = 0x1408069800000091ull;
    const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
    double worst_z = 0;
    for (int k = 0; k < 20000; ++k) {
        const uint32_t t = (uint32_t)(rng() % 1000), i = (uint32_t)(rng() % 4632), blk = (uint32_t)(rng() % 64);
        float z[4]; double zo[4];
        normal4(key, t, i, blk, z);
        shwfs_oracle_normal4(seed, t, i, blk, zo);
        for (int q = 0; q < 4; ++q) {
            const double e = std::fabs((double)z[q] - zo[q]);
            if (!(e <= 2e-6 * (1.0 + std::fabs(zo[q])))) FAIL("normal deviate (t=%u i=%u blk=%u q=%d): %.9g vs %.9g", t, i, blk, q, z[q], zo[q]);
            worst_z = std::fmax(worst_z, e);
        }
    }
    {
        double B[256], counts[256];
        for (int q = 0; q < 256; ++q) B[q] = (double)(float)(std::ldexp((double)(rng() % 100000), -14));
        const double F = 5.0, ron = 3.0;
        shwfs_oracle_add_noise(B, 16, F, ron, seed, 7u, 11u, counts);
        for (int C = 0; C < 16; ++C) {
            float col[16];
            for (int R = 0; R < 16; ++R) col[R] = (float)B[R * 16 + C];
            add_noise_col16(col, C, key, 7u, 11u, (float)F, (float)(ron * ron), 0);
            for (int R = 0; R < 16; ++R) {
                const double sig = std::sqrt(F * B[R * 16 + C] + ron * ron);
                if (!(std::fabs((double)col[R] - counts[R * 16 + C]) <= 1e-5 * sig + 1e-6 * std::fabs(counts[R * 16 + C])))
                    FAIL("Gaussian-limit count at (R=%d,C=%d): %.9g vs %.9g", R, C, col[R], counts[R * 16 + C]);
            }
        }
    }
    /* ---- Poisson draws: the column routine of the kernels against the oracle, pixel by pixel ---- */
    long clear = 0, unclear = 0, unclear_diff = 0;
    const double rates[] = {0.02, 0.3, 1.0, 3.0, 9.5, 29.0, 31.0, 75.0, 300.0, 2500.0};
    for (double base : rates)
        for (int rep = 0; rep < 40; ++rep) {
            const uint32_t t = (uint32_t)(rng() % 1000), i = (uint32_t)(rng() % 4632);
            for (int C = 0; C < 16; ++C) {
                float col[16], rate[16];
                for (int R = 0; R < 16; ++R) { rate[R] = (float)(base * (0.5 + (double)(rng() % 1000) / 1000.0)); col[R] = rate[R]; }
                add_noise_col16(col, C, key, t, i, 1.0f, 0.0f, 1);                       /* F = 1, no read noise */
                for (int R = 0; R < 16; ++R) {
                    double margin;
                    const uint32_t p = (uint32_t)(16 * C + R);
                    const long want = shwfs_oracle_poisson_draw((double)rate[R], seed, t, i, p, &margin);
                    const bool is_clear = margin > 1e-4 + 1e-5 * rate[R];
                    const double d = std::fabs((double)col[R] - (double)want);
                    if (col[R] != std::floor(col[R]) || col[R] < 0.f) FAIL("count %.9g is not a non-negative integer", col[R]);
                    if (is_clear) {
                        ++clear;
                        if (d != 0.0) FAIL("rate %.6g (t=%u i=%u p=%u): %g vs oracle %ld, margin %.3g", rate[R], t, i, p, col[R], want, margin);
                    } else {
                        ++unclear;
                        if (d != 0.0) ++unclear_diff;
                        if (rate[R] < 29.9f && d > 1.0) FAIL("unclear inversion draw differs by %g counts", d);
                        if (d > 8.0 * std::sqrt((double)rate[R]) + 2.0) FAIL("unclear rejection draw differs by %g counts", d);
                    }
                }
            }
        }
    /* unclear draws are rare: the clearance 1e-4 + 1e-5 rate is a few per cent of a count only at the rates of thousands */
    if (!(unclear <= 0.06 * (clear + unclear))) FAIL("%ld of %ld draws unclear", unclear, clear + unclear);
    std::printf("ok philox 20000 blocks, worst deviate error %.2g, %ld clear Poisson draws identical, %ld unclear (%ld differ)\n",
                worst_z, clear, unclear, unclear_diff);
    return 0;
}
