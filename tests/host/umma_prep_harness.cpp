/*
 * umma_prep_harness.cpp -- the part of the tensor-core DM-phase path (csrc/dm_umma.cu) that has a
 * host form: umma_split_modes_kernel and umma_split_coef_kernel, which build the operands of dm_umma_kernel -- every
 * fp32 value split x = hi + lo into two TF32 numbers and laid out in the tensor core's canonical K-major no-swizzle
 * tiles [k/4][row/8][row%8][k%4] -- cut out of the .cu file as text ("umma_prep_extract.inc", written by
 * tests/test_kernels_host.py; the one PTX instruction cvt.rna.tf32.f32 restated as round-to-nearest, ties away, to 10
 * mantissa bits) and run on the SIMT machine of simt.h.  The tcgen05 kernel itself has no host form; what is checked
 * here is what it is fed and the arithmetic claim of its header:
 *   - every hi and lo is a TF32 number (13 low mantissa bits zero), the padding (modes >= M, pixels >= NN, frames >= T)
 *     is exactly zero, and every element sits where the layout formula says;
 *   - C = A_hi B_hi + A_hi B_lo + A_lo B_hi, summed exactly (double) from the tiles as the MMA reads them, equals
 *     sum_m coef[t][m] modes[i][m][px] to ~2^-22 relative, while the hi terms alone are ~2^-11 off.
 * usage: umma_prep_harness nsub M NN NP T  ->  "ok <split error> <single-pass error>", errors relative to max |C|.
 * Test infrastructure only.
 */
#include "simt.h"

#include "../../paper_1408_0698_b200/csrc/internal.h"

static inline float host_tf32_rna(float x)
{
    uint32_t u;
    std::memcpy(&u, &x, 4);
    u = (u + 0x1000u) & ~0x1FFFu;            /* nearest, ties away from zero, on the magnitude */
    std::memcpy(&x, &u, 4);
    return x;
}

namespace {
#include "umma_prep_extract.inc"
}

static bool is_tf32(float x)
{
    uint32_t u;
    std::memcpy(&u, &x, 4);
    return (u & 0x1FFFu) == 0;
}

int main(int argc, char **argv)
{
    if (argc != 6) return 2;
    const int nsub = std::atoi(argv[1]), M = std::atoi(argv[2]), NN = std::atoi(argv[3]), NP = std::atoi(argv[4]), T = std::atoi(argv[5]);
    const int nkb = (M + UM_KB - 1) / UM_KB, mt = (T + UM_MT - 1) / UM_MT;
    std::mt19937 rng(76u);
    std::normal_distribution<float> G(0.f, 1.f);
    std::vector<float> modes((size_t)nsub * M * NN), coef((size_t)T * M);
    for (auto &v : modes) v = G(rng);
    for (auto &v : coef) v = 0.5f * G(rng);
    std::vector<float> B((size_t)nsub * nkb * 2 * UM_KB * NP, NAN), A((size_t)mt * nkb * 2 * UM_KB * UM_MT, NAN);
    if (!simt::launch2d(nsub, nkb, 256, 0, simt::RANDOM, 1u,
                        [&]() { umma_split_modes_kernel(modes.data(), M, NN, NP, nkb, B.data()); }, 8) ||
        !simt::launch2d(mt, nkb, 256, 0, simt::RANDOM, 2u,
                        [&]() { umma_split_coef_kernel(coef.data(), M, T, M, nkb, A.data()); }, 8)) {
        std::printf("FAIL: dead-lock\n");
        return 1;
    }
    for (float v : B) if (!(is_tf32(v))) { std::printf("FAIL: a mode operand is not a TF32 number (or was never written)\n"); return 1; }
    for (float v : A) if (!(is_tf32(v))) { std::printf("FAIL: a coefficient operand is not a TF32 number (or was never written)\n"); return 1; }

    /* element (row, k) of a canonical tile of `rows` rows: [k/4][row/8][row%8][k%4] */
    auto at = [](const float *tile, int row, int k, int rows) { return tile[(k / 4) * (rows * 4) + (row / 8) * 32 + (row % 8) * 4 + (k % 4)]; };
    double worst3 = 0, worst1 = 0, cmax = 0;
    for (int i = 0; i < nsub; ++i)
        for (int t = 0; t < mt * UM_MT; ++t)
            for (int px = 0; px < NP; ++px) {
                double c3 = 0, c1 = 0, exact = 0;
                for (int kb = 0; kb < nkb; ++kb) {
                    const float *bh = B.data() + ((size_t)i * nkb + kb) * 2 * UM_KB * NP, *bl = bh + UM_KB * NP;
                    const float *ah = A.data() + ((size_t)(t / UM_MT) * nkb + kb) * 2 * UM_KB * UM_MT, *al = ah + UM_KB * UM_MT;
                    for (int k = 0; k < UM_KB; ++k) {
                        const double a_h = at(ah, t % UM_MT, k, UM_MT), a_l = at(al, t % UM_MT, k, UM_MT);
                        const double b_h = at(bh, px, k, NP), b_l = at(bl, px, k, NP);
                        c3 += a_h * b_h + a_h * b_l + a_l * b_h;
                        c1 += a_h * b_h;
                        const int m = kb * UM_KB + k;
                        if (m < M && t < T && px < NN) exact += (double)coef[(size_t)t * M + m] * (double)modes[((size_t)i * M + m) * NN + px];
                        else if (a_h * b_h != 0.0 || a_l * b_h != 0.0 || a_h * b_l != 0.0) { std::printf("FAIL: padding is not zero\n"); return 1; }
                    }
                }
                worst3 = std::max(worst3, std::fabs(c3 - exact));
                worst1 = std::max(worst1, std::fabs(c1 - exact));
                cmax = std::max(cmax, std::fabs(exact));
            }
    std::printf("ok %.3e %.3e\n", worst3 / cmax, worst1 / cmax);
    return 0;
}
