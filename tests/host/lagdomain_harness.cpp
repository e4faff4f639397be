/*
 * lagdomain_harness.cpp -- host-side parity of the device code that follows the autocorrelation in the lag-domain
 * path against the float64 oracle's own chain O2..O9 (oracle/shwfs_oracle.c, linked in as a C object):
 *     csrc/field.cuh      H2   field_value (range reduction to +-1/2 turn, fast sincos)
 *     csrc/wk_common.cuh  H5 + x half of H6   finish_row (scalar) and finish_row2 (packed, staged table row in the
 *                         visiting order of term_lag / term_m / term_first);  y half of H6   ytransform16
 *     csrc/cog.cuh        H7 + H8   cog16, its half-warp xor shuffles simulated (see shuffle16 below)
 * compiled AS THEY ARE for the host, and
 *     csrc/wk.cu          H0   wk_table_kernel, the float64 table M, cut out of the .cu file as text
 *                         ("wk_table_extract.inc", written by tests/test_lagdomain_host.py) and run with ONE simulated
 *                         thread per block (its loops stride by blockDim.x; the dynamic shared array is a plain buffer).
 * What the harness supplies itself: the autocorrelation G of the device-made fp32 field, by the plain double sums of
 * its definition (the kernels' own sums: tests/test_wk_acc_host.py), and -- as a cross-check of the table kernel only
 * -- M from the formula of DESIGN.md 6.1
 *     M[ly,lx] = Z[ly,lx] beta(ly) beta(lx) / P^2 (x 2 for ly >= 1),  beta(l) = sum_{alpha<b} w^(alpha l),
 *     Z = DFT of the spatial kernel at (-ly,-lx), or (-1)^(ly+lx) without kernels,   w = exp(2 pi i / P).
 * So a green run says:
 * the identity B[R,C] = Re sum G M w_D^(R ly + C lx) with its centring, binning and aliasing mod 16, AS THE DEVICE
 * CODE EVALUATES IT, reproduces the oracle's binned image to 1e-4 of the peak and its slopes to 1e-3 px (north_star).
 * Built and run by tests/test_lagdomain_host.py (gcc + g++, no GPU).  Test infrastructure only.
 */
#include <cuda_runtime.h>

#include <cmath>
#include <complex>
#include <cstdio>
#include <random>
#include <vector>

/* ---- shims ---- */
extern "C" void __sincosf(float x, float *s, float *c) noexcept { *s = sinf(x); *c = cosf(x); }
static inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
static inline float2 __fadd2_rn(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
static inline float2 __fmul2_rn(float2 a, float2 b) { return make_float2(a.x * b.x, a.y * b.y); }
static inline float2 __ldg(const float2 *p) { return *p; }
static inline size_t __cvta_generic_to_shared(const void *p) { return (size_t)p; }
/* cog16's shuffles: the 16 lanes are run one after the other, several passes over; shuffle number k of lane L records
 * its operand and returns what lane L ^ o recorded at its shuffle k in the previous pass.  The operand of shuffle k
 * depends on shuffles < k only, so after k + 1 passes it is right: 17 passes settle the 16 shuffles of cog16. */
static int g_lane, g_shfl_idx;
static float g_rec[2][16][32];
static int g_pass;
static inline float __shfl_xor_sync(unsigned, float v, int o)
{
    const int k = g_shfl_idx++;
    g_rec[g_pass & 1][g_lane][k] = v;
    return g_rec[(g_pass & 1) ^ 1][g_lane ^ o][k];
}

#include "../../paper_1408_0698_b200/csrc/wk_common.cuh"
#include "../../paper_1408_0698_b200/csrc/field.cuh"
#include "../../paper_1408_0698_b200/csrc/cog.cuh"

/* wk_table_kernel on the host: one thread per block */
struct Dim { unsigned x, y, z; };
static Dim threadIdx = {0, 0, 0}, blockIdx = {0, 0, 0}, blockDim = {1, 1, 1};
static inline void __syncthreads() {}
static inline void sincospi(double x, double *s, double *c) { *s = std::sin(M_PI * x); *c = std::cos(M_PI * x); }
static double2 tmp[64 * 63];                   /* the kernel's `extern __shared__ double2 tmp[]`: [P][2n-1] */
#include "wk_table_extract.inc"

extern "C" {
void shwfs_oracle_field(const float *phase_frame, const float *amplitude, int N, int n, int P, int sy, int sx,
                        double c_phi, double *e);
int shwfs_oracle_dft2(const double *in, double *out, int P, int sign);
void shwfs_oracle_intensity(const double *E, int P, double *I);
int shwfs_oracle_convolve_fft(const double *I, const float *K, int P, double *C);
void shwfs_oracle_centre(const double *C, int P, double *Sh);
void shwfs_oracle_bin(const double *Sh, int P, int b, double *B);
void shwfs_oracle_threshold_cog(const double *B, int D, double tau, int mode, double *slope_xy);
}

using namespace shwfs;
typedef std::complex<double> cd;

static std::mt19937 rng(140806u);
static double worst_img = 0, worst_slope = 0, worst_table = 0;

template <int MODE>
static float2 shuffle16(const float (&B)[16][16], float tau)
{
    float2 out[16];
    for (g_pass = 0; g_pass < 18; ++g_pass)
        for (g_lane = 0; g_lane < 16; ++g_lane) {
            float bcol[16];
            for (int R = 0; R < 16; ++R) bcol[R] = B[R][g_lane];
            g_shfl_idx = 0;
            out[g_lane] = cog16<MODE>(bcol, g_lane, tau);
        }
    return out[0];
}

/* one spot of an n x n patch padded to P, binned b x b to 16 x 16; with_kernel: a random positive asymmetric kernel */
template <int n>
static bool one_spot(int P, int b, bool with_kernel, float tau, int mode, float phase_scale)
{
    constexpr int LX = 2 * n - 1;
    const int N = n, D = P / b;
    std::uniform_real_distribution<float> U(0.f, 1.f);
    std::vector<float> phase(n * n), amp(n * n), K((size_t)P * P, 0.f);
    for (int q = 0; q < n * n; ++q) { phase[q] = phase_scale * (U(rng) - 0.5f); amp[q] = U(rng) < 0.15f ? 0.f : 0.5f + 0.5f * U(rng); }
    if (with_kernel) {
        double s = 0;
        for (int y = 0; y < P; ++y)
            for (int x = 0; x < P; ++x) {
                const double dy = y - P / 2 - 0.7, dx = x - P / 2 + 1.3;
                const double v = std::exp(-(dy * dy / 18.0 + dx * dx / 5.0 + 0.2 * dx * dy)) * (0.8 + 0.4 * U(rng));
                K[(size_t)y * P + x] = (float)v; s += v;
            }
        for (auto &v : K) v = (float)(v / s);
    }
    /* ---- oracle: O2 .. O9 ---- */
    std::vector<double> e((size_t)2 * P * P), I((size_t)P * P), C((size_t)P * P), Sh((size_t)P * P), Bo((size_t)D * D);
    shwfs_oracle_field(phase.data(), amp.data(), N, n, P, 0, 0, 1.0, e.data());
    if (shwfs_oracle_dft2(e.data(), e.data(), P, -1)) return false;
    shwfs_oracle_intensity(e.data(), P, I.data());
    if (with_kernel) { if (shwfs_oracle_convolve_fft(I.data(), K.data(), P, C.data())) return false; } else C = I;
    shwfs_oracle_centre(C.data(), P, Sh.data());
    shwfs_oracle_bin(Sh.data(), P, b, Bo.data());
    double so[2];
    shwfs_oracle_threshold_cog(Bo.data(), D, tau, mode, so);

    /* ---- device code on the host ---- */
    const float turns = (float)(1.0 / (2.0 * M_PI)), ramp_unit = 0.5f / (float)P;
    std::vector<cd> ef(n * n);
    for (int j = 0; j < n; ++j)
        for (int k = 0; k < n; ++k) {
            const float2 f = field_value(phase[j * n + k], amp[j * n + k], turns, (float)(j + k) * ramp_unit);     /* H2 */
            ef[j * n + k] = cd(f.x, f.y);
        }
    /* table M, layout [a][ly] as on the device */
    const cd w = std::polar(1.0, 2.0 * M_PI / P);
    std::vector<float2> M((size_t)LX * n);
    for (int ly = 0; ly < n; ++ly)
        for (int a = 0; a < LX; ++a) {
            const int lx = a - (n - 1);
            cd Z = ((ly + lx) & 1) ? -1.0 : 1.0;
            if (with_kernel) {
                Z = 0;
                for (int qy = 0; qy < P; ++qy)
                    for (int qx = 0; qx < P; ++qx)
                        Z += (double)K[(size_t)qy * P + qx] * std::pow(w, -(double)((qy * ly + qx * lx) % P));
            }
            cd by = 0, bx = 0;
            for (int al = 0; al < b; ++al) { by += std::pow(w, (double)(al * ly)); bx += std::pow(w, (double)(al * lx)); }
            const cd m = Z * by * bx / (double)(P * P) * (ly >= 1 ? 2.0 : 1.0);
            M[(size_t)a * n + ly] = make_float2((float)m.real(), (float)m.imag());
        }
    /* H0 as the device builds it; must agree with the formula, and is what the product below uses */
    {
        std::vector<float2> Md((size_t)LX * n);
        blockIdx.x = 0;
        wk_table_kernel(with_kernel ? K.data() : nullptr, with_kernel ? 1 : 0, n, P, b, Md.data());
        double mscale = 0;
        for (const float2 &v : M) mscale = std::fmax(mscale, std::hypot((double)v.x, (double)v.y));
        for (size_t q = 0; q < M.size(); ++q) {
            const double e = std::hypot((double)Md[q].x - M[q].x, (double)Md[q].y - M[q].y) / mscale;
            worst_table = std::fmax(worst_table, e);
            if (!(e <= 1e-6)) { std::printf("FAIL: n=%d P=%d b=%d kernel=%d: table entry %zu off by %.3g of the largest\n", n, P, b, (int)with_kernel, q, e); return false; }
        }
        M = Md;
    }
    float Bs[16][16], Bp[16][16];
    float Hs[n][32], Hp[n][32];
    for (int ly = 0; ly < n; ++ly) {
        float2 acc[LX];
        for (int a = 0; a < LX; ++a) {                                                   /* G[ly][lx]: its definition */
            const int lx = a - (n - 1);
            cd g = 0;
            for (int j = 0; j + ly < n; ++j)
                for (int k = 0; k < n; ++k)
                    if (k + lx >= 0 && k + lx < n) g += ef[j * n + k] * std::conj(ef[(j + ly) * n + k + lx]);
            acc[a] = make_float2((float)g.real(), (float)g.imag());
        }
        finish_row<n>(acc, M.data() + ly, Hs[ly]);                                       /* scalar: table read in place */
        alignas(16) float staged[2 * (LX + 1)] = {0};
        for (int k = 0; k < LX; ++k) {                                                   /* what mrow_stage copies */
            const float2 mv = M[(size_t)term_lag<n>(k) * n + ly];
            staged[2 * k] = mv.x; staged[2 * k + 1] = mv.y;
        }
        alignas(16) float hp[32];
        finish_row2<n>(acc, staged, hp);                                                 /* packed: staged row */
        for (int q = 0; q < 32; ++q) Hp[ly][q] = hp[q];
    }
    for (int C16 = 0; C16 < 16; ++C16) {
        float bs[16], bp[16];
        ytransform16<n>([&](int m) { return make_float2(Hs[m][2 * C16], Hs[m][2 * C16 + 1]); }, bs);
        ytransform16<n>([&](int m) { return make_float2(Hp[m][2 * C16], Hp[m][2 * C16 + 1]); }, bp);
        for (int R = 0; R < 16; ++R) { Bs[R][C16] = bs[R]; Bp[R][C16] = bp[R]; }
    }
    double peak = 0;
    for (double v : Bo) peak = std::fmax(peak, v);
    for (int R = 0; R < 16; ++R)
        for (int C16 = 0; C16 < 16; ++C16) {
            const double es = std::fabs(Bs[R][C16] - Bo[R * D + C16]) / peak, ep = std::fabs(Bp[R][C16] - Bo[R * D + C16]) / peak;
            worst_img = std::fmax(worst_img, std::fmax(es, ep));
            if (!(es <= 1e-4) || !(ep <= 1e-4)) {
                std::printf("FAIL: n=%d P=%d b=%d kernel=%d: binned image (R=%d,C=%d) off by %.3g / %.3g of the peak\n", n, P, b, (int)with_kernel, R, C16, es, ep);
                return false;
            }
        }
    const float2 sl = mode == 0 ? shuffle16<0>(Bp, tau) : shuffle16<1>(Bp, tau);
    const double es = std::fmax(std::fabs(sl.x - so[0]), std::fabs(sl.y - so[1]));
    worst_slope = std::fmax(worst_slope, es);
    /* mode 1 (hard mask) is compared only where no pixel sits within rounding of the threshold */
    bool near = false;
    if (mode == 1) for (double v : Bo) if (std::fabs(v - tau * peak) < 1e-5 * peak) near = true;
    if (!near && !(es <= 1e-3)) { std::printf("FAIL: n=%d P=%d b=%d mode=%d: slopes off by %.3g px\n", n, P, b, mode, es); return false; }
    return true;
}

int main()
{
    /* the visiting order of the table product covers every lag once and puts it on lx mod 16 */
    {
        constexpr int n = 10, LX = 2 * n - 1;
        int seen[LX] = {0};
        for (int k = 0; k < LX; ++k) {
            const int a = term_lag<n>(k), m = term_m<n>(k);
            if (a < 0 || a >= LX || m != (((a - (n - 1)) % 16) + 16) % 16) { std::printf("FAIL: term order at %d\n", k); return 1; }
            if (term_first<n>(k) != (k == 0 || term_m<n>(k - 1) != m)) { std::printf("FAIL: term_first at %d\n", k); return 1; }
            seen[a] += 1;
        }
        for (int a = 0; a < LX; ++a) if (seen[a] != 1) { std::printf("FAIL: lag %d visited %d times\n", a, seen[a]); return 1; }
    }
    int spots = 0;
    for (int rep = 0; rep < 6; ++rep) {
        const float ps = rep < 3 ? 6.0f : 120.0f;                 /* a few radians, and the +-60 rad of the MAORY screens */
        const float tau = rep % 2 ? 0.1f : 0.0f;
        const int mode = rep == 5 ? 1 : 0;
        if (!one_spot<8>(16, 1, false, tau, mode, ps)) return 1;      /* config 1 */
        if (!one_spot<10>(32, 2, true, tau, mode, ps)) return 1;      /* configs 3, 4 */
        if (!one_spot<10>(32, 2, false, tau, mode, ps)) return 1;
        if (!one_spot<16>(32, 2, false, tau, mode, ps)) return 1;     /* config 2 sizes */
        if (!one_spot<16>(64, 4, true, tau, mode, ps)) return 1;      /* config 5 */
        if (!one_spot<12>(32, 2, true, tau, mode, ps)) return 1;
        spots += 6;
    }
    std::printf("ok %d spots, device table within %.3g of the formula, worst image error %.3g of the peak, worst slope error %.3g px\n",
                spots, worst_table, worst_img, worst_slope);
    return 0;
}
