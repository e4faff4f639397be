/*
 * fft_regs.cuh -- register-resident power-of-two complex FFTs with compile-time twiddles.
 *
 * Every index is a compile-time constant after unrolling, so the arrays live in registers, the
 * bit-reversal is free (renaming) and multiplications by 1, +-i and (1+-i)/sqrt(2) are special-cased.
 * Used by the lag-domain D-point transforms (H6 of include/shwfs.h in Fourier form) and by the
 * literal P x P chain (H3, H5).  X[k] = sum_m x[m] exp(SIGN * 2*pi*i * m*k / L).
 */
#ifndef SHWFS_FFT_REGS_CUH_
#define SHWFS_FFT_REGS_CUH_

namespace shwfs {

/* cos(2*pi*k/64), k = 0..16 (quarter wave); everything else by symmetry. */
__host__ __device__ constexpr float qcos64(int k)
{
    constexpr float t[17] = {1.000000000e+00f, 9.951847267e-01f, 9.807852804e-01f, 9.569403357e-01f,
                             9.238795325e-01f, 8.819212643e-01f, 8.314696123e-01f, 7.730104534e-01f,
                             7.071067812e-01f, 6.343932842e-01f, 5.555702330e-01f, 4.713967368e-01f,
                             3.826834324e-01f, 2.902846773e-01f, 1.950903220e-01f, 9.801714033e-02f,
                             0.0f};
    return t[k];
}
/* cos / sin of 2*pi*k/64 for k in [0,64) */
__host__ __device__ constexpr float cos64(int k)
{
    k &= 63;
    return k <= 16 ? qcos64(k) : k <= 32 ? -qcos64(32 - k) : k <= 48 ? -qcos64(k - 32) : qcos64(64 - k);
}
__host__ __device__ constexpr float sin64(int k) { return cos64(k - 16); }

__host__ __device__ constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }
__host__ __device__ constexpr int bitrev(int v, int bits)
{
    int r = 0;
    for (int q = 0; q < bits; ++q) r |= ((v >> q) & 1) << (bits - 1 - q);
    return r;
}

/* (re,im) *= exp(2*pi*i*K64/64), K64 compile-time */
template <int K64>
__device__ __forceinline__ void twiddle(float &re, float &im)
{
    constexpr int k = K64 & 63;
    if constexpr (k == 0) {
    } else if constexpr (k == 16) { float t = re; re = -im; im = t; }
    else if constexpr (k == 32) { re = -re; im = -im; }
    else if constexpr (k == 48) { float t = re; re = im; im = -t; }
    else if constexpr (k == 8)  { float a = re, b = im; re = (a - b) * 0.70710678118654752f; im = (a + b) * 0.70710678118654752f; }
    else if constexpr (k == 24) { float a = re, b = im; re = (a + b) * -0.70710678118654752f; im = (a - b) * 0.70710678118654752f; }
    else if constexpr (k == 40) { float a = re, b = im; re = (b - a) * 0.70710678118654752f; im = (a + b) * -0.70710678118654752f; }
    else if constexpr (k == 56) { float a = re, b = im; re = (a + b) * 0.70710678118654752f; im = (b - a) * 0.70710678118654752f; }
    else {
        constexpr float c = cos64(k), s = sin64(k);
        float a = re, b = im;
        re = fmaf(a, c, -b * s);
        im = fmaf(a, s, b * c);
    }
}

/* One decimation-in-frequency stage over blocks of LEN inside an L-point array.
 * NZ: inputs with index >= NZ are known to be zero (only honoured when LEN == L). */
template <int L, int LEN, int SIGN, int NZ>
__device__ __forceinline__ void dif_stage(float (&re)[L], float (&im)[L])
{
    constexpr int half = LEN / 2;
#pragma unroll
    for (int base = 0; base < L; base += LEN) {
#pragma unroll
        for (int q = 0; q < half; ++q) {
            const int i0 = base + q, i1 = base + q + half;
            float dr, di;
            if (LEN == L && i1 >= NZ) {          /* second operand is zero: u+0, (u-0)*w */
                if (LEN == L && i0 >= NZ) { re[i0] = 0.f; im[i0] = 0.f; re[i1] = 0.f; im[i1] = 0.f; continue; }
                dr = re[i0]; di = im[i0];
            } else {
                float ur = re[i0], ui = im[i0], vr = re[i1], vi = im[i1];
                re[i0] = ur + vr; im[i0] = ui + vi;
                dr = ur - vr; di = ui - vi;
            }
            re[i1] = dr; im[i1] = di;
        }
    }
}

/* helper to apply the stage twiddles with compile-time indices */
template <int L, int LEN, int SIGN, int BASE, int Q>
struct TwApply {
    __device__ __forceinline__ static void run(float (&re)[L], float (&im)[L])
    {
        constexpr int half = LEN / 2;
        constexpr int k64 = ((SIGN > 0 ? Q : -Q) * (64 / LEN)) & 63;
        twiddle<k64>(re[BASE + Q + half], im[BASE + Q + half]);
        if constexpr (Q + 1 < half) TwApply<L, LEN, SIGN, BASE, Q + 1>::run(re, im);
        else if constexpr (BASE + LEN < L) TwApply<L, LEN, SIGN, BASE + LEN, 0>::run(re, im);
    }
};

template <int L, int LEN, int SIGN, int NZ>
struct DifRec {
    __device__ __forceinline__ static void run(float (&re)[L], float (&im)[L])
    {
        dif_stage<L, LEN, SIGN, NZ>(re, im);
        if constexpr (LEN > 2) {
            TwApply<L, LEN, SIGN, 0, 0>::run(re, im);
            DifRec<L, LEN / 2, SIGN, L>::run(re, im);
        }
    }
};

/* In-place L-point DIF FFT.  Output element k is left at position bitrev(k): use fft_out_index<L>(k). */
template <int L, int SIGN, int NZ = L>
__device__ __forceinline__ void fft_dif(float (&re)[L], float (&im)[L])
{
    static_assert(L >= 2 && L <= 64 && (L & (L - 1)) == 0, "L must be a power of two <= 64");
    DifRec<L, L, SIGN, NZ>::run(re, im);
}

template <int L>
__host__ __device__ constexpr int fft_out_index(int k) { return bitrev(k, ilog2(L)); }

}  // namespace shwfs
#endif
