/*
 * fft_regs.cuh -- register-resident power-of-two complex FFTs with compile-time twiddles.
 *
 * Every index is a compile-time constant after unrolling, so the arrays live in registers, the
 * bit-reversal is free (renaming) and multiplications by 1 and +-i are special-cased.
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

/* ---------------------------------------------------------------------------------------------------------
 * Radix-2 decimation in time with fused multiply-adds.  A butterfly (a + w b, a - w b) with w = c + i s costs
 * six FFMA when the twiddle is taken in tangent form, w b = c ((br - t bi) + i (bi + t br)), t = s / c
 * (cotangent form when |c| < |s|), against four operations for the product and four for the sums: 388
 * floating-point instructions at L = 32 (the decimation-in-frequency form this replaced compiled to ~440).
 * The array is addressed through the bit reversal (element i of the decimated order lives in register
 * bitrev(i)): natural-order input, output k at position fft_out_index<L>(k).  Inputs with index >= NZ are
 * known zeros and are never read: a block whose inputs are all zero is skipped, a butterfly whose second
 * operand is zero is a copy -- with NZ <= L/2 the whole first stage costs nothing.
 * ------------------------------------------------------------------------------------------------------- */
template <int L, int SIGN, int NZ, int S, int I>
struct DitBf {
    __device__ __forceinline__ static void run(float (&re)[L], float (&im)[L])
    {
        constexpr int bits = ilog2(L);
        constexpr int h = 1 << (S - 1);
        constexpr int j = I % h;
        constexpr int i0 = (I / h) * 2 * h + j, i1 = i0 + h;
        constexpr int p0 = bitrev(i0, bits), p1 = bitrev(i1, bits);
        /* the block of h elements around i holds a partial transform of the inputs bitrev(block): all zero
         * iff the smallest of them is >= NZ */
        constexpr bool az = bitrev((i0 / h) * h, bits) >= NZ;
        constexpr bool bz = bitrev((i1 / h) * h, bits) >= NZ;
        constexpr int k64 = ((SIGN > 0 ? j : -j) * (64 / (2 * h))) & 63;
        if constexpr (az) {
            static_assert(!az || bz, "prefix of non-zero inputs");
        } else if constexpr (bz) {
            re[p1] = re[p0]; im[p1] = im[p0];
        } else {
            const float ar = re[p0], ai = im[p0], br = re[p1], bi = im[p1];
            if constexpr (k64 == 0) {
                re[p0] = ar + br; im[p0] = ai + bi; re[p1] = ar - br; im[p1] = ai - bi;
            } else if constexpr (k64 == 16) {           /* w = +i: w b = (-bi, br) */
                re[p0] = ar - bi; im[p0] = ai + br; re[p1] = ar + bi; im[p1] = ai - br;
            } else if constexpr (k64 == 48) {           /* w = -i: w b = (bi, -br) */
                re[p0] = ar + bi; im[p0] = ai - br; re[p1] = ar - bi; im[p1] = ai + br;
            } else {
                constexpr float c = cos64(k64), s = sin64(k64);
                constexpr bool tanform = (c < 0 ? -c : c) >= (s < 0 ? -s : s);
                if constexpr (tanform) {
                    constexpr float t = (float)((double)s / (double)c);
                    const float p = fmaf(-t, bi, br), q = fmaf(t, br, bi);
                    re[p0] = fmaf(c, p, ar); im[p0] = fmaf(c, q, ai);
                    re[p1] = fmaf(-c, p, ar); im[p1] = fmaf(-c, q, ai);
                } else {
                    constexpr float ct = (float)((double)c / (double)s);
                    const float p = fmaf(ct, br, -bi), q = fmaf(ct, bi, br);
                    re[p0] = fmaf(s, p, ar); im[p0] = fmaf(s, q, ai);
                    re[p1] = fmaf(-s, p, ar); im[p1] = fmaf(-s, q, ai);
                }
            }
        }
        if constexpr (I + 1 < L / 2) DitBf<L, SIGN, NZ, S, I + 1>::run(re, im);
        else if constexpr ((1 << S) < L) DitBf<L, SIGN, NZ, S + 1, 0>::run(re, im);
    }
};

/* In-place L-point FFT: X[k] = sum_m x[m] exp(SIGN 2 pi i m k / L) is left at position fft_out_index<L>(k). */
template <int L, int SIGN, int NZ = L>
__device__ __forceinline__ void fft_fma(float (&re)[L], float (&im)[L])
{
    static_assert(L >= 2 && L <= 64 && (L & (L - 1)) == 0, "L must be a power of two <= 64");
    static_assert(NZ >= 1 && NZ <= L, "at least one non-zero input");
    DitBf<L, SIGN, NZ, 1, 0>::run(re, im);
}

template <int L>
__host__ __device__ constexpr int fft_out_index(int k) { return bitrev(k, ilog2(L)); }

/* ---------------------------------------------------------------------------------------------------------
 * The same transform on packed complex registers (float2 = (re, im) in an even register pair), sm_100a.
 * Blackwell's FP32x2 instructions (FFMA2 / FADD2 / FMUL2) take a 64-bit register pair per operand, a scalar
 * immediate broadcast to both halves, and a per-operand half swizzle with per-half negation (SASS
 * `-R8.F32x2.LO_HI.NP`), so multiplication by +-i costs nothing and a complex rotation is ONE instruction:
 *     w b = c (b + t (-b_i, b_r)),  t = s / c      ->  pq = FFMA2((-b_i, b_r), t, b)
 *     a +- w b                                      ->  FFMA2(pq, +-c, a)
 * A general butterfly is 3 instructions instead of 6, a trivial one (w = 1, +-i) 2 FADD2 instead of 4 FADD:
 * 194 instructions at L = 32 (162 pruned to 16 inputs) against 388 (324).  The FMA pipe does the same work
 * (an FP32x2 instruction occupies it for two cycles); what is halved is the issue slots, which is what
 * bounded the line transforms (profiles/r02_pf32.md: issue 76 %, FMA pipe 59 %).  Arithmetic and
 * rounding are those of fft_fma, element for element.
 * ------------------------------------------------------------------------------------------------------- */
__device__ __forceinline__ float2 rot_pi2(float2 b) { return make_float2(-b.y, b.x); }     /* +i b */
__device__ __forceinline__ float2 rot_mi2(float2 b) { return make_float2(b.y, -b.x); }     /* -i b */
__device__ __forceinline__ float2 neg2(float2 b) { return make_float2(-b.x, -b.y); }
__device__ __forceinline__ float2 bc2(float c) { return make_float2(c, c); }

template <int L, int SIGN, int NZ, int S, int I>
struct DitBf2 {
    __device__ __forceinline__ static void run(float2 (&z)[L])
    {
        constexpr int bits = ilog2(L);
        constexpr int h = 1 << (S - 1);
        constexpr int j = I % h;
        constexpr int i0 = (I / h) * 2 * h + j, i1 = i0 + h;
        constexpr int p0 = bitrev(i0, bits), p1 = bitrev(i1, bits);
        constexpr bool az = bitrev((i0 / h) * h, bits) >= NZ;
        constexpr bool bz = bitrev((i1 / h) * h, bits) >= NZ;
        constexpr int k64 = ((SIGN > 0 ? j : -j) * (64 / (2 * h))) & 63;
        if constexpr (az) {
            static_assert(!az || bz, "prefix of non-zero inputs");
        } else if constexpr (bz) {
            z[p1] = z[p0];
        } else {
            const float2 a = z[p0], b = z[p1];
            if constexpr (k64 == 0) {
                z[p0] = __fadd2_rn(a, b); z[p1] = __fadd2_rn(a, neg2(b));
            } else if constexpr (k64 == 16) {           /* w = +i */
                z[p0] = __fadd2_rn(a, rot_pi2(b)); z[p1] = __fadd2_rn(a, rot_mi2(b));
            } else if constexpr (k64 == 48) {           /* w = -i */
                z[p0] = __fadd2_rn(a, rot_mi2(b)); z[p1] = __fadd2_rn(a, rot_pi2(b));
            } else {
                constexpr float c = cos64(k64), s = sin64(k64);
                constexpr bool tanform = (c < 0 ? -c : c) >= (s < 0 ? -s : s);
                if constexpr (tanform) {
                    constexpr float t = (float)((double)s / (double)c);
                    const float2 pq = __ffma2_rn(rot_pi2(b), bc2(t), b);          /* (br - t bi, bi + t br) */
                    z[p0] = __ffma2_rn(pq, bc2(c), a); z[p1] = __ffma2_rn(pq, bc2(-c), a);
                } else {
                    constexpr float ct = (float)((double)c / (double)s);
                    const float2 pq = __ffma2_rn(b, bc2(ct), rot_pi2(b));         /* (ct br - bi, ct bi + br) */
                    z[p0] = __ffma2_rn(pq, bc2(s), a); z[p1] = __ffma2_rn(pq, bc2(-s), a);
                }
            }
        }
        if constexpr (I + 1 < L / 2) DitBf2<L, SIGN, NZ, S, I + 1>::run(z);
        else if constexpr ((1 << S) < L) DitBf2<L, SIGN, NZ, S + 1, 0>::run(z);
    }
};

/* In-place L-point FFT on packed complex registers; output k at position fft_out_index<L>(k). */
template <int L, int SIGN, int NZ = L>
__device__ __forceinline__ void fft_fma2(float2 (&z)[L])
{
    static_assert(L >= 2 && L <= 64 && (L & (L - 1)) == 0, "L must be a power of two <= 64");
    static_assert(NZ >= 1 && NZ <= L, "at least one non-zero input");
    DitBf2<L, SIGN, NZ, 1, 0>::run(z);
}

/* The same transform of x = xr + i xi given as two scalar arrays: the first stage (w = 1 everywhere) is done with
 * scalar additions that write the (re, im) pairs, the rest is packed.  For inputs that are produced one scalar at
 * a time (wk_fft.cu step C: two real columns into one complex transform): asking for them as register pairs
 * pins 2L registers for as long as the first half is live, this form lets them sit anywhere.                */
template <int L, int SIGN>
__device__ __forceinline__ void fft_fma2_split(const float (&xr)[L], const float (&xi)[L], float2 (&z)[L])
{
    static_assert(L >= 4 && L <= 64 && (L & (L - 1)) == 0, "L must be a power of two in 4..64");
    constexpr int bits = ilog2(L);
#pragma unroll
    for (int I = 0; I < L / 2; ++I) {
        const int p0 = bitrev(2 * I, bits), p1 = bitrev(2 * I + 1, bits);
        z[p0] = make_float2(xr[p0] + xr[p1], xi[p0] + xi[p1]);
        z[p1] = make_float2(xr[p0] - xr[p1], xi[p0] - xi[p1]);
    }
    DitBf2<L, SIGN, L, 2, 0>::run(z);
}

}  // namespace shwfs
#endif
