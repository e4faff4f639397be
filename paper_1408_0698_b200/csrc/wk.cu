/*
 * wk.cu -- Wiener-Khinchin (lag-domain) form of the Shack-Hartmann hot path, sm_100a.
 *
 * What it computes is H1..H8 of include/shwfs.h ("The WF is split into sub-apertures and
 * the spot computed by FFT for each sensor sub-aperture ... a convolution for a gaussian ... the
 * centroid computed on the final image to retrieve the slopes").  How: the binned, centred, convolved
 * image B is linear in the intensity I = |DFT(e)|^2 / P^2, and the DFT of I is the (aperiodic)
 * autocorrelation of the n x n field e (invariant I13 of SURVEY.md 8(c)).  Writing w = exp(2*pi*i/P),
 * w_D = exp(2*pi*i/D), D = P/b:
 *
 *     G[ly,lx]  = sum_{j,k} e[j,k] * conj(e[j+ly, k+lx])              |ly|,|lx| < n          (H3+H4)
 *     B[R,C]    = sum_{ly,lx} G[ly,lx] * M_i[ly,lx] * w_D^(R*ly + C*lx)                      (H5+H6)
 *     M_i[l]    = Z_i[l] * beta(ly) * beta(lx) / P^2,   beta(l) = sum_{alpha<b} w^(alpha*l),
 *     Z_i[l]    = sum_q K_i[q] w^(-q.l)  with kernels,  (-1)^(ly+lx) without
 *
 * G[-l] = conj(G[l]) and M[-l] = conj(M[l]) (K real), so only ly >= 0 is computed and the factor 2
 * for ly >= 1 is folded into M.  The result equals the literal P x P FFT chain up to fp32 rounding
 * for ANY P >= n (the identity is one of trigonometric polynomials), costs n^2(n+1)/2 * n complex
 * MACs instead of three P x P transforms, and needs a D x D rather than P x P final transform.
 * DESIGN.md section 6 has the derivation, the thread mapping and the flop counts.
 */
#include <stdio.h>

#include "internal.h"
#include "fft_regs.cuh"
#include "field.cuh"
#include "cog.cuh"
#include "noise.cuh"
#include "wk_common.cuh"

namespace {

using namespace shwfs;

/* ------------------------------------------------------------------------------------------------
 * Table M (float64 on the device, stored as float2).  One CTA per subaperture (or one CTA in all
 * when there are no kernels).  Layout M[i][a][ly], a = lx + n - 1: lag row ly is a column, so that the threads of
 * wk_fft.cu (thread = lag row) read 16 consecutive entries per load instead of 16 rows 8(2n-1) bytes apart.
 * ---------------------------------------------------------------------------------------------- */
__global__ void wk_table_kernel(const float *__restrict__ K, int has_k, int n, int P, int b,
                                float2 *__restrict__ M)
{
    extern __shared__ double2 tmp[];           /* [P][2n-1]: row-wise partial transform of K */
    const int LX = 2 * n - 1;
    const int i = blockIdx.x;
    if (has_k) {
        const float *Ki = K + (size_t)i * P * P;
        for (int idx = threadIdx.x; idx < P * LX; idx += blockDim.x) {
            const int qy = idx / LX, lx = idx % LX - (n - 1);
            double sr = 0.0, si = 0.0;
            for (int qx = 0; qx < P; ++qx) {
                const int m = ((qx * lx) % P + P) % P;        /* w^(-qx*lx) */
                double s, c;
                sincospi(-2.0 * (double)m / (double)P, &s, &c);
                const double kv = (double)Ki[qy * P + qx];
                sr += kv * c;
                si += kv * s;
            }
            tmp[idx] = make_double2(sr, si);
        }
        __syncthreads();
    }
    const double inv_pp = 1.0 / ((double)P * (double)P);
    for (int idx = threadIdx.x; idx < n * LX; idx += blockDim.x) {
        const int ly = idx / LX, a = idx % LX, lx = a - (n - 1);
        double zr, zi;
        if (has_k) {
            zr = 0.0; zi = 0.0;
            for (int qy = 0; qy < P; ++qy) {
                const int m = (qy * ly) % P;                   /* w^(-qy*ly) */
                double s, c;
                sincospi(-2.0 * (double)m / (double)P, &s, &c);
                const double2 t = tmp[qy * LX + a];
                zr += t.x * c - t.y * s;
                zi += t.x * s + t.y * c;
            }
        } else {
            zr = ((ly + lx) & 1) ? -1.0 : 1.0;
            zi = 0.0;
        }
        double byr = 0.0, byi = 0.0, bxr = 0.0, bxi = 0.0;     /* beta(ly), beta(lx) */
        for (int al = 0; al < b; ++al) {
            double s, c;
            sincospi(2.0 * (double)((al * ly) % P) / (double)P, &s, &c);
            byr += c; byi += s;
            sincospi(2.0 * (double)(((al * lx) % P + P) % P) / (double)P, &s, &c);
            bxr += c; bxi += s;
        }
        const double br = byr * bxr - byi * bxi, bi = byr * bxi + byi * bxr;
        const double scale = inv_pp * (ly >= 1 ? 2.0 : 1.0);
        M[(size_t)i * n * LX + a * n + ly] = make_float2((float)((zr * br - zi * bi) * scale),
                                                         (float)((zr * bi + zi * br) * scale));
    }
}

/* ------------------------------------------------------------------------------------------------
 * Specialised kernel: n in {8,10,16}, D = 16.  One CTA = 32 consecutive spots g = i*T + t (frame
 * fastest, so the 32 lanes of a warp mostly share one subaperture's table M_i), n/2 warps.
 *
 *   phase 0  thread = (pixel pair, spot group): H1 gather as 8-byte loads (all of a thread's loads in
 *            flight at once), H2 sincos, field e -> shared memory.
 *   phase 1  lane = spot, warp c = lag-row class {c, n-c} (class 0 = {0, n/2}): the thread
 *            accumulates G[ly, -(n-1)..n-1] for its lag rows in registers, one row pair (j, j+ly)
 *            at a time (2n-1 independent complex accumulators, 4 n^2 FFMA per 2*2n/4 LDS.128), then
 *            multiplies by M_i[ly,:], aliases lx mod 16 and does the 16-point x-transform in
 *            registers: H[ly][C] -> shared memory.  Lag row 0 is Hermitian in lx (G[0,-lx] =
 *            conj G[0,lx]), so only lx >= 0 is accumulated there: every class costs 4 n^3 FFMA.
 *   phase 2  half-warp = spot, lane = detector column C: 16-point y-transform (real part) of
 *            H[0..n-1][C], then H7/H8 with half-warp shuffles; lane 0 writes the two slopes.
 * ---------------------------------------------------------------------------------------------- */
template <int n>
struct WkCfg {
    static constexpr int LX = 2 * n - 1;
    static constexpr int NW = n / 2;
    static constexpr int THREADS = 32 * NW;
    static constexpr int SPOTS = 32;
    static constexpr int NP = n * n / 2;                    /* pixel pairs (float4 of e) per spot        */
    static constexpr int SG = THREADS / NP;                 /* spot groups in phase 0: 4 / 3 / 2         */
    static constexpr int ITEMS = (SPOTS + SG - 1) / SG;     /* spots per phase-0 thread: 8 / 11 / 16     */
    static constexpr int ES = (((2 * n * n) / 4) | 1) * 4;  /* floats per spot; /4 odd => LDS.128 conflict-free */
    /* multi-layer instances: the raw lag rows G pile up over the sub-layers in shared memory, one row of RS floats
     * per lag row (2n-1 complex lags, and room for the 16 complex values of H that replace them after the last
     * sub-layer); GS/2 odd => the lane-strided 8-byte accesses are conflict-free                              */
    static constexpr int RS = 2 * LX > 32 ? 2 * LX : 32;
    static constexpr int GS = n * RS + (((n * RS / 2) & 1) ? 0 : 2);
    static constexpr int HA = (((NW * 32) / 4) | 1) * 4;    /* the NW rows of the first pass only (plain ones) */
    static_assert(n % 2 == 0 && n <= 16, "n must be even and <= 16");
    static_assert(NW * 32 <= ES, "the second-pass rows of H must fit in the field buffer they replace");
};

/* Shared memory of one CTA.  Plain instances (SPLIT): the rows of H produced by the second pass overwrite the
 * field buffer once every warp is done reading it, so only the first-pass rows need room of their own --
 * 47 KB instead of 68 KB at n = 10, a fourth CTA per SM.  EXT instances accumulate H across sub-layers while
 * the field buffer is rewritten, and keep the two apart.                                                  */
template <int n, bool SPLIT>
struct WkSmem {
    using Cfg = WkCfg<n>;
    static constexpr int HSTRIDE = SPLIT ? Cfg::HA : Cfg::GS;
    static constexpr size_t BYTES = sizeof(float) * (size_t)(Cfg::SPOTS * Cfg::ES + Cfg::SPOTS * HSTRIDE) + sizeof(int4) * Cfg::SPOTS;
    static constexpr int BY_SMEM = (int)((227 * 1024) / (BYTES + 1024));
    /* the plain n = 16 instance needs 196 registers x 256 threads: one CTA per SM whatever the memory says */
    static constexpr int MIN_CTAS = n == 16 ? 1 : (BY_SMEM < 1 ? 1 : BY_SMEM);
};

template <int n>
__device__ __forceinline__ void load_row(const float *__restrict__ p, float (&r)[2 * n])
{
#pragma unroll
    for (int q = 0; q < (2 * n) / 4; ++q) {
        const float4 v = reinterpret_cast<const float4 *>(p)[q];
        r[4 * q] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w;
    }
}

/* G[lx] += e1[k] * conj(e2[k2]),  lx = k2 - k, all n^2 products of one row pair.  With e1 = a + ib,
 * conj(e2) = c - id, s = a + b, t = c - d the product is (ac + bd) + i(st - ac + bd): three real products
 * instead of four.  X = sum ac and Y = sum bd share one packed FFMA2 (sm_100a fma.rn.f32x2 on the
 * (re,im) register pairs exactly as LDS.128 delivers them), Z = sum st is a scalar FFMA; G = (X + Y) +
 * i(Z - X + Y) is formed once per lag row (lag_value).  3 FMA-pipe cycles and 2 issue slots per complex
 * MAC instead of 4 and 4.                                                                                */
template <int n>
struct LagAcc {
    float2 xy[2 * n - 1];
    float z[2 * n - 1];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int a = 0; a < 2 * n - 1; ++a) { xy[a] = make_float2(0.f, 0.f); z[a] = 0.f; }
    }
    __device__ __forceinline__ float2 lag_value(int a) const
    {
        return make_float2(xy[a].x + xy[a].y, (z[a] - xy[a].x) + xy[a].y);
    }
};

template <int n>
__device__ __forceinline__ void load_row2(const float *__restrict__ p, float2 (&r)[n])
{
#pragma unroll
    for (int q = 0; q < n / 2; ++q) {
        const float4 v = reinterpret_cast<const float4 *>(p)[q];
        r[2 * q] = make_float2(v.x, v.y);
        r[2 * q + 1] = make_float2(v.z, v.w);
    }
}

template <int n>
__device__ __forceinline__ void rowpair_acc(const float *__restrict__ p1, const float *__restrict__ p2, LagAcc<n> &A)
{
    float2 e1[n], e2[n];
    float s[n], t[n];
    load_row2<n>(p1, e1);
    load_row2<n>(p2, e2);
#pragma unroll
    for (int k = 0; k < n; ++k) { s[k] = e1[k].x + e1[k].y; t[k] = e2[k].x - e2[k].y; }
#pragma unroll
    for (int k = 0; k < n; ++k) {
#pragma unroll
        for (int k2 = 0; k2 < n; ++k2) {
            const int a = k2 - k + n - 1;
            A.xy[a] = __ffma2_rn(e1[k], e2[k2], A.xy[a]);
            A.z[a] = fmaf(s[k], t[k2], A.z[a]);
        }
    }
}

/* lag row 0: the row against itself, lx >= 0 only (G[0,-lx] = conj G[0,lx]; G[0,0] is real) */
template <int n>
__device__ __forceinline__ void rowself_acc(const float *__restrict__ p, LagAcc<n> &A)
{
    float2 e[n];
    float s[n], t[n];
    load_row2<n>(p, e);
#pragma unroll
    for (int k = 0; k < n; ++k) { s[k] = e[k].x + e[k].y; t[k] = e[k].x - e[k].y; }
#pragma unroll
    for (int k = 0; k < n; ++k) {
#pragma unroll
        for (int k2 = 0; k2 < n; ++k2) {
            if (k2 < k) continue;
            const int a = k2 - k + n - 1;
            A.xy[a] = __ffma2_rn(e[k], e[k2], A.xy[a]);
            if (k2 > k) A.z[a] = fmaf(s[k], t[k2], A.z[a]);
        }
    }
}

/* EXTK: 0 = plain sensor; 1 = extensions on one (sub-)layer (noise, DM residual, a single sodium layer): same
 * shared-memory layout and occupancy as the plain instance; 2 = several sodium sub-layers: H accumulates over
 * the layers in a buffer of its own.                                                                     */
template <int n, int MODE, int EXTK>
__global__ void __launch_bounds__(WkCfg<n>::THREADS, WkSmem<n, (EXTK < 2)>::MIN_CTAS) wk_measure_kernel(const WkArgs A)
{
    constexpr bool EXT = EXTK > 0;
    using Cfg = WkCfg<n>;
    constexpr bool SPLIT = EXTK < 2;
    constexpr int HSTRIDE = WkSmem<n, SPLIT>::HSTRIDE;
    extern __shared__ __align__(16) float smem[];
    float *ebuf = smem;
    float *hbuf = smem + Cfg::SPOTS * Cfg::ES;
    int4 *s_info = reinterpret_cast<int4 *>(hbuf + Cfg::SPOTS * HSTRIDE);   /* {patch offset, t, i, -} */

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g0 = blockIdx.x * Cfg::SPOTS;

    if (tid < Cfg::SPOTS) {
        const int g = g0 + tid;
        int i = -1, t = 0, off = 0;
        if (g < A.total) {
            i = g / A.T;
            t = g - i * A.T;
            const int2 yx = A.valid[i];
            off = yx.x * n * A.N + yx.y * n;
        }
        s_info[tid] = make_int4(off, t, i, 0);
    }
    __syncthreads();

    const int n_layers = EXTK == 2 && A.L > 0 ? A.L : 1;      /* A.L == 0: single-layer sensor (noise only) */
    const bool sodium = EXT && A.L > 0;
#pragma unroll 1
    for (int layer = 0; layer < n_layers; ++layer) {
    if (EXT && layer > 0) __syncthreads();        /* every warp is done reading the previous layer's field */
    /* ---- phase 0: H1 gather + H2 field.  Thread = pixel pair q2 of the spots sg, sg+SG, ... ---- */
    {
        const int sg = tid / Cfg::NP, q2 = tid - sg * Cfg::NP;
        if (sg < Cfg::SG) {
            const int j = q2 / (n / 2), kk = q2 - j * (n / 2);
            const int poff = j * A.N + 2 * kk;
            const float ramp0 = (float)(j + 2 * kk) * A.ramp_unit, ramp1 = ramp0 + A.ramp_unit;
            /* EXT: pixel offsets from the patch centre and the sub-layer's curvature term (reading B1) */
            const float dj = (float)j - 0.5f * (float)(n - 1), dk0 = (float)(2 * kk) - 0.5f * (float)(n - 1);
            const float lq = sodium ? A.sod_q[layer] : 0.f, lsw = sodium ? A.sod_sw[layer] : 1.f;
            const float quad0 = lq * (dj * dj + dk0 * dk0), quad1 = lq * (dj * dj + (dk0 + 1.f) * (dk0 + 1.f));
            float2 ph[Cfg::ITEMS];
            int aoff[Cfg::ITEMS];
#pragma unroll
            for (int r = 0; r < Cfg::ITEMS; ++r) {
                const int s = sg + r * Cfg::SG;
                aoff[r] = -1;
                ph[r] = make_float2(0.f, 0.f);
                if (s < Cfg::SPOTS) {
                    const int4 inf = s_info[s];
                    if (inf.z >= 0) {
                        aoff[r] = inf.x + poff;
                        ph[r] = __ldg(reinterpret_cast<const float2 *>(A.phase + (size_t)inf.y * A.frame_stride
                                                                       + (EXT ? (size_t)layer * A.layer_stride : 0) + aoff[r]));
                    }
                }
            }
            if (EXT && A.dm_patch != nullptr) {
                /* PAPER.md:76 "the residual phase (the open loop wavefront subtracted by the DM)" */
#pragma unroll
                for (int r = 0; r < Cfg::ITEMS; ++r) {
                    const int s = sg + r * Cfg::SG;
                    if (s < Cfg::SPOTS && aoff[r] >= 0) {
                        const int4 inf = s_info[s];
                        const float2 d = __ldg(reinterpret_cast<const float2 *>(A.dm_patch)
                                               + ((size_t)inf.y * A.nsub + inf.z) * Cfg::NP + q2);
                        ph[r].x -= d.x; ph[r].y -= d.y;
                    }
                }
            }
            float2 am = make_float2(0.f, 0.f);
            int acur = -1;
#pragma unroll
            for (int r = 0; r < Cfg::ITEMS; ++r) {
                const int s = sg + r * Cfg::SG;
                if (s < Cfg::SPOTS) {
                    float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (aoff[r] >= 0) {
                        if (aoff[r] != acur) {          /* amplitude patch changes only with the subaperture */
                            acur = aoff[r];
                            am = __ldg(reinterpret_cast<const float2 *>(A.amp + acur));
                        }
                        float2 e0, e1;
                        if (EXTK == 2) {
                            /* several sub-layers: sodium is on by construction.  (Written as if (sodium) .. else ..
                             * this compiled to BOTH field evaluations per pixel: twice the sincos.) */
                            const float2 g = __ldg(A.sod_g + (size_t)layer * A.nsub + s_info[s].z);
                            const float lin = fmaf(g.x, dk0, g.y * dj);
                            e0 = field_value(ph[r].x, am.x * lsw, A.turns, ramp0 - (lin + quad0));
                            e1 = field_value(ph[r].y, am.y * lsw, A.turns, ramp1 - (lin + g.x + quad1));
                        } else if (sodium) {
                            const float2 g = __ldg(A.sod_g + (size_t)layer * A.nsub + s_info[s].z);
                            const float lin = fmaf(g.x, dk0, g.y * dj);
                            e0 = field_value(ph[r].x, am.x * lsw, A.turns, ramp0 - (lin + quad0));
                            e1 = field_value(ph[r].y, am.y * lsw, A.turns, ramp1 - (lin + g.x + quad1));
                        } else {
                            e0 = field_value(ph[r].x, am.x, A.turns, ramp0);
                            e1 = field_value(ph[r].y, am.y, A.turns, ramp1);
                        }
                        e = make_float4(e0.x, e0.y, e1.x, e1.y);
                    }
                    reinterpret_cast<float4 *>(ebuf + s * Cfg::ES)[q2] = e;
                }
            }
        }
    }
    __syncthreads();

    /* ---- phase 1: autocorrelation rows, table product, x-transform ---- */
    {
        const float *eb = ebuf + lane * Cfg::ES;
        float *hb = hbuf + lane * HSTRIDE;
        const int i = max(s_info[lane].z, 0);
        const float2 *Mi = A.M + (size_t)i * A.mstride;
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            const int ly = pass == 0 ? warp : (warp == 0 ? n / 2 : n - warp);
            LagAcc<n> L;
            L.clear();
            if (ly == 0) {
#pragma unroll 1
                for (int j = 0; j < n; ++j) rowself_acc<n>(eb + j * 2 * n, L);
            } else {
#pragma unroll 1
                for (int j = 0; j < n - ly; ++j) rowpair_acc<n>(eb + j * 2 * n, eb + (j + ly) * 2 * n, L);
            }
            float2 acc[Cfg::LX];
            if (ly == 0) {
                acc[n - 1] = make_float2(L.xy[n - 1].x + L.xy[n - 1].y, 0.f);
#pragma unroll
                for (int lx = 1; lx < n; ++lx) {
                    const float2 g = L.lag_value(n - 1 + lx);
                    acc[n - 1 + lx] = g;
                    acc[n - 1 - lx] = make_float2(g.x, -g.y);
                }
            } else {
#pragma unroll
                for (int a = 0; a < Cfg::LX; ++a) acc[a] = L.lag_value(a);
            }
            if (SPLIT) {
                /* first pass: row slot = warp in the H buffer; second pass: same slot in the field buffer,
                 * once every warp has finished reading the field */
                if (pass == 1) __syncthreads();
                finish_row<n>(acc, Mi + ly, (pass == 0 ? hb : ebuf + lane * Cfg::ES) + warp * 32);
            } else {
                /* several sub-layers: everything up to the table product is linear in the intensity, so the raw
                 * lag row piles up in shared memory and only the last sub-layer pays the table product and
                 * the x-transform (whose 16 complex values then take the row's place) */
                float2 *grow = reinterpret_cast<float2 *>(hb + ly * Cfg::RS);
                if (layer > 0) {
#pragma unroll
                    for (int a = 0; a < Cfg::LX; ++a) { const float2 g = grow[a]; acc[a].x += g.x; acc[a].y += g.y; }
                }
                if (layer + 1 < n_layers) {
#pragma unroll
                    for (int a = 0; a < Cfg::LX; ++a) grow[a] = acc[a];
                } else {
                    finish_row<n, true>(acc, Mi + ly, hb + ly * Cfg::RS);
                }
            }
        }
    }
    }   /* sub-layers */
    __syncthreads();

    /* ---- phase 2: y-transform (real part), threshold, centre of gravity ---- */
    {
        const int half = lane >> 4, C = lane & 15;
        for (int s = warp * 2 + half; s < Cfg::SPOTS; s += 2 * Cfg::NW) {
            const float *hb = hbuf + s * HSTRIDE + 2 * C;
            const float *hb2 = ebuf + s * Cfg::ES + 2 * C;       /* SPLIT: second-pass rows */
            float yr[16], yi[16];
#pragma unroll
            for (int m = 0; m < 16; ++m) {
                if (m < n) {
                    /* lag row m sits in slot m (first pass), 0 (m = n/2) or n - m (second pass) */
                    const float *src = !SPLIT ? hb + m * Cfg::RS
                                     : m < n / 2 ? hb + m * 32 : hb2 + (m == n / 2 ? 0 : n - m) * 32;
                    const float2 v = *reinterpret_cast<const float2 *>(src);
                    yr[m] = v.x; yi[m] = v.y;
                } else { yr[m] = 0.f; yi[m] = 0.f; }
            }
            fft_fma<16, +1, n>(yr, yi);          /* B[R,C] = Re sum_m H[m][C] w_16^(R m) */
            float bcol[16];
#pragma unroll
            for (int R = 0; R < 16; ++R) bcol[R] = yr[fft_out_index<16>(R)];
            const int4 inf = s_info[s];
            const size_t o = (size_t)inf.y * A.nsub + max(inf.z, 0);
            if (inf.z >= 0 && A.binned) {
#pragma unroll
                for (int R = 0; R < 16; ++R) A.binned[(o * 16 + R) * 16 + C] = bcol[R];
            }
            if (EXT && A.flux > 0.f) {
                add_noise_col16(bcol, C, A.key, A.t0 + (unsigned)inf.y, (unsigned)max(inf.z, 0), A.flux, A.ron2, A.photon_model);
                if (inf.z >= 0 && A.noisy) {
#pragma unroll
                    for (int R = 0; R < 16; ++R) A.noisy[(o * 16 + R) * 16 + C] = bcol[R];
                }
            }
            const float2 sl = cog16<MODE>(bcol, C, A.tau);
            if (inf.z >= 0 && C == 0) reinterpret_cast<float2 *>(A.slopes)[o] = sl;
        }
    }
}

/* ------------------------------------------------------------------------------------------------
 * Size-generic kernel (any even or odd n <= 32, any D <= 32): one CTA of 128 threads per spot, the
 * same three steps written as plain loops.  Slow; it exists so that every size the ABI accepts has
 * a kernel, and as an independently written cross-check of the specialised instances.
 * ---------------------------------------------------------------------------------------------- */
constexpr int GEN_THREADS = 128;

__global__ void __launch_bounds__(GEN_THREADS) wk_generic_kernel(const WkArgs A, int n, int D)
{
    extern __shared__ __align__(16) float smem[];
    const int LX = 2 * n - 1;
    float2 *e = reinterpret_cast<float2 *>(smem);           /* [n*n]   */
    float2 *S = e + n * n;                                  /* [n*LX]  */
    float2 *tw = S + n * LX;                                /* [D]     */
    float *B = reinterpret_cast<float *>(tw + D);           /* [D*D]   */
    float *red = B + D * D;                                 /* [3*GEN_THREADS] */

    const int tid = threadIdx.x;
    const int g = blockIdx.x;
    const int i = g / A.T, t = g - i * A.T;
    const int2 yx = A.valid[i];
    const int off = yx.x * n * A.N + yx.y * n;

    for (int m = tid; m < D; m += GEN_THREADS) {
        float s, c;
        sincospif(2.f * (float)m / (float)D, &s, &c);
        tw[m] = make_float2(c, s);
    }
    const float2 *Mi = A.M + (size_t)i * A.mstride;
    const int n_layers = A.L > 0 ? A.L : 1;                /* A.L == 0: the plain single-layer sensor */
    for (int layer = 0; layer < n_layers; ++layer) {
    __syncthreads();
    for (int q = tid; q < n * n; q += GEN_THREADS) {
        const int j = q / n, k = q - j * n, o = off + j * A.N + k;
        float extra = 0.f, sw = 1.f;
        if (A.L > 0) {                                     /* sub-layer's analytic phase, turns (reading B1) */
            const float2 g = A.sod_g[(size_t)layer * A.nsub + i];
            const float dj = (float)j - 0.5f * (float)(n - 1), dk = (float)k - 0.5f * (float)(n - 1);
            extra = g.x * dk + g.y * dj + A.sod_q[layer] * (dj * dj + dk * dk);
            sw = A.sod_sw[layer];
        }
        float pv = A.phase[(size_t)t * A.frame_stride + (size_t)layer * A.layer_stride + o];
        if (A.dm_patch != nullptr) pv -= A.dm_patch[((size_t)t * A.nsub + i) * (n * n) + q];   /* residual */
        e[q] = field_value(pv, A.amp[o] * sw, A.turns, (float)(j + k) * A.ramp_unit - extra);
    }
    __syncthreads();

    for (int idx = tid; idx < n * LX; idx += GEN_THREADS) {
        const int ly = idx / LX, lx = idx - ly * LX - (n - 1);
        const int k_lo = lx < 0 ? -lx : 0, k_hi = lx < 0 ? n : n - lx;
        float gr = 0.f, gi = 0.f;
        for (int j = 0; j + ly < n; ++j)
            for (int k = k_lo; k < k_hi; ++k) {
                const float2 u = e[j * n + k], v = e[(j + ly) * n + k + lx];
                gr = fmaf(u.x, v.x, fmaf(u.y, v.y, gr));     /* u * conj(v) */
                gi = fmaf(u.y, v.x, fmaf(-u.x, v.y, gi));
            }
        const float2 mv = Mi[(idx - ly * LX) * n + ly];
        float2 sv = make_float2(gr * mv.x - gi * mv.y, gr * mv.y + gi * mv.x);
        if (layer > 0) { sv.x += S[idx].x; sv.y += S[idx].y; }      /* sub-layer arrays piled up */
        S[idx] = sv;
    }
    }   /* sub-layers */
    __syncthreads();

    for (int px = tid; px < D * D; px += GEN_THREADS) {
        const int R = px / D, C = px - R * D;
        float acc = 0.f;
        for (int ly = 0; ly < n; ++ly)
            for (int a = 0; a < LX; ++a) {
                int m = (R * ly + C * (a - (n - 1))) % D;
                if (m < 0) m += D;
                const float2 w = tw[m], s = S[ly * LX + a];
                acc += s.x * w.x - s.y * w.y;
            }
        B[px] = acc;
    }
    __syncthreads();
    const size_t o = (size_t)t * A.nsub + i;
    if (A.binned)
        for (int px = tid; px < D * D; px += GEN_THREADS) A.binned[o * D * D + px] = B[px];
    if (A.flux > 0.f) {                                    /* detector noise, pixel p = C*D + R (noise.cuh) */
        for (int px = tid; px < D * D; px += GEN_THREADS) {
            const int R = px / D, C = px - R * D, p = C * D + R;
            float z[4];
            normal4(A.key, A.t0 + (unsigned)t, (unsigned)i, (unsigned)(p >> 2), z);
            if (A.photon_model == 1) {
                const uint4 x = philox4x32_10(make_uint4((unsigned)(p >> 1), (unsigned)i, A.t0 + (unsigned)t, 1u), A.key);
                B[px] = fmaf(sqrtf(A.ron2), z[p & 3], poisson_count(B[px], A.flux, x, A.key, A.t0 + (unsigned)t, (unsigned)i, (unsigned)p));
            } else {
                B[px] = noisy_count(B[px], A.flux, A.ron2, z[p & 3]);
            }
            if (A.noisy) A.noisy[o * D * D + px] = B[px];
        }
        __syncthreads();
    }

    /* H7: peak */
    float mx = -INFINITY;
    for (int px = tid; px < D * D; px += GEN_THREADS) mx = fmaxf(mx, B[px]);
    red[tid] = mx;
    __syncthreads();
    for (int o = GEN_THREADS / 2; o >= 1; o >>= 1) {
        if (tid < o) red[tid] = fmaxf(red[tid], red[tid + o]);
        __syncthreads();
    }
    const float thr = A.tau * red[0];
    __syncthreads();
    /* H8: centre of gravity */
    const float ref = 0.5f * (float)(D - 1);
    float sw = 0.f, sx = 0.f, sy = 0.f;
    for (int px = tid; px < D * D; px += GEN_THREADS) {
        const int R = px / D, C = px - R * D;
        const float v = B[px];
        const float w = A.mode == 0 ? fmaxf(v - thr, 0.f) : (v >= thr ? v : 0.f);
        sw += w;
        sx = fmaf(w, (float)C - ref, sx);
        sy = fmaf(w, (float)R - ref, sy);
    }
    red[tid] = sw; red[GEN_THREADS + tid] = sx; red[2 * GEN_THREADS + tid] = sy;
    __syncthreads();
    for (int o = GEN_THREADS / 2; o >= 1; o >>= 1) {
        if (tid < o) {
            red[tid] += red[tid + o];
            red[GEN_THREADS + tid] += red[GEN_THREADS + tid + o];
            red[2 * GEN_THREADS + tid] += red[2 * GEN_THREADS + tid + o];
        }
        __syncthreads();
    }
    if (tid == 0) {
        const float w = red[0];
        A.slopes[2 * o] = w == 0.f ? 0.f : red[GEN_THREADS] / w;
        A.slopes[2 * o + 1] = w == 0.f ? 0.f : red[2 * GEN_THREADS] / w;
    }
}

template <int n, int MODE, int EXTK>
cudaError_t launch_special_mode(shwfs_handle *h, const WkArgs &A, cudaStream_t st)
{
    using Cfg = WkCfg<n>;
    static char name[64];
    if (!name[0]) snprintf(name, sizeof(name), "wk_measure_kernel<%d,%d,%d>", n, MODE, EXTK);
    h->last_kernel = name;
    static shwfs_once_per_device attr;
    int dev;
    if (attr.pending(&dev)) {
        cudaError_t e = cudaFuncSetAttribute(wk_measure_kernel<n, MODE, EXTK>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)WkSmem<n, (EXTK < 2)>::BYTES);
        if (e != cudaSuccess) return e;
        attr.mark(dev);
    }
    const int grid = (A.total + Cfg::SPOTS - 1) / Cfg::SPOTS;
    wk_measure_kernel<n, MODE, EXTK><<<grid, Cfg::THREADS, WkSmem<n, (EXTK < 2)>::BYTES, st>>>(A);
    return cudaGetLastError();
}

template <int n>
cudaError_t launch_special(shwfs_handle *h, const WkArgs &A, cudaStream_t st)
{
    if (A.L > 1)
        return A.mode == 0 ? launch_special_mode<n, 0, 2>(h, A, st) : launch_special_mode<n, 1, 2>(h, A, st);
    if (A.L > 0 || A.flux > 0.f || A.dm_patch != nullptr)
        return A.mode == 0 ? launch_special_mode<n, 0, 1>(h, A, st) : launch_special_mode<n, 1, 1>(h, A, st);
    return A.mode == 0 ? launch_special_mode<n, 0, 0>(h, A, st) : launch_special_mode<n, 1, 0>(h, A, st);
}

}  // namespace

int shwfs_wk_supported(const shwfs_handle *h, int generic)
{
    if (generic) return h->n <= 32 && h->D <= 32;
    return h->D == 16 && (h->n == 8 || h->n == 10 || h->n == 16);
}

cudaError_t shwfs_wk_build_table(shwfs_handle *h, cudaStream_t st)
{
    const int LX = 2 * h->n - 1;
    const int blocks = h->has_kernels ? h->nsub : 1;
    const size_t smem = h->has_kernels ? sizeof(double2) * (size_t)h->P * LX : 0;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(wk_table_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    wk_table_kernel<<<blocks, 128, smem, st>>>(h->d_kernels, h->has_kernels, h->n, h->P, h->b, h->d_wk_table);
    return cudaGetLastError();
}

cudaError_t shwfs_wk_launch(shwfs_handle *h, const float *phase, int T, int call_T, float *slopes, float *binned,
                            float *noisy, unsigned t_base, const float *dm_patch, int generic, cudaStream_t st)
{
    WkArgs A;
    A.phase = phase; A.amp = h->d_amp; A.valid = h->d_valid; A.M = h->d_wk_table;
    A.slopes = slopes; A.binned = binned;
    A.frame_stride = (long long)h->N * h->N;
    A.sod_g = h->d_sod_g; A.noisy = noisy; A.layer_stride = 0; A.L = h->sod_L;
    for (int l = 0; l < SHWFS_MAX_LAYERS; ++l) { A.sod_q[l] = h->sod_q[l]; A.sod_sw[l] = h->sod_sw[l]; }
    if (h->sod_L > 0 && !h->sod_shared) { A.layer_stride = A.frame_stride; A.frame_stride *= h->sod_L; }
    A.flux = h->nz_flux; A.ron2 = h->nz_ron * h->nz_ron; A.photon_model = h->nz_model;
    A.key = make_uint2((unsigned)h->nz_seed, (unsigned)(h->nz_seed >> 32));
    A.t0 = h->nz_first_frame + t_base;
    A.dm_patch = dm_patch;
    A.patch = h->d_patch;
    A.sched = h->d_sched;
    A.T = T; A.N = h->N; A.nsub = h->nsub; A.mstride = h->wk_table_stride;
    A.total = T * h->nsub; A.mode = h->mode;
    A.tau = h->tau;
    A.turns = (float)((double)h->c_phi / 6.283185307179586476925286766559);
    A.ramp_unit = 0.5f / (float)h->P;
    if (A.total == 0) return cudaSuccess;
    h->launches += 1;
    /* n = 8, 10 under SHWFS_ALGO_AUTO: direct sums win on batches (1.0e9 against 0.7e9 spots/s at config 4), but a call of
     * one or two frames (the closed-loop step) is less than a wave of their 32-spot CTAs and runs at the latency of one
     * CTA; the half-warp-per-spot FFT instance spreads it over four times as many CTAs without CTA barriers */
    if (!generic && !h->algo_explicit && h->algo == SHWFS_ALGO_WK && h->D == 16 && (h->n == 8 || h->n == 10)) {
        const long long call_spots = (long long)(call_T > T ? call_T : T) * h->nsub;
        if (call_spots <= 64LL * h->sms) return shwfs_wk_fft_launch(h, A, h->n, st);
    }
    if (h->algo != SHWFS_ALGO_WK && !generic && shwfs_wk_fft_supported(h))   /* explicit WK: direct sums */
        return shwfs_wk_fft_launch(h, A, h->n, st);
    if (!generic && shwfs_wk_supported(h, 0)) {
        switch (h->n) {
        case 8: return launch_special<8>(h, A, st);
        case 10: return launch_special<10>(h, A, st);
        case 16: return launch_special<16>(h, A, st);
        default: return cudaErrorInvalidValue;
        }
    }
    const int n = h->n, D = h->D, LX = 2 * n - 1;
    const size_t smem = sizeof(float2) * (size_t)(n * n + n * LX + D) + sizeof(float) * (size_t)(D * D + 3 * GEN_THREADS);
    h->last_kernel = "wk_generic_kernel";
    wk_generic_kernel<<<A.total, GEN_THREADS, smem, st>>>(A, n, D);
    return cudaGetLastError();
}
