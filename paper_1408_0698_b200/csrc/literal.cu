/*
 * literal.cu -- the Shack-Hartmann chain in the literal order of PAPER.md:91, sm_100a:
 *   "The WF is split into sub-apertures and the spot computed by FFT for each sensor sub-aperture ...
 *    a convolution for a gaussian of the desired properties ... the centroid computed on the final
 *    image to retrieve the slopes."
 * i.e. H1 gather, H2 field, H3 zero-padded P x P FFT, H4 |.|^2, H5 FFT -> x K^ -> inverse FFT,
 * H6 centre + bin, H7 threshold, H8 centre of gravity (include/shwfs.h), all in one kernel; only the
 * phase patch is read from and the two slopes written to HBM (plus K^_i, L2-resident over frames).
 *
 * Thread mapping: P threads per spot, thread r owns ONE LINE of the P x P tile in registers.  A 1-D
 * pass is a register-resident radix-2 DIF FFT with compile-time twiddles (fft_regs.cuh); a 2-D
 * transform is row pass -> transpose through padded shared memory -> column pass.  Because the
 * column pass of one transform leaves thread u holding column u, the next transform starts with its
 * column pass in place, so the three transforms of the elongated chain need three transposes, not six:
 *     rows(e) T cols -> |.|^2 -> cols(I) T rows -> x K^ -> rows^-1 T cols^-1 -> C
 * The first transform is input-pruned (lines >= n are zero: their first butterfly stage is free).
 * It is the timed path when there are no elongation kernels and n >= 16 (config 2), the producer of
 * the stage-0/1 debug images, and an independently written cross-check of the lag-domain path (wk.cu).
 */
#include "internal.h"
#include "fft_regs.cuh"
#include "field.cuh"

namespace {

using namespace shwfs;

constexpr int LIT_THREADS = 128;

struct LitArgs {
    const float *phase;
    const float *amp;
    const int2 *valid;
    const float2 *khat;       /* [nsub][u'][v'] = DFT of the re-centred kernel / P^2, or null */
    float *slopes;
    float *img;               /* stage output or null */
    long long frame_stride;
    int T, N, nsub, total, mode, n, b, D, stage;
    float tau, turns, ramp_unit;
};

/* L-point FFT, natural order in and out (the bit-reversal is a compile-time renaming). */
template <int L, int SIGN, int NZ = L>
__device__ __forceinline__ void fft_nat(float (&re)[L], float (&im)[L])
{
    fft_fma<L, SIGN, NZ>(re, im);
#pragma unroll
    for (int k = 0; k < L; ++k) {
        const int q = fft_out_index<L>(k);
        if (q > k) {
            float t = re[k]; re[k] = re[q]; re[q] = t;
            t = im[k]; im[k] = im[q]; im[q] = t;
        }
    }
}

/* Reduction over the P threads of one spot.  P <= 32: xor shuffles inside the aligned lane segment;
 * P == 64: two warps combined through shared memory (every thread of the CTA takes the barriers). */
template <int P, class Op>
__device__ __forceinline__ float group_reduce(float v, Op op, float *red)
{
    constexpr int W = P < 32 ? P : 32;
#pragma unroll
    for (int o = W / 2; o >= 1; o >>= 1) v = op(v, __shfl_xor_sync(0xffffffffu, v, o));
    if constexpr (P > 32) {
        const int warp = threadIdx.x >> 5;
        __syncthreads();
        if ((threadIdx.x & 31) == 0) red[warp] = v;
        __syncthreads();
        v = op(red[warp & ~1], red[warp | 1]);
    }
    return v;
}

template <int P>
struct LitCfg {
    static constexpr int SPB = LIT_THREADS / P;    /* spots per CTA */
    static constexpr int LD = P + 1;               /* padded line length: transposes are conflict-free */
    static constexpr int TILE = P * LD;            /* float2 elements per spot */
    static constexpr size_t SMEM = sizeof(float2) * (size_t)SPB * TILE + sizeof(float) * (LIT_THREADS / 32);
};

template <int P, int NZ>
__global__ void __launch_bounds__(LIT_THREADS) literal_kernel(const LitArgs A)
{
    using Cfg = LitCfg<P>;
    extern __shared__ __align__(16) float2 lit_smem[];
    const int tid = threadIdx.x, sp = tid / P, r = tid % P;
    float2 *tile = lit_smem + sp * Cfg::TILE;
    float *red = reinterpret_cast<float *>(lit_smem + Cfg::SPB * Cfg::TILE);
    constexpr int LD = Cfg::LD, HP = P / 2;
    constexpr float inv_pp = 1.0f / ((float)P * (float)P);

    const int g = blockIdx.x * Cfg::SPB + sp;
    const bool live = g < A.total;
    int i = 0, t = 0;
    if (live) { i = g / A.T; t = g - i * A.T; }

    float re[P], im[P];

    /* ---- H1 gather + H2 field: thread r < n owns patch row r ---- */
#pragma unroll
    for (int k = 0; k < P; ++k) { re[k] = 0.f; im[k] = 0.f; }
    if (live && r < A.n) {
        const int2 yx = A.valid[i];
        const size_t o = (size_t)(yx.x * A.n + r) * A.N + (size_t)yx.y * A.n;
        const float *pp = A.phase + (size_t)t * A.frame_stride + o;
        const float *pa = A.amp + o;
#pragma unroll
        for (int k = 0; k < NZ; ++k) {
            if (k < A.n) {
                const float2 e = field_value(__ldg(pp + k), __ldg(pa + k), A.turns, (float)(r + k) * A.ramp_unit);
                re[k] = e.x; im[k] = e.y;
            }
        }
    }

    /* ---- H3: rows, transpose, columns (pruned: only the first NZ inputs of a line can be non-zero) ---- */
    fft_nat<P, -1, NZ>(re, im);
#pragma unroll
    for (int u = 0; u < P; ++u) tile[r * LD + u] = make_float2(re[u], im[u]);
    __syncthreads();
#pragma unroll
    for (int v = 0; v < P; ++v) {
        if (v < NZ) { const float2 f = tile[v * LD + r]; re[v] = f.x; im[v] = f.y; }
        else { re[v] = 0.f; im[v] = 0.f; }
    }
    fft_nat<P, -1, NZ>(re, im);

    /* ---- H4: thread u = r holds I[v][u] in re[v] ---- */
#pragma unroll
    for (int v = 0; v < P; ++v) { re[v] = (re[v] * re[v] + im[v] * im[v]) * inv_pp; im[v] = 0.f; }

    const size_t spot = (size_t)t * A.nsub + i;
    if (A.stage == 0 && live) {
#pragma unroll
        for (int v = 0; v < P; ++v) A.img[(spot * P + (v ^ HP)) * P + (r ^ HP)] = re[v];
    }

    /* ---- H5: C = I (*) K_i as columns(I), transpose, rows, x K^, rows^-1, transpose, columns^-1 ---- */
    if (A.khat != nullptr) {
        fft_nat<P, -1>(re, im);
        __syncthreads();
#pragma unroll
        for (int v = 0; v < P; ++v) tile[v * LD + r] = make_float2(re[v], im[v]);
        __syncthreads();
#pragma unroll
        for (int u = 0; u < P; ++u) { const float2 f = tile[r * LD + u]; re[u] = f.x; im[u] = f.y; }
        fft_nat<P, -1>(re, im);
        const float2 *kh = A.khat + (size_t)i * P * P + r;       /* thread v' = r, element u' */
#pragma unroll
        for (int u = 0; u < P; ++u) {
            const float2 k = __ldg(kh + u * P);
            const float x = re[u], y = im[u];
            re[u] = fmaf(x, k.x, -y * k.y);
            im[u] = fmaf(x, k.y, y * k.x);
        }
        fft_nat<P, +1>(re, im);
        __syncthreads();
#pragma unroll
        for (int u = 0; u < P; ++u) tile[r * LD + u] = make_float2(re[u], im[u]);
        __syncthreads();
#pragma unroll
        for (int v = 0; v < P; ++v) { const float2 f = tile[v * LD + r]; re[v] = f.x; im[v] = f.y; }
        fft_nat<P, +1>(re, im);                                   /* re[v] = C[v][u = r] (K^ carries 1/P^2) */
    }
    if (A.stage == 1 && live) {
#pragma unroll
        for (int v = 0; v < P; ++v) A.img[(spot * P + (v ^ HP)) * P + (r ^ HP)] = re[v];
    }

    /* ---- H6: centre (roll by P/2 = xor on a power of two) and b x b binning through shared memory ---- */
    __syncthreads();
    float *Sh = reinterpret_cast<float *>(tile);                  /* [P][LD] floats */
    float *Bb = Sh + P * LD;                                      /* [D*D] floats   */
#pragma unroll
    for (int v = 0; v < P; ++v) Sh[(v ^ HP) * LD + (r ^ HP)] = re[v];
    __syncthreads();
    const int D = A.D, b = A.b, DD = D * D;
    float mx = -INFINITY;
    for (int p = r; p < DD; p += P) {
        const int R = p / D, Cc = p - R * D;
        float s = 0.f;
        for (int al = 0; al < b; ++al)
            for (int be = 0; be < b; ++be) s += Sh[(b * R + al) * LD + b * Cc + be];
        Bb[p] = s;
        mx = fmaxf(mx, s);
    }
    /* ---- H7 + H8 ---- */
    mx = group_reduce<P>(mx, [](float a, float c) { return fmaxf(a, c); }, red);
    const float thr = A.tau * mx, ref = 0.5f * (float)(D - 1);
    float sw = 0.f, sx = 0.f, sy = 0.f;
    for (int p = r; p < DD; p += P) {
        const int R = p / D, Cc = p - R * D;
        const float v = Bb[p];
        const float w = A.mode == 0 ? fmaxf(v - thr, 0.f) : (v >= thr ? v : 0.f);
        sw += w;
        sx = fmaf(w, (float)Cc - ref, sx);
        sy = fmaf(w, (float)R - ref, sy);
        if (A.stage == 2 && live) A.img[spot * DD + p] = v;
    }
    auto add = [](float a, float c) { return a + c; };
    sw = group_reduce<P>(sw, add, red);
    sx = group_reduce<P>(sx, add, red);
    sy = group_reduce<P>(sy, add, red);
    if (live && r == 0)
        reinterpret_cast<float2 *>(A.slopes)[spot] = sw == 0.f ? make_float2(0.f, 0.f) : make_float2(sx / sw, sy / sw);
}

/* ------------------------------------------------------------------------------------------------
 * K^ table (float64 on the device, once per handle): K^_i[v',u'] = sum_q K_i[q] w^(-(q - P/2).(v',u')) / P^2,
 * the DFT of the kernel re-centred so that index (P/2,P/2) is the origin (reading A9, step O5), with the
 * 1/P^2 of the inverse transform folded in.  Stored transposed, [i][u'][v'], so that the P threads of a
 * spot (thread = v') read it coalesced.  One CTA per subaperture, separable O(P^3).
 * ---------------------------------------------------------------------------------------------- */
__global__ void literal_khat_kernel(const float *__restrict__ K, int P, float2 *__restrict__ khat)
{
    extern __shared__ double2 ksm[];
    double2 *tw = ksm;              /* [P]  w^-m */
    double2 *tmp = ksm + P;         /* [P][P]: tmp[qy][u'] */
    const float *Ki = K + (size_t)blockIdx.x * P * P;
    for (int m = threadIdx.x; m < P; m += blockDim.x) {
        double s, c;
        sincospi(-2.0 * (double)m / (double)P, &s, &c);
        tw[m] = make_double2(c, s);
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < P * P; idx += blockDim.x) {
        const int qy = idx / P, u = idx % P;
        double sr = 0.0, si = 0.0;
        for (int qx = 0; qx < P; ++qx) {
            const double2 w = tw[(qx * u) % P];
            const double kv = (double)Ki[qy * P + qx];
            sr += kv * w.x; si += kv * w.y;
        }
        tmp[idx] = make_double2(sr, si);
    }
    __syncthreads();
    const double inv_pp = 1.0 / ((double)P * (double)P);
    for (int idx = threadIdx.x; idx < P * P; idx += blockDim.x) {
        const int u = idx / P, v = idx % P;                /* output [u'][v'] */
        double zr = 0.0, zi = 0.0;
        for (int qy = 0; qy < P; ++qy) {
            const double2 w = tw[(qy * v) % P], tq = tmp[qy * P + u];
            zr += tq.x * w.x - tq.y * w.y;
            zi += tq.x * w.y + tq.y * w.x;
        }
        const double sgn = ((u + v) & 1) ? -inv_pp : inv_pp;    /* w^(+(P/2)(u'+v')) = (-1)^(u'+v') */
        khat[(size_t)blockIdx.x * P * P + idx] = make_float2((float)(zr * sgn), (float)(zi * sgn));
    }
}

template <int P, int NZ>
cudaError_t launch_literal(const LitArgs &A, cudaStream_t st)
{
    using Cfg = LitCfg<P>;
    cudaError_t e = cudaFuncSetAttribute(literal_kernel<P, NZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
    if (e != cudaSuccess) return e;
    const int grid = (A.total + Cfg::SPB - 1) / Cfg::SPB;
    literal_kernel<P, NZ><<<grid, LIT_THREADS, Cfg::SMEM, st>>>(A);
    return cudaGetLastError();
}

template <int P>
cudaError_t launch_literal_p(const LitArgs &A, cudaStream_t st)
{
    return 2 * A.n <= P ? launch_literal<P, P / 2>(A, st) : launch_literal<P, P>(A, st);
}

}  // namespace

int shwfs_literal_supported(const shwfs_handle *h)
{
    return h->P == 8 || h->P == 16 || h->P == 32 || h->P == 64;
}

cudaError_t shwfs_literal_build_khat(shwfs_handle *h, cudaStream_t st)
{
    const int P = h->P;
    const size_t smem = sizeof(double2) * (size_t)(P + P * P);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(literal_khat_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    literal_khat_kernel<<<h->nsub, 256, smem, st>>>(h->d_kernels, P, h->d_khat);
    return cudaGetLastError();
}

cudaError_t shwfs_literal_launch(shwfs_handle *h, const float *phase, int T, float *slopes, int stage,
                                 float *img, cudaStream_t st)
{
    LitArgs A;
    A.phase = phase; A.amp = h->d_amp; A.valid = h->d_valid;
    A.khat = h->has_kernels ? h->d_khat : nullptr;
    A.slopes = slopes; A.img = img;
    A.frame_stride = (long long)h->N * h->N;
    A.T = T; A.N = h->N; A.nsub = h->nsub; A.total = T * h->nsub; A.mode = h->mode;
    A.n = h->n; A.b = h->b; A.D = h->D; A.stage = img ? stage : -1;
    A.tau = h->tau;
    A.turns = (float)((double)h->c_phi / 6.283185307179586476925286766559);
    A.ramp_unit = 0.5f / (float)h->P;
    if (A.total == 0) return cudaSuccess;
    if (h->has_kernels && !h->d_khat) return cudaErrorInvalidValue;
    h->launches += 1;
    h->last_kernel = h->P == 8 ? "literal_kernel<8>" : h->P == 16 ? "literal_kernel<16>" : h->P == 32 ? "literal_kernel<32>" : "literal_kernel<64>";
    switch (h->P) {
    case 8: return launch_literal_p<8>(A, st);
    case 16: return launch_literal_p<16>(A, st);
    case 32: return launch_literal_p<32>(A, st);
    case 64: return launch_literal_p<64>(A, st);
    default: return cudaErrorInvalidValue;
    }
}
