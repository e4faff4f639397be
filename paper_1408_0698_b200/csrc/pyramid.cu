/*
 * pyramid.cu -- pyramid wavefront sensor (include/pyrwfs.h), sm_100a.
 *
 * Steps Q1..Q7 of include/pyrwfs.h.  The work is two Np x Np complex transforms per (frame, modulation point);
 * both are done as hand-written "four-step" FFTs inside a CTA: a line of L = R*R points (R = 16 or 32) is owned
 * by R threads, each holding R points in registers; a line transform is
 *     R-point register FFT over m (x = j + R m)  ->  twiddle w_L^(j p)  ->  exchange through shared memory
 *     ->  R-point register FFT over j            ->  thread p holds X[p + R q], q = 0..R-1,
 * which is again the "thread j holds x[j + R m]" layout, so a forward and an inverse transform chain with no
 * reshuffle in between (the pyramid mask is applied in registers there).  Eight lines per CTA, so that the
 * transposed hand-over between the row and column passes moves 64-byte segments.
 *
 *   pyr_rows_kernel   Q1 field of 8 pupil rows (input-pruned: N <= L/2 non-zero points) -> FFT over x ->
 *                     A1[tk][u][y]            (y < N: only the N non-zero rows exist)
 *   pyr_cols_kernel   8 columns u: FFT over y (input-pruned) -> Q3 mask -> inverse FFT over v ->
 *                     A2[tk][r][u]            (r: the 2N rows that hold the four pupil copies, output-pruned)
 *   pyr_final_kernel  8 rows r, loop over the K modulation points: inverse FFT over u -> |.|^2 accumulated in
 *                     registers (Q4, Q5) -> I2[t][r][c] on the 2N x 2N pixels of the four copies
 *   pyr_bin_kernel    Q6 b x b block sums -> Q[t][a][b][Y][X];  pyr_signal_kernel  Q7 (one CTA per frame).
 * A1 / A2 live in scratch owned by the handle (L2-sized chunks of frames); only the phase is read from and the
 * signals written to HBM by the caller's buffers.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <type_traits>

#include "internal.h"
#include "fft_regs.cuh"
#include "../../include/pyrwfs.h"

struct pyrwfs_handle {
    int N, Np, R, s, bp, Sp, K, nvalid, device;
    float r_mod, D_pix, c_phi;
    int64_t launches;
    float *d_amp;            /* [N*N] */
    int2 *d_valid;           /* [nvalid] (Y, X) */
    int32_t *h_valid;
    float2 *d_tw;            /* [Np] exp(+2 pi i m / Np) */
    float2 *d_mod;           /* [max(K,1)] (r_mod cos th_k / D_pix, r_mod sin th_k / D_pix): turns per pixel */
    int Kp;                  /* number of modulation points actually run: max(K, 1) */
    int chunk;               /* frames per pass through the scratch */
    float2 *d_A1;            /* [chunk*Kp][Np][N]   */
    float2 *d_A2;            /* [chunk*Kp][2N][Np]  */
    float *d_I2;             /* [chunk][2N][2N]     */
    float *d_Q;              /* [chunk][2][2][Sp][Sp] */
};

namespace {

using namespace shwfs;

constexpr int PY_LINES = 8;

/* natural-order copy of a transform result: out[k] = X[k] */
template <int R>
__device__ __forceinline__ void unscramble(float2 (&z)[R])
{
#pragma unroll
    for (int k = 0; k < R; ++k) {
        const int q = fft_out_index<R>(k);
        if (q > k) { const float2 t = z[k]; z[k] = z[q]; z[q] = t; }
    }
}

/* a * w on packed registers: a_r (w_r, w_i) + a_i (-w_i, w_r), two FP32x2 instructions (fft_regs.cuh) */
__device__ __forceinline__ float2 cmul2(float2 a, float2 w)
{
    return __ffma2_rn(bc2(a.y), rot_pi2(w), __fmul2_rn(bc2(a.x), w));
}

/* All products W0 * g^q, q = 0 .. 2^BITS - 1, from the BITS table values pw[b] = g^(2^b): a depth-first walk over
 * the binary expansions of q, one complex product per q and no product more than BITS deep (the rounding of a
 * q-fold recurrence would be q deep), a handful of registers live.  emit(q, w) is called once per q with q a
 * compile-time constant.  Replaces one table lookup per q: at 32 lookups per thread and line with addresses
 * scattered over the table, the L1 data pipe of pyr_cols_kernel ran at 80 % of its wavefront peak and
 * long_scoreboard was its first stall (profiles/r02_pyramid.md). */
template <int BITS>
struct PowWalk {
    template <int Q, int B, typename F>
    __device__ __forceinline__ static void node(float2 w, const float2 (&pw)[BITS], F &emit)
    {
        emit(std::integral_constant<int, Q>(), w);
        if constexpr (B >= 0) below<Q, B>(w, pw, emit);
    }
    /* children of Q: set one more bit among bits B .. 0 */
    template <int Q, int B, typename F>
    __device__ __forceinline__ static void below(float2 w, const float2 (&pw)[BITS], F &emit)
    {
        node<Q + (1 << B), B - 1>(cmul2(w, pw[B]), pw, emit);
        if constexpr (B > 0) below<Q, B - 1>(w, pw, emit);
    }
    template <typename F>
    __device__ __forceinline__ static void run(float2 w0, const float2 (&pw)[BITS], F emit)
    {
        node<0, BITS - 1>(w0, pw, emit);
    }
};

/* One L = R*R point transform of the line owned by the R threads j = 0..R-1 (all in one warp), on packed
 * (re, im) registers with FP32x2 butterflies (fft_fma2).
 * In : z[m] = x[j + R m] (natural order; entries m >= NZ are zero).
 * Out: z[q] = X[p + R q], p = this thread's index (natural order).
 * X[k] = sum_x x[x] exp(SIGN 2 pi i x k / L).  `line` is this line's R*(R+2) float2 of shared memory.
 * The twiddles w_L^(j p), p = 0..R-1, are the powers of w_L^j: log2 R table reads and a PowWalk.            */
template <int R, int SIGN, int NZ>
__device__ __forceinline__ void line_fft(float2 (&z)[R], int j, float2 *__restrict__ line,
                                         const float2 *__restrict__ tw)
{
    constexpr int L = R * R, BITS = ilog2(R);
    fft_fma2<R, SIGN, NZ>(z);
    float2 pw[BITS];
#pragma unroll
    for (int b = 0; b < BITS; ++b) {
        pw[b] = __ldg(tw + ((j << b) & (L - 1)));                       /* w_L^(j 2^b), conjugated for SIGN < 0 */
        if (SIGN < 0) pw[b].y = -pw[b].y;
    }
    PowWalk<BITS>::run(make_float2(1.f, 0.f), pw, [&](auto pc, float2 w) {
        constexpr int p = decltype(pc)::value;
        float2 a = z[fft_out_index<R>(p)];
        if (p > 0) a = cmul2(a, w);
        line[p * (R + 2) + j] = a;
    });
    __syncwarp();
#pragma unroll
    for (int jj = 0; jj < R; jj += 2) {                                 /* this thread is now p = j */
        const float4 v = *reinterpret_cast<const float4 *>(line + j * (R + 2) + jj);   /* row stride R+2: 16-byte rows */
        z[jj] = make_float2(v.x, v.y); z[jj + 1] = make_float2(v.z, v.w);
    }
    __syncwarp();
    fft_fma2<R, SIGN, R>(z);
    unscramble<R>(z);
}

/* index of pupil-plane coordinate c (row or column) among the 2N kept ones, or -1 (Q6: copies at +s and -s) */
__device__ __forceinline__ int kept_index(int c, int N, int Np, int s)
{
    const int d1 = c - s;
    if (d1 >= 0 && d1 < N) return d1;
    const int d2 = (c + s) & (Np - 1);
    return d2 < N ? N + d2 : -1;
}

struct PyArgs {
    const float *phase;      /* first frame of this chunk */
    const float *amp;
    const float2 *tw, *mod;
    float2 *A1, *A2;
    float *I2;
    int N, Np, s, Kp, Tc;
    float turns;             /* phase_to_rad / 2 pi */
    float scale;             /* 1 / (Kp * Np^4): Q4 normalisation and Q5 average */
};

/* ---- Q1 + row half of Q2: grid (ceil(N/8), Tc*Kp), block 8*R ------------------------------------------- */
template <int R>
__global__ void __launch_bounds__(PY_LINES * R) pyr_rows_kernel(const PyArgs A)
{
    constexpr int L = R * R, NZ = R / 2;
    extern __shared__ __align__(16) float2 py_smem[];
    const int tid = threadIdx.x, b = tid / R, j = tid % R;
    const int tk = blockIdx.y, t = tk / A.Kp, k = tk - t * A.Kp;
    const int y0 = blockIdx.x * PY_LINES, y = y0 + b;
    float2 z[R];
#pragma unroll
    for (int m = 0; m < R; ++m) z[m] = make_float2(0.f, 0.f);
    if (y < A.N) {
        const float2 md = __ldg(A.mod + k);                   /* modulation tilt, turns per pixel */
        const float *pp = A.phase + ((size_t)t * A.N + y) * A.N;
        const float *pa = A.amp + (size_t)y * A.N;
#pragma unroll
        for (int m = 0; m < NZ; ++m) {
            const int x = j + R * m;
            if (x < A.N) {
                float u = fmaf(__ldg(pp + x), A.turns, fmaf(md.x, (float)x, md.y * (float)y));
                u -= rintf(u);
                float sn, cs;
                __sincosf(u * 6.283185307179586f, &sn, &cs);
                const float a = __ldg(pa + x);
                z[m] = make_float2(a * cs, a * sn);
            }
        }
    }
    line_fft<R, -1, NZ>(z, j, py_smem + b * R * (R + 2), A.tw);
    __syncthreads();
    /* transposed hand-over: stage[u][b] (row padded to 9), then 64-byte segments of A1[tk][u][y0..y0+7] */
    float2 *stage = py_smem;
#pragma unroll
    for (int q = 0; q < R; ++q) stage[(j + R * q) * (PY_LINES + 1) + b] = z[q];
    __syncthreads();
    float2 *dst = A.A1 + (size_t)tk * L * A.N;
    for (int e = tid; e < L * PY_LINES; e += PY_LINES * R) {
        const int u = e / PY_LINES, bb = e - u * PY_LINES;
        if (y0 + bb < A.N) dst[(size_t)u * A.N + y0 + bb] = stage[u * (PY_LINES + 1) + bb];
    }
}

/* ---- column half of Q2, Q3 mask, column half of Q4: grid (Np/8, Tc*Kp) ---------------------------------- */
template <int R>
__global__ void __launch_bounds__(PY_LINES * R, 2) pyr_cols_kernel(const PyArgs A)
{
    constexpr int L = R * R, NZ = R / 2;
    extern __shared__ __align__(16) float2 py_smem[];
    const int tid = threadIdx.x, b = tid / R, j = tid % R;
    const int tk = blockIdx.y, u0 = blockIdx.x * PY_LINES, u = u0 + b;
    float2 z[R];
#pragma unroll
    for (int m = 0; m < R; ++m) z[m] = make_float2(0.f, 0.f);
    const float2 *src = A.A1 + ((size_t)tk * L + u) * A.N;
#pragma unroll
    for (int m = 0; m < NZ; ++m) {
        const int y = j + R * m;
        if (y < A.N) z[m] = __ldg(src + y);
    }
    float2 *line = py_smem + b * R * (R + 2);
    line_fft<R, -1, NZ>(z, j, line, A.tw);
    /* Q3: exp(-2 pi i s (|u~| + |v~|) / Np) at v = j + R q.  |v~| = v for q < R/2 and L - v above, so the phase
     * index runs s (ua + j) + (R s) q over the lower half of q and s (ua - j) - (R s) q over the upper one: two
     * table reads for the ends and a PowWalk over the powers of w^(R s) for each half. */
    {
        constexpr int HB = ilog2(R) - 1, H = R / 2;
        const int ua = u < L / 2 ? u : L - u;
        float2 st[HB], stc[HB];
#pragma unroll
        for (int b = 0; b < HB; ++b) {
            st[b] = __ldg(A.tw + ((A.s * R << b) & (L - 1)));           /* w^(R s 2^b) */
            stc[b] = make_float2(st[b].x, -st[b].y);
        }
        float2 lo = __ldg(A.tw + ((A.s * (ua + j)) & (L - 1)));                     /* q = 0   */
        float2 hi = __ldg(A.tw + ((A.s * (ua - j) - A.s * R * H) & (L - 1)));        /* q = R/2 */
        lo.y = -lo.y; hi.y = -hi.y;                                     /* the mask is the conjugate */
        PowWalk<HB>::run(lo, stc, [&](auto qc, float2 w) { constexpr int q = decltype(qc)::value; z[q] = cmul2(z[q], w); });
        PowWalk<HB>::run(hi, st, [&](auto qc, float2 w) { constexpr int q = decltype(qc)::value; z[H + q] = cmul2(z[H + q], w); });
    }
    line_fft<R, +1, R>(z, j, line, A.tw);
    __syncthreads();
    float2 *stage = py_smem;                                   /* stage[y'][b] */
#pragma unroll
    for (int q = 0; q < R; ++q) stage[(j + R * q) * (PY_LINES + 1) + b] = z[q];
    __syncthreads();
    float2 *dst = A.A2 + (size_t)tk * 2 * A.N * L;
    /* only the 2N kept rows are written: row r < N is pupil-plane row r + s, row N + d is row (d - s) mod Np
     * (the inverse of kept_index; the two ranges are disjoint by the create-time checks on s) */
    for (int e = tid; e < 2 * A.N * PY_LINES; e += PY_LINES * R) {
        const int r = e / PY_LINES, bb = e - r * PY_LINES;
        const int yy = r < A.N ? r + A.s : (r - A.N - A.s) & (L - 1);
        dst[(size_t)r * L + u0 + bb] = stage[yy * (PY_LINES + 1) + bb];
    }
}

/* ---- row half of Q4, |.|^2, Q5: grid (2N/8 rounded up, Tc) ---------------------------------------------- */
template <int R>
__global__ void __launch_bounds__(PY_LINES * R, 2) pyr_final_kernel(const PyArgs A)
{
    constexpr int L = R * R;
    extern __shared__ __align__(16) float2 py_smem[];
    const int tid = threadIdx.x, b = tid / R, j = tid % R;
    const int t = blockIdx.y, r = blockIdx.x * PY_LINES + b, rows = 2 * A.N;
    const bool live = r < rows;
    float acc[R];
#pragma unroll
    for (int q = 0; q < R; ++q) acc[q] = 0.f;
    float2 *line = py_smem + b * R * (R + 2);
    for (int k = 0; k < A.Kp; ++k) {
        float2 z[R];
        const float2 *src = A.A2 + (((size_t)t * A.Kp + k) * rows + (live ? r : 0)) * L;
#pragma unroll
        for (int m = 0; m < R; ++m) z[m] = live ? __ldg(src + j + R * m) : make_float2(0.f, 0.f);
        line_fft<R, +1, R>(z, j, line, A.tw);
#pragma unroll
        for (int q = 0; q < R; ++q) acc[q] = fmaf(z[q].x, z[q].x, fmaf(z[q].y, z[q].y, acc[q]));
    }
    if (live) {
        float *dst = A.I2 + ((size_t)t * rows + r) * rows;
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const int c = kept_index(j + R * q, A.N, L, A.s);
            if (c >= 0) dst[c] = acc[q] * A.scale;
        }
    }
}

/* ---- Q6: Q[t][a][b][Y][X] = block sums of I2: one thread per output ------------------------------------ */
__global__ void pyr_bin_kernel(const float *__restrict__ I2, int N, int bp, int Sp, int Tc, float *__restrict__ Q)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int per = 4 * Sp * Sp;
    if (idx >= Tc * per) return;
    const int t = idx / per, rem = idx - t * per;
    const int ab = rem / (Sp * Sp), yx = rem - ab * Sp * Sp, Y = yx / Sp, X = yx - Y * Sp;
    const int ia = ab >> 1, ib = ab & 1, rows = 2 * N;
    const float *src = I2 + ((size_t)t * rows + ia * N + Y * bp) * rows + ib * N + X * bp;
    float sum = 0.f;
    for (int dy = 0; dy < bp; ++dy)
        for (int dx = 0; dx < bp; ++dx) sum += src[(size_t)dy * rows + dx];
    Q[idx] = sum;
}

/* ---- Q7: one CTA per frame ------------------------------------------------------------------------------ */
__global__ void __launch_bounds__(256) pyr_signal_kernel(const float *__restrict__ Q, const int2 *__restrict__ valid,
                                                         int nvalid, int Sp, float *__restrict__ signals)
{
    __shared__ float red[256];
    const int t = blockIdx.x, tid = threadIdx.x, SS = Sp * Sp;
    const float *q = Q + (size_t)t * 4 * SS;
    float tot = 0.f;
    for (int i = tid; i < nvalid; i += 256) {
        const int o = valid[i].x * Sp + valid[i].y;
        tot += (q[o] + q[SS + o]) + (q[2 * SS + o] + q[3 * SS + o]);
    }
    red[tid] = tot;
    __syncthreads();
    for (int o = 128; o >= 1; o >>= 1) {
        if (tid < o) red[tid] += red[tid + o];
        __syncthreads();
    }
    const float inv = (float)nvalid / red[0];                 /* 1 / I0 */
    for (int i = tid; i < nvalid; i += 256) {
        const int o = valid[i].x * Sp + valid[i].y;
        const float pp = q[o], pm = q[SS + o], mp = q[2 * SS + o], mm = q[3 * SS + o];   /* [a][b] */
        signals[((size_t)t * nvalid + i) * 2] = ((pp + mp) - (pm + mm)) * inv;
        signals[((size_t)t * nvalid + i) * 2 + 1] = ((pp + pm) - (mp + mm)) * inv;
    }
}

template <int R>
cudaError_t run_chunk(pyrwfs_handle *h, const float *phase, int Tc, float *signals, float *q_out, cudaStream_t st)
{
    constexpr int L = R * R;
    PyArgs A;
    A.phase = phase; A.amp = h->d_amp; A.tw = h->d_tw; A.mod = h->d_mod;
    A.A1 = h->d_A1; A.A2 = h->d_A2; A.I2 = h->d_I2;
    A.N = h->N; A.Np = h->Np; A.s = h->s; A.Kp = h->Kp; A.Tc = Tc;
    A.turns = (float)((double)h->c_phi / 6.283185307179586476925286766559);
    A.scale = (float)(1.0 / ((double)h->Kp * pow((double)h->Np, 4.0)));
    const size_t smem = sizeof(float2) * (size_t)(L * (PY_LINES + 1) > PY_LINES * R * (R + 2) ? L * (PY_LINES + 1)
                                                                                              : PY_LINES * R * (R + 2));
    static shwfs_once_per_device attr;
    int dev;
    if (attr.pending(&dev)) {
        cudaError_t e = cudaFuncSetAttribute(pyr_rows_kernel<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(pyr_cols_kernel<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(pyr_final_kernel<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr.mark(dev);
    }
    const int threads = PY_LINES * R;
    pyr_rows_kernel<R><<<dim3((h->N + PY_LINES - 1) / PY_LINES, Tc * h->Kp), threads, smem, st>>>(A);
    pyr_cols_kernel<R><<<dim3(L / PY_LINES, Tc * h->Kp), threads, smem, st>>>(A);
    pyr_final_kernel<R><<<dim3((2 * h->N + PY_LINES - 1) / PY_LINES, Tc), threads, smem, st>>>(A);
    const int nq = Tc * 4 * h->Sp * h->Sp;
    float *Q = q_out ? q_out : h->d_Q;
    pyr_bin_kernel<<<(nq + 255) / 256, 256, 0, st>>>(h->d_I2, h->N, h->bp, h->Sp, Tc, Q);
    if (signals) pyr_signal_kernel<<<Tc, 256, 0, st>>>(Q, h->d_valid, h->nvalid, h->Sp, signals);
    h->launches += signals ? 5 : 4;
    return cudaGetLastError();
}

}  // namespace

namespace {

void pyr_free(pyrwfs_handle *h)
{
    if (!h) return;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != h->device) cudaSetDevice(h->device);
    cudaFree(h->d_amp); cudaFree(h->d_valid); cudaFree(h->d_tw); cudaFree(h->d_mod);
    cudaFree(h->d_A1); cudaFree(h->d_A2); cudaFree(h->d_I2); cudaFree(h->d_Q);
    free(h->h_valid);
    if (prev >= 0 && prev != h->device) cudaSetDevice(prev);
    delete h;
    cudaGetLastError();
}

#define PY_TRY(call, where)                                                          \
    do {                                                                             \
        cudaError_t e_ = (call);                                                     \
        if (e_ != cudaSuccess) {                                                     \
            shwfs_note_cuda_error(e_, where);                                        \
            rc = (e_ == cudaErrorMemoryAllocation) ? SHWFS_ENOMEM : SHWFS_ECUDA;     \
            goto fail;                                                               \
        }                                                                            \
    } while (0)

int pyr_run(pyrwfs_handle *h, const float *phase, int T, float *signals, float *q_out, cudaStream_t st)
{
    const size_t fr = (size_t)h->N * h->N, qper = (size_t)4 * h->Sp * h->Sp;
    for (int t0 = 0; t0 < T; t0 += h->chunk) {
        const int tc = T - t0 < h->chunk ? T - t0 : h->chunk;
        float *sg = signals ? signals + (size_t)t0 * h->nvalid * 2 : nullptr;
        float *qo = q_out ? q_out + (size_t)t0 * qper : nullptr;
        cudaError_t e = h->R == 32 ? run_chunk<32>(h, phase + (size_t)t0 * fr, tc, sg, qo, st)
                                   : run_chunk<16>(h, phase + (size_t)t0 * fr, tc, sg, qo, st);
        if (e != cudaSuccess) { shwfs_note_cuda_error(e, "pyramid kernels"); return SHWFS_ECUDA; }
    }
    return SHWFS_OK;
}

}  // namespace

extern "C" {

int pyrwfs_create(const pyrwfs_config *c, pyrwfs_handle **out)
{
    if (!c || !out || !c->amplitude) return SHWFS_EINVAL;
    const int N = c->n_pupil, Np = c->pad, s = c->separation, bp = c->bin;
    if (N <= 0 || bp <= 0 || N % bp || s <= 0 || c->mod_points < 0) return SHWFS_EINVAL;
    if (!(c->pupil_diameter_px > 0.f) || !isfinite(c->mod_radius) || c->mod_radius < 0.f ||
        !isfinite(c->phase_to_rad) || !isfinite(c->min_illum)) return SHWFS_EINVAL;
    if (Np != 256 && Np != 1024) return (Np > 0 && (Np & (Np - 1)) == 0) ? SHWFS_EUNSUPPORTED : SHWFS_EINVAL;
    if (2 * N > Np || 2 * s < N || 2 * s + N > Np) return SHWFS_EINVAL;
    const int Sp = N / bp;
    int32_t *valid = (int32_t *)malloc(sizeof(int32_t) * 2 * (size_t)Sp * Sp);
    if (!valid) return SHWFS_ENOMEM;
    int nv = 0;
    for (int Y = 0; Y < Sp; ++Y)
        for (int X = 0; X < Sp; ++X) {
            double sum = 0.0;
            for (int dy = 0; dy < bp; ++dy)
                for (int dx = 0; dx < bp; ++dx) sum += (double)c->amplitude[(size_t)(Y * bp + dy) * N + X * bp + dx];
            if (sum / ((double)bp * bp) >= (double)c->min_illum) { valid[2 * nv] = Y; valid[2 * nv + 1] = X; ++nv; }
        }
    if (nv == 0) { free(valid); return SHWFS_EINVAL; }
    pyrwfs_handle *h = new (std::nothrow) pyrwfs_handle();
    if (!h) { free(valid); return SHWFS_ENOMEM; }
    memset(h, 0, sizeof(*h));
    h->N = N; h->Np = Np; h->R = Np == 1024 ? 32 : 16; h->s = s; h->bp = bp; h->Sp = Sp; h->K = c->mod_points;
    h->nvalid = nv; h->h_valid = valid;
    h->r_mod = c->mod_radius; h->D_pix = c->pupil_diameter_px; h->c_phi = c->phase_to_rad;
    const bool modulated = h->K > 0 && h->r_mod > 0.f;
    h->Kp = modulated ? h->K : 1;
    int rc = SHWFS_OK;
    float2 *tw = nullptr, *md = nullptr;
    {
        PY_TRY(cudaGetDevice(&h->device), "cudaGetDevice");
        const size_t per_frame = sizeof(float2) * (size_t)h->Kp * ((size_t)Np * N + (size_t)2 * N * Np) +
                                 sizeof(float) * ((size_t)4 * N * N + (size_t)4 * Sp * Sp);
        size_t chunk = ((size_t)1536 << 20) / per_frame;
        if (chunk < 1) chunk = 1;
        if (chunk > 64) chunk = 64;
        h->chunk = (int)chunk;
        tw = (float2 *)malloc(sizeof(float2) * Np);
        md = (float2 *)malloc(sizeof(float2) * h->Kp);
        if (!tw || !md) { rc = SHWFS_ENOMEM; goto fail; }
        for (int m = 0; m < Np; ++m) {
            const double a = 6.283185307179586476925286766559 * (double)m / (double)Np;
            tw[m] = make_float2((float)cos(a), (float)sin(a));
        }
        for (int k = 0; k < h->Kp; ++k) {
            const double th = 6.283185307179586476925286766559 * ((double)k + 0.5) / (double)h->Kp;
            const double r = modulated ? (double)h->r_mod / (double)h->D_pix : 0.0;
            md[k] = make_float2((float)(r * cos(th)), (float)(r * sin(th)));
        }
        PY_TRY(cudaMalloc(&h->d_amp, sizeof(float) * (size_t)N * N), "cudaMalloc(pyr amplitude)");
        PY_TRY(cudaMemcpy(h->d_amp, c->amplitude, sizeof(float) * (size_t)N * N, cudaMemcpyHostToDevice), "cudaMemcpy");
        PY_TRY(cudaMalloc(&h->d_valid, sizeof(int2) * (size_t)nv), "cudaMalloc(pyr valid)");
        PY_TRY(cudaMemcpy(h->d_valid, valid, sizeof(int2) * (size_t)nv, cudaMemcpyHostToDevice), "cudaMemcpy");
        PY_TRY(cudaMalloc(&h->d_tw, sizeof(float2) * Np), "cudaMalloc(pyr twiddles)");
        PY_TRY(cudaMemcpy(h->d_tw, tw, sizeof(float2) * Np, cudaMemcpyHostToDevice), "cudaMemcpy");
        PY_TRY(cudaMalloc(&h->d_mod, sizeof(float2) * h->Kp), "cudaMalloc(pyr modulation)");
        PY_TRY(cudaMemcpy(h->d_mod, md, sizeof(float2) * h->Kp, cudaMemcpyHostToDevice), "cudaMemcpy");
        PY_TRY(cudaMalloc(&h->d_A1, sizeof(float2) * chunk * h->Kp * Np * N), "cudaMalloc(pyr A1)");
        PY_TRY(cudaMalloc(&h->d_A2, sizeof(float2) * chunk * h->Kp * 2 * N * Np), "cudaMalloc(pyr A2)");
        PY_TRY(cudaMalloc(&h->d_I2, sizeof(float) * chunk * 4 * N * N), "cudaMalloc(pyr I2)");
        PY_TRY(cudaMalloc(&h->d_Q, sizeof(float) * chunk * 4 * Sp * Sp), "cudaMalloc(pyr Q)");
    }
    free(tw); free(md);
    *out = h;
    return SHWFS_OK;
fail:
    free(tw); free(md);
    pyr_free(h);
    return rc;
}

int pyrwfs_destroy(pyrwfs_handle *h)
{
    if (!h) return SHWFS_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != h->device) cudaSetDevice(h->device);
    cudaDeviceSynchronize();
    if (prev >= 0 && prev != h->device) cudaSetDevice(prev);
    pyr_free(h);
    return SHWFS_OK;
}

int pyrwfs_num_pixels(const pyrwfs_handle *h, int32_t *nvalid)
{
    if (!h || !nvalid) return SHWFS_EINVAL;
    *nvalid = h->nvalid;
    return SHWFS_OK;
}

int pyrwfs_valid_list(const pyrwfs_handle *h, int32_t *yx_host)
{
    if (!h || !yx_host) return SHWFS_EINVAL;
    memcpy(yx_host, h->h_valid, sizeof(int32_t) * 2 * (size_t)h->nvalid);
    return SHWFS_OK;
}

int pyrwfs_launch_count(const pyrwfs_handle *h, int64_t *count)
{
    if (!h || !count) return SHWFS_EINVAL;
    *count = h->launches;
    return SHWFS_OK;
}

/* pyrwfs_measure / pyrwfs_debug_quadrants launch on the current device: it has to be the handle's */
static bool pyr_on_device(const pyrwfs_handle *h)
{
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == h->device;
}

int pyrwfs_measure(pyrwfs_handle *h, const float *phase_dev, int32_t T, float *signals_dev, void *cuda_stream)
{
    if (!h || T < 0) return SHWFS_EINVAL;
    if (T == 0) return SHWFS_OK;
    if (!phase_dev || !signals_dev || !pyr_on_device(h)) return SHWFS_EINVAL;
    return pyr_run(h, phase_dev, T, signals_dev, nullptr, (cudaStream_t)cuda_stream);
}

int pyrwfs_debug_quadrants(pyrwfs_handle *h, const float *phase_dev, int32_t T, float *out_dev, void *cuda_stream)
{
    if (!h || T < 0) return SHWFS_EINVAL;
    if (T == 0) return SHWFS_OK;
    if (!phase_dev || !out_dev || !pyr_on_device(h)) return SHWFS_EINVAL;
    return pyr_run(h, phase_dev, T, nullptr, out_dev, (cudaStream_t)cuda_stream);
}

}  // extern "C"
