/*
 * wk_kernel_harness.cpp -- the lag-domain kernels of csrc/wk.cu run WHOLE on the host: wk_table_kernel (H0, the
 * float64 table M), wk_measure_kernel<n, MODE, EXTK> (the headline kernel of configs 3/4: H1 .. H8 of
 * include/shwfs.h, one CTA of n/2 warps per 32 spots, four barrier-fenced phases, second-pass rows of H written over
 * the field buffer) and wk_generic_kernel, cut out of the .cu file as text ("wk_kernel_extract.inc", written by
 * tests/test_kernels_host.py) with the headers they include compiled as they are, on the coroutine SIMT machine of
 * simt.h -- every thread of every CTA, its shared memory, __syncthreads and half-warp shuffles.
 *
 * Likewise wkf_kernel of csrc/wk_fft.cu (config 5's kernel, and what SHWFS_ALGO_AUTO gives one- and two-frame calls at
 * n = 8, 10: the autocorrelation by 32-point FFTs, a half-warp per spot, six steps on one shared-memory tile fenced
 * by __syncwarp only), cut out as "wkf_kernel_extract.inc": the one-tile-per-CTA register-gather instances and the
 * persistent TMA instance with its dynamic deal.  Its table row staging (mrow_stage / mrow_wait of wk_common.cuh:
 * 2n-1 cp.async copies of 8 bytes, inline PTX) is restated below as the plain copies it performs.
 *
 * usage: wk_kernel_harness in.bin out.bin
 *   in.bin   int32[14] {N, n, P, b, T, nsub, mode, has_k, kernel, order, seed, L, grid, lazy_tma}, float[2] {tau, c_phi},
 *            kernel: 0 wk_measure_kernel, 1 wk_generic_kernel, 2 wkf_kernel (one tile per CTA), 3 wkf_kernel (TMA,
 *            persistent, `grid` CTAs)
 *            float sod_q[8], sod_sw[8], phase[T*(L > 0 && !shared ? L : 1)*N*N], amp[N*N],
 *            int32 valid[nsub*2] (sy, sx), float K[has_k ? nsub*P*P : 0], float sod_g[L*nsub*2]
 *            after sod_sw: float[2] {flux, ron}, int32[5] {shared wavefront, photon_model, seed low, seed high, has_dm};
 *            after sod_g: float dm_patch[has_dm ? T*nsub*n*n : 0] (subtracted from the wavefront in H1)
 *   out.bin  slopes[T*nsub*2], binned[T*nsub*D*D], noisy[flux > 0 ? T*nsub*D*D : 0]
 * What the harness supplies itself is what the launchers (host code of wk.cu) do: the WkArgs and the grids.
 * The comparison with the float64 oracle is the Python test's.  Test infrastructure only.
 */
#include "simt.h"

#include "../../paper_1408_0698_b200/csrc/internal.h"
#include "../../paper_1408_0698_b200/csrc/fft_regs.cuh"
#include "../../paper_1408_0698_b200/csrc/field.cuh"
#include "../../paper_1408_0698_b200/csrc/cog.cuh"
#include "../../paper_1408_0698_b200/csrc/noise.cuh"
#include "../../paper_1408_0698_b200/csrc/wk_common.cuh"
#include "../../paper_1408_0698_b200/csrc/sweep.cuh"

namespace {
using namespace shwfs;
#include "wk_kernel_extract.inc"

/* what the cp.async copies of mrow_stage do: entry k of the staged row is M_i[term_lag(k)][ly] */
template <int n>
void host_mrow_stage(const float2 *Mcol, float *dst)
{
    for (int k = 0; k < 2 * n - 1; ++k) reinterpret_cast<float2 *>(dst)[k] = Mcol[term_lag<n>(k) * n];
}
inline void host_mrow_wait() {}
#include "wkf_kernel_extract.inc"

struct Job {
    int N, n, P, b, T, nsub, mode, has_k, kernel, order, seed, L, grid, lazy;
    float tau, c_phi;
    float sod_q[8], sod_sw[8];
    float flux, ron;
    int shared, photon_model;
    unsigned seed_lo, seed_hi;
    int has_dm;
};

template <int n, int MODE, int EXTK>
bool run(const Job &J, const WkArgs &A)
{
    using Cfg = WkCfg<n>;
    const int grid = (A.total + Cfg::SPOTS - 1) / Cfg::SPOTS;
    return simt::launch(grid, Cfg::THREADS, WkSmem<n, (EXTK < 2)>::BYTES, (simt::Order)J.order, (unsigned)J.seed,
                        [&]() { wk_measure_kernel<n, MODE, EXTK>(A); });
}

template <int n>
bool special(const Job &J, const WkArgs &A)
{
    if (A.L > 1) return A.mode == 0 ? run<n, 0, 2>(J, A) : run<n, 1, 2>(J, A);
    if (A.L > 0 || A.flux > 0.f || A.dm_patch != nullptr) return A.mode == 0 ? run<n, 0, 1>(J, A) : run<n, 1, 1>(J, A);
    return A.mode == 0 ? run<n, 0, 0>(J, A) : run<n, 1, 0>(J, A);
}

template <int n, int MODE, int EXTK>
bool run_wkf_ext(const Job &J, const WkArgs &A, const CUtensorMap *map)
{
    return simt::launch((A.total + WF_SPOTS - 1) / WF_SPOTS, WF_THREADS, EXTK == 2 ? 2 * WF_SMEM : WF_SMEM, (simt::Order)J.order,
                        (unsigned)J.seed, [&]() { wkf_kernel<n, MODE, EXTK, false>(A, *map); });
}

template <int n, int MODE>
bool run_wkf(const Job &J, const WkArgs &A, const CUtensorMap *map)
{
    if (A.L > 1) return run_wkf_ext<n, MODE, 2>(J, A, map);
    if (A.L > 0 || A.flux > 0.f || A.dm_patch != nullptr) return run_wkf_ext<n, MODE, 1>(J, A, map);
    if constexpr (n == 16) {
        if (J.kernel == 3)
            return simt::launch(J.grid, WF_THREADS, WF_SMEM + WF_STAGE + 1024, (simt::Order)J.order, (unsigned)J.seed,
                                [&]() { wkf_kernel<n, MODE, 0, true>(A, *map); });
    }
    return simt::launch((A.total + WF_SPOTS - 1) / WF_SPOTS, WF_THREADS, WF_SMEM, (simt::Order)J.order, (unsigned)J.seed,
                        [&]() { wkf_kernel<n, MODE, 0, false>(A, *map); });
}

template <int n>
bool wkf(const Job &J, const WkArgs &A, const CUtensorMap *map)
{
    return A.mode == 0 ? run_wkf<n, 0>(J, A, map) : run_wkf<n, 1>(J, A, map);
}
}  // namespace

int main(int argc, char **argv)
{
    if (argc != 3) return 2;
    static_assert(SHWFS_MAX_LAYERS == 8, "the job header carries 8 sub-layers");
    FILE *f = std::fopen(argv[1], "rb");
    if (!f) return 2;
    Job J;
    if (std::fread(&J, 4, 14, f) != 14 || std::fread(&J.tau, 4, 25, f) != 25) return 2;
    const int D = J.P / J.b, LX = 2 * J.n - 1, layers = J.L > 0 && !J.shared ? J.L : 1;
    const size_t NN = (size_t)J.N * J.N, total = (size_t)J.T * J.nsub;
    std::vector<float> phase(NN * J.T * layers), amp(NN), K(J.has_k ? (size_t)J.nsub * J.P * J.P : 0);
    std::vector<int2> valid(J.nsub);
    std::vector<float2> sod_g((size_t)J.L * J.nsub);
    if (std::fread(phase.data(), 4, phase.size(), f) != phase.size() || std::fread(amp.data(), 4, NN, f) != NN ||
        std::fread(valid.data(), 8, valid.size(), f) != valid.size() || std::fread(K.data(), 4, K.size(), f) != K.size() ||
        std::fread(sod_g.data(), 8, sod_g.size(), f) != sod_g.size()) return 2;
    std::vector<float> dm_patch(J.has_dm ? total * J.n * J.n : 0);      /* [T][nsub][n*n], as dm_phase_kernel leaves it */
    if (std::fread(dm_patch.data(), 4, dm_patch.size(), f) != dm_patch.size()) return 2;
    std::fclose(f);

    /* H0: as shwfs_wk_build_table launches it */
    const int blocks = J.has_k ? J.nsub : 1;
    std::vector<float2> M((size_t)blocks * LX * J.n);
    if (!simt::launch(blocks, 128, J.has_k ? sizeof(double2) * (size_t)J.P * LX : 0, (simt::Order)J.order, (unsigned)J.seed,
                      [&]() { wk_table_kernel(K.data(), J.has_k, J.n, J.P, J.b, M.data()); })) {
        std::printf("FAIL: the table launch dead-locked\n");
        return 1;
    }

    std::vector<float> slopes(total * 2, NAN), binned(total * D * D, NAN);
    WkArgs A;
    std::memset(&A, 0, sizeof(A));
    A.phase = phase.data(); A.amp = amp.data(); A.valid = valid.data(); A.M = M.data();
    A.slopes = slopes.data(); A.binned = binned.data();
    A.frame_stride = (long long)NN;
    A.sod_g = sod_g.data(); A.L = J.L;
    for (int l = 0; l < 8; ++l) { A.sod_q[l] = J.sod_q[l]; A.sod_sw[l] = J.sod_sw[l]; }
    if (J.L > 0 && !J.shared) { A.layer_stride = A.frame_stride; A.frame_stride *= J.L; }
    std::vector<float> noisy(J.flux > 0.f ? total * D * D : 0, NAN);
    A.flux = J.flux; A.ron2 = J.ron * J.ron; A.photon_model = J.photon_model;
    A.key = make_uint2(J.seed_lo, J.seed_hi);
    A.t0 = 0;
    A.noisy = J.flux > 0.f ? noisy.data() : nullptr;
    A.dm_patch = J.has_dm ? dm_patch.data() : nullptr;
    A.T = J.T; A.N = J.N; A.nsub = J.nsub; A.mstride = J.has_k ? LX * J.n : 0;
    A.total = (int)total; A.mode = J.mode;
    A.tau = J.tau;
    A.turns = (float)((double)J.c_phi / 6.283185307179586476925286766559);
    A.ramp_unit = 0.5f / (float)J.P;

    /* the patch table and chunk counters of the handle (api.cu, shwfs_create) */
    std::vector<int2> patch(J.nsub);
    for (int i = 0; i < J.nsub; ++i) {
        const int y0 = valid[i].x * J.n, x0 = valid[i].y * J.n;
        bool lit = true;
        for (int j = 0; j < J.n && lit; ++j)
            for (int k = 0; k < J.n; ++k)
                if (amp[(size_t)(y0 + j) * J.N + x0 + k] != 1.0f) { lit = false; break; }
        patch[i] = make_int2(x0 | (lit ? SHWFS_PATCH_LIT : 0), y0);
    }
    int sched[2] = {0, 0};
    A.patch = patch.data();
    A.sched = sched;
    CUtensorMap map;
    std::memset(&map, 0, sizeof(map));
    const simt::TmaMap tm{phase.data(), J.N, J.T, 16};
    std::memcpy(&map, &tm, sizeof(tm));
    simt::lazy_tma = J.lazy != 0;

    bool ok = false;
    if (J.kernel >= 2) {
        if (D != 16 || (J.kernel == 3 && J.n != 16)) { std::printf("FAIL: no such instance\n"); return 1; }
        switch (J.n) {
        case 8: ok = wkf<8>(J, A, &map); break;
        case 10: ok = wkf<10>(J, A, &map); break;
        case 12: ok = wkf<12>(J, A, &map); break;
        case 14: ok = wkf<14>(J, A, &map); break;
        case 16: ok = wkf<16>(J, A, &map); break;
        default: return 2;
        }
        if (sched[0] != 0 || sched[1] != 0) { std::printf("FAIL: chunk counters not re-armed\n"); return 1; }
        if (!simt::g_pending.empty()) { std::printf("FAIL: a requested box was never waited for\n"); return 1; }
        if (J.kernel == 3 && simt::g_boxes != (long)total) { std::printf("FAIL: %ld boxes for %zu spots\n", simt::g_boxes, total); return 1; }
    } else if (J.kernel == 1) {
        const size_t smem = sizeof(float2) * (size_t)(J.n * J.n + J.n * LX + D) + sizeof(float) * (size_t)(D * D + 3 * GEN_THREADS);
        ok = simt::launch(A.total, GEN_THREADS, smem, (simt::Order)J.order, (unsigned)J.seed,
                          [&]() { wk_generic_kernel(A, J.n, D); });
    } else {
        if (D != 16) { std::printf("FAIL: the specialised kernel is for D = 16\n"); return 1; }
        switch (J.n) {
        case 8: ok = special<8>(J, A); break;
        case 10: ok = special<10>(J, A); break;
        case 16: ok = special<16>(J, A); break;
        default: return 2;
        }
    }
    if (!ok) { std::printf("FAIL: the launch dead-locked\n"); return 1; }

    f = std::fopen(argv[2], "wb");
    if (!f) return 2;
    std::fwrite(slopes.data(), 4, slopes.size(), f);
    std::fwrite(binned.data(), 4, binned.size(), f);
    std::fwrite(noisy.data(), 4, noisy.size(), f);
    std::fclose(f);
    std::printf("ok switches %ld\n", simt::g_switches);
    return 0;
}
