// Kernels and launchers of the smoother; the tile-level device code is in mg_tile_gs.cuh (shared with the
// fused small-level kernel of mg_tail.cu).
#include <algorithm>
#include <cstdlib>

#include "mg_strip_gs.cuh"

namespace mgb {

namespace {

// x_out = S^NS (x_in - [PC] P e_c);  zero: x_in is the zero vector and is not read.
// EPI = 1: additionally d_c = R (A x_out - b) on the next coarser level (ccode = its point codes, dc = d_c).
// EPI = 2: additionally w = A x_out (dc = w).
// BX x BY < tile: several CTAs per tile (blockIdx = tile * blocks-per-tile + block).
template <int NS, bool PC, int EPI, int BX, int BY, int XIM>
__global__ void __launch_bounds__(GT, 2) k_gs(LevelDev lv, VecRef xin_r, VecRef xout_r, VecRef b_r, const double* __restrict__ ec,
                                              int xin_zero, const uint16_t* __restrict__ ccode, double* __restrict__ dc,
                                              const int* __restrict__ stop, const int* __restrict__ tlist) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int pl = blockIdx.y;
    if (stopped(stop, pl)) return;
    lv = plane_of(lv, pl);
    const int64_t cps = (int64_t)(lv.ntiles_coarse + 1) * TS;      // plane stride of the next coarser level
    if (PC) ec += pl * cps;
    if (EPI == 1) dc += pl * cps; else if (EPI == 2) dc += pl * lv.nslots;
    constexpr int NBX = TX / BX, NSUB = NBX * (TY / BY);
    const int ti = blockIdx.x / NSUB, sub = blockIdx.x - ti * NSUB;
    const int t = tlist != nullptr ? tlist[ti] : ti;            // the launch covers a list of tiles, or all of them
    gs_tile<NS, PC, false, EPI, BX, BY, XIM>(lv, t, resolve(xin_r, pl), resolve(xout_r, pl), resolve(b_r, pl), ec, xin_zero, smem_raw, nullptr, ccode, dc,
                                       (sub % NBX) * BX, (sub / NBX) * BY);
}

__global__ void k_copy(VecRef sr, VecRef dr, int64_t n) {
    const double* __restrict__ s = resolve(sr, blockIdx.y);
    double* __restrict__ d = resolve(dr, blockIdx.y);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) d[k] = s[k];
}

// Levels of at most SUB_MAX_TILES tiles are latency bound (7-25 us per launch whatever the tile count,
// profiles/r01c_small_levels.md): they run with one CTA per SBX x SBY block, 8 CTAs per tile.
constexpr int SBX = 16, SBY = 16;      // 8 CTAs per tile: levels of at most 40 tiles on 148 SMs (sms * 10 / 37)
constexpr int MBX = 32, MBY = 16;      // 4 CTAs per tile: at most one wave at 2 CTAs per SM (tiles <= sms / 2)
constexpr int HBX = 64, HBY = 16;      // 2 CTAs per tile: one wave up to `sms` tiles

// cost of a general tile in units of an interior tile, per fused variant (measured on config 4, B200): k = 0 sweeps + defect + restriction,
// 1 correction + sweeps, 2 correction + sweeps + apply, 3 plain sweeps.  MG_B200_STRIP_GEN_COST_<k> overrides (tuning runs).
inline double strip_gen_cost(int k) {
    static double v[4] = {-1.0, -1.0, -1.0, -1.0};
    static const double dflt[4] = {2.5, 2.5, 2.5, 2.5};
    if (v[k] < 0.0) {
        const char* names[4] = {"MG_B200_STRIP_GEN_COST_0", "MG_B200_STRIP_GEN_COST_1", "MG_B200_STRIP_GEN_COST_2", "MG_B200_STRIP_GEN_COST_3"};
        const char* e = getenv(names[k]);
        v[k] = e ? atof(e) : dflt[k];
    }
    return v[k];
}
inline bool no_strips() { static const bool v = getenv("MG_B200_NO_STRIPS") != nullptr; return v; }

template <int NS, bool PC, int EPI, int BX, int BY, int XIM>
void launch_blk_x(const Launch& L, const LevelDev& lv, VecRef xin, VecRef xout, VecRef b, const double* ec, bool zero,
                  const uint16_t* ccode, double* dc) {
    constexpr size_t smem = Geo<NS, PC, EPI, BX, BY>::SMEM;
    ensure_dyn_smem((const void*)k_gs<NS, PC, EPI, BX, BY, XIM>, smem);
    if (XIM != 2 && BX == TX && BY == TY && !no_strips()) {
        // large level: interior and general tiles by the register-tiled kernel, guard-list overflow tiles by the tile code.  Halos
        // (even: column pairs): interior 2 NS + epilogue (2 defect restriction, 1 apply), general 3 NS + 1 (correction) + epilogue
        constexpr int EH = EPI == 1 ? 2 : (EPI == 2 ? 1 : 0);
        constexpr int SH = (2 * NS + EH + 1) / 2 * 2, GH = (3 * NS + (PC ? 1 : 0) + EH + 1) / 2 * 2;
        constexpr int K = SH <= 4 ? 0 : 1;                  // work lists: interior = all inner within 4 (K = 0) / 6 (K = 1) cells of the tile
        static_assert(SH <= 6 && GH <= 8, "work lists and the overflow rule cover halos up to 6 / 8");
        const int nint = lv.nint[K], ngen = lv.ngen[K], novf = lv.ntiles - nint - ngen, sms = dev_info().sms;
        if (novf > 0) {
            k_gs<NS, PC, EPI, BX, BY, XIM><<<dim3(novf, L.planes), GT, smem, L.stream>>>(lv, xin, xout, b, ec, zero ? 1 : 0, ccode, dc, L.stop, lv.tlist[K] + nint + ngen);
            if (L.counter) *L.counter += 1;
        }
        if (nint + ngen > 0) {
            // one launch: the first ggen CTAs walk the general tiles, the rest the interior tiles; a general tile costs
            // about STRIP_GEN_COST interior ones (wider halo, boundary phases), the SMs are split in that proportion
            using SI = SGeo<SH>; using SGG = SGeo<GH>;
            constexpr size_t ssm = std::max(SI::smem(PC, false), SGG::smem(PC, true));
            constexpr int nthreads = std::max(SI::NT, SGG::NT);
            const int grid = (int)std::min<int64_t>(sms, (int64_t)(nint + ngen) * L.planes);
            int ggen = 0;
            if (ngen > 0) {
                const double wg = ngen * strip_gen_cost(EPI == 1 ? 0 : (PC ? (EPI == 2 ? 2 : 1) : 3));
                ggen = std::max(1, std::min(ngen * L.planes, (int)(grid * wg / (wg + nint) + 0.5)));
                if (nint > 0) ggen = std::min(ggen, grid - 1);
            }
            if (L.planes > 1) {
                ensure_dyn_smem((const void*)k_gs_strip<NS, SH, GH, PC, EPI, true, XIM == 1>, ssm);
                k_gs_strip<NS, SH, GH, PC, EPI, true, XIM == 1><<<grid, nthreads, ssm, L.stream>>>(lv, lv.smeta[K], nint, lv.smeta[K] + (size_t)SMETA * nint, ngen, ggen, L.planes,
                                                                                      xin, xout, b, ec, zero ? 1 : 0, ccode, dc, L.stop);
            } else {
                ensure_dyn_smem((const void*)k_gs_strip<NS, SH, GH, PC, EPI, false, XIM == 1>, ssm);
                k_gs_strip<NS, SH, GH, PC, EPI, false, XIM == 1><<<grid, nthreads, ssm, L.stream>>>(lv, lv.smeta[K], nint, lv.smeta[K] + (size_t)SMETA * nint, ngen, ggen, 1,
                                                                                       xin, xout, b, ec, zero ? 1 : 0, ccode, dc, L.stop);
            }
            if (L.counter) *L.counter += 1;
        }
        return;
    }
    const int grid = lv.ntiles * (TX / BX) * (TY / BY);
    k_gs<NS, PC, EPI, BX, BY, XIM><<<dim3(grid, L.planes), GT, smem, L.stream>>>(lv, xin, xout, b, ec, zero ? 1 : 0, ccode, dc, L.stop, nullptr);
    if (L.counter) *L.counter += 1;
}

// two-field form (xi = 1): kernels compiled without xi; three-field form (Eq. 3): with it
template <int NS, bool PC, int EPI, int BX, int BY>
void launch_blk(const Launch& L, const LevelDev& lv, VecRef xin, VecRef xout, VecRef b, const double* ec, bool zero,
                const uint16_t* ccode, double* dc) {
    if (lv.xi != nullptr) launch_blk_x<NS, PC, EPI, BX, BY, 1>(L, lv, xin, xout, b, ec, zero, ccode, dc);
    else launch_blk_x<NS, PC, EPI, BX, BY, 0>(L, lv, xin, xout, b, ec, zero, ccode, dc);
}

template <int NS, bool PC, int EPI = 0>
void launch_ns(const Launch& L, const LevelDev& lv, VecRef xin, VecRef xout, VecRef b, const double* ec, bool zero,
               const uint16_t* ccode = nullptr, double* dc = nullptr) {
    static const bool no_sub = getenv("MG_B200_NO_SUBBLOCKS") != nullptr;
    const int sms = dev_info().sms;
    const int SUB_MAX_TILES = sms * 10 / 37, MID_MAX_TILES = sms / 2, HALF_MAX_TILES = sms;
    // layout study (profiles/r02_layout.md): MG_B200_FORCE_BLOCK = 1 / 2 / 3 / 4 forces 16x16 / 32x16 / 64x16 / whole-tile CTAs of the
    // shared-memory tile code on every level
    static const int force = getenv("MG_B200_FORCE_BLOCK") ? atoi(getenv("MG_B200_FORCE_BLOCK")) : 0;
    if (force == 1) return launch_blk<NS, PC, EPI, SBX, SBY>(L, lv, xin, xout, b, ec, zero, ccode, dc);
    if (force == 2) return launch_blk<NS, PC, EPI, MBX, MBY>(L, lv, xin, xout, b, ec, zero, ccode, dc);
    if (force == 3) return launch_blk<NS, PC, EPI, HBX, HBY>(L, lv, xin, xout, b, ec, zero, ccode, dc);
    const int64_t nt = (int64_t)lv.ntiles * L.planes;       // tiles of all planes: what fills the machine
    if (nt <= SUB_MAX_TILES && !no_sub) launch_blk<NS, PC, EPI, SBX, SBY>(L, lv, xin, xout, b, ec, zero, ccode, dc);
    else if (nt <= MID_MAX_TILES && !no_sub) launch_blk<NS, PC, EPI, MBX, MBY>(L, lv, xin, xout, b, ec, zero, ccode, dc);
    else if (nt <= HALF_MAX_TILES && !no_sub) launch_blk<NS, PC, EPI, HBX, HBY>(L, lv, xin, xout, b, ec, zero, ccode, dc);
    else launch_blk<NS, PC, EPI, TX, TY>(L, lv, xin, xout, b, ec, zero, ccode, dc);
}

}  // namespace

void launch_gs_fused(const Launch& L, const LevelDev& lv, VecRef x_in, VecRef x_out, VecRef b, int sweeps, bool x_in_zero,
                     const LevelDev* coarse, double* d_coarse, double* w_out) {
    if (coarse != nullptr) {                                  // + restricted defect of the result
        if (sweeps == 2) launch_ns<2, false, 1>(L, lv, x_in, x_out, b, nullptr, x_in_zero, coarse->code, d_coarse);
        else launch_ns<1, false, 1>(L, lv, x_in, x_out, b, nullptr, x_in_zero, coarse->code, d_coarse);
        return;
    }
    if (w_out != nullptr) {                                   // + w = A x_out
        if (sweeps == 2) launch_ns<2, false, 2>(L, lv, x_in, x_out, b, nullptr, x_in_zero, nullptr, w_out);
        else launch_ns<1, false, 2>(L, lv, x_in, x_out, b, nullptr, x_in_zero, nullptr, w_out);
        return;
    }
    if (sweeps == 2) launch_ns<2, false>(L, lv, x_in, x_out, b, nullptr, x_in_zero);
    else launch_ns<1, false>(L, lv, x_in, x_out, b, nullptr, x_in_zero);
}

void launch_gs_correct(const Launch& L, const LevelDev& lv, const double* e_coarse, VecRef x_in, VecRef x_out, VecRef b, int sweeps,
                       double* w_out) {
    if (w_out != nullptr) {                                   // + w = A x_out
        if (sweeps == 2) launch_ns<2, true, 2>(L, lv, x_in, x_out, b, e_coarse, false, nullptr, w_out);
        else launch_ns<1, true, 2>(L, lv, x_in, x_out, b, e_coarse, false, nullptr, w_out);
        return;
    }
    if (sweeps == 2) launch_ns<2, true>(L, lv, x_in, x_out, b, e_coarse, false);
    else launch_ns<1, true>(L, lv, x_in, x_out, b, e_coarse, false);
}

void launch_copy(const Launch& L, VecRef src, VecRef dst, int64_t n) {
    k_copy<<<dim3((int)std::min<int64_t>((n + 255) / 256, dev_info().sms * 8), L.planes), 256, 0, L.stream>>>(src, dst, n);
    if (L.counter) *L.counter += 1;
}

}  // namespace mgb
