// S6, optional (MG_SETUP_FUSED_TAIL): the small levels of the V-cycle in ONE cooperative kernel.  The steps of
// all levels >= s0 (smoothing, defect + restriction, coarsest solve, correction + smoothing) are a short
// program (TailProgram) interpreted by a grid that stays resident: one CTA per tile, grid.sync() between
// steps instead of kernel boundaries.  Measured on B200 (profiles/r01c_small_levels.md): a step on one tile
// takes 7-16 us of single-SM work however it is launched, so removing the ~2 us launch gaps does not pay for
// the lower occupancy of the cooperative kernel; the unfused graph is the default.  The tile-level device code is exactly the one the
// stand-alone kernels use (mg_tile_gs.cuh, mg_tile_ops.cuh), so results are bit-identical to the
// unfused path.  (The paper sends the coarsest system to the CPU at every cycle, and
// reports the small levels + transfers as ~30 % of kernel time.)
#include <cooperative_groups.h>

#include "mg_tile_gs.cuh"
#include "mg_tile_ops.cuh"

namespace cg = cooperative_groups;

namespace mgb {

namespace {

__device__ __forceinline__ double* tail_ptr(double* p, double* topx, double* topb) {
    return p == TAIL_TOPX ? topx : (p == TAIL_TOPB ? topb : p);
}

template <int NS, bool PC, bool DR>
__device__ __forceinline__ void tail_gs(const LevelDev& lv, const TailOp& op, const double* xin, double* xout, const double* b,
                                        unsigned char* smem, const int* meta, const uint16_t* ccode) {
    if ((int)blockIdx.x < op.ntiles) gs_tile<NS, PC, true, DR>(lv, blockIdx.x, xin, xout, b, op.ec, op.zero, smem, meta, ccode, op.dc);
}

// The grid has one CTA per tile of the largest level involved, so on every level a CTA owns at most the tile
// t = blockIdx.x.  All tile tables it will ever need are fetched once, up front, in one wave of
// independent loads: afterwards a step costs one batch of vector loads, the on-chip work and the grid barrier.
__global__ void __launch_bounds__(GT, 1) k_tail(const LevelDev* __restrict__ levs, int s0, int nlev, TailProgram prog, TailCoarse cs,
                                                VecRef topx_r, VecRef topb_r, const int* __restrict__ stop) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ LevelDev slev[TAIL_MAX_LEVELS];
    __shared__ int smeta[TAIL_MAX_LEVELS][META_INTS];
    if (stop != nullptr && *stop) return;          // uniform over the grid: nobody reaches a grid.sync()
    cg::grid_group grid = cg::this_grid();
    const int tid = threadIdx.x, t = blockIdx.x;
    {   // ---- preload: level descriptors, then the tables of tile t on every level
        const int nl = nlev - s0;
        constexpr int LW = sizeof(LevelDev) / 4;
        for (int k = tid; k < nl * LW; k += GT) reinterpret_cast<int*>(slev)[k] = reinterpret_cast<const int*>(levs + s0)[k];
        __syncthreads();
        for (int k = tid; k < nl * META_INTS; k += GT) {
            const int li = k / META_INTS, m = k - li * META_INTS;
            const LevelDev& lv = slev[li];
            int v = 0;
            if (t < lv.ntiles) {
                if (m < META_PT) v = lv.tnb[9 * t + m];
                else if (m < META_ODD) { if (li + 1 < nl) v = lv.ptab[9 * t + (m - META_PT)]; }
                else if (m < META_FLAG) v = lv.tij[2 * t + (m - META_ODD)] & 1;
                else if (m == META_FLAG) v = lv.tflag[t];
                else if (li > 0) {                 // this tile as the coarse side; the fine level is li - 1
                    const LevelDev& fl = slev[li - 1];
                    if (m < META_FTN) v = lv.ctab[9 * t + (m - META_CT)];
                    else if (m < META_RING) {
                        const int q = (m - META_FTN) / 9, kk = (m - META_FTN) - 9 * q;
                        const int ft = lv.ctab[9 * t + ((q >> 1) + 1) * 3 + (q & 1) + 1];
                        v = (ft == lv.ntiles_fine) ? ft : fl.tnb[9 * ft + kk];
                    } else if (m < META_RING + 20) {
                        const int r = (m - META_RING) / 4, d = (m - META_RING) - 4 * r;
                        const int cti = r == 0 ? 0 : (r == 1 ? 3 : (r == 2 ? 6 : (r == 3 ? 1 : 2)));   // SW, W, W', S, S'
                        const int ft = lv.ctab[9 * t + cti];
                        const int nbi = d == 0 ? 3 : (d == 1 ? 5 : (d == 2 ? 1 : 7));                  // W, E, S, N
                        v = (ft == lv.ntiles_fine) ? ft : fl.tnb[9 * ft + nbi];
                    }
                }
            }
            smeta[li][m] = v;
        }
        __syncthreads();
    }
    double* topx = topx_r.base ? resolve(topx_r) : nullptr;
    double* topb = topb_r.base ? resolve(topb_r) : nullptr;
    for (int i = 0; i < prog.nops; i++) {
        const TailOp op = prog.op[i];
        const LevelDev& lv = slev[op.level - s0];
        const int* meta = smeta[op.level - s0];
        double* a = tail_ptr(op.a, topx, topb);
        double* b = tail_ptr(op.b, topx, topb);
        double* c = tail_ptr(op.c, topx, topb);
        if (op.type == TAIL_GS) {                  // a = x_in, b = x_out, c = right-hand side
            const uint16_t* ccode = op.pc == 2 ? slev[op.level + 1 - s0].code : nullptr;
            if (op.ns == 2) {
                if (op.pc == 1) tail_gs<2, true, false>(lv, op, a, b, c, smem_raw, meta, ccode);
                else if (op.pc == 2) tail_gs<2, false, true>(lv, op, a, b, c, smem_raw, meta, ccode);
                else tail_gs<2, false, false>(lv, op, a, b, c, smem_raw, meta, ccode);
            } else {
                if (op.pc == 1) tail_gs<1, true, false>(lv, op, a, b, c, smem_raw, meta, ccode);
                else if (op.pc == 2) tail_gs<1, false, true>(lv, op, a, b, c, smem_raw, meta, ccode);
                else tail_gs<1, false, false>(lv, op, a, b, c, smem_raw, meta, ccode);
            }
        } else if (op.type == TAIL_DR) {           // a = x, c = right-hand side (fine), b = restricted defect (coarse)
            if (t < op.ntiles) defect_restrict_tile<true>(lv, slev[op.level + 1 - s0], t, a, c, b, smem_raw, smeta[op.level + 1 - s0]);
        } else if (op.type == TAIL_COARSE) {       // b = A^-1 a on the coarsest level (rule C)
            if (t == 0) {
                const int n = cs.n;
                double* sb = reinterpret_cast<double*>(smem_raw);
                __syncthreads();
                for (int r = tid; r < n; r += blockDim.x) sb[r] = __ldca(a + cs.cslot[r]);
                __syncthreads();
                const int warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
                for (int r = warp; r < n; r += nw) {
                    double acc = 0.0;
                    for (int k = lane; k < n; k += 32) acc += cs.Ainv[(size_t)r * n + k] * sb[k];
                    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
                    if (lane == 0) b[cs.cslot[r]] = acc;
                }
            }
        } else {                                   // TAIL_COPY: b = a
            for (int64_t k = (int64_t)blockIdx.x * blockDim.x + tid; k < op.n; k += (int64_t)gridDim.x * blockDim.x) b[k] = __ldca(a + k);
        }
        grid.sync();
    }
}

size_t tail_smem() {
    size_t m = DR_SMEM;
    m = std::max(m, Geo<2, true>::SMEM_COH);
    m = std::max(m, Geo<2, false>::SMEM_COH);
    m = std::max(m, Geo<1, true>::SMEM_COH);
    m = std::max(m, Geo<1, false>::SMEM_COH);
    m = std::max(m, Geo<2, false, 1>::SMEM_COH);
    m = std::max(m, Geo<1, false, 1>::SMEM_COH);
    return m;
}

}  // namespace

int tail_max_grid() {
    // per device: the caller (mg_setup) stores the result in the handle
    const size_t smem = tail_smem();
    if (ensure_dyn_smem((const void*)k_tail, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    int per_sm = 0;
    if (!dev_info().coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_tail, GT, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    return per_sm * dev_info().sms;
}

cudaError_t launch_tail(const Launch& L, const LevelDev* d_levs, int s0, int nlev, const TailProgram& prog, const TailCoarse& cs,
                        VecRef topx, VecRef topb, int grid) {
    if (nlev - s0 > TAIL_MAX_LEVELS) return cudaErrorInvalidValue;
    const LevelDev* levs = d_levs;
    TailProgram p = prog;
    TailCoarse c = cs;
    const int* stop = L.stop;
    void* args[] = {(void*)&levs, (void*)&s0, (void*)&nlev, (void*)&p, (void*)&c, (void*)&topx, (void*)&topb, (void*)&stop};
    cudaError_t e = cudaLaunchCooperativeKernel((const void*)k_tail, dim3(grid), dim3(GT), args, tail_smem(), L.stream);
    if (L.counter) *L.counter += 1;
    return e;
}

}  // namespace mgb
