// Tile-level device code of the operator rows (rules D1-D3) and of the fused defect + full-weighting
// restriction, shared by the kernels of mg_kernels.cu and the fused small-level kernel of mg_tail.cu.
#pragma once
#include "mg_device.h"

namespace mgb {
namespace {

#ifndef MGB_LDV
#define MGB_LDV
template <bool COH>
__device__ __forceinline__ double ldv(const double* p) { return COH ? __ldca(p) : __ldg(p); }
#endif

constexpr int NT = 512;                 // threads per CTA: 64 x 8, four rows per thread
constexpr int ROWS_PER_PASS = NT / TX;  // 8

// slot of the point at local offset (lx, ly) in [-TX, 2TX) x [-TY, 2TY) relative to tile whose 3x3
// neighbour table is tn[9]
__device__ __forceinline__ int64_t nslot(const int* tn, int lx, int ly) {
    const int ox = (lx < 0) ? -1 : (lx >= TX ? 1 : 0);
    const int oy = (ly < 0) ? -1 : (ly >= TY ? 1 : 0);
    return (int64_t)tn[(oy + 1) * 3 + ox + 1] * TS + (ly - oy * TY) * TX + (lx - ox * TX);
}

// Rule D3 / Eq. 14-16: upstream value of a Neumann guard. Returns sum over non-self nodes of w*x,
// the weight on the point itself and the distance delta = h |n| (h for the fallback).
__device__ __forceinline__ void neumann_row(uint16_t code, const int* tn, int lx, int ly, const double* __restrict__ x,
                                            double h, double& sum, double& wself, double& delta) {
    const int tnR = ((code >> 2) & 7) - 2, tnZ = ((code >> 5) & 7) - 2;
    sum = 0.0; wself = 0.0;
    if (code & (1 << 8)) {                                  // fallback: mean of the inner 4-neighbours
        const int mask = (code >> 9) & 15;
        if (mask & 1) sum += x[nslot(tn, lx - 1, ly)];
        if (mask & 2) sum += x[nslot(tn, lx + 1, ly)];
        if (mask & 4) sum += x[nslot(tn, lx, ly - 1)];
        if (mask & 8) sum += x[nslot(tn, lx, ly + 1)];
        sum = sum / (double)__popc(mask);
        delta = h;
        return;
    }
    int ox[2], oy[2], nx, ny; double wx, wy;
    if (tnR & 1) { nx = 2; ox[0] = 0; ox[1] = tnR; wx = 0.5; } else { nx = 1; ox[0] = tnR / 2; ox[1] = 0; wx = 1.0; }
    if (tnZ & 1) { ny = 2; oy[0] = 0; oy[1] = tnZ; wy = 0.5; } else { ny = 1; oy[0] = tnZ / 2; oy[1] = 0; wy = 1.0; }
    const double w = wx * wy;
    for (int b = 0; b < ny; b++)
        for (int a = 0; a < nx; a++) {
            if (ox[a] == 0 && oy[b] == 0) { wself += w; continue; }
            sum += w * x[nslot(tn, lx + ox[a], ly + oy[b])];
        }
    delta = h * sqrt(0.25 * (double)(tnR * tnR + tnZ * tnZ));
}

// ---------------------------------------------------------------------------------- S1 apply / residual
// (A x) at cell (lx, ly) of tile t (slot s), rules D1-D3.  Neighbours inside the tile are s +- 1, s +- TX;
// only the tile-edge lanes go through the neighbour table.
// Inner row of rule D1 with every load issued unconditionally (all neighbour slots exist in memory: missing
// tiles map to the null tile), so that the loads of all cells a thread handles overlap.
struct Nb4 { int w, e, s, n; };   // ids of the W, E, S, N neighbour tiles, held in registers (branch-free edge handling)
__device__ __forceinline__ Nb4 nb4(const int* tn) { return Nb4{tn[3], tn[5], tn[1], tn[7]}; }
__device__ __forceinline__ Nb4 nbr4(const int* r) { return Nb4{r[0], r[1], r[2], r[3]}; }   // packed W, E, S, N

template <bool COH>
__device__ __forceinline__ double inner_row(const LevelDev& lv, const Nb4 nb, int lx, int ly, int64_t s, const double* __restrict__ x) {
    const int64_t eW = (int64_t)nb.w * TS + ly * TX + (TX - 1), eE = (int64_t)nb.e * TS + ly * TX;
    const int64_t eS = (int64_t)nb.s * TS + (TY - 1) * TX + lx, eN = (int64_t)nb.n * TS + lx;
    const int64_t sW = (lx > 0) ? s - 1 : eW;
    const int64_t sE = (lx < TX - 1) ? s + 1 : eE;
    const int64_t sS = (ly > 0) ? s - TX : eS;
    const int64_t sN = (ly < TY - 1) ? s + TX : eN;
    const double cl = __ldg(lv.c + s);
    const double kap = lv.xi ? lv.kappa * __ldg(lv.xi + s) : lv.kappa;     // xi_{i,j} / (2 h^2), Eq. 10
    const double aW = kap * (cl + __ldg(lv.c + sW)), aE = kap * (cl + __ldg(lv.c + sE));
    const double aS = kap * (cl + __ldg(lv.c + sS)), aN = kap * (cl + __ldg(lv.c + sN));
    const double xl = ldv<COH>(x + s);                                     // difference form (rule D1)
    return row_d1(__ldg(lv.lam + s), xl, aW, ldv<COH>(x + sW), aE, ldv<COH>(x + sE), aS, ldv<COH>(x + sS), aN, ldv<COH>(x + sN));
}

// ---------------------------------------------------------------------------------- S1 + S3 fused
// d_c = R (A x - b): one CTA per COARSE tile computes the defect of the (2 TX + 1) x (2 TY + 1) fine cells it
// needs into shared memory (never to HBM), then every coarse inner point gathers its 3 x 3 full-weighting
// stencil (rule T2: fine non-inner points contribute 0, coarse guard rows are 0).
constexpr int DRW = 2 * TX + 1, DRH = 2 * TY + 1, DRS = DRW + 1;      // fine x in [-1, 2TX), y in [-1, 2TY); padded row
constexpr size_t DR_SMEM = (size_t)DRH * DRS * sizeof(double);

template <bool COH>
__device__ __forceinline__ double defect_cell(const LevelDev& fine, const Nb4 tn, int ft, int lx, int ly, const double* __restrict__ x,
                                              const double* __restrict__ b) {
    const int64_t s = (int64_t)ft * TS + ly * TX + lx;
    const uint16_t code = __ldg(fine.code + s);
    const double d = inner_row<COH>(fine, tn, lx, ly, s, x) - ldv<COH>(b + s);
    return ((code & 3) == C_INNER) ? d : 0.0;
}

template <bool COH>
__device__ __forceinline__ void defect_restrict_tile(const LevelDev& fine, const LevelDev& coarse, int t, const double* __restrict__ x,
                                                     const double* __restrict__ b, double* __restrict__ dc, unsigned char* smem_raw,
                                                     const int* meta = nullptr) {
    double* sd = reinterpret_cast<double*>(smem_raw);
    __shared__ int ct[9];
    __shared__ int ftn[4][9];
    const int tid = threadIdx.x;
    __syncthreads();
    if (meta != nullptr) {                 // tables preloaded by the caller (fused small-level kernel)
        if (tid < 9) ct[tid] = meta[META_CT + tid];
        if (tid < 36) ftn[tid / 9][tid % 9] = meta[META_FTN + tid];
    } else {
        if (tid < 9) ct[tid] = coarse.ctab[9 * t + tid];
        __syncthreads();
        if (tid < 36) {
            const int q = tid / 9, k = tid - 9 * q;
            const int ft = ct[((q >> 1) + 1) * 3 + (q & 1) + 1];
            ftn[q][k] = (ft == coarse.ntiles_fine) ? ft : fine.tnb[9 * ft + k];   // the null tile has no table (and is never used)
        }
    }
    __syncthreads();
    const int lx = tid % TX;
    // the 2 x 2 fine tiles under the coarse tile
#pragma unroll
    for (int q = 0; q < 4; q++) {
        const int qx = q & 1, qy = q >> 1;
        const int ft = ct[(qy + 1) * 3 + qx + 1];
        const Nb4 nbq = nb4(ftn[q]);
        double dv[TY / ROWS_PER_PASS];
#pragma unroll
        for (int p = 0; p < TY / ROWS_PER_PASS; p++) dv[p] = defect_cell<COH>(fine, nbq, ft, lx, tid / TX + p * ROWS_PER_PASS, x, b);
#pragma unroll
        for (int p = 0; p < TY / ROWS_PER_PASS; p++) sd[(qy * TY + tid / TX + p * ROWS_PER_PASS + 1) * DRS + qx * TX + lx + 1] = dv[p];
    }
    // west column (fine x = -1) and south row (fine y = -1): cells of the neighbouring fine tiles
    if (tid < DRH) {
        const int fy = tid - 1;
        const int cy = fy < 0 ? 0 : (fy < TY ? 1 : 2);
        const int ft = ct[cy * 3 + 0];
        sd[tid * DRS] = (ft == coarse.ntiles_fine) ? 0.0 : defect_cell<COH>(fine, meta != nullptr ? nbr4(meta + META_RING + 4 * cy) : nb4(fine.tnb + 9 * ft), ft, TX - 1, fy - (cy - 1) * TY, x, b);
    } else if (tid >= 128 && tid < 128 + 2 * TX) {
        const int fx = tid - 128;
        const int cx = fx < TX ? 1 : 2;
        const int ft = ct[cx];
        sd[fx + 1] = (ft == coarse.ntiles_fine) ? 0.0 : defect_cell<COH>(fine, meta != nullptr ? nbr4(meta + META_RING + 4 * (2 + cx)) : nb4(fine.tnb + 9 * ft), ft, fx - (cx - 1) * TX, TY - 1, x, b);
    }
    __syncthreads();
#pragma unroll
    for (int p = 0; p < TY / ROWS_PER_PASS; p++) {
        const int ly = tid / TX + p * ROWS_PER_PASS;
        const int64_t s = (int64_t)t * TS + ly * TX + lx;
        double acc = 0.0;
        if ((coarse.code[s] & 3) == C_INNER) {
#pragma unroll
            for (int dy = -1; dy <= 1; dy++)
#pragma unroll
                for (int dx = -1; dx <= 1; dx++) {
                    const double w = (dx == 0 ? 2.0 : 1.0) * (dy == 0 ? 2.0 : 1.0) * 0.0625;
                    acc += w * sd[(2 * ly + dy + 1) * DRS + 2 * lx + dx + 1];
                }
        }
        dc[s] = acc;
    }
}

}  // namespace
}  // namespace mgb
