// S2 (+S4): red-black-boundary Gauss-Seidel (gauss_seidel_rbb), NS full sweeps fused into
// ONE pass over memory, optionally preceded in the same pass by the coarse-grid correction
// x <- x - P e_c with set_bnds_hom (rule T3).
//
// One CTA per tile loads the tile plus a halo of H cells of x, c and the point codes into shared memory,
// then runs red / black / boundary phases entirely on-chip; the region in which values are valid shrinks by
// one cell per phase (temporal blocking), halo cells are recomputed redundantly with exactly the
// arithmetic the owning CTA uses, so the result does not depend on the tiling.  x is double-buffered
// (x_in -> x_out): a neighbouring CTA may still be reading the old values.
//
// Shared-memory layout is COLOUR-SPLIT: cell (rx, ry) of the region lives at
// colour * NC + ry * RWC + (rx >> 1), colour = (rx + ry) & 1, so that a warp updating 32 consecutive red
// cells reads its W/E/S/N black neighbours at unit stride (no bank conflicts, no stride-2 access).
// Every thread owns a FIXED set of cells (ROUNDS per colour) for the whole kernel: b and 1/a_ll of its
// inner cells stay in registers across all sweeps, the phase geometry is compile-time, and guard cells
// are collected once into a compact list, so the colour phases contain no global loads, no integer
// divisions and no fp64 divisions.
//
// HBM traffic per point and launch: x in 8 (0 when x_in is known to be zero) + c 8 + b 8 + lambda 8 +
// x out 8 + code 2 (+ e_c 2 with the fused correction), against 64 B per sweep of the three-loop
// formulation.
#pragma once
#include "mg_device.h"

namespace mgb {
namespace {

// Vector loads: read-only path (ld.global.nc) in the stand-alone kernels; in the fused small-level kernel the
// vectors are written by other CTAs earlier in the SAME launch, so they take ordinary coherent loads (ld.global.ca; grid.sync() orders them).
#ifndef MGB_LDV
#define MGB_LDV
template <bool COH>
__device__ __forceinline__ double ldv(const double* p) { return COH ? __ldca(p) : __ldg(p); }
#endif

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// XIM: how the tile code learns whether the level carries the paper's third field xi (Eq. 3):
// 0 two-field form, 1 three-field form (both compile-time, so the two-field kernels carry no trace of xi),
// 2 decided at run time from lv.xi (fused small-level kernel, latency bound).
template <int XIM>
__device__ __forceinline__ bool has_xi(const LevelDev& lv) { return XIM == 2 ? (lv.xi != nullptr) : (XIM == 1); }

constexpr int GT = 512;     // threads per CTA
constexpr int GCAP = GUARD_CAP;   // guard-list capacity per CTA; beyond it the guard phase scans the owned cells

// EPI: epilogue after the sweeps.  1 (DR): the launch also restricts the defect of its result (needs x two cells beyond
// the tile).  2 (AP): the launch also writes w = A x_out (needs one cell beyond the tile): the operator apply of the
// Arnoldi step, fused into the last smoothing launch of the preconditioner cycle.
// BX x BY: the block of the tile one CTA produces (the whole tile, or a sub-block on small levels where
// latency, not throughput, decides: more CTAs per tile).
template <int NS, bool PC, int EPI = 0, int BX = TX, int BY = TY>
struct Geo {
    static constexpr int H = 3 * NS + (PC ? 1 : 0) + (EPI == 1 ? 2 : (EPI == 2 ? 1 : 0));
    static constexpr int RW = BX + 2 * H;
    static constexpr int RH = BY + 2 * H;
    static constexpr int BW = BX, BH = BY;
    static constexpr int RWC = RW / 2;              // cells per colour and row
    static constexpr int NC = RH * RWC;             // cells per colour
    static constexpr int RN = 2 * NC;
    static constexpr int ROUNDS = (NC + GT - 1) / GT;
    static constexpr size_t SMEM = (size_t)RN * (2 * sizeof(double) + sizeof(uint16_t)) + (size_t)GCAP * (sizeof(double) + sizeof(uint16_t));
    // the batched staging of the fused small-level kernel keeps the prolongated correction in a third array
    static constexpr size_t SMEM_COH = SMEM + (PC ? (size_t)RN * sizeof(double) : 0);
};

// Interior tiles (every cell within 2*NS of the tile is an inner point; flagged by the host setup) take a
// fast path: no guard phase, so the valid region shrinks by 2 instead of 3 cells per sweep (halo 2*NS), and
// no point codes are needed at all.
template <int NS, int EPI = 0, int BX = TX, int BY = TY>
struct GeoF {
    static constexpr int H = 2 * NS + (EPI == 1 ? 2 : (EPI == 2 ? 1 : 0));
    static constexpr int RW = BX + 2 * H;
    static constexpr int RH = BY + 2 * H;
    static constexpr int BW = BX, BH = BY;
    static constexpr int RWC = RW / 2;
    static constexpr int NC = RH * RWC;
    static constexpr int RN = 2 * NC;
    static constexpr int ROUNDS = (NC + GT - 1) / GT;
};

// global slot of region cell (rx, ry); region origin is (-H, -H) relative to the tile
template <int H>
__device__ __forceinline__ int64_t region_slot(const int* tn, int rx, int ry) {
    const int lx = rx - H, ly = ry - H;
    const int ox = (lx < 0) ? -1 : (lx >= TX ? 1 : 0);
    const int oy = (ly < 0) ? -1 : (ly >= TY ? 1 : 0);
    return (int64_t)tn[(oy + 1) * 3 + ox + 1] * TS + (ly - oy * TY) * TX + (lx - ox * TX);
}

template <class G>
__device__ __forceinline__ int cidx(int rx, int ry) {
    return ((rx + ry) & 1) * G::NC + ry * G::RWC + (rx >> 1);
}

// Rule D3 on the shared-memory region: sum over the non-self stencil nodes of w * v, weight on the point
// itself, distance delta (h |n|, or h for the fallback).
template <class G>
__device__ __forceinline__ void neumann_smem(uint16_t code, int rx, int ry, const double* v, double h, double& sum, double& wself,
                                             double& delta) {
    const int tnR = ((code >> 2) & 7) - 2, tnZ = ((code >> 5) & 7) - 2;
    sum = 0.0; wself = 0.0;
    if (code & (1 << 8)) {
        const int mask = (code >> 9) & 15;
        if (mask & 1) sum += v[cidx<G>(rx - 1, ry)];
        if (mask & 2) sum += v[cidx<G>(rx + 1, ry)];
        if (mask & 4) sum += v[cidx<G>(rx, ry - 1)];
        if (mask & 8) sum += v[cidx<G>(rx, ry + 1)];
        sum = sum / (double)__popc(mask);
        delta = h;
        return;
    }
    int ox[2], oy[2], nx, ny; double wx, wy;
    if (tnR & 1) { nx = 2; ox[0] = 0; ox[1] = tnR; wx = 0.5; } else { nx = 1; ox[0] = tnR / 2; ox[1] = 0; wx = 1.0; }
    if (tnZ & 1) { ny = 2; oy[0] = 0; oy[1] = tnZ; wy = 0.5; } else { ny = 1; oy[0] = tnZ / 2; oy[1] = 0; wy = 1.0; }
    const double wgt = wx * wy;
    for (int bb = 0; bb < ny; bb++)
        for (int aa = 0; aa < nx; aa++) {
            if (ox[aa] == 0 && oy[bb] == 0) { wself += wgt; continue; }
            sum += wgt * v[cidx<G>(rx + ox[aa], ry + oy[bb])];
        }
    delta = h * sqrt(0.25 * (double)(tnR * tnR + tnZ * tnZ));
}

__device__ __forceinline__ int64_t parent_slot9(const int* pt, int cx, int cy) {
    const int ox = (cx < 0) ? -1 : (cx >= TX ? 1 : 0);
    const int oy = (cy < 0) ? -1 : (cy >= TY ? 1 : 0);
    return (int64_t)pt[(oy + 1) * 3 + ox + 1] * TS + (cy - oy * TY) * TX + (cx - ox * TX);
}

// Fused defect restriction (rules D4 + T2), run after the sweeps of a pre-smoothing launch: every
// thread forms d = A x - b (difference form of rule D1) for its own inner cells of the tile and of the one-cell
// ring around it, parks it in the (no longer needed) c array, and the 32 x 16 coarse points under the tile
// gather their 3 x 3 full-weighting stencils; coarse guard rows get 0.  `breg` still holds b.
template <class G, bool GENERAL, int XIM>
__device__ __forceinline__ void restrict_epilogue(const LevelDev& lv, const int* tn, const int* pt, const int* odd, const double* sx,
                                                  double* sc, const uint16_t* scode, double (&breg)[2][G::ROUNDS], double kappa,
                                                  const uint16_t* __restrict__ ccode, double* __restrict__ dc, int bx0, int by0) {
    constexpr int H = G::H, RW = G::RW, RH = G::RH, RWC = G::RWC, NC = G::NC, ROUNDS = G::ROUNDS, BX = G::BW, BY = G::BH;
    const int tid = threadIdx.x;
    // Interior tiles (no boundary phase): the black cells were updated last from the current red values, so
    // their defect is zero up to rounding; only the red defects are formed and gathered.
    constexpr int NCOL = GENERAL ? 2 : 1;
#pragma unroll
    for (int col = 0; col < NCOL; col++)
#pragma unroll
        for (int r = 0; r < ROUNDS; r++) {
            const int q = tid + r * GT;
            double d = 0.0;
            if (q < NC) {
                const int ry = q / RWC, k = q - ry * RWC, tpar = (ry + col) & 1, rx = 2 * k + tpar;
                const int own = col * NC + q, ob = (1 - col) * NC + q;
                const bool inner = GENERAL ? ((scode[own] & 3) == C_INNER) : true;
                if (inner && min(min(rx, RW - 1 - rx), min(ry, RH - 1 - ry)) >= H - 1) {
                    const int64_t gs = region_slot<H>(tn, rx + bx0, ry + by0);
                    const double lam = __ldg(lv.lam + gs);
                    const bool hx = has_xi<XIM>(lv);
                    const double xi = hx ? __ldg(lv.xi + gs) : 1.0;                  // breg holds b / xi (three-field form)
                    // __dmul_rn: never contracted into the sums below, so the run-time and compile-time xi variants agree bit for bit
                    const double kap = hx ? __dmul_rn(kappa, xi) : kappa, bl = hx ? __dmul_rn(breg[col][r], xi) : breg[col][r];
                    const double cl = sc[own], xl = sx[own];
                    const double aW = kap * (cl + sc[ob + tpar - 1]), aE = kap * (cl + sc[ob + tpar]);
                    const double aS = kap * (cl + sc[ob - RWC]), aN = kap * (cl + sc[ob + RWC]);
                    d = __dsub_rn(row_d1(lam, xl, aW, sx[ob + tpar - 1], aE, sx[ob + tpar], aS, sx[ob - RWC], aN, sx[ob + RWC]), bl);
                }
            }
            breg[col][r] = d;
        }
    __syncthreads();
#pragma unroll
    for (int col = 0; col < NCOL; col++)
#pragma unroll
        for (int r = 0; r < ROUNDS; r++) {
            const int q = tid + r * GT;
            if (q < NC) sc[col * NC + q] = breg[col][r];
        }
    __syncthreads();
    const int ptile = pt[4];                                  // the coarse tile this fine tile lies under
    if (ptile == lv.ntiles_coarse) return;                    // no coarse point here
    for (int i = tid; i < (BX / 2) * (BY / 2); i += GT) {
        const int cyl = i / (BX / 2), cxl = i - cyl * (BX / 2);
        const int rx = 2 * cxl + H, ry = 2 * cyl + H;
        const int64_t cs = (int64_t)ptile * TS + (odd[1] * (TY / 2) + by0 / 2 + cyl) * TX + odd[0] * (TX / 2) + bx0 / 2 + cxl;
        double acc = 0.0;
        if ((__ldg(ccode + cs) & 3) == C_INNER) {
#pragma unroll
            for (int dy = -1; dy <= 1; dy++)
#pragma unroll
                for (int dx = -1; dx <= 1; dx++) {
                    if (!GENERAL && ((dx + dy) & 1)) continue;      // black neighbours of a (red) coarse point: zero
                    const double w = (dx == 0 ? 2.0 : 1.0) * (dy == 0 ? 2.0 : 1.0) * 0.0625;
                    acc += w * sc[cidx<G>(rx + dx, ry + dy)];
                }
        }
        dc[cs] = acc;
    }
}

// Fused operator apply (rules D1-D3, the same rows as k_apply): every thread forms (A x) for its own cells of the tile
// from the smoothed x in shared memory (lambda is the only extra load), parks it in the no longer needed c array,
// and the tile is written out coalesced.  `breg` is reused as scratch.
template <class G, bool GENERAL, int XIM>
__device__ __forceinline__ void apply_epilogue(const LevelDev& lv, int t, const int* tn, const double* sx, double* sc, const uint16_t* scode,
                                               double (&breg)[2][G::ROUNDS], double kappa, double* __restrict__ wout, int bx0, int by0) {
    constexpr int H = G::H, RW = G::RW, RH = G::RH, RWC = G::RWC, NC = G::NC, ROUNDS = G::ROUNDS, BX = G::BW, BY = G::BH;
    const int tid = threadIdx.x;
#pragma unroll
    for (int col = 0; col < 2; col++)
#pragma unroll
        for (int r = 0; r < ROUNDS; r++) {
            const int q = tid + r * GT;
            double v = 0.0;
            if (q < NC) {
                const int ry = q / RWC, k = q - ry * RWC, tpar = (ry + col) & 1, rx = 2 * k + tpar;
                if (min(min(rx, RW - 1 - rx), min(ry, RH - 1 - ry)) >= H) {          // a cell of the tile (block)
                    const int own = col * NC + q, ob = (1 - col) * NC + q;
                    const uint16_t code = GENERAL ? scode[own] : (uint16_t)C_INNER;
                    const int kind = code & 3;
                    if (kind == C_INNER) {
                        const int64_t gs = region_slot<H>(tn, rx + bx0, ry + by0);
                        const double lam = __ldg(lv.lam + gs);
                        const double kap = has_xi<XIM>(lv) ? __dmul_rn(kappa, __ldg(lv.xi + gs)) : kappa;     // xi_{i,j} / (2 h^2), Eq. 10
                        const double cl = sc[own], xl = sx[own];
                        const double aW = kap * (cl + sc[ob + tpar - 1]), aE = kap * (cl + sc[ob + tpar]);
                        const double aS = kap * (cl + sc[ob - RWC]), aN = kap * (cl + sc[ob + RWC]);
                        v = row_d1(lam, xl, aW, sx[ob + tpar - 1], aE, sx[ob + tpar], aS, sx[ob - RWC], aN, sx[ob + RWC]);
                    } else if (kind == C_DIR) v = sx[own];
                    else if (kind == C_NEU) {
                        double sum, wself, delta;
                        neumann_smem<G>(code, rx, ry, sx, lv.h, sum, wself, delta);
                        const double xl = sx[own];
                        v = (sum + wself * xl - xl) / delta;
                    }
                }
            }
            breg[col][r] = v;
        }
    __syncthreads();
#pragma unroll
    for (int col = 0; col < 2; col++)
#pragma unroll
        for (int r = 0; r < ROUNDS; r++) {
            const int q = tid + r * GT;
            if (q < NC) sc[col * NC + q] = breg[col][r];
        }
    __syncthreads();
    for (int idx = tid; idx < BX * BY; idx += GT) {
        const int ly = idx / BX, lx = idx - ly * BX;
        wout[(int64_t)t * TS + (by0 + ly) * TX + bx0 + lx] = sc[cidx<G>(lx + H, ly + H)];
    }
}

// e = (P e_c) at fine cell (lx, ly) relative to the tile (may lie in the halo): bilinear, weights
// 1 / (1/2, 1/2) / (1/4 x 4) in the order (cx, cy), (cx+1, cy), (cx, cy+1), (cx+1, cy+1); absent parents hold 0.
// Branch-free (unused parents alias the first one with weight 0) so that the loads of all cells overlap.
template <bool COH>
__device__ __forceinline__ double prolong_e(const int* pt, int odd0, int odd1, int lx, int ly, const double* __restrict__ ec) {
    const int cx = odd0 * (TX / 2) + (lx >> 1), cy = odd1 * (TY / 2) + (ly >> 1);
    const bool ax = lx & 1, ay = ly & 1;
    const int64_t p00 = parent_slot9(pt, cx, cy);
    const int64_t p10 = ax ? parent_slot9(pt, cx + 1, cy) : p00;
    const int64_t p01 = ay ? parent_slot9(pt, cx, cy + 1) : p00;
    const int64_t p11 = (ax && ay) ? parent_slot9(pt, cx + 1, cy + 1) : p00;
    const double w00 = (ax ? 0.5 : 1.0) * (ay ? 0.5 : 1.0);
    const double w10 = ax ? w00 : 0.0, w01 = ay ? w00 : 0.0, w11 = (ax && ay) ? w00 : 0.0;
    return w00 * ldv<COH>(ec + p00) + w10 * ldv<COH>(ec + p10) + w01 * ldv<COH>(ec + p01) + w11 * ldv<COH>(ec + p11);
}

// x_out = S^NS (x_in - [PC] P e_c);  zero: x_in is the zero vector and is not read.
template <int NS, bool PC, bool COH, int EPI = 0, int BX = TX, int BY = TY, int XIM = 2>
__device__ __forceinline__ void gs_general(const LevelDev& lv, int t, const double* __restrict__ xin, double* __restrict__ xout,
                                           const double* __restrict__ b, const double* __restrict__ ec, int xin_zero,
                                           unsigned char* smem_raw, const int* meta = nullptr,
                                           const uint16_t* __restrict__ ccode = nullptr, double* __restrict__ dc = nullptr,
                                           int bx0 = 0, int by0 = 0) {
    using G = Geo<NS, PC, EPI, BX, BY>;
    constexpr bool DR = EPI == 1, AP = EPI == 2;
    constexpr int H = G::H, RW = G::RW, RH = G::RH, RWC = G::RWC, NC = G::NC, RN = G::RN, ROUNDS = G::ROUNDS;
    static_assert(ROUNDS * 2 * 4 <= 32, "activity nibbles must fit one word");
    double* sx = reinterpret_cast<double*>(smem_raw);
    double* sc = sx + RN;
    double* gb = sc + RN;
    double* se = gb + GCAP;                                  // (PC, batched staging) prolongated correction
    uint16_t* scode = reinterpret_cast<uint16_t*>(se + ((PC && COH) ? RN : 0));
    uint16_t* glist = scode + RN;
    __shared__ int tn[9];
    __shared__ int pt[9];
    __shared__ int odd[2];
    __shared__ int gcount;
    const int tid = threadIdx.x;
    __syncthreads();                       // shared memory may still be in use by a previous tile of this CTA
    if (meta != nullptr) {                 // tile tables preloaded by the caller (fused small-level kernel)
        if (tid < 9) { tn[tid] = meta[META_TN + tid]; pt[tid] = meta[META_PT + tid]; }
        if (tid < 2) odd[tid] = meta[META_ODD + tid];
    } else {
        if (tid < 9) {
            tn[tid] = lv.tnb[9 * t + tid];
            if (PC || DR) pt[tid] = lv.ptab[9 * t + tid];
        }
        if (tid < 2 && (PC || DR)) odd[tid] = lv.tij[2 * t + tid] & 1;
    }
    if (tid == 0) gcount = 0;
    __syncthreads();

    double breg[2][ROUNDS], rd[2][ROUNDS];
    unsigned act = 0;      // per (colour, round) nibble: bits 0-1 number of sweeps the cell takes part in, bit 2 row parity term
    if constexpr (COH) {
        // ---- global loads, one batch per colour: code, x, c, b, 1/a_ll and (PC) the coarse parents of every owned
        // cell are requested before any of them is used.  b and 1/a_ll stay in registers, the rest goes to shared memory.
    #pragma unroll
        for (int col = 0; col < 2; col++) {
            uint16_t codes[ROUNDS];
            double xv[ROUNDS], cv[ROUNDS], ev[ROUNDS], xiv[ROUNDS];
    #pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                const int q = min(tid + r * GT, NC - 1);
                const int ry = q / RWC, k = q - ry * RWC, rx = 2 * k + ((ry + col) & 1);
                const int64_t s = region_slot<H>(tn, rx + bx0, ry + by0);
                codes[r] = __ldg(lv.code + s);
                xv[r] = (!PC && xin_zero) ? 0.0 : ldv<COH>(xin + s);
                cv[r] = __ldg(lv.c + s);
                breg[col][r] = ldv<COH>(b + s);
                xiv[r] = has_xi<XIM>(lv) ? __ldg(lv.xi + s) : 1.0;
                rd[col][r] = __ldg(lv.rd + s);
                ev[r] = PC ? prolong_e<COH>(pt, odd[0], odd[1], rx - H + bx0, ry - H + by0, ec) : 0.0;
            }
    #pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                const int q = tid + r * GT;
                if (q >= NC) continue;
                const int ry = q / RWC, k = q - ry * RWC, tpar = (ry + col) & 1, rx = 2 * k + tpar;
                const int idx = col * NC + q;
                const int kind = codes[r] & 3;
                scode[idx] = codes[r];
                sx[idx] = xv[r];
                sc[idx] = cv[r];
                if (PC) se[idx] = (kind == C_INNER) ? ev[r] : 0.0;
                if (kind == C_INNER) {
                    const int marg = min(min(rx, RW - 1 - rx), min(ry, RH - 1 - ry));
                    const int base = 1 + col + (PC ? 1 : 0);
                    const int nsw = marg >= base ? min(NS, (marg - base) / 3 + 1) : 0;
                    act |= (unsigned)(nsw | (tpar << 2)) << (4 * (col * ROUNDS + r));
                    if (has_xi<XIM>(lv)) breg[col][r] = __ddiv_rn(breg[col][r], xiv[r]);    // the smoother's row is divided by xi
                } else if (kind != C_ABSENT) {
                    const int pos = atomicAdd(&gcount, 1);
                    if (pos < GCAP) { glist[pos] = (uint16_t)(ry * RW + rx); gb[pos] = breg[col][r]; }
                }
            }
        }
        if (PC) {
            // ---- coarse-grid correction x <- x - e on the whole region; guards of e by the homogeneous
            // Eq. 11 / Eq. 16 (set_bnds_hom)
            __syncthreads();
    #pragma unroll
            for (int col = 0; col < 2; col++)
    #pragma unroll
                for (int r = 0; r < ROUNDS; r++) {
                    const int q = tid + r * GT;
                    if (q >= NC) continue;
                    const int idx = col * NC + q;
                    const uint16_t code = scode[idx];
                    const int kind = code & 3;
                    if (kind == C_INNER) sx[idx] -= se[idx];
                    else if (kind == C_NEU) {
                        const int ry = q / RWC, k = q - ry * RWC, rx = 2 * k + ((ry + col) & 1);
                        if (rx >= 1 && rx < RW - 1 && ry >= 1 && ry < RH - 1) {      // edge guards are outside the valid region anyway
                            double sum, wself, delta;
                            neumann_smem<G>(code, rx, ry, se, lv.h, sum, wself, delta);
                            sx[idx] -= sum / (1.0 - wself);
                        }
                    }
                }
        }
    } else {
        if (PC) {
            // ---- coarse-grid correction on the whole region: e = P e_c on inner cells (bilinear, absent parents
            // hold 0), homogeneous Eq. 11 / Eq. 16 on guards (set_bnds_hom), x <- x - e.  e is staged in sc.
    #pragma unroll
            for (int col = 0; col < 2; col++)
    #pragma unroll
                for (int r = 0; r < ROUNDS; r++) {
                    const int q = tid + r * GT;
                    if (q >= NC) continue;
                    const int ry = q / RWC, k = q - ry * RWC, rx = 2 * k + ((ry + col) & 1);
                    const int64_t s = region_slot<H>(tn, rx + bx0, ry + by0);
                    const uint16_t code = __ldg(lv.code + s);
                    const int idx = col * NC + q;
                    scode[idx] = code;
                    sx[idx] = ldv<COH>(xin + s);
                    double e = 0.0;
                    if ((code & 3) == C_INNER) {
                        const int lx = rx - H + bx0, ly = ry - H + by0;
                        const int cx = odd[0] * (TX / 2) + (lx >> 1), cy = odd[1] * (TY / 2) + (ly >> 1);
                        const int ax = lx & 1, ay = ly & 1;
                        if (!ax && !ay) e = ldv<COH>(ec + parent_slot9(pt, cx, cy));
                        else if (ax && !ay) e = 0.5 * ldv<COH>(ec + parent_slot9(pt, cx, cy)) + 0.5 * ldv<COH>(ec + parent_slot9(pt, cx + 1, cy));
                        else if (!ax && ay) e = 0.5 * ldv<COH>(ec + parent_slot9(pt, cx, cy)) + 0.5 * ldv<COH>(ec + parent_slot9(pt, cx, cy + 1));
                        else e = 0.25 * ldv<COH>(ec + parent_slot9(pt, cx, cy)) + 0.25 * ldv<COH>(ec + parent_slot9(pt, cx + 1, cy)) +
                                 0.25 * ldv<COH>(ec + parent_slot9(pt, cx, cy + 1)) + 0.25 * ldv<COH>(ec + parent_slot9(pt, cx + 1, cy + 1));
                    }
                    sc[idx] = e;
                }
            __syncthreads();
    #pragma unroll
            for (int col = 0; col < 2; col++)
    #pragma unroll
                for (int r = 0; r < ROUNDS; r++) {
                    const int q = tid + r * GT;
                    if (q >= NC) continue;
                    const int idx = col * NC + q;
                    const uint16_t code = scode[idx];
                    const int kind = code & 3;
                    if (kind == C_INNER) sx[idx] -= sc[idx];
                    else if (kind == C_NEU) {
                        const int ry = q / RWC, k = q - ry * RWC, rx = 2 * k + ((ry + col) & 1);
                        if (rx >= 1 && rx < RW - 1 && ry >= 1 && ry < RH - 1) {      // edge guards are outside the valid region anyway
                            double sum, wself, delta;
                            neumann_smem<G>(code, rx, ry, sc, lv.h, sum, wself, delta);
                            sx[idx] -= sum / (1.0 - wself);
                        }
                    }
                }
            __syncthreads();
        }

        // ---- stage c (and x, codes if not done above); b and lambda of the owned inner cells go to registers
    #pragma unroll
        for (int col = 0; col < 2; col++)
    #pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                breg[col][r] = 0.0; rd[col][r] = 0.0;
                const int q = tid + r * GT;
                if (q >= NC) continue;
                const int ry = q / RWC, k = q - ry * RWC, tpar = (ry + col) & 1, rx = 2 * k + tpar;
                const int64_t s = region_slot<H>(tn, rx + bx0, ry + by0);
                const int idx = col * NC + q;
                uint16_t code;
                if (PC) code = scode[idx];
                else {
                    code = __ldg(lv.code + s);
                    scode[idx] = code;
                    sx[idx] = xin_zero ? 0.0 : ldv<COH>(xin + s);
                }
                sc[idx] = __ldg(lv.c + s);
                const int kind = code & 3;
                if (kind == C_INNER) {
                    const int marg = min(min(rx, RW - 1 - rx), min(ry, RH - 1 - ry));
                    const int base = 1 + col + (PC ? 1 : 0);
                    const int nsw = marg >= base ? min(NS, (marg - base) / 3 + 1) : 0;
                    if (nsw > 0) {
                        breg[col][r] = ldv<COH>(b + s); rd[col][r] = __ldg(lv.rd + s);
                        if (has_xi<XIM>(lv)) breg[col][r] = __ddiv_rn(breg[col][r], __ldg(lv.xi + s));
                    }
                    if ((DR && marg >= H - 1) || (AP && marg >= H)) prefetch_l2(lv.lam + s);     // read by the restriction epilogue
                    act |= (unsigned)(nsw | (tpar << 2)) << (4 * (col * ROUNDS + r));
                } else if (kind != C_ABSENT) {
                    const int pos = atomicAdd(&gcount, 1);
                    if (pos < GCAP) { glist[pos] = (uint16_t)(ry * RW + rx); gb[pos] = ldv<COH>(b + s); }
                }
            }
    }
    __syncthreads();
    const double kappa = lv.kappa;
    const int ng = gcount;

#pragma unroll
    for (int sweep = 0; sweep < NS; sweep++) {
        // ---- red (colour 0), then black (colour 1)
#pragma unroll
        for (int col = 0; col < 2; col++) {
#pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                const unsigned nib = (act >> (4 * (col * ROUNDS + r))) & 15u;
                if (sweep < (int)(nib & 3u)) {
                    const int q = tid + r * GT, tpar = (nib >> 2) & 1;
                    const int own = col * NC + q, ob = (1 - col) * NC + q;
                    const double cl = sc[own];
                    double acc = (cl + sc[ob + tpar - 1]) * sx[ob + tpar - 1];
                    acc = fma(cl + sc[ob + tpar], sx[ob + tpar], acc);
                    acc = fma(cl + sc[ob - RWC], sx[ob - RWC], acc);
                    acc = fma(cl + sc[ob + RWC], sx[ob + RWC], acc);
                    sx[own] = fma(kappa, acc, breg[col][r]) * rd[col][r];
                }
            }
            __syncthreads();
        }
        // ---- boundary points (Eq. 11, Eq. 16 solved for the point)
        if (ng > 0) {
            const int m = 3 * sweep + 3 + (PC ? 1 : 0);
            if (ng <= GCAP) {
                for (int g = tid; g < ng; g += GT) {
                    const int cell = glist[g];
                    const int ry = cell / RW, rx = cell - ry * RW;
                    if (min(min(rx, RW - 1 - rx), min(ry, RH - 1 - ry)) < m) continue;
                    const int idx = cidx<G>(rx, ry);
                    const uint16_t code = scode[idx];
                    if ((code & 3) == C_DIR) sx[idx] = gb[g];
                    else {
                        double sum, wself, delta;
                        neumann_smem<G>(code, rx, ry, sx, lv.h, sum, wself, delta);
                        sx[idx] = neumann_point(sum, delta, gb[g], wself);
                    }
                }
            } else {                                   // list overflow: every thread scans its own cells
                for (int col = 0; col < 2; col++)
                    for (int r = 0; r < ROUNDS; r++) {
                        const int q = tid + r * GT;
                        if (q >= NC) continue;
                        const int idx = col * NC + q;
                        const uint16_t code = scode[idx];
                        const int kind = code & 3;
                        if (kind != C_DIR && kind != C_NEU) continue;
                        const int ry = q / RWC, k = q - ry * RWC, rx = 2 * k + ((ry + col) & 1);
                        if (min(min(rx, RW - 1 - rx), min(ry, RH - 1 - ry)) < m) continue;
                        const double bv = ldv<COH>(b + region_slot<H>(tn, rx + bx0, ry + by0));
                        if (kind == C_DIR) sx[idx] = bv;
                        else {
                            double sum, wself, delta;
                            neumann_smem<G>(code, rx, ry, sx, lv.h, sum, wself, delta);
                            sx[idx] = neumann_point(sum, delta, bv, wself);
                        }
                    }
            }
            __syncthreads();
        }
    }
    // ---- write the tile back (absent slots carry the zeros they were loaded with)
    for (int idx = tid; idx < BX * BY; idx += GT) {
        const int ly = idx / BX, lx = idx - ly * BX;
        xout[(int64_t)t * TS + (by0 + ly) * TX + bx0 + lx] = sx[cidx<G>(lx + H, ly + H)];
    }
    if (DR) restrict_epilogue<G, true, XIM>(lv, tn, pt, odd, sx, sc, scode, breg, kappa, ccode, dc, bx0, by0);
    if (AP) apply_epilogue<G, true, XIM>(lv, t, tn, sx, sc, scode, breg, kappa, dc, bx0, by0);
}

// Interior tile: all cells of the region are inner points.
template <int NS, bool PC, bool COH, int EPI = 0, int BX = TX, int BY = TY, int XIM = 2>
__device__ __forceinline__ void gs_fast(const LevelDev& lv, int t, const double* __restrict__ xin, double* __restrict__ xout,
                                        const double* __restrict__ b, const double* __restrict__ ec, int xin_zero,
                                        unsigned char* smem_raw, const int* meta = nullptr,
                                           const uint16_t* __restrict__ ccode = nullptr, double* __restrict__ dc = nullptr,
                                           int bx0 = 0, int by0 = 0) {
    using G = GeoF<NS, EPI, BX, BY>;
    constexpr bool DR = EPI == 1, AP = EPI == 2;
    constexpr int H = G::H, RW = G::RW, RH = G::RH, RWC = G::RWC, NC = G::NC, RN = G::RN, ROUNDS = G::ROUNDS;
    static_assert(ROUNDS * 2 * 4 <= 32, "activity nibbles must fit one word");
    double* sx = reinterpret_cast<double*>(smem_raw);
    double* sc = sx + RN;
    double* sce = sc + RN;                                   // (PC) coarse values under the region
    constexpr int CM = (H + 1) / 2, CW = BX / 2 + (H - 1) / 2 + CM + 2, CHH = BY / 2 + (H - 1) / 2 + CM + 2;
    static_assert((size_t)(2 * RN + CW * CHH) * sizeof(double) <= Geo<NS, true, EPI, BX, BY>::SMEM, "coarse stage must fit the PC allocation");
    __shared__ int tn[9];
    __shared__ int pt[9];
    __shared__ int odd[2];
    const int tid = threadIdx.x;
    __syncthreads();
    if (meta != nullptr) {                 // tile tables preloaded by the caller (fused small-level kernel)
        if (tid < 9) { tn[tid] = meta[META_TN + tid]; pt[tid] = meta[META_PT + tid]; }
        if (tid < 2) odd[tid] = meta[META_ODD + tid];
    } else {
        if (tid < 9) {
            tn[tid] = lv.tnb[9 * t + tid];
            if (PC || DR) pt[tid] = lv.ptab[9 * t + tid];
        }
        if (tid < 2 && (PC || DR)) odd[tid] = lv.tij[2 * t + tid] & 1;
    }
    __syncthreads();
    double breg[2][ROUNDS], rd[2][ROUNDS];
    unsigned act = 0;
    if constexpr (COH) {
    #pragma unroll
        for (int col = 0; col < 2; col++) {                         // one batch of independent loads per colour
            double xv[ROUNDS], cv[ROUNDS];
    #pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                const int q = min(tid + r * GT, NC - 1);
                const int ry = q / RWC, k = q - ry * RWC, rx = 2 * k + ((ry + col) & 1);
                const int64_t s = region_slot<H>(tn, rx + bx0, ry + by0);
                xv[r] = xin_zero ? 0.0 : ldv<COH>(xin + s);
                cv[r] = __ldg(lv.c + s);
                breg[col][r] = ldv<COH>(b + s);
                if (has_xi<XIM>(lv)) breg[col][r] = __ddiv_rn(breg[col][r], __ldg(lv.xi + s));
                rd[col][r] = __ldg(lv.rd + s);
                if (PC) xv[r] -= prolong_e<COH>(pt, odd[0], odd[1], rx - H + bx0, ry - H + by0, ec);   // x <- x - P e_c
            }
    #pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                const int q = tid + r * GT;
                if (q >= NC) continue;
                const int ry = q / RWC, k = q - ry * RWC, tpar = (ry + col) & 1, rx = 2 * k + tpar;
                const int idx = col * NC + q;
                sx[idx] = xv[r];
                sc[idx] = cv[r];
                const int marg = min(min(rx, RW - 1 - rx), min(ry, RH - 1 - ry));
                const int base = 1 + col;
                const int nsw = marg >= base ? min(NS, (marg - base) / 2 + 1) : 0;
                act |= (unsigned)(nsw | (tpar << 2)) << (4 * (col * ROUNDS + r));
            }
        }
    } else {
        if (PC)                                             // coarse values under the region, staged once
            for (int i = tid; i < CW * CHH; i += GT) {
                const int ccy = i / CW, ccx = i - ccy * CW;
                sce[i] = ldv<COH>(ec + parent_slot9(pt, odd[0] * (TX / 2) + bx0 / 2 + ccx - CM, odd[1] * (TY / 2) + by0 / 2 + ccy - CM));
            }
    #pragma unroll
        for (int col = 0; col < 2; col++)
    #pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                breg[col][r] = 0.0; rd[col][r] = 0.0;
                const int q = tid + r * GT;
                if (q >= NC) continue;
                const int ry = q / RWC, k = q - ry * RWC, tpar = (ry + col) & 1, rx = 2 * k + tpar;
                const int64_t s = region_slot<H>(tn, rx + bx0, ry + by0);
                const int idx = col * NC + q;
                const double x = xin_zero ? 0.0 : ldv<COH>(xin + s);
                sx[idx] = x;
                sc[idx] = __ldg(lv.c + s);
                const int marg = min(min(rx, RW - 1 - rx), min(ry, RH - 1 - ry));
                const int base = 1 + col;
                const int nsw = marg >= base ? min(NS, (marg - base) / 2 + 1) : 0;
                if (nsw > 0) {
                    breg[col][r] = ldv<COH>(b + s); rd[col][r] = __ldg(lv.rd + s);
                    if (has_xi<XIM>(lv)) breg[col][r] = __ddiv_rn(breg[col][r], __ldg(lv.xi + s));
                }
                if ((DR && marg >= H - 1) || (AP && marg >= H)) prefetch_l2(lv.lam + s);         // read by the restriction epilogue
                act |= (unsigned)(nsw | (tpar << 2)) << (4 * (col * ROUNDS + r));
            }
    }
    __syncthreads();
    if (PC && !COH) {
        // x <- x - P e_c on the owned cells (bilinear; all cells of an interior tile are inner):
        // weights 1 / (1/2, 1/2) / (1/4 x 4) over the parents (cx, cy), (cx+1, cy), (cx, cy+1), (cx+1, cy+1)
#pragma unroll
        for (int col = 0; col < 2; col++)
#pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                const int q = tid + r * GT;
                if (q >= NC) continue;
                const int ry = q / RWC, k = q - ry * RWC, rx = 2 * k + ((ry + col) & 1);
                const int lx = rx - H, ly = ry - H;
                const double* p = sce + ((ly >> 1) + CM) * CW + (lx >> 1) + CM;
                const int ax = lx & 1, ay = ly & 1;
                double e;
                if (!ax && !ay) e = p[0];
                else if (ax && !ay) e = 0.5 * p[0] + 0.5 * p[1];
                else if (!ax && ay) e = 0.5 * p[0] + 0.5 * p[CW];
                else e = 0.25 * p[0] + 0.25 * p[1] + 0.25 * p[CW] + 0.25 * p[CW + 1];
                sx[col * NC + q] -= e;
            }
        __syncthreads();
    }
    const double kappa = lv.kappa;
#pragma unroll
    for (int sweep = 0; sweep < NS; sweep++)
#pragma unroll
        for (int col = 0; col < 2; col++) {
#pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                const unsigned nib = (act >> (4 * (col * ROUNDS + r))) & 15u;
                if (sweep < (int)(nib & 3u)) {
                    const int q = tid + r * GT, tpar = (nib >> 2) & 1;
                    const int own = col * NC + q, ob = (1 - col) * NC + q;
                    const double cl = sc[own];
                    double acc = (cl + sc[ob + tpar - 1]) * sx[ob + tpar - 1];
                    acc = fma(cl + sc[ob + tpar], sx[ob + tpar], acc);
                    acc = fma(cl + sc[ob - RWC], sx[ob - RWC], acc);
                    acc = fma(cl + sc[ob + RWC], sx[ob + RWC], acc);
                    sx[own] = fma(kappa, acc, breg[col][r]) * rd[col][r];
                }
            }
            __syncthreads();
        }
    for (int idx = tid; idx < BX * BY; idx += GT) {
        const int ly = idx / BX, lx = idx - ly * BX;
        xout[(int64_t)t * TS + (by0 + ly) * TX + bx0 + lx] = sx[cidx<G>(lx + H, ly + H)];
    }
    if (DR) restrict_epilogue<G, false, XIM>(lv, tn, pt, odd, sx, sc, nullptr, breg, kappa, ccode, dc, bx0, by0);
    if (AP) apply_epilogue<G, false, XIM>(lv, t, tn, sx, sc, nullptr, breg, kappa, dc, bx0, by0);
}

template <int NS, bool PC, bool COH, int EPI = 0, int BX = TX, int BY = TY, int XIM = 2>
__device__ __forceinline__ void gs_tile(const LevelDev& lv, int t, const double* __restrict__ xin, double* __restrict__ xout,
                                        const double* __restrict__ b, const double* __restrict__ ec, int xin_zero,
                                        unsigned char* smem_raw, const int* meta = nullptr,
                                           const uint16_t* __restrict__ ccode = nullptr, double* __restrict__ dc = nullptr,
                                           int bx0 = 0, int by0 = 0) {
    const int flag = meta != nullptr ? meta[META_FLAG] : lv.tflag[t];
    constexpr int need = 1 << (NS - 1 + (EPI ? 1 : 0));         // interior halo 2 NS (+ 1 or 2, rounded up to the next flag)
    if (flag & need) gs_fast<NS, PC, COH, EPI, BX, BY, XIM>(lv, t, xin, xout, b, ec, xin_zero, smem_raw, meta, ccode, dc, bx0, by0);
    else gs_general<NS, PC, COH, EPI, BX, BY, XIM>(lv, t, xin, xout, b, ec, xin_zero, smem_raw, meta, ccode, dc, bx0, by0);
}

}  // namespace
}  // namespace mgb
