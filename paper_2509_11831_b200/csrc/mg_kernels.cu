// Tile kernels of the multigrid hierarchy (sm_100a) other than the smoother: operator apply / residual (S1),
// the unfused transfers used by the single-step entry points and by cycles with nu_pre = 0 or nu_post = 0
// (defect + restriction S1+S3, restriction S3, prolongation + set_bnds_hom + correction S4), coefficient
// restriction (U1), diagonal (U2), permutations (B1).  One CTA per active tile; halo values come from the
// neighbour tiles through the per-tile 3x3 table (missing tiles map to the all-absent null tile).  Inside the
// cycle S3 and S4 are fused into the smoother launches (mg_tile_gs.cuh).
#include "mg_tile_ops.cuh"

#include <algorithm>

namespace mgb {

namespace {

template <int MODE>
__global__ void __launch_bounds__(NT, 3) k_apply(LevelDev lv, VecRef xr, VecRef br, VecRef yr, const int* __restrict__ stop) {
    __shared__ int tn[9];
    const int pl = blockIdx.y;
    if (stopped(stop, pl)) return;
    lv = plane_of(lv, pl);
    const int t = blockIdx.x;
    if (threadIdx.x < 9) tn[threadIdx.x] = lv.tnb[9 * t + threadIdx.x];
    __syncthreads();
    const double* __restrict__ x = resolve(xr, pl);
    const double* __restrict__ b = (MODE != 0) ? resolve(br, pl) : nullptr;
    double* __restrict__ y = resolve(yr, pl);
    const int lx = threadIdx.x % TX;
    constexpr int NP = TY / ROWS_PER_PASS;
    const Nb4 nb = nb4(tn);
    uint16_t codes[NP];
    double ax[NP], bv[NP];
#pragma unroll
    for (int p = 0; p < NP; p++) {                          // all loads of the thread's four cells in one batch
        const int ly = threadIdx.x / TX + p * ROWS_PER_PASS;
        const int64_t s = (int64_t)t * TS + ly * TX + lx;
        codes[p] = __ldg(lv.code + s);
        ax[p] = inner_row<false>(lv, nb, lx, ly, s, x);            // Eq. 10 with 1/h^2
        bv[p] = (MODE != 0) ? __ldg(b + s) : 0.0;
    }
#pragma unroll
    for (int p = 0; p < NP; p++) {
        const int ly = threadIdx.x / TX + p * ROWS_PER_PASS;
        const int64_t s = (int64_t)t * TS + ly * TX + lx;
        const int kind = codes[p] & 3;
        double v = (kind == C_INNER) ? ax[p] : 0.0;
        if (kind == C_DIR) v = x[s];                        // Eq. 11
        else if (kind == C_NEU) {                           // Eq. 16
            double sum, wself, delta;
            neumann_row(codes[p], tn, lx, ly, x, lv.h, sum, wself, delta);
            const double xl = x[s];
            v = (sum + wself * xl - xl) / delta;
        }
        if (kind == C_ABSENT) y[s] = 0.0;
        else if (MODE == 0) y[s] = v;
        else if (MODE == 1) y[s] = bv[p] - v;
        else y[s] = v - bv[p];
    }
}

// (S2, the smoother, lives in mg_smoother.cu)

// ---------------------------------------------------------------------------------- S3 restriction (rule T2)
// One CTA per COARSE tile. Fine point (2 lxc + dx, 2 lyc + dy) lives in one of the 3x3 fine tiles of ctab.
__device__ __forceinline__ int64_t fine_slot(const int* ct, int fx, int fy) {   // fx in [-1, 2TX), fy in [-1, 2TY)
    const int cx = (fx < 0) ? 0 : (fx < TX ? 1 : 2);
    const int cy = (fy < 0) ? 0 : (fy < TY ? 1 : 2);
    return (int64_t)ct[cy * 3 + cx] * TS + (fy - (cy - 1) * TY) * TX + (fx - (cx - 1) * TX);
}

__global__ void __launch_bounds__(NT) k_restrict(LevelDev fine, LevelDev coarse, const double* __restrict__ df, double* __restrict__ dc, const int* __restrict__ stop) {
    __shared__ int ct[9];
    const int pl = blockIdx.y;
    if (stopped(stop, pl)) return;
    df += pl * fine.nslots; dc += pl * coarse.nslots;
    const int t = blockIdx.x;
    if (threadIdx.x < 9) ct[threadIdx.x] = coarse.ctab[9 * t + threadIdx.x];
    __syncthreads();
    const int lx = threadIdx.x % TX;
#pragma unroll
    for (int p = 0; p < TY / ROWS_PER_PASS; p++) {
        const int ly = threadIdx.x / TX + p * ROWS_PER_PASS;
        const int64_t s = (int64_t)t * TS + ly * TX + lx;
        const int kind = coarse.code[s] & 3;
        double acc = 0.0;
        if (kind == C_INNER) {
#pragma unroll
            for (int dy = -1; dy <= 1; dy++)
#pragma unroll
                for (int dx = -1; dx <= 1; dx++) {
                    const int64_t fs = fine_slot(ct, 2 * lx + dx, 2 * ly + dy);
                    const double w = (dx == 0 ? 2.0 : 1.0) * (dy == 0 ? 2.0 : 1.0) * 0.0625;
                    if ((fine.code[fs] & 3) == C_INNER) acc += w * df[fs];
                }
        }
        dc[s] = acc;        // coarse guard rows and absent slots: 0
    }
}

__global__ void __launch_bounds__(NT) k_defect_restrict(LevelDev fine, LevelDev coarse, VecRef xr, VecRef br, double* __restrict__ dc,
                                                        const int* __restrict__ stop) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int pl = blockIdx.y;
    if (stopped(stop, pl)) return;
    defect_restrict_tile<false>(plane_of(fine, pl), coarse, blockIdx.x, resolve(xr, pl), resolve(br, pl), dc + pl * coarse.nslots, smem_raw);
}

// ---------------------------------------------------------------------------------- U1 coefficient restriction (rule T4)
__global__ void __launch_bounds__(NT) k_restrict_coeff(LevelDev fine, LevelDev coarse) {
    __shared__ int ct[9];
    fine = plane_of(fine, blockIdx.y); coarse = plane_of(coarse, blockIdx.y);
    const int t = blockIdx.x;
    if (threadIdx.x < 9) ct[threadIdx.x] = coarse.ctab[9 * t + threadIdx.x];
    __syncthreads();
    const int lx = threadIdx.x % TX;
#pragma unroll
    for (int p = 0; p < TY / ROWS_PER_PASS; p++) {
        const int ly = threadIdx.x / TX + p * ROWS_PER_PASS;
        const int64_t s = (int64_t)t * TS + ly * TX + lx;
        double sl = 0.0, sc = 0.0, sw = 0.0, sx = 0.0;
        if ((coarse.code[s] & 3) != C_ABSENT) {
#pragma unroll
            for (int dy = -1; dy <= 1; dy++)
#pragma unroll
                for (int dx = -1; dx <= 1; dx++) {
                    const int64_t fs = fine_slot(ct, 2 * lx + dx, 2 * ly + dy);
                    const double w = (dx == 0 ? 2.0 : 1.0) * (dy == 0 ? 2.0 : 1.0) * 0.0625;
                    if ((fine.code[fs] & 3) != C_ABSENT) {
                        sl += w * fine.lam[fs]; sc += w * fine.c[fs]; sw += w;
                        if (fine.xi) sx += w * fine.xi[fs];
                    }
                }
            sl /= sw; sc /= sw; sx /= sw;
        }
        coarse.lam[s] = sl;
        coarse.c[s] = sc;
        if (fine.xi) coarse.xi[s] = sx;
    }
}


// ---------------------------------------------------------------------------------- U2 diagonal (rule D1)
// rd = 1 / a_ll, a_ll = lambda + a_W + a_E + a_S + a_N summed in this order; read by the smoother instead
// of lambda (same traffic, no division in the sweeps).
__global__ void __launch_bounds__(NT) k_diag(LevelDev lv) {
    __shared__ int tn[9];
    lv = plane_of(lv, blockIdx.y);
    const int t = blockIdx.x;
    if (threadIdx.x < 9) tn[threadIdx.x] = lv.tnb[9 * t + threadIdx.x];
    __syncthreads();
    const int lx = threadIdx.x % TX;
#pragma unroll
    for (int p = 0; p < TY / ROWS_PER_PASS; p++) {
        const int ly = threadIdx.x / TX + p * ROWS_PER_PASS;
        const int64_t s = (int64_t)t * TS + ly * TX + lx;
        double r = 0.0;
        if ((lv.code[s] & 3) == C_INNER) {
            const double cl = lv.c[s];
            const double xi = lv.xi ? lv.xi[s] : 1.0;
            const double kap = lv.xi ? lv.kappa * xi : lv.kappa;                 // xi_{i,j} / (2 h^2), Eq. 10
            const double aW = kap * (cl + lv.c[nslot(tn, lx - 1, ly)]), aE = kap * (cl + lv.c[nslot(tn, lx + 1, ly)]);
            const double aS = kap * (cl + lv.c[nslot(tn, lx, ly - 1)]), aN = kap * (cl + lv.c[nslot(tn, lx, ly + 1)]);
            r = xi / (lv.lam[s] + aW + aE + aS + aN);                            // the smoother's row is divided by xi
        }
        lv.rd[s] = r;
    }
}

// ---------------------------------------------------------------------------------- S4 prolongation (rule T3)
__device__ __forceinline__ int64_t parent_slot(const int* pt, int cx, int cy) {   // cx in [-TX, 2TX), cy in [-TY, 2TY)
    const int ox = (cx < 0) ? -1 : (cx >= TX ? 1 : 0);
    const int oy = (cy < 0) ? -1 : (cy >= TY ? 1 : 0);
    return (int64_t)pt[(oy + 1) * 3 + ox + 1] * TS + (cy - oy * TY) * TX + (cx - ox * TX);
}

// Phase A: e = P e_c on fine inner points (bilinear; absent parents hold 0), 0 elsewhere.
__global__ void __launch_bounds__(NT) k_prolong(LevelDev fine, const double* __restrict__ ec, double* __restrict__ ef, const int* __restrict__ stop) {
    __shared__ int pt[9];
    const int pl = blockIdx.y;
    if (stopped(stop, pl)) return;
    ec += pl * ((int64_t)(fine.ntiles_coarse + 1) * TS); ef += pl * fine.nslots;
    __shared__ int odd[2];
    const int t = blockIdx.x;
    if (threadIdx.x < 9) pt[threadIdx.x] = fine.ptab[9 * t + threadIdx.x];
    if (threadIdx.x < 2) odd[threadIdx.x] = fine.tij[2 * t + threadIdx.x] & 1;
    __syncthreads();
    const int lx = threadIdx.x % TX;
    const int cx = odd[0] * (TX / 2) + (lx >> 1);
#pragma unroll
    for (int p = 0; p < TY / ROWS_PER_PASS; p++) {
        const int ly = threadIdx.x / TX + p * ROWS_PER_PASS;
        const int64_t s = (int64_t)t * TS + ly * TX + lx;
        double e = 0.0;
        if ((fine.code[s] & 3) == C_INNER) {
            const int cy = odd[1] * (TY / 2) + (ly >> 1);
            const int ax = lx & 1, ay = ly & 1;
            if (!ax && !ay) e = ec[parent_slot(pt, cx, cy)];
            else if (ax && !ay) e = 0.5 * ec[parent_slot(pt, cx, cy)] + 0.5 * ec[parent_slot(pt, cx + 1, cy)];
            else if (!ax && ay) e = 0.5 * ec[parent_slot(pt, cx, cy)] + 0.5 * ec[parent_slot(pt, cx, cy + 1)];
            else e = 0.25 * ec[parent_slot(pt, cx, cy)] + 0.25 * ec[parent_slot(pt, cx + 1, cy)] +
                     0.25 * ec[parent_slot(pt, cx, cy + 1)] + 0.25 * ec[parent_slot(pt, cx + 1, cy + 1)];
        }
        ef[s] = e;
    }
}

// Phase B: set_bnds_hom on the guards of e (homogeneous Eq. 11 / Eq. 16), then x <- x - e.
__global__ void __launch_bounds__(NT) k_correct(LevelDev fine, const double* __restrict__ ef, VecRef xr, const int* __restrict__ stop) {
    __shared__ int tn[9];
    const int pl = blockIdx.y;
    if (stopped(stop, pl)) return;
    ef += pl * fine.nslots;
    const int t = blockIdx.x;
    if (threadIdx.x < 9) tn[threadIdx.x] = fine.tnb[9 * t + threadIdx.x];
    __syncthreads();
    double* __restrict__ x = resolve(xr, pl);
    const int lx = threadIdx.x % TX;
#pragma unroll
    for (int p = 0; p < TY / ROWS_PER_PASS; p++) {
        const int ly = threadIdx.x / TX + p * ROWS_PER_PASS;
        const int64_t s = (int64_t)t * TS + ly * TX + lx;
        const uint16_t code = fine.code[s];
        const int kind = code & 3;
        if (kind == C_INNER) x[s] -= ef[s];
        else if (kind == C_NEU) {
            double sum, wself, delta;
            neumann_row(code, tn, lx, ly, ef, fine.h, sum, wself, delta);
            x[s] -= sum / (1.0 - wself);
        }
    }
}

// ---------------------------------------------------------------------------------- small helpers
__global__ void k_zero(VecRef xr, int64_t n) {
    double* x = resolve(xr, blockIdx.y);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) x[k] = 0.0;
}
// user order <-> tile layout; plane p: user vectors at p * n, tiled vectors at p * ps
__global__ void k_gather(const double* __restrict__ src, const int32_t* __restrict__ slot, double* __restrict__ dst, int64_t n, int64_t ps) {
    src += blockIdx.y * n; dst += blockIdx.y * ps;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) dst[slot[k]] = src[k];
}
// gather of a coefficient field with the admissibility test of PAPER.md:51: mode 1: finite; mode 2: finite and > 0.
// A violation sets *bad (bit 0 lambda, bit 1 c, bit 2 xi, given by `bit`); the values are copied regardless.
__global__ void k_gather_check(const double* __restrict__ src, const int32_t* __restrict__ slot, double* __restrict__ dst, int64_t n,
                               int64_t ps, int mode, int bit, int* __restrict__ bad) {
    src += blockIdx.y * n; dst += blockIdx.y * ps;
    bool any = false;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        const double v = src[k];
        dst[slot[k]] = v;
        any |= !isfinite(v) || (mode == 2 && !(v > 0.0));
    }
    if (any) atomicOr(bad, bit);
}
__global__ void k_scatter(const double* __restrict__ src, const int32_t* __restrict__ slot, double* __restrict__ dst, int64_t n, int64_t ps) {
    src += blockIdx.y * ps; dst += blockIdx.y * n;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) dst[k] = src[slot[k]];
}

inline int grid1d(int64_t n) { return (int)std::min<int64_t>((n + 255) / 256, dev_info().sms * 8); }
inline void count(const Launch& L, int k = 1) { if (L.counter) *L.counter += k; }

}  // namespace

void launch_apply(const Launch& L, const LevelDev& lv, VecRef x, VecRef b, VecRef y, int mode) {
    const dim3 g(lv.ntiles, L.planes);
    if (mode == 0) k_apply<0><<<g, NT, 0, L.stream>>>(lv, x, b, y, L.stop);
    else if (mode == 1) k_apply<1><<<g, NT, 0, L.stream>>>(lv, x, b, y, L.stop);
    else k_apply<2><<<g, NT, 0, L.stream>>>(lv, x, b, y, L.stop);
    count(L);
}

void launch_restrict(const Launch& L, const LevelDev& fine, const LevelDev& coarse, const double* d_fine, double* d_coarse) {
    k_restrict<<<dim3(coarse.ntiles, L.planes), NT, 0, L.stream>>>(fine, coarse, d_fine, d_coarse, L.stop);
    count(L);
}

void launch_defect_restrict(const Launch& L, const LevelDev& fine, const LevelDev& coarse, VecRef x, VecRef b, double* d_coarse) {
    ensure_dyn_smem((const void*)k_defect_restrict, DR_SMEM);
    k_defect_restrict<<<dim3(coarse.ntiles, L.planes), NT, DR_SMEM, L.stream>>>(fine, coarse, x, b, d_coarse, L.stop);
    count(L);
}

void launch_prolong_correct(const Launch& L, const LevelDev& fine, const LevelDev& coarse, const double* e_coarse,
                            double* e_fine_tmp, VecRef x_fine) {
    (void)coarse;
    k_prolong<<<dim3(fine.ntiles, L.planes), NT, 0, L.stream>>>(fine, e_coarse, e_fine_tmp, L.stop);
    k_correct<<<dim3(fine.ntiles, L.planes), NT, 0, L.stream>>>(fine, e_fine_tmp, x_fine, L.stop);
    count(L, 2);
}

void launch_restrict_coeff(const Launch& L, const LevelDev& fine, const LevelDev& coarse) {
    k_restrict_coeff<<<dim3(coarse.ntiles, L.planes), NT, 0, L.stream>>>(fine, coarse);
    count(L);
}

void launch_diag(const Launch& L, const LevelDev& lv) {
    k_diag<<<dim3(lv.ntiles, L.planes), NT, 0, L.stream>>>(lv);
    count(L);
}

void launch_zero(const Launch& L, VecRef x, int64_t n) {
    k_zero<<<dim3(grid1d(n), L.planes), 256, 0, L.stream>>>(x, n);
    count(L);
}
void launch_gather(const Launch& L, const double* src, const int32_t* slot, double* dst, int64_t n, int64_t ps) {
    k_gather<<<dim3(grid1d(n), L.planes), 256, 0, L.stream>>>(src, slot, dst, n, ps);
    count(L);
}
void launch_gather_check(const Launch& L, const double* src, const int32_t* slot, double* dst, int64_t n, int64_t ps, int mode, int bit, int* bad) {
    k_gather_check<<<dim3(grid1d(n), L.planes), 256, 0, L.stream>>>(src, slot, dst, n, ps, mode, bit, bad);
    count(L);
}
void launch_scatter(const Launch& L, const double* src, const int32_t* slot, double* dst, int64_t n, int64_t ps) {
    k_scatter<<<dim3(grid1d(n), L.planes), 256, 0, L.stream>>>(src, slot, dst, n, ps);
    count(L);
}

}  // namespace mgb
