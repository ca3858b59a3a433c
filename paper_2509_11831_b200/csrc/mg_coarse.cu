// Coarsest-level direct solve on the device (rule C).  The paper factorises the
// coarsest matrix on the CPU at every update and round-trips the right-hand side at every cycle
// (PAPER.md:217); here the dense operator is assembled, inverted (Gauss-Jordan with partial pivoting,
// one CTA) at update time, and the cycle applies the inverse with one small kernel: no host step.
#include <cooperative_groups.h>

#include <algorithm>

#include "mg_device.h"

namespace mgb {

namespace {

constexpr int CT = 1024;

__device__ __forceinline__ int64_t gslot(const int32_t* tn, int lx, int ly) {
    const int ox = (lx < 0) ? -1 : (lx >= TX ? 1 : 0);
    const int oy = (ly < 0) ? -1 : (ly >= TY ? 1 : 0);
    return (int64_t)tn[(oy + 1) * 3 + ox + 1] * TS + (ly - oy * TY) * TX + (lx - ox * TX);
}

// W = [A | I], row-major n x 2n; one thread per row (rules D1-D3).
__global__ void k_coarse_assemble(LevelDev lv, const int32_t* __restrict__ cslot, const int32_t* __restrict__ slot2row,
                                  int n, double* __restrict__ W) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    lv = plane_of(lv, blockIdx.y);
    W += blockIdx.y * coarse_work_doubles(n);
    double* row = W + (size_t)r * 2 * n;
    for (int k = 0; k < 2 * n; k++) row[k] = 0.0;
    row[n + r] = 1.0;
    const int64_t s = cslot[r];
    const int t = (int)(s / TS), ly = (int)(s % TS) / TX, lx = (int)(s % TS) % TX;
    const int32_t* tn = lv.tnb + 9 * t;
    const uint16_t code = lv.code[s];
    const int kind = code & 3;
    if (kind == C_INNER) {
        const int64_t sn[4] = {gslot(tn, lx - 1, ly), gslot(tn, lx + 1, ly), gslot(tn, lx, ly - 1), gslot(tn, lx, ly + 1)};
        const double cl = lv.c[s];
        double all = lv.lam[s];
        double a[4];
        const double kap = lv.xi ? lv.kappa * lv.xi[s] : lv.kappa;           // xi_{i,j} / (2 h^2), Eq. 10
        for (int d = 0; d < 4; d++) { a[d] = kap * (cl + lv.c[sn[d]]); }
        all = lv.lam[s] + a[0] + a[1] + a[2] + a[3];
        row[r] = all;
        for (int d = 0; d < 4; d++) row[slot2row[sn[d]]] = -a[d];
    } else if (kind == C_DIR) {
        row[r] = 1.0;
    } else {
        const int tnR = ((code >> 2) & 7) - 2, tnZ = ((code >> 5) & 7) - 2;
        if (code & (1 << 8)) {
            const int mask = (code >> 9) & 15;
            const double w = 1.0 / (double)__popc(mask), delta = lv.h;
            const int dx[4] = {-1, 1, 0, 0}, dy[4] = {0, 0, -1, 1};
            for (int d = 0; d < 4; d++)
                if (mask & (1 << d)) row[slot2row[gslot(tn, lx + dx[d], ly + dy[d])]] = w / delta;
            row[r] = -1.0 / delta;
        } else {
            int ox[2], oy[2], nx, ny; double wx, wy;
            if (tnR & 1) { nx = 2; ox[0] = 0; ox[1] = tnR; wx = 0.5; } else { nx = 1; ox[0] = tnR / 2; ox[1] = 0; wx = 1.0; }
            if (tnZ & 1) { ny = 2; oy[0] = 0; oy[1] = tnZ; wy = 0.5; } else { ny = 1; oy[0] = tnZ / 2; oy[1] = 0; wy = 1.0; }
            const double w = wx * wy, delta = lv.h * sqrt(0.25 * (double)(tnR * tnR + tnZ * tnZ));
            double wself = 0.0;
            for (int b = 0; b < ny; b++)
                for (int a = 0; a < nx; a++) {
                    if (ox[a] == 0 && oy[b] == 0) { wself += w; continue; }
                    row[slot2row[gslot(tn, lx + ox[a], ly + oy[b])]] = w / delta;
                }
            row[r] = (wself - 1.0) / delta;
        }
    }
}

// In-place Gauss-Jordan with partial pivoting (first maximum wins ties) on W = [A | I] -> [I | A^-1].
// One CTA; when [A | I] fits (n <= ~110) it is worked on in shared memory, so a pivot step costs three
// barriers instead of three global-memory round trips.
__global__ void __launch_bounds__(CT) k_coarse_invert(int n, double* __restrict__ Wg, double* __restrict__ Ainv, int in_smem, int* __restrict__ bad) {
    extern __shared__ __align__(16) double wsm[];
    __shared__ double fac[1024];
    __shared__ double redv[CT / 32];
    __shared__ int redi[CT / 32];
    __shared__ int piv;
    const int tid = threadIdx.x, n2 = 2 * n;
    Wg += blockIdx.y * coarse_work_doubles(n); Ainv += (size_t)blockIdx.y * n * n;
    double* W = Wg;
    if (in_smem) {
        for (int e = tid; e < n * n2; e += CT) wsm[e] = Wg[e];
        W = wsm;
        __syncthreads();
    }
    for (int k = 0; k < n; k++) {
        // pivot search over rows k..n-1 of column k
        double best = -1.0; int bi = n;
        for (int r = k + tid; r < n; r += CT) {
            const double v = fabs(W[(size_t)r * n2 + k]);
            if (v > best) { best = v; bi = r; }
        }
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_down_sync(0xffffffffu, best, o);
            const int oi = __shfl_down_sync(0xffffffffu, bi, o);
            if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
        }
        if ((tid & 31) == 0) { redv[tid >> 5] = best; redi[tid >> 5] = bi; }
        __syncthreads();
        if (tid == 0) {
            double b = redv[0]; int i = redi[0];
            for (int w = 1; w < CT / 32; w++)
                if (redv[w] > b || (redv[w] == b && redi[w] < i)) { b = redv[w]; i = redi[w]; }
            piv = i < n ? i : k;        // a column of NaNs (inadmissible coefficients, MG_ECOEFF) has no maximum: stay in bounds
            if (!(b > 0.0) || isinf(b)) atomicOr(bad, 8);      // zero or non-finite pivot: the coarsest operator is singular (the oracle's -2)
        }
        __syncthreads();
        const int p = piv;
        if (p != k)
            for (int c = tid; c < n2; c += CT) {
                const double a = W[(size_t)k * n2 + c];
                W[(size_t)k * n2 + c] = W[(size_t)p * n2 + c];
                W[(size_t)p * n2 + c] = a;
            }
        __syncthreads();
        const double inv = 1.0 / W[(size_t)k * n2 + k];
        for (int r = tid; r < n; r += CT) fac[r] = (r == k) ? 0.0 : W[(size_t)r * n2 + k];
        __syncthreads();
        for (int c = tid; c < n2; c += CT) W[(size_t)k * n2 + c] *= inv;
        __syncthreads();
        for (int e = tid; e < n * n2; e += CT) {
            const int r = e / n2, c = e - r * n2;
            const double f = fac[r];
            if (f != 0.0) W[e] -= f * W[(size_t)k * n2 + c];
        }
        __syncthreads();
    }
    for (int e = tid; e < n * n; e += CT) Ainv[e] = W[(size_t)(e / n) * n2 + n + (e % n)];
}

// The same elimination for coarsest levels that do not fit one CTA's shared memory (n > ~110; the paper keeps
// ~400 points on its coarsest level): a cooperative grid in which every CTA owns a slab of COLUMNS of
// [A | I] in shared memory for the whole elimination.  A pivot step needs only column k and the pivot index
// from the CTA that owns column k: it publishes them (double-buffered) before the one grid barrier of the
// step.  Same arithmetic and pivot rule as k_coarse_invert.
constexpr int CIT = 256;
__global__ void __launch_bounds__(CIT) k_coarse_invert_coop(int n, int cpb, const double* __restrict__ Wg, double* __restrict__ Ainv,
                                                            double* colbuf, int* pivbuf, int* __restrict__ bad) {
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    extern __shared__ __align__(16) double csm[];
    double* sc = csm;                       // [cpb][n], column-major slab
    double* fac = sc + (size_t)cpb * n;     // column k as published
    double* rowk = fac + n;                 // [cpb] scaled pivot-row entries of the own columns
    double* oldk = rowk + cpb;              // [cpb] row-k entries before the swap
    __shared__ double redv[CIT / 32];
    __shared__ int redi[CIT / 32];
    const int tid = threadIdx.x, n2 = 2 * n;
    const int c0 = blockIdx.x * cpb, nc = max(0, min(cpb, n2 - c0));
    for (int e = tid; e < nc * n; e += CIT) { const int c = e / n, r = e - c * n; sc[e] = Wg[(size_t)r * n2 + c0 + c]; }
    __syncthreads();
    auto publish = [&](int k) {             // called by every thread of the CTA that owns column k
        const double* col = sc + (size_t)(k - c0) * n;
        double best = -1.0; int bi = n;
        for (int r = k + tid; r < n; r += CIT) { const double v = fabs(col[r]); if (v > best) { best = v; bi = r; } }
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_down_sync(0xffffffffu, best, o);
            const int oi = __shfl_down_sync(0xffffffffu, bi, o);
            if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
        }
        if ((tid & 31) == 0) { redv[tid >> 5] = best; redi[tid >> 5] = bi; }
        __syncthreads();
        if (tid == 0) {
            double b = redv[0]; int i = redi[0];
            for (int w = 1; w < CIT / 32; w++)
                if (redv[w] > b || (redv[w] == b && redi[w] < i)) { b = redv[w]; i = redi[w]; }
            pivbuf[k & 1] = i < n ? i : k;   // as above
            if (!(b > 0.0) || isinf(b)) atomicOr(bad, 8);
        }
        for (int r = tid; r < n; r += CIT) colbuf[(size_t)(k & 1) * n + r] = col[r];
        __syncthreads();
    };
    if (0 >= c0 && 0 < c0 + nc) publish(0);
    grid.sync();
    for (int k = 0; k < n; k++) {
        for (int r = tid; r < n; r += CIT) fac[r] = __ldcg(colbuf + (size_t)(k & 1) * n + r);
        const int p = __ldcg(pivbuf + (k & 1));
        __syncthreads();
        const double inv = 1.0 / fac[p];
        const double fk = fac[k];           // after the swap this is the column-k entry of row p
        if (tid < nc) { oldk[tid] = sc[(size_t)tid * n + k]; rowk[tid] = sc[(size_t)tid * n + p] * inv; }
        __syncthreads();
        for (int e = tid; e < nc * n; e += CIT) {
            const int c = e / n, r = e - c * n;
            double v;
            if (r == k) v = rowk[c];
            else if (r == p) v = (fk != 0.0) ? oldk[c] - fk * rowk[c] : oldk[c];
            else { const double f = fac[r]; v = (f != 0.0) ? sc[e] - f * rowk[c] : sc[e]; }
            sc[e] = v;
        }
        __syncthreads();
        if (k + 1 < n && k + 1 >= c0 && k + 1 < c0 + nc) publish(k + 1);
        grid.sync();
    }
    for (int e = tid; e < nc * n; e += CIT) {
        const int c = e / n, r = e - c * n;
        if (c0 + c >= n) Ainv[(size_t)r * n + (c0 + c - n)] = sc[e];
    }
}

// x = A^-1 b on the coarsest level; vectors in the tile layout, rows addressed through cslot.
__global__ void __launch_bounds__(CT) k_coarse_solve(const double* __restrict__ Ainv, const int32_t* __restrict__ cslot, int n,
                                                     VecRef br, VecRef xr, const int* __restrict__ stop) {
    __shared__ double sb[1024];
    const int pl = blockIdx.y;
    if (stopped(stop, pl)) return;
    Ainv += (size_t)pl * n * n;
    const double* __restrict__ b = resolve(br, pl);
    double* __restrict__ x = resolve(xr, pl);
    for (int r = threadIdx.x; r < n; r += CT) sb[r] = b[cslot[r]];
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int r = warp; r < n; r += CT / 32) {
        double acc = 0.0;
        for (int c = lane; c < n; c += 32) acc += Ainv[(size_t)r * n + c] * sb[c];
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        if (lane == 0) x[cslot[r]] = acc;
    }
}

}  // namespace

void launch_coarse_factor(const Launch& L, const LevelDev& lv, const int32_t* cslot, const int32_t* slot2row, int n,
                          double* work, double* Ainv, int* bad) {
    k_coarse_assemble<<<dim3((n + 127) / 128, L.planes), 128, 0, L.stream>>>(lv, cslot, slot2row, n, work);
    const size_t wbytes = (size_t)n * 2 * n * sizeof(double);
    const int in_smem = wbytes <= 200 * 1024;
    ensure_dyn_smem((const void*)k_coarse_invert, 200 * 1024);
    ensure_dyn_smem((const void*)k_coarse_invert_coop, 200 * 1024);
    const int coop_sms = dev_info().coop ? dev_info().sms : 0;
    if (!in_smem && coop_sms > 0) {                           // column slabs over a cooperative grid
        int G = std::min(coop_sms, (2 * n + 3) / 4);
        int cpb = (2 * n + G - 1) / G;
        G = (2 * n + cpb - 1) / cpb;
        const size_t smem = ((size_t)cpb * n + n + 2 * (size_t)cpb) * sizeof(double);
        if (smem <= 200 * 1024) {
            for (int pl = 0; pl < L.planes; pl++) {           // one cooperative grid per plane
                double* wp = work + (size_t)pl * coarse_work_doubles(n);
                double* colbuf = wp + (size_t)2 * n * n;      // 2 n doubles + 2 ints behind [A | I] (allocated by mg_setup)
                int* pivbuf = reinterpret_cast<int*>(colbuf + 2 * n);
                const double* Wg = wp;
                double* ai = Ainv + (size_t)pl * n * n;
                void* args[] = {(void*)&n, (void*)&cpb, (void*)&Wg, (void*)&ai, (void*)&colbuf, (void*)&pivbuf, (void*)&bad};
                cudaLaunchCooperativeKernel((const void*)k_coarse_invert_coop, dim3(G), dim3(CIT), args, smem, L.stream);
            }
            if (L.counter) *L.counter += 1 + L.planes;
            return;
        }
    }
    k_coarse_invert<<<dim3(1, L.planes), CT, in_smem ? wbytes : 0, L.stream>>>(n, work, Ainv, in_smem, bad);
    if (L.counter) *L.counter += 2;
}

void launch_coarse_solve(const Launch& L, const double* Ainv, const int32_t* cslot, int n, VecRef b_tiled, VecRef x_tiled) {
    k_coarse_solve<<<dim3(1, L.planes), CT, 0, L.stream>>>(Ainv, cslot, n, b_tiled, x_tiled, L.stop);
    if (L.counter) *L.counter += 1;
}

}  // namespace mgb
