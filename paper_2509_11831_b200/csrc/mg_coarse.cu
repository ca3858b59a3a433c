// Coarsest-level direct solve on the device (rule C).  The paper factorises the
// coarsest matrix on the CPU at every update and round-trips the right-hand side at every cycle
// (PAPER.md:217); here the dense operator is assembled, inverted (Gauss-Jordan with partial pivoting,
// one CTA) at update time, and the cycle applies the inverse with one small kernel: no host step.
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
        for (int d = 0; d < 4; d++) { a[d] = lv.kappa * (cl + lv.c[sn[d]]); }
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
__global__ void __launch_bounds__(CT) k_coarse_invert(int n, double* __restrict__ Wg, double* __restrict__ Ainv, int in_smem) {
    extern __shared__ __align__(16) double wsm[];
    __shared__ double fac[1024];
    __shared__ double redv[CT / 32];
    __shared__ int redi[CT / 32];
    __shared__ int piv;
    const int tid = threadIdx.x, n2 = 2 * n;
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
            piv = i;
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

// x = A^-1 b on the coarsest level; vectors in the tile layout, rows addressed through cslot.
__global__ void __launch_bounds__(CT) k_coarse_solve(const double* __restrict__ Ainv, const int32_t* __restrict__ cslot, int n,
                                                     VecRef br, VecRef xr, const int* __restrict__ stop) {
    __shared__ double sb[1024];
    if (stop != nullptr && *stop) return;
    const double* __restrict__ b = resolve(br);
    double* __restrict__ x = resolve(xr);
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
                          double* work, double* Ainv) {
    k_coarse_assemble<<<(n + 127) / 128, 128, 0, L.stream>>>(lv, cslot, slot2row, n, work);
    const size_t wbytes = (size_t)n * 2 * n * sizeof(double);
    const int in_smem = wbytes <= 200 * 1024;
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_coarse_invert, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        configured = true;
    }
    k_coarse_invert<<<1, CT, in_smem ? wbytes : 0, L.stream>>>(n, work, Ainv, in_smem);
    if (L.counter) *L.counter += 2;
}

void launch_coarse_solve(const Launch& L, const double* Ainv, const int32_t* cslot, int n, VecRef b_tiled, VecRef x_tiled) {
    k_coarse_solve<<<1, CT, 0, L.stream>>>(Ainv, cslot, n, b_tiled, x_tiled, L.stop);
    if (L.counter) *L.counter += 1;
}

}  // namespace mgb
